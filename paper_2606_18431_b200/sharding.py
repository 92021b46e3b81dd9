"""Multi-GPU plumbing: replicas are independent units, so the path shards by
replica with no data-path collective; only four scalars are reduced for reporting.  Holds no scheduler arithmetic."""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(rank: int, world: int, replicas_per_rank: int) -> range:
    """Replica (= seed) indices simulated by `rank`: contiguous blocks of `replicas_per_rank` (weak scaling)."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    return range(rank * replicas_per_rank, (rank + 1) * replicas_per_rank)


def shard_workload(make_workload, rank: int, world: int, replicas_per_rank: int, n_requests: int):
    """The sub-workload of `rank` out of make_workload(n_seeds=world * replicas_per_rank, n_requests=...)."""
    wl = make_workload(n_seeds=replicas_per_rank * world, n_requests=n_requests)
    return wl if world == 1 else wl.select(shard_range(rank, world, replicas_per_rank))


def aggregate(request_steps_timed: float, request_steps_all: float, ms: float, t_e2e: float, device, world: int):
    """Whole-job totals: request-steps SUMMED over ranks, times taken as the MAX over ranks."""
    tot = torch.tensor([float(request_steps_timed), float(request_steps_all), float(ms), float(t_e2e)],
                       dtype=torch.float64, device=device)
    if world > 1:
        s_ = tot.clone(); dist.all_reduce(s_, dist.ReduceOp.SUM)
        m_ = tot.clone(); dist.all_reduce(m_, dist.ReduceOp.MAX)
        return s_[0].item(), s_[1].item(), m_[2].item(), m_[3].item()
    return tot[0].item(), tot[1].item(), tot[2].item(), tot[3].item()


def gather_replica_stats(table, device, world: int):
    """The one exchange of the job: every rank's [R_rank][W] per-replica statistics, concatenated
    in rank order (= replica order of the unsharded job) on every rank.  `table`: int64 numpy array; returns numpy."""
    import numpy as np
    t = torch.as_tensor(np.ascontiguousarray(table, dtype=np.int64), device=device)
    if world == 1:
        return t.cpu().numpy()
    out = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(out, t)
    return torch.cat(out, 0).cpu().numpy()
