"""N > 1 path on CPU (gloo, world_size 2): replicas shard by seed with no data-path collective.
The two ranks go through bench.py's own control flow -- its argument parser, its rank layout check, the shard
selection, the reduction of the totals and the final gather of the per-replica statistics --;
the shards are disjoint, cover the job, hold exactly the traces of the unsharded workload, the reported totals are
request-steps summed / times max'ed over ranks and the gathered table is the unsharded job's, in replica order.  The
oracle stands in for the CUDA path here (no GPU in this tier): a replica's schedule does not depend on which replicas
run beside it (pin P14)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_18431_b200 import sharding as SH
from paper_2606_18431_b200 import workloads as W

R_PER_RANK, N_REQ, ITERS = 3, 48, 400


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from oracle import oracle as O
    args = bench.parse(["--gpus", str(world), "--replicas", str(R_PER_RANK), "--requests", str(N_REQ)])
    assert bench.rank_layout(args, os.environ) == (rank, world, rank)
    wl = SH.shard_workload(W.config5, rank, world, args.replicas, args.requests)
    tr = wl.traces()
    o = O.OracleSim(wl.sim, wl.replicas, tr)
    o.step(ITERS)
    st = o.stats()
    rs = sum(s["request_steps"] for s in st)
    dg = o.digest()
    o.close()
    tot = SH.aggregate(rs, rs, 10.0 + rank, 1.0 + rank, "cpu", world)
    table = np.array([[s[c] for c in bench.COLS] for s in st], np.int64)          # bench.py's per-replica table
    job = SH.gather_replica_stats(table, "cpu", world)                               # the one exchange of the job
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), a=tr[0], digest=dg, rs=rs, tot=np.asarray(tot),
             seeds=wl.trace_seeds, job=job)
    dist.barrier()
    dist.destroy_process_group()


def test_shard_range_partitions_the_job():
    for world in (1, 2, 4, 8):
        got = [i for g in range(world) for i in SH.shard_range(g, world, 5)]
        assert got == list(range(5 * world))
    with pytest.raises(ValueError):
        SH.shard_range(2, 2, 5)


def test_two_rank_gloo_sharding(tmp_path, oracle_mod):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    parts = [np.load(tmp_path / f"rank{g}.npz") for g in range(world)]
    # one process, the whole job
    wl = W.config5(n_seeds=R_PER_RANK * world, n_requests=N_REQ)
    tr = wl.traces()
    o = oracle_mod.OracleSim(wl.sim, wl.replicas, tr)
    o.step(ITERS)
    import bench
    rs_all = sum(s["request_steps"] for s in o.stats())
    st_all = np.array([[s[c] for c in bench.COLS] for s in o.stats()], np.int64)
    dg_all = o.digest()
    o.close()
    assert np.array_equal(np.concatenate([p["seeds"] for p in parts]), wl.trace_seeds)
    assert np.array_equal(np.concatenate([p["a"] for p in parts]), tr[0])
    assert np.array_equal(np.concatenate([p["digest"] for p in parts]), dg_all)      # same schedules, sharded or not
    assert sum(int(p["rs"]) for p in parts) == rs_all
    for p in parts:                                                                  # every rank sees the job totals
        assert p["tot"][0] == rs_all and p["tot"][1] == rs_all
        assert p["tot"][2] == 11.0 and p["tot"][3] == 2.0                            # max over ranks
        assert np.array_equal(p["job"], st_all)                                      # and the whole job's statistics


def test_bench_launch_line_and_rank_layout():
    """`python bench.py --gpus N` outside torchrun re-executes itself under the contract's launch line (one rank per
    GPU, rendezvous on 127.0.0.1); under a launcher `--gpus` must agree with WORLD_SIZE."""
    import bench
    args = bench.parse(["--gpus", "4", "--steps", "2"])
    cmd = bench.torchrun_command(args, ["--gpus", "4", "--steps", "2"], 29511)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"]
    assert cmd[cmd.index("--nproc-per-node") + 1] == "4" and cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[cmd.index("--master-port") + 1] == "29511" and cmd[-4:] == ["--gpus", "4", "--steps", "2"]
    assert os.path.basename(cmd[cmd.index("29511") + 1]) == "bench.py"
    assert bench.rank_layout(args, {"RANK": "3", "WORLD_SIZE": "4", "LOCAL_RANK": "3"}) == (3, 4, 3)
    with pytest.raises(SystemExit):
        bench.rank_layout(args, {"RANK": "0", "WORLD_SIZE": "2", "LOCAL_RANK": "0"})
    assert bench.rank_layout(bench.parse([]), {}) == (0, 1, 0)
