"""Seeded synthetic workloads (input generators only).

This module serves BOTH the CUDA path and the CPU oracle with the same inputs and
holds none of the scheduler's arithmetic: it only draws request traces
(arrival_us, prompt_tok, decode_tok) and lists the simulator / replica
parameters of the five configurations of BASELINE.json.  It imports numpy only.

The traces stand in for the paper's Azure conversation/code, ShareGPT and s1k
workloads, which are not available; shapes follow
BASELINE.json:configs and Fig. 1 (prefill light-tailed, decode light- or
heavy-tailed).  Recipe (also in DESIGN.md Sec. 4):

  rng = numpy.random.default_rng([config_id, seed])      one generator per trace
  draw order: lengths first, then inter-arrivals
  tokens  = clip(rint(x), lo, hi);  D <- max(1, min(D, B*blk - P))
  arrival = rint(cumsum(gaps) * 1e6) microseconds (int64)
  "cost-model capacity" lambda_cap = 1 / s_bar with
     F_bar = mean(D*(P + D/2)) / mean(D)          time-average resident tokens of a sequence
     n_ref = min(M, B*blk / F_bar)                sequences the KV pool sustains
     s_bar = c_pf*mean(P) + mean(D)*(c_dec + c0/n_ref)   service time per request, means over the trace
"""
from __future__ import annotations

import dataclasses
import math
from typing import Callable, Dict, List, Optional, Sequence

import numpy as np

POLICY_FCFS, POLICY_SRPT, POLICY_BOOST, POLICY_LAS, POLICY_SJF, POLICY_SPF, POLICY_DISTBOOST, POLICY_SARATHI = 0, 1, 2, 3, 4, 5, 6, 7
SIG_UNIFIED, SIG_PHASE, SIG_REMAINING = 0, 1, 2
QUANT_GEOMETRIC, QUANT_EXACT = 0, 1
PRE_RECOMPUTE, PRE_SWAP, PRE_AUTO = 0, 1, 2

#: defaults shared by every configuration (DESIGN.md Sec. 3 "Defaults")
SIM_DEFAULTS = dict(
    block_tokens=16, max_batch=256, chunk_tokens=1024, token_budget=1024,
    c0_us=5000, c_prefill_tok_us=20, c_decode_seq_us=10,
    preempt_mode=PRE_RECOMPUTE, swap_ns_per_block=5243, swap_pool_blocks=0,
    bin_tokens=256, tok_us=5000,
)

REPLICA_FIELDS = ("trace_id", "policy", "guard", "signal_mode", "quant_mode", "hysteresis_us", "gamma")


def make_replicas(n: int, **kw) -> Dict[str, np.ndarray]:
    """Replica parameter table (struct of arrays) with BOOST defaults."""
    rep = dict(
        trace_id=np.arange(n, dtype=np.int64),
        policy=np.full(n, POLICY_BOOST, np.int64),
        guard=np.ones(n, np.int64),
        signal_mode=np.full(n, SIG_UNIFIED, np.int64),
        quant_mode=np.full(n, QUANT_GEOMETRIC, np.int64),
        hysteresis_us=np.full(n, 100_000, np.int64),
        gamma=np.full(n, 0.3, np.float64),
    )
    for k, v in kw.items():
        rep[k] = np.broadcast_to(np.asarray(v, dtype=rep[k].dtype), (n,)).copy()
    return rep


@dataclasses.dataclass
class Workload:
    """A simulator configuration + replica table + a trace generator."""
    name: str
    config_id: int
    sim: Dict[str, int]                 # n_replicas, n_traces, max_requests, queue_cap, kv_blocks, ...
    replicas: Dict[str, np.ndarray]     # REPLICA_FIELDS, each [R]
    trace_fn: Callable[[int], tuple]    # seed -> (arrival_us[N], prompt[N], decode[N])
    trace_seeds: np.ndarray             # seed of trace t
    description: str = ""

    @property
    def R(self) -> int:
        return int(self.sim["n_replicas"])

    def traces(self, workers: int = 1):
        """Return (arrival_us[int64 NT,N], prompt[int32 NT,N], decode[int32 NT,N], n_req[uint32 NT])."""
        NT, N = int(self.sim["n_traces"]), int(self.sim["max_requests"])
        a = np.zeros((NT, N), np.int64)
        p = np.ones((NT, N), np.int32)
        d = np.ones((NT, N), np.int32)
        n = np.full(NT, N, np.uint32)
        seeds = [int(s) for s in self.trace_seeds]
        if workers > 1 and NT >= 4 * workers:
            import multiprocessing as mp
            chunks = np.array_split(np.arange(NT), workers * 4)
            global _POOL_FN
            _POOL_FN = self.trace_fn            # inherited by the forked workers (closures do not pickle)
            with mp.get_context("fork").Pool(workers) as pool:
                parts = pool.map(_gen_chunk, [[seeds[i] for i in ch] for ch in chunks])
            for ch, (pa, pp, pd) in zip(chunks, parts):
                a[ch], p[ch], d[ch] = pa, pp, pd
        else:
            for t, s in enumerate(seeds):
                a[t], p[t], d[t] = self.trace_fn(s)
        return a, p, d, n

    def select(self, replica_ids: Sequence[int]) -> "Workload":
        """Sub-workload holding only the given replicas (and the traces they use).
        Results of a replica do not depend on which other replicas run beside it."""
        ids = np.asarray(replica_ids, np.int64)
        used, inv = np.unique(self.replicas["trace_id"][ids], return_inverse=True)
        rep = {k: v[ids].copy() for k, v in self.replicas.items()}
        rep["trace_id"] = inv.astype(np.int64)
        sim = dict(self.sim, n_replicas=len(ids), n_traces=len(used))
        return Workload(self.name + f"[{len(ids)} replicas]", self.config_id, sim, rep, self.trace_fn,
                        self.trace_seeds[used], self.description)


_POOL_FN = None


def _gen_chunk(seeds):
    out = [_POOL_FN(s) for s in seeds]
    return (np.stack([o[0] for o in out]), np.stack([o[1] for o in out]), np.stack([o[2] for o in out]))


# ----------------------------------------------------------------------------- length mixes

def _lognormal_tokens(rng, n, mu, sigma, lo, hi):
    return np.clip(np.rint(rng.lognormal(mu, sigma, n)), lo, hi).astype(np.int64)


def _chat_lengths(rng, n):
    """Chat mix (config 2): P ~ LN(6.5, 0.9) in [16, 4096], D ~ LN(5.0, 0.8) in [1, 4096]."""
    return _lognormal_tokens(rng, n, 6.5, 0.9, 16, 4096), _lognormal_tokens(rng, n, 5.0, 0.8, 1, 4096)


def _reasoning_lengths(rng, n):
    """Reasoning mix (config 3): P ~ LN(6.0, 0.8) in [16, 4096]; D = 70% LN(6.0, 1.0) /
    30% Pareto(alpha 1.3, x_min 1024), clipped to [1, 32768]."""
    P = _lognormal_tokens(rng, n, 6.0, 0.8, 16, 4096)
    pick = rng.random(n)
    ln = rng.lognormal(6.0, 1.0, n)
    par = 1024.0 * (1.0 - rng.random(n)) ** (-1.0 / 1.3)
    D = np.clip(np.rint(np.where(pick < 0.7, ln, par)), 1, 32768).astype(np.int64)
    return P, D


def _fit_kv(P, D, kv_tokens):
    return np.maximum(1, np.minimum(D, kv_tokens - P))


def capacity_rate(P, D, sim) -> float:
    """lambda_cap (requests / s) of the stated cost model for this trace's own requests."""
    P = P.astype(np.float64); D = D.astype(np.float64)
    fbar = float(np.mean(D * (P + D / 2.0)) / np.mean(D))
    n_ref = min(float(sim["max_batch"]), sim["kv_blocks"] * sim["block_tokens"] / fbar)
    sbar_us = sim["c_prefill_tok_us"] * float(np.mean(P)) + float(np.mean(D)) * (
        sim["c_decode_seq_us"] + sim["c0_us"] / n_ref)
    return 1e6 / sbar_us


def _poisson_arrivals(rng, n, rate):
    return np.rint(np.cumsum(rng.exponential(1.0 / rate, n)) * 1e6).astype(np.int64)


def _mmpp2_arrivals(rng, n, mean_rate, hi=2.0, lo=0.3, sojourn_s=30.0):
    """2-state MMPP by time change: alternate exponential sojourns (mean 30 s) at rates
    hi*lam and lo*lam, lam = mean_rate / ((hi+lo)/2); a unit-rate Poisson stream is mapped
    through the inverse of the piecewise-linear cumulative intensity (exact sample)."""
    lam = mean_rate / ((hi + lo) / 2.0)
    start_hi = rng.random() < 0.5
    u = np.cumsum(rng.exponential(1.0, n))
    m = int(n / (mean_rate * sojourn_s) * 3) + 16
    while True:
        dur = rng.exponential(sojourn_s, m)
        k = np.arange(m)
        rates = np.where((k % 2 == 0) == start_hi, hi * lam, lo * lam)
        big = np.concatenate([[0.0], np.cumsum(dur * rates)])
        if big[-1] > u[-1]:
            break
        m *= 2
    tb = np.concatenate([[0.0], np.cumsum(dur)])
    return np.rint(np.interp(u, big, tb) * 1e6).astype(np.int64)


# ----------------------------------------------------------------------------- the five configs

def _sim(R, NT, N, Q, B, **kw):
    s = dict(SIM_DEFAULTS, n_replicas=R, n_traces=NT, max_requests=N, queue_cap=Q, kv_blocks=B)
    s.update(kw)
    return s


def config1() -> Workload:
    """1 replica, 256 requests, boost policy, Poisson 4 req/s, recompute, seed 0."""
    sim = _sim(1, 1, 256, 256, 2048)

    def gen(seed):
        rng = np.random.default_rng([1, seed])
        P = _lognormal_tokens(rng, 256, 6.0, 0.8, 16, 4096)
        D = _fit_kv(P, _lognormal_tokens(rng, 256, 5.5, 1.0, 1, 8192), 2048 * 16)
        return _poisson_arrivals(rng, 256, 4.0), P.astype(np.int32), D.astype(np.int32)

    return Workload("config1: 1 replica x 256 requests, boost", 1, sim, make_replicas(1), gen,
                    np.array([0]), "smoke + full-oracle parity")


def config2(n_seeds: int = 1024) -> Workload:
    """Chat-heavy mix, seeds x {FCFS, SRPT(perfect lengths), BOOST} side by side, 80% load."""
    N, B = 4000, 8192
    sim = _sim(3 * n_seeds, n_seeds, N, 2048, B)

    def gen(seed):
        rng = np.random.default_rng([2, seed])
        P, D = _chat_lengths(rng, N)
        D = _fit_kv(P, D, B * 16)
        lam = 0.8 * capacity_rate(P, D, sim)
        return _poisson_arrivals(rng, N, lam), P.astype(np.int32), D.astype(np.int32)

    R = 3 * n_seeds
    j = np.arange(R) % 3
    rep = make_replicas(
        R, trace_id=np.arange(R) // 3,
        policy=np.array([POLICY_FCFS, POLICY_SRPT, POLICY_BOOST])[j],
        guard=(j == 2).astype(np.int64), hysteresis_us=np.where(j == 2, 100_000, 0))
    return Workload(f"config2: chat mix, {n_seeds} seeds x 3 policies x {N} requests", 2, sim, rep, gen,
                    np.arange(n_seeds))


def config3(n_seeds: int = 4096) -> Workload:
    """Reasoning-heavy mix, bursty MMPP-2 arrivals, swap-vs-recompute preemption."""
    N, B = 4000, 6144
    sim = _sim(n_seeds, n_seeds, N, 2048, B, preempt_mode=PRE_AUTO, swap_pool_blocks=B)

    def gen(seed):
        rng = np.random.default_rng([3, seed])
        P, D = _reasoning_lengths(rng, N)
        D = _fit_kv(P, D, B * 16)
        lam = 0.8 * capacity_rate(P, D, sim)
        return _mmpp2_arrivals(rng, N, lam), P.astype(np.int32), D.astype(np.int32)

    return Workload(f"config3: reasoning mix, MMPP-2, {n_seeds} replicas x {N} requests", 3, sim,
                    make_replicas(n_seeds), gen, np.arange(n_seeds))


def config4(n_seeds: int = 1024, n_gamma: int = 16) -> Workload:
    """Distribution shift (chat -> reasoning at request 1000) + memory pressure; gamma sweep as batch dim."""
    N, B = 2000, 2048
    R = n_seeds * n_gamma
    sim = _sim(R, n_seeds, N, 2048, B)

    def gen(seed):
        rng = np.random.default_rng([4, seed])
        P1, D1 = _chat_lengths(rng, N // 2)
        P2, D2 = _reasoning_lengths(rng, N - N // 2)
        P = np.concatenate([P1, P2]); D = _fit_kv(P, np.concatenate([D1, D2]), B * 16)
        lam = 0.8 * capacity_rate(P, D, sim)
        return _poisson_arrivals(rng, N, lam), P.astype(np.int32), D.astype(np.int32)

    gam = 10.0 ** (-2.0 + 4.0 * np.arange(n_gamma) / max(1, n_gamma - 1))
    rep = make_replicas(R, trace_id=np.arange(R) // n_gamma, gamma=gam[np.arange(R) % n_gamma])
    return Workload(f"config4: shift + pressure, {n_seeds} seeds x {n_gamma} gamma x {N} requests", 4, sim,
                    rep, gen, np.arange(n_seeds))


def config5(n_seeds: int = 65536, n_requests: int = 8192) -> Workload:
    """Scale stress: 50/50 chat/reasoning, Poisson at 95% load, queue cap 2048."""
    N, B = n_requests, 16384
    sim = _sim(n_seeds, n_seeds, N, 2048, B, preempt_mode=PRE_AUTO, swap_pool_blocks=B)

    def gen(seed):
        rng = np.random.default_rng([5, seed])
        Pc, Dc = _chat_lengths(rng, N)
        Pr, Dr = _reasoning_lengths(rng, N)
        is_chat = rng.random(N) < 0.5
        P = np.where(is_chat, Pc, Pr); D = _fit_kv(P, np.where(is_chat, Dc, Dr), B * 16)
        lam = 0.95 * capacity_rate(P, D, sim)
        return _poisson_arrivals(rng, N, lam), P.astype(np.int32), D.astype(np.int32)

    return Workload(f"config5: scale stress, {n_seeds} replicas x {N} requests", 5, sim,
                    make_replicas(n_seeds), gen, np.arange(n_seeds))


def starvation(n_seeds: int = 1, n_requests: int = 2000, load: float = 0.99) -> Workload:
    """Test-only shape of the paper's starvation experiment:
    90% short (~125 prefill / 100 decode) + 10% long (2k / 6k), Poisson at rho ~ 0.99."""
    N, B = n_requests, 4096
    sim = _sim(n_seeds, n_seeds, N, 2048, B)

    def gen(seed):
        rng = np.random.default_rng([6, seed])
        long_ = rng.random(N) < 0.1
        P = np.where(long_, 2000, np.clip(np.rint(rng.normal(125, 10, N)), 16, 4096)).astype(np.int64)
        D = np.where(long_, 6000, np.clip(np.rint(rng.normal(100, 10, N)), 1, 4096)).astype(np.int64)
        lam = load * capacity_rate(P, D, sim)
        return _poisson_arrivals(rng, N, lam), P.astype(np.int32), D.astype(np.int32)

    return Workload(f"starvation shape, {n_seeds} replicas x {N} requests", 6, sim, make_replicas(n_seeds), gen,
                    np.arange(n_seeds))


def routed_cluster(n_replicas: int = 8, n_requests_total: int = 6000, dispatch: str = "round_robin", load: float = 0.9,
                   seed: int = 0, kv_blocks: int = 4096):
    """Global dispatch in front of per-replica scheduling (Tables 9-10: "the routing policy is
    exogenous", the part that keeps replicas independent): ONE global Poisson stream at
    load x n_replicas x lambda_cap (50/50 chat / reasoning mix) is split over the replicas by a router that does not
    look at replica state -- "round_robin" (request i -> replica i mod R) or "random" (seeded uniform choice).
    Join-the-shortest-queue looks at queue lengths at arrival time and would couple the replicas: not built.
    Returns (workload, traces) with ragged per-replica request counts (traces[3])."""
    if dispatch not in ("round_robin", "random"):
        raise ValueError("dispatch must be 'round_robin' or 'random'")
    R, T = int(n_replicas), int(n_requests_total)
    rng = np.random.default_rng([7, seed])
    Pc, Dc = _chat_lengths(rng, T)
    Pr, Dr = _reasoning_lengths(rng, T)
    is_chat = rng.random(T) < 0.5
    P = np.where(is_chat, Pc, Pr); D = _fit_kv(P, np.where(is_chat, Dc, Dr), kv_blocks * 16)
    sim0 = _sim(R, R, 1, 2048, kv_blocks, preempt_mode=PRE_AUTO, swap_pool_blocks=kv_blocks)
    arr = _poisson_arrivals(rng, T, load * R * capacity_rate(P, D, sim0))
    dest = (np.arange(T) % R) if dispatch == "round_robin" else rng.integers(0, R, T)
    counts = np.bincount(dest, minlength=R)
    N = int(max(1, counts.max()))
    a = np.zeros((R, N), np.int64); p = np.ones((R, N), np.int32); d = np.ones((R, N), np.int32)
    for r in range(R):
        sel = np.nonzero(dest == r)[0]                  # arrival order is kept inside a replica
        a[r, :len(sel)], p[r, :len(sel)], d[r, :len(sel)] = arr[sel], P[sel], D[sel]
    sim = dict(sim0, max_requests=N, queue_cap=min(N, 2048))
    wl = Workload(f"routed cluster: {R} replicas, {T} requests, {dispatch}", 7, sim, make_replicas(R),
                  lambda s_: (a[s_], p[s_], d[s_]), np.arange(R))
    return wl, (a, p, d, counts.astype(np.uint32)), (arr, P.astype(np.int32), D.astype(np.int32), dest)


def by_id(config_id: int, **kw) -> Workload:
    return {1: config1, 2: config2, 3: config3, 4: config4, 5: config5, 6: starvation}[config_id](**kw)


def custom(arrival_us, prompt, decode, sim_overrides: Optional[dict] = None,
           replicas: Optional[Dict[str, np.ndarray]] = None, name: str = "custom") -> Workload:
    """Wrap explicit trace arrays ([NT][N] or [N]) as a Workload (tests)."""
    a = np.atleast_2d(np.asarray(arrival_us, np.int64))
    p = np.atleast_2d(np.asarray(prompt, np.int32))
    d = np.atleast_2d(np.asarray(decode, np.int32))
    NT, N = a.shape
    rep = replicas if replicas is not None else make_replicas(NT)
    R = len(rep["trace_id"])
    sim = _sim(R, NT, N, max(1, min(N, 2048)), 2048)
    sim.update(sim_overrides or {})
    sim["n_replicas"], sim["n_traces"], sim["max_requests"] = R, NT, N
    return Workload(name, 0, sim, rep, lambda s: (a[s], p[s], d[s]), np.arange(NT))
