"""Shared test helpers: small seeded memory-pressured traces (inputs only, no scheduler arithmetic)."""
import json
import os

import numpy as np

from paper_2606_18431_b200 import workloads as W


def pressure_workload(seed, n=60, kv_blocks=48, policy=W.POLICY_BOOST, gamma=0.3, guard=1, delta=100_000,
                      preempt=W.PRE_RECOMPUTE, mean_gap_us=8000, pmax=300, dmax=200, n_replicas=1,
                      signal=W.SIG_UNIFIED, quant=W.QUANT_GEOMETRIC, bin_tokens=64, **sim_kw):
    """n requests with P in [1,pmax], D in [1,dmax] against a tiny KV pool => frequent evictions."""
    rng = np.random.default_rng([99, seed])
    P = rng.integers(1, pmax + 1, n)
    D = rng.integers(1, dmax + 1, n)
    cap = kv_blocks * 16
    P = np.minimum(P, cap - 1)
    D = np.maximum(1, np.minimum(D, cap - P))
    a = np.cumsum(rng.exponential(mean_gap_us, n)).astype(np.int64)
    rep = W.make_replicas(n_replicas, trace_id=0, policy=policy, gamma=gamma, guard=guard, hysteresis_us=delta,
                          signal_mode=signal, quant_mode=quant)
    sim = dict(kv_blocks=kv_blocks, queue_cap=max(1, min(n, 2048)), preempt_mode=preempt, bin_tokens=bin_tokens,
               swap_pool_blocks=kv_blocks, max_batch=16, chunk_tokens=64, token_budget=96)
    sim.update(sim_kw)
    return W.custom(a, P, D, sim, rep, name=f"pressure{seed}")


GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def hand_cases():
    """The hand-worked schedules of tests/golden/hand_traces.{md,json} (inputs and expected numbers, all typed by hand)."""
    with open(os.path.join(GOLD, "hand_traces.json")) as f:
        return json.load(f)["cases"]


def hand_workload(case):
    sim = dict(block_tokens=16, c0_us=1000, c_prefill_tok_us=10, c_decode_seq_us=100, queue_cap=8)
    sim.update(case["sim"])
    rep = W.make_replicas(1, hysteresis_us=0, **case["replica"])
    return W.custom(case["arrival_us"], case["prompt"], case["decode"], sim, rep, name=case["name"])
