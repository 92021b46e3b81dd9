"""Pins for the CPU oracle: what the paper and the mathematics fix, checked without the CUDA path.

Each test cites the passage or the DESIGN.md rule it pins.  None of them calls the oracle to
produce its own expected value: expectations are hand-worked numbers (tests/golden), closed forms,
50-digit evaluations, textbook recursions, brute force, or invariants.
"""
import itertools
import json
import math
import os
from decimal import Decimal, getcontext
from functools import lru_cache

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_18431_b200 import workloads as W
from tests.helpers import GOLD, hand_cases, hand_workload, pressure_workload


def run_wl(wl, **kw):
    sim = O.OracleSim.from_workload(wl)
    sim.run(**kw)
    return sim


# ------------------------------------------------------------------ hand-worked schedules

HAND = hand_cases()
_hand_workload = hand_workload


@pytest.mark.parametrize("case", HAND, ids=[c["name"] for c in HAND])
def test_hand_worked_schedule(case):
    """Algorithm 1 on hand-derived schedules, tests/golden/hand_traces.md."""
    wl = _hand_workload(case)
    exp = case["expect"]
    sim = O.OracleSim.from_workload(wl)
    costs = []
    while True:
        info, _ = sim.step_replica(0)
        if not info["executed"]:
            break
        costs.append(info["cost_us"])
    assert costs == exp["step_costs_us"]
    tf, tl, ne, neu = sim.per_request()
    n = len(case["prompt"])
    assert tf[0, :n].tolist() == exp["t_first_us"]
    assert tl[0, :n].tolist() == exp["t_last_us"]
    assert ne[0, :n].tolist() == exp["n_evict"]
    if "n_evict_unforced" in exp:
        assert neu[0, :n].tolist() == exp["n_evict_unforced"]
    st = sim.stats()[0]
    for k in ("iterations", "request_steps", "t_end_us", "tokens_lost", "prefill_tokens", "decode_seqs",
              "evict_recompute", "evict_swap") + (("swapins",) if "swapins" in exp else ()):
        assert st[k] == exp[k], k
    assert st["done"] == 1 and st["n_completed"] == n


def test_hand_traces_file_consistent():
    """The hand file must satisfy work conservation by itself (guards against typos in the fixture)."""
    for c in HAND:
        e = c["expect"]
        work = sum(p + d - 1 for p, d in zip(c["prompt"], c["decode"]))
        assert e["prefill_tokens"] + e["decode_seqs"] == work + e["tokens_lost"], c["name"]
        assert sum(e["step_costs_us"]) <= e["t_end_us"]
        assert len(e["step_costs_us"]) == e["iterations"]


# ------------------------------------------------------------------ P1 quantiser (Eq. 8)

def test_quantiser_closed_form_and_paper_example():
    """Eq. 8 and 'for a 10k decode length at most 6 swap opportunities under k=256'."""
    k = 256
    what = lambda w: k * 2 ** O.quant_bin(w, k)
    assert [what(w) for w in (0, 1, 255, 256, 511, 512, 1023, 1024, 10000, 36864)] == \
           [256, 256, 256, 256, 256, 512, 512, 1024, 8192, 32768]
    values = sorted({what(w) for w in range(0, 10001)})
    assert values == [256, 512, 1024, 2048, 4096, 8192]
    assert len(values) == 6 == 1 + math.floor(math.log2(10000 / 256))
    for kk in (1, 16, 64, 256, 1000):
        for w in list(range(0, 3000, 7)) + [10 ** 5, 2 ** 31 - 1]:
            b = O.quant_bin(w, kk)
            assert b == math.floor(math.log2(max(w, kk) / kk)) or abs(math.log2(max(w, kk) / kk) - round(math.log2(max(w, kk) / kk))) < 1e-9
            assert kk * 2 ** b <= max(w, kk) < kk * 2 ** (b + 1)       # the defining property of the floor
    # QUANTIZE listing prints k*2^floor(log2(max{1, s/k})): same function
    for w in range(0, 5000, 13):
        assert what(w) == k * 2 ** math.floor(math.log2(max(1.0, w / k)))


# ------------------------------------------------------------------ P2 boost table (Eq. 2)

def _boost_exact_us(gamma, w_tokens, tok_us):
    getcontext().prec = 60
    x = Decimal(w_tokens) * Decimal(tok_us) / Decimal(10 ** 6)
    g = Decimal(repr(float(gamma)))
    one = Decimal(1)
    b = (one / (one - (-g * x).exp())).ln() / g
    return b * Decimal(10 ** 6)


@pytest.mark.parametrize("gamma", [1e-7, 0.01, 0.1, 0.3, 1.0, 3.0, 10.0, 100.0])
def test_boost_table_against_50_digit_eq2(gamma):
    """Eq. 2: b = (1/gamma) log(1/(1-exp(-gamma w))), fixed point in us, within 1 us."""
    tok = 5000
    for w in [1, 2, 17, 255, 256, 512, 1024, 2048, 4096, 8192, 16384, 32768, 65536]:
        exact = _boost_exact_us(gamma, w, tok)
        got = O.boost_us(gamma, w, tok)
        tol = max(Decimal(1), exact * Decimal(10) ** -12)
        assert abs(Decimal(got) - exact) <= tol, (gamma, w, got, exact)


def test_boost_table_shape_and_limits():
    """Boost is weakly decreasing in attained service (Lemma A.1 precondition), -> 0 as gamma*w -> inf,
    ~ (1/gamma) ln(1/(gamma w)) for gamma*w << 1; gamma = +inf gives 0 (FCFS)."""
    tok = 5000
    for gamma in (0.01, 0.1, 0.3, 1.0, 10.0):
        v = [O.boost_us(gamma, 256 * 2 ** b, tok) for b in range(0, 24)]
        assert all(v[i] >= v[i + 1] for i in range(len(v) - 1))
        assert v[-1] == 0
    assert O.boost_us(float("inf"), 256, tok) == 0
    assert O.boost_us(10.0, 256, tok) == 0      # exp(-12.8)/10 s = 0.28 us rounds to 0: gamma >= 10 is FCFS here
    assert O.boost_us(1.0, 256, tok) == round(-math.log(1 - math.exp(-1.28)) * 1e6)
    g, w = 1e-6, 10
    x = w * tok * 1e-6
    approx = (1 / g) * math.log(1 / (g * x)) * 1e6
    assert abs(O.boost_us(g, w, tok) - approx) / approx < 1e-6
    assert O.boost_us(0.3, 0, tok) == 1 << 60


def test_boost_lut_of_sim_matches_helper():
    wl = W.config1()
    sim = O.OracleSim.from_workload(wl)
    lut = sim.boost_lut(0)
    assert len(lut) == 64
    for b in range(0, 30):
        assert lut[b] == O.boost_us(0.3, 256 * 2 ** b, 5000)
    assert lut[40] == 0


# ------------------------------------------------------------------ P3/P4/P5 limits

def _same_schedule(sa, sb):
    assert sa.digest().tolist() == sb.digest().tolist()
    for x, y in zip(sa.per_request()[:3], sb.per_request()[:3]):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("seed", range(6))
def test_gamma_large_is_fcfs(seed):
    """'high gamma (100) mimics FCFS': boost table == 0 => identical schedule under memory pressure."""
    a = run_wl(pressure_workload(seed, policy=W.POLICY_BOOST, gamma=1000.0))
    b = run_wl(pressure_workload(seed, policy=W.POLICY_FCFS))
    assert not a.boost_lut(0).any()
    _same_schedule(a, b)
    assert a.stats()[0]["evict_recompute"] > 0


@pytest.mark.parametrize("seed", range(6))
def test_gamma_small_is_las(seed):
    """'low gamma (0.01) mimics LAS': vanilla boost (EXACT quantiser, G3), gamma -> 0+."""
    kw = dict(guard=0, delta=0, quant=W.QUANT_EXACT)
    a = run_wl(pressure_workload(seed, policy=W.POLICY_BOOST, gamma=1e-7, **kw))
    b = run_wl(pressure_workload(seed, policy=W.POLICY_LAS, **kw))
    _same_schedule(a, b)
    assert b.stats()[0]["evict_recompute"] > 0


@pytest.mark.parametrize("seed", range(6))
def test_unbounded_boost_on_remaining_size_is_srpt(seed):
    """north_star: an infinite-boost-on-size limit reproduces SRPT with perfect lengths."""
    kw = dict(guard=0, delta=0, quant=W.QUANT_EXACT)
    a = run_wl(pressure_workload(seed, policy=W.POLICY_BOOST, gamma=1e-7, signal=W.SIG_REMAINING, **kw))
    b = run_wl(pressure_workload(seed, policy=W.POLICY_SRPT, **kw))
    _same_schedule(a, b)
    assert b.stats()[0]["evict_recompute"] > 0


def test_policies_differ_when_they_should():
    """Sanity for the three limit tests: FCFS, SRPT and LAS do not coincide on these traces."""
    d = {p: run_wl(pressure_workload(0, policy=p, guard=0, delta=0)).digest()[0]
         for p in (W.POLICY_FCFS, W.POLICY_SRPT, W.POLICY_LAS)}
    assert len(set(d.values())) == 3


def test_hysteresis_eq7_and_key_formula():
    """Eq. 7: a newcomer j preempts the running request only if Phi(j) < Phi(curr) - delta;
    key = a - b_gamma(w~).  Keys are checked against a 60-digit evaluation of Eq. 2 and the
    iteration at which the newcomer first overtakes is predicted from it."""
    tok, gamma, a1 = 5000, 1.0, 1500
    sim_kw = dict(block_tokens=16, c0_us=1000, c_prefill_tok_us=10, c_decode_seq_us=100, queue_cap=8, kv_blocks=3,
                  max_batch=8, chunk_tokens=64, token_budget=64, tok_us=tok)
    b = lambda w: int((_boost_exact_us(gamma, w, tok)).to_integral_value(rounding="ROUND_HALF_UP"))
    for delta in (0, 100_000):
        rep = W.make_replicas(1, policy=W.POLICY_BOOST, gamma=gamma, guard=0, hysteresis_us=delta,
                              quant_mode=W.QUANT_EXACT)
        wl = W.custom([0, a1], [30, 30], [10, 2], sim_kw, rep)
        sim = O.OracleSim.from_workload(wl)
        first_overtake = None
        for it in range(1, 40):
            info, ents = sim.step_replica(0)
            if not info["executed"]:
                break
            ids = [e["id"] for e in ents]
            if ids == [1, 0] and first_overtake is None:
                first_overtake = (it, ents)
        assert first_overtake is not None
        it, ents = first_overtake
        e1, e0 = ents
        # r1 is fresh (d=0, not resident): key = a1 - b(30); r0 is resident with P+d tokens: key = 0 - b(P+d) - delta
        assert e1["resident_before"] == 0 and abs(e1["key"] - (a1 - b(30))) <= 1
        sig0 = e0["bin"]                                       # EXACT quantiser: bin == signal == P + d
        assert e0["resident_before"] == 1 and abs(e0["key"] - (0 - b(sig0) - delta)) <= 1
        assert e0["evict"] == 1                                 # B = 3 blocks cannot hold both
        # predicted switch point: smallest P+d (>= 32, the signal when r1 is first seen) with a1 - b(30) < -b(sig) - delta
        pred = next(s for s in range(32, 41) if a1 - b(30) < -b(s) - delta)
        assert sig0 == pred
        assert (delta == 0 and pred == 32) or (delta == 100_000 and pred == 34)


# ------------------------------------------------------------------ P6/P7 invariants + walk structure

MODES = [(W.POLICY_BOOST, 1, W.PRE_RECOMPUTE), (W.POLICY_BOOST, 1, W.PRE_AUTO), (W.POLICY_SRPT, 0, W.PRE_SWAP),
         (W.POLICY_FCFS, 0, W.PRE_RECOMPUTE), (W.POLICY_BOOST, 0, W.PRE_SWAP)]


@pytest.mark.parametrize("seed", range(4))
@pytest.mark.parametrize("policy,guard,pre", MODES)
def test_kv_capacity_walk_structure_and_work_conservation(seed, policy, guard, pre):
    """KV occupancy never exceeds capacity (U + dU <= B at PAPER.md:452); admission order
    (PAPER.md:438-441); victims from the back (M8); work conservation."""
    wl = pressure_workload(seed, policy=policy, guard=guard, preempt=pre, swap_ns_per_block=40_000,
                           swap_pool_blocks=20)
    s = wl.sim
    B, blk, M, T, c = s["kv_blocks"], s["block_tokens"], s["max_batch"], s["token_budget"], s["chunk_tokens"]
    a, P, D, _ = wl.traces()
    sim = O.OracleSim.from_workload(wl)
    cached = {}
    dtok = {}
    tot_cost = 0
    t_prev_end, all_done_prev = None, True
    emitted = 0
    n_steps = 0
    while True:
        info, ents = sim.step_replica(0)
        if not info["executed"]:
            break
        n_steps += 1
        # clock: contiguous unless the replica was empty (idle jump, M6)
        if t_prev_end is not None and not all_done_prev:
            assert info["t_start_us"] == t_prev_end
        if t_prev_end is not None:
            assert info["t_start_us"] >= t_prev_end
        assert info["t_end_us"] == info["t_start_us"] + info["cost_us"]
        tot_cost += info["cost_us"]
        # order: ascending (class, key, id); locked class only for residents
        keys = [(e["klass"], e["key"], e["id"]) for e in ents]
        assert keys == sorted(keys)
        for e in ents:
            assert e["klass"] in (0, 1)
            if e["klass"] == 0:
                assert e["resident_before"] == 1 and guard == 1
        # admission walk structure
        adm = [e for e in ents if e["want"] > 0]
        assert ents[0]["want"] > 0                                  # the head always runs: no empty batch
        assert len(adm) <= M and sum(e["want"] for e in adm) <= T
        foot = 0
        for e in adm:
            before = cached.get(e["id"], 0)
            assert 1 <= e["want"] <= c
            foot += -(-(before + e["want"]) // blk)
        assert foot == info["claimed_blocks"] <= B
        # no leap-frogging past a blocked newcomer: admitted non-residents are a prefix of the non-residents
        seen_skipped_new = False
        for e in ents:
            if e["resident_before"] == 0:
                if e["want"] == 0:
                    seen_skipped_new = True
                else:
                    assert not seen_skipped_new
        # victims: non-admitted residents, taken from the back of the order
        nonadm_res = [e for e in ents if e["want"] == 0 and e["resident_before"] == 1]
        flags = [e["evict"] != 0 for e in nonadm_res]
        assert flags == sorted(flags)                               # False... then True...: a suffix
        for e in ents:
            if e["evict"]:
                assert e["want"] == 0 and e["resident_before"] == 1 and e["resident_after"] == 0
                if e["evict"] == 1:
                    assert e["cached_after"] == 0
                assert pre != W.PRE_RECOMPUTE or e["evict"] == 1
        # minimality: keeping the first victim as well would overflow
        kept = sum(-(-cached[e["id"]] // blk) for e in nonadm_res if not e["evict"])
        assert kept + info["claimed_blocks"] <= B
        vict = [e for e in nonadm_res if e["evict"]]
        if vict:
            assert kept + -(-cached[vict[0]["id"]] // blk) + info["claimed_blocks"] > B
        # KV occupancy after the step, recomputed from the dump
        occ = sum(-(-e["cached_after"] // blk) for e in ents if e["resident_after"])
        assert occ == info["kv_resident_after"] <= B
        for e in ents:
            cached[e["id"]] = e["cached_after"]
            emitted += e["d_after"] - dtok.get(e["id"], 0)
            dtok[e["id"]] = e["d_after"]
        all_done_prev = all(e["d_after"] == D[0, e["id"]] for e in ents)
        t_prev_end = info["t_end_us"]
    st = sim.stats()[0]
    n = len(P[0])
    assert st["done"] == 1 and st["n_completed"] == n and st["iterations"] == n_steps
    assert st["swap_used"] == 0 and st["evict_swap"] == st["swapins"]
    assert st["prefill_tokens"] + st["decode_seqs"] == int((P[0] + D[0] - 1).sum()) + st["tokens_lost"]
    assert st["tokens_emitted"] == emitted == int(D[0].sum())
    assert st["t_end_us"] >= tot_cost
    assert st["evict_recompute"] + st["evict_swap"] > 0
    if pre == W.PRE_RECOMPUTE:
        assert st["evict_swap"] == 0
    tf, tl, ne, neu = sim.per_request()
    assert (tf[0] >= a[0]).all() and (tl[0] >= tf[0]).all()
    assert int(ne[0].sum()) == st["evict_recompute"] + st["evict_swap"]


def test_swap_pool_never_overflows():
    wl = pressure_workload(3, policy=W.POLICY_SRPT, guard=0, delta=0, preempt=W.PRE_SWAP, swap_pool_blocks=6)
    sim = O.OracleSim.from_workload(wl)
    seen_fallback = False
    for _ in range(100000):
        info, ents = sim.step_replica(0)
        if not info["executed"]:
            break
        st = sim.stats()[0]
        assert 0 <= st["swap_used"] <= 6
        seen_fallback |= any(e["evict"] == 1 for e in ents)
    assert seen_fallback and st["evict_swap"] > 0      # the pool filled up at least once => recompute fallback


# ------------------------------------------------------------------ P8 textbook single server

@pytest.mark.parametrize("seed", range(5))
def test_gg1_fifo_lindley(seed):
    """M=1, P=1, zero token costs, FCFS: the replica is a G/G/1 FIFO queue with service D_i*c0:
    C_i = max(a_i, C_{i-1}) + D_i*c0 (Lindley), TTFT_i = max(a_i, C_{i-1}) + c0 - a_i."""
    rng = np.random.default_rng([8, seed])
    n, c0 = 200, 5000
    D = rng.integers(1, 12, n)
    a = np.cumsum(rng.exponential(30000, n)).astype(np.int64)
    wl = W.custom(a, np.ones(n, np.int32), D, dict(
        max_batch=1, kv_blocks=1 << 20, c0_us=c0, c_prefill_tok_us=0, c_decode_seq_us=0, queue_cap=n),
        W.make_replicas(1, policy=W.POLICY_FCFS, guard=0, hysteresis_us=0))
    sim = run_wl(wl)
    tf, tl, _, _ = sim.per_request()
    C_prev = 0
    for i in range(n):
        start = max(int(a[i]), C_prev)
        C_prev = start + int(D[i]) * c0
        assert tl[0, i] == C_prev and tf[0, i] == start + c0
    assert sim.stats()[0]["t_end_us"] == C_prev


# ------------------------------------------------------------------ P9 brute force on tiny traces

def _brute_optima(arr, D):
    """Slotted single server: exhaustive DP over every work-conserving preemptive slot schedule."""
    n = len(D)

    @lru_cache(None)
    def best(t, rem):
        if not any(rem):
            return 0, 0
        avail = [j for j in range(n) if rem[j] and arr[j] <= t]
        if not avail:
            return best(min(arr[j] for j in range(n) if rem[j]), rem)
        bs, bm = None, None
        for j in avail:
            r2 = rem[:j] + (rem[j] - 1,) + rem[j + 1:]
            s, m = best(t + 1, r2)
            if rem[j] == 1:
                flow = t + 1 - arr[j]
            else:
                flow = 0
            bs = s + flow if bs is None else min(bs, s + flow)
            bm = max(m, flow) if bm is None else min(bm, max(m, flow))
        return bs, bm

    # min of sum and min of max are separate optimisations; compute each with its own recursion
    @lru_cache(None)
    def best_sum(t, rem):
        if not any(rem):
            return 0
        avail = [j for j in range(n) if rem[j] and arr[j] <= t]
        if not avail:
            return best_sum(min(arr[j] for j in range(n) if rem[j]), rem)
        return min((t + 1 - arr[j] if rem[j] == 1 else 0) + best_sum(t + 1, rem[:j] + (rem[j] - 1,) + rem[j + 1:])
                   for j in avail)

    @lru_cache(None)
    def best_max(t, rem):
        if not any(rem):
            return 0
        avail = [j for j in range(n) if rem[j] and arr[j] <= t]
        if not avail:
            return best_max(min(arr[j] for j in range(n) if rem[j]), rem)
        return min(max((t + 1 - arr[j] if rem[j] == 1 else 0), best_max(t + 1, rem[:j] + (rem[j] - 1,) + rem[j + 1:]))
                   for j in avail)

    return best_sum(0, tuple(D)), best_max(0, tuple(D))


@pytest.mark.parametrize("seed", range(40))
def test_bruteforce_tiny_traces(seed):
    """Single server, arrivals on the c0 grid, N <= 5, D <= 4: over ALL preemptive slot schedules SRPT attains the
    minimum total response time and FCFS the minimum maximum response time (classical results the paper builds
    on); the oracle's schedules must attain those optima."""
    rng = np.random.default_rng([9, seed])
    n = int(rng.integers(2, 6))
    D = [int(x) for x in rng.integers(1, 5, n)]
    arr = sorted(int(x) for x in rng.integers(0, 7, n))
    c0 = 1000
    opt_sum, opt_max = _brute_optima(tuple(arr), D)
    res = {}
    for pol in (W.POLICY_SRPT, W.POLICY_FCFS):
        wl = W.custom(np.array(arr) * c0, np.ones(n, np.int32), D, dict(
            max_batch=1, kv_blocks=1 << 16, c0_us=c0, c_prefill_tok_us=0, c_decode_seq_us=0, queue_cap=n),
            W.make_replicas(1, policy=pol, guard=0, hysteresis_us=0))
        sim = run_wl(wl)
        _, tl, _, _ = sim.per_request()
        res[pol] = (tl[0, :n] - np.array(arr) * c0) // c0
        assert ((tl[0, :n] - np.array(arr) * c0) % c0 == 0).all()
    assert int(res[W.POLICY_SRPT].sum()) == opt_sum
    assert int(res[W.POLICY_FCFS].max()) == opt_max


# ------------------------------------------------------------------ baselines SJF / SPF as static keys

@pytest.mark.parametrize("seed", range(20))
def test_sjf_spf_are_shortest_processing_time_first(seed):
    """Single server, all jobs present at time 0: shortest-processing-time-first minimises the total completion time
    (Smith's rule, 1 || sum C_j).  SJF sees job size = output length D (one token per slot); SPF sees job size =
    prompt length P (one prefill token per slot, single-token outputs).  Both must attain the brute-force optimum
    over ALL slot schedules, which is also the closed form sum_k (n - k) s_(k) over the sorted sizes."""
    rng = np.random.default_rng([14, seed])
    n = int(rng.integers(2, 6))
    size = [int(x) for x in rng.integers(1, 5, n)]
    c0 = 1000
    opt_sum, _ = _brute_optima(tuple([0] * n), size)
    closed = sum((n - k) * v for k, v in enumerate(sorted(size)))
    assert opt_sum == closed
    sjf = W.custom(np.zeros(n, np.int64), np.ones(n, np.int32), size, dict(
        max_batch=1, kv_blocks=1 << 16, c0_us=c0, c_prefill_tok_us=0, c_decode_seq_us=0, queue_cap=n),
        W.make_replicas(1, policy=W.POLICY_SJF, guard=0, hysteresis_us=0))
    spf = W.custom(np.zeros(n, np.int64), size, np.ones(n, np.int32), dict(
        max_batch=1, chunk_tokens=1, token_budget=1, kv_blocks=1 << 16, c0_us=c0, c_prefill_tok_us=0,
        c_decode_seq_us=0, queue_cap=n),
        W.make_replicas(1, policy=W.POLICY_SPF, guard=0, hysteresis_us=0))
    for wl in (sjf, spf):
        sim = run_wl(wl)
        _, tl, _, _ = sim.per_request()
        assert (tl[0, :n] % c0 == 0).all()
        assert int(tl[0, :n].sum()) // c0 == opt_sum
        # the completion order is the size order (ties by id)
        assert list(np.argsort(tl[0, :n], kind="stable")) == sorted(range(n), key=lambda i: (size[i], i))


def test_sjf_preempts_by_total_length_not_by_remaining():
    """A static key: a job of length 3 arriving while a job of length 4 has 1 token left still preempts it (SRPT
    would not) -- the difference between SJF with perfect lengths and SRPT."""
    c0 = 1000
    arr, D = np.array([0, 3]) * c0, [4, 3]
    out = {}
    for pol in (W.POLICY_SJF, W.POLICY_SRPT):
        wl = W.custom(arr, np.ones(2, np.int32), D, dict(
            max_batch=1, kv_blocks=1 << 16, c0_us=c0, c_prefill_tok_us=0, c_decode_seq_us=0, queue_cap=2),
            W.make_replicas(1, policy=pol, guard=0, hysteresis_us=0))
        out[pol] = [int(x) // c0 for x in run_wl(wl).per_request()[1][0, :2]]
    assert out[W.POLICY_SJF] == [7, 6]        # job 0 runs slots 0-2, waits for job 1 (slots 3-5), finishes in slot 6
    assert out[W.POLICY_SRPT] == [4, 7]       # job 0 (1 left) keeps the server, job 1 runs slots 4-6


# ------------------------------------------------------------------ P10 Eq. 6 arg-min subset

@pytest.mark.parametrize("seed", range(10))
def test_admitted_set_is_argmin_subset(seed):
    """Eq. 6: with KV and token budget non-binding the batch is the size-min(n,M) subset of
    minimum total priority."""
    rng = np.random.default_rng([10, seed])
    n, M = int(rng.integers(4, 11)), int(rng.integers(1, 6))
    P = rng.integers(1, 3000, n)
    D = rng.integers(2, 50, n)
    a = np.sort(rng.choice(1000, n, replace=False)).astype(np.int64)      # all present from iteration 2 on
    wl = W.custom(a + 10_000_000, P, D, dict(
        max_batch=M, kv_blocks=1 << 20, token_budget=1 << 20, chunk_tokens=1 << 20, queue_cap=n),
        W.make_replicas(1, policy=W.POLICY_BOOST, gamma=0.05))
    sim = O.OracleSim.from_workload(wl)
    # first iteration with every request present: step until all n have been ingested
    for _ in range(1000):
        info, ents = sim.step_replica(0)
        if info["n_active"] == n:
            break
    assert info["n_active"] == n
    prio = {e["id"]: (e["klass"], e["key"]) for e in ents}
    assert len(set(prio.values())) == n                      # distinct => unique optimum
    got = frozenset(e["id"] for e in ents if e["want"] > 0)
    m = min(n, M)
    # locked (class 0) requests precede everything: lexicographic (class, key) sum
    best = min(itertools.combinations(range(n), m),
               key=lambda S: (sum(prio[i][0] for i in S), sum(prio[i][1] for i in S)))
    assert got == frozenset(best)


# ------------------------------------------------------------------ P11 MemGuard logarithmic bound

@pytest.mark.parametrize("seed", range(8))
@pytest.mark.parametrize("policy", [W.POLICY_BOOST, W.POLICY_SRPT, W.POLICY_LAS, W.POLICY_SJF, W.POLICY_SPF])
def test_memguard_logarithmic_preemption_bound(seed, policy):
    """'request i can trigger at most 1 + floor(log2(S_i/k)) priority-revision points':
    evictions of a request that was not locked (unforced) are bounded by that number."""
    k = 32
    wl = pressure_workload(seed, n=80, policy=policy, guard=1, gamma=0.02, bin_tokens=k, kv_blocks=40)
    _, P, D, _ = wl.traces()
    sim = run_wl(wl)
    _, _, ne, neu = sim.per_request()
    S = (P[0] + D[0]).astype(np.int64)
    bound = 1 + np.floor(np.log2(np.maximum(S, k) / k)).astype(np.int64)
    assert (neu[0] <= bound).all()
    assert (neu[0] <= ne[0]).all()
    assert int(ne[0].sum()) > 0


# ------------------------------------------------------------------ P12 Lemma A.1 invariant

def test_assigned_boost_at_most_b_of_half_attained():
    """'it assigns a job of attained service a a boost of at most b_gamma(a/2)'."""
    tok, k = 5000, 256
    for gamma in (0.01, 0.3, 1.0):
        for sig in [256, 300, 511, 512, 1000, 4095, 4096, 10000, 36864]:
            assigned = O.boost_us(gamma, k * 2 ** O.quant_bin(sig, k), tok)
            getcontext().prec = 50
            half = _boost_exact_us(gamma, Decimal(sig) / 2, tok)
            assert Decimal(assigned) <= half + 1


# ------------------------------------------------------------------ P13 percentiles

def test_percentile_is_inverted_cdf():
    """t_p = inf{t : Fbar(t) <= (100-p)/100} == numpy's 'inverted_cdf'."""
    rng = np.random.default_rng(13)
    for m in [1, 2, 3, 7, 10, 99, 100, 101, 1000, 4000]:
        x = np.sort(rng.integers(0, 10 ** 9, m))
        for p in (50, 90, 99):
            assert O.percentile_nearest_rank(x, p) == int(np.percentile(x, p, method="inverted_cdf"))


def test_stats_percentiles_from_outputs():
    wl = W.config2(n_seeds=1)
    a, P, D, _ = wl.traces()
    sim = run_wl(wl)
    tf, tl, _, _ = sim.per_request()
    for r, st in enumerate(sim.stats()):
        ttft = tf[r] - a[0]
        ttlt = tl[r] - a[0]
        for i, p in enumerate((50, 90, 99)):
            assert st["ttft_us"][i] == int(np.percentile(ttft, p, method="inverted_cdf"))
            assert st["ttlt_us"][i] == int(np.percentile(ttlt, p, method="inverted_cdf"))
            assert st["ttlt_s"][i] == pytest.approx(st["ttlt_us"][i] * 1e-6, rel=1e-15)
        assert st["mean_ttlt_s"] == pytest.approx(float(ttlt.mean()) * 1e-6, rel=1e-12)
        assert st["mean_tbt_s"] == pytest.approx(float((tl[r] - tf[r]).sum()) / float((D[0] - 1).sum()) * 1e-6, rel=1e-12)


def test_tbt_histogram_bins_and_percentiles():
    """M11: log-linear histogram, 7 sub-bits: every gap lies in [edge, edge*(1+2^-7)); percentile from the histogram
    is within 2^-7 of the exact pooled nearest-rank gap."""
    for g in list(range(0, 2000)) + [2 ** k + d for k in range(8, 40) for d in (-1, 0, 1, 12345 % (2 ** k))]:
        b = O.tbt_bin(g)
        lo = O.tbt_edge(b)
        hi = O.tbt_edge(b + 1)
        assert lo <= g < hi and 0 <= b < O.TBT_BINS
        assert hi - lo <= max(1, lo >> 7)
    # pooled gaps rebuilt from per-step emission times
    wl = pressure_workload(2, n=60)
    sim = O.OracleSim.from_workload(wl)
    last, dprev, gaps = {}, {}, []
    while True:
        info, ents = sim.step_replica(0)
        if not info["executed"]:
            break
        for e in ents:
            if e["d_after"] > dprev.get(e["id"], 0):
                if e["d_after"] >= 2:
                    gaps.append(info["t_end_us"] - last[e["id"]])
                last[e["id"]] = info["t_end_us"]
                dprev[e["id"]] = e["d_after"]
    hist = sim.tbt_hist(0)
    assert int(hist.sum()) == len(gaps)
    ref = np.bincount([O.tbt_bin(g) for g in gaps], minlength=O.TBT_BINS)
    assert np.array_equal(hist, ref)
    st = sim.stats()[0]
    gs = np.sort(np.array(gaps))
    for i, p in enumerate((50, 90, 99)):
        exact = int(np.percentile(gs, p, method="inverted_cdf"))
        assert st["tbt_us"][i] <= exact < st["tbt_us"][i] * (1 + 2 ** -7) + 1


# ------------------------------------------------------------------ P14 batch invariance (oracle side)

def test_oracle_batch_invariance():
    """A replica's schedule does not depend on the other replicas, on its index, on Q >= peak, or on step granularity."""
    base = W.config2(n_seeds=2)
    full = run_wl(base)
    dg = full.digest()
    sub = base.select([4, 1])
    s2 = run_wl(sub)
    assert s2.digest().tolist() == [dg[4], dg[1]]
    peak = max(s["peak_active"] for s in full.stats())
    small_q = base.select([4, 1]); small_q.sim = dict(small_q.sim, queue_cap=peak)
    assert run_wl(small_q).digest().tolist() == [dg[4], dg[1]]
    s3 = O.OracleSim.from_workload(sub)
    for k in (1, 7, 1000, 100000):
        s3.step(k)
    assert s3.digest().tolist() == [dg[4], dg[1]]


def test_queue_cap_defers_arrivals():
    """M6: arrivals wait in the trace while the window is full; nothing is lost."""
    wl = pressure_workload(5, n=80, mean_gap_us=500, queue_cap=8)
    sim = run_wl(wl)
    st = sim.stats()[0]
    assert st["peak_active"] == 8 and st["n_completed"] == 80


# ------------------------------------------------------------------ loader validation

def test_loader_rejects_bad_traces():
    ok = dict(kv_blocks=64, queue_cap=4)
    good = W.custom([0, 10], [5, 5], [5, 5], ok)
    O.OracleSim.from_workload(good)
    with pytest.raises(O.OracleError) as e:
        O.OracleSim.from_workload(W.custom([10, 0], [5, 5], [5, 5], ok))
    assert e.value.code == -5
    for P, D in (([0, 5], [5, 5]), ([5, 5], [0, 5]), ([5, 1000], [5, 100])):
        with pytest.raises(O.OracleError) as e:
            O.OracleSim.from_workload(W.custom([0, 10], P, D, ok))
        assert e.value.code == -6


def test_workload_generators_are_seeded_and_feasible():
    for cid, kw in [(1, {}), (2, dict(n_seeds=2)), (3, dict(n_seeds=2)), (4, dict(n_seeds=2, n_gamma=3)),
                    (5, dict(n_seeds=2, n_requests=512)), (6, dict(n_seeds=1))]:
        wl = W.by_id(cid, **kw)
        a, P, D, n = wl.traces()
        a2, P2, D2, _ = wl.traces()
        assert np.array_equal(a, a2) and np.array_equal(P, P2) and np.array_equal(D, D2)
        assert (np.diff(a, axis=1) >= 0).all() and (a >= 0).all()
        assert (P >= 1).all() and (D >= 1).all()
        assert ((P + D + 15) // 16 <= wl.sim["kv_blocks"]).all()
        assert len(wl.replicas["gamma"]) == wl.R
        assert wl.replicas["trace_id"].max() == wl.sim["n_traces"] - 1
    # parallel generation gives the same arrays
    wl = W.config2(n_seeds=16)
    x = wl.traces(workers=1); y = wl.traces(workers=2)
    assert all(np.array_equal(u, v) for u, v in zip(x, y))


# ------------------------------------------------------------------ DistBoost (Phase 1 strawman, rule M14)

@pytest.mark.parametrize("seed", range(5))
@pytest.mark.parametrize("gamma", [0.05, 3.0])
def test_distboost_single_slot_is_non_preemptive_fifo(seed, gamma):
    """Eq. 5 selects the decode batch first.  With one slot and one-token prompts a request enters
    the decode queue in its first slot and then holds the server until it completes; equal prompts give equal
    prefill boosts, so the prefill queue is FIFO: the replica is the G/G/1 FIFO queue of the Lindley recursion,
    whatever gamma -- the inter-queue head-of-line blocking the paper describes."""
    rng = np.random.default_rng([15, seed])
    n, c0 = 150, 5000
    D = rng.integers(1, 12, n)
    a = np.cumsum(rng.exponential(30000, n)).astype(np.int64)
    wl = W.custom(a, np.ones(n, np.int32), D, dict(
        max_batch=1, kv_blocks=1 << 20, c0_us=c0, c_prefill_tok_us=0, c_decode_seq_us=0, queue_cap=n),
        W.make_replicas(1, policy=W.POLICY_DISTBOOST, guard=0, hysteresis_us=0, gamma=gamma))
    sim = run_wl(wl)
    tf, tl, _, _ = sim.per_request()
    C_prev = 0
    for i in range(n):
        start = max(int(a[i]), C_prev)
        C_prev = start + int(D[i]) * c0
        assert tl[0, i] == C_prev and tf[0, i] == start + c0


def test_distboost_two_queues_eq3_to_eq6():
    """Every iteration: the order is the decode queue (requests that emitted their first token) by the time they
    entered it (Eq. 4), then the prefill queue by a - b_gamma(prompt) (Eq. 3); the batch is a prefix of it (Eq. 5-6)."""
    wl = pressure_workload(3, n=120, kv_blocks=4096, policy=W.POLICY_DISTBOOST, guard=0, gamma=0.3)
    tr = wl.traces()
    a, P = tr[0][0], tr[1][0]
    o = O.OracleSim(wl.sim, wl.replicas, tr)
    first = {}
    k, tok = int(wl.sim["bin_tokens"]), int(wl.sim["tok_us"])
    seen_mixed = False
    for it in range(20000):
        info, rows = o.step_replica(0)
        if not info["executed"]:
            break
        dec = [r for r in rows if r["id"] in first]
        pre = [r for r in rows if r["id"] not in first]
        assert [r["id"] for r in rows] == [r["id"] for r in dec] + [r["id"] for r in pre]      # decode queue first
        assert all(r["klass"] == 0 and r["key"] == first[r["id"]] for r in dec)               # Eq. 4
        for r in pre:                                                                          # Eq. 3
            assert r["klass"] == 1 and r["key"] == int(a[r["id"]]) - O.boost_us(0.3, k * 2 ** O.quant_bin(int(P[r["id"]]), k), tok)
        assert [(r["key"], r["id"]) for r in dec] == sorted((r["key"], r["id"]) for r in dec)
        assert [(r["key"], r["id"]) for r in pre] == sorted((r["key"], r["id"]) for r in pre)
        adm = [r["want"] > 0 for r in rows]
        assert adm == sorted(adm, reverse=True)                                                # KV ample: a prefix
        seen_mixed |= bool(dec) and bool(pre)
        for r in rows:                                                                         # entering the decode queue
            if r["id"] not in first and r["d_after"] >= 1:
                first[r["id"]] = info["t_end_us"]
    assert seen_mixed
    tf = o.per_request()[0][0]
    assert all(tf[i] == t for i, t in first.items())
    o.close()


# ------------------------------------------------------------------ M16 Sarathi

@pytest.mark.parametrize("seed", range(4))
def test_sarathi_single_slot_is_non_preemptive_fifo(seed):
    """Decode-prioritised: with one slot and one-token prompts a request that has started decoding holds
    the server until it completes, and the prefill queue is first come first served: the G/G/1 FIFO queue of the
    Lindley recursion."""
    rng = np.random.default_rng([16, seed])
    n, c0 = 120, 5000
    D = rng.integers(1, 12, n)
    a = np.cumsum(rng.exponential(30000, n)).astype(np.int64)
    wl = W.custom(a, np.ones(n, np.int32), D, dict(
        max_batch=1, kv_blocks=1 << 20, c0_us=c0, c_prefill_tok_us=0, c_decode_seq_us=0, queue_cap=n),
        W.make_replicas(1, policy=W.POLICY_SARATHI, guard=0, hysteresis_us=0))
    tf, tl, _, _ = run_wl(wl).per_request()
    C_prev = 0
    for i in range(n):
        start = max(int(a[i]), C_prev)
        C_prev = start + int(D[i]) * c0
        assert tl[0, i] == C_prev and tf[0, i] == start + c0


def test_sarathi_decode_round_robin():
    """"Round-robin ordering in the decode": the decode queue is ordered by the time of the request's last
    token (tracked here from the per-iteration records), so whoever was left out of an iteration -- the KV pool is
    small -- goes in front of those that were served in it; the prefill queue behind it is first come first served."""
    wl = pressure_workload(2, n=140, kv_blocks=40, policy=W.POLICY_SARATHI, guard=0, delta=0, mean_gap_us=3000)
    tr = wl.traces()
    a = tr[0][0]
    o = O.OracleSim(wl.sim, wl.replicas, tr)
    t_last, d_seen = {}, {}
    left_out_then_first = 0
    prev_left, prev_served = set(), set()
    for it in range(200000):
        info, rows = o.step_replica(0)
        if not info["executed"]:
            break
        started = [r for r in rows if r["klass"] == 0]
        fresh = [r for r in rows if r["klass"] == 1]
        assert [r["id"] for r in rows] == [r["id"] for r in started] + [r["id"] for r in fresh]      # decode-prioritised
        assert all(d_seen.get(r["id"], 0) >= 1 for r in started) and all(d_seen.get(r["id"], 0) == 0 for r in fresh)
        assert all(r["key"] == t_last[r["id"]] for r in started)                                    # round robin
        assert all(r["key"] == int(a[r["id"]]) for r in fresh)                                      # FCFS prefill
        assert [(r["key"], r["id"]) for r in started] == sorted((r["key"], r["id"]) for r in started)
        assert [(r["key"], r["id"]) for r in fresh] == sorted((r["key"], r["id"]) for r in fresh)
        pos = {r["id"]: j for j, r in enumerate(started)}
        for x in prev_left:
            for y in prev_served:
                if x in pos and y in pos:
                    assert pos[x] < pos[y]
                    left_out_then_first += 1
        prev_left = {r["id"] for r in started if r["want"] == 0}
        prev_served = {r["id"] for r in started if r["want"] > 0 and r["d_after"] > d_seen.get(r["id"], 0)}
        for r in rows:
            if r["d_after"] > d_seen.get(r["id"], 0):
                t_last[r["id"]] = info["t_end_us"]
            d_seen[r["id"]] = r["d_after"]
    assert left_out_then_first > 50 and o.stats()[0]["n_completed"] == 140


@pytest.mark.parametrize("seed", range(3))
def test_sarathi_is_distboost_without_boost_when_the_batch_cap_does_not_bind(seed):
    """Decode first, chunked prefill piggy-backing first come first served: that is DistBoost (Eq. 3-6) with b_gamma = 0
    (gamma = +inf) except for the order INSIDE the decode queue (round robin vs entry time), which only matters when
    the batch cap, the token budget or the KV capacity cut the decode queue."""
    wl_s = pressure_workload(seed, n=150, kv_blocks=1 << 16, policy=W.POLICY_SARATHI, guard=0, delta=0, max_batch=256,
                             chunk_tokens=64, token_budget=1 << 15)
    wl_d = pressure_workload(seed, n=150, kv_blocks=1 << 16, policy=W.POLICY_DISTBOOST, guard=0, delta=0, gamma=float("inf"),
                             max_batch=256, chunk_tokens=64, token_budget=1 << 15)
    s, d = run_wl(wl_s), run_wl(wl_d)
    for x, y in zip(s.per_request(), d.per_request()):
        assert np.array_equal(x, y)
    assert s.stats()[0]["t_end_us"] == d.stats()[0]["t_end_us"]
