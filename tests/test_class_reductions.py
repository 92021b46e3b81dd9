"""Pins of rule M15 (preemption time) and of the per-class reductions (Tables 3-5,
PAPER.md:549-560, 604-620) on the oracle -- CPU only -- and their GPU parity.

* hand-worked: the preemption times read off the hand-derived schedules of tests/golden/hand_traces.md;
* closed form: with a KV pool of ONE block and one-token prompts only one request can hold the device, every own
  iteration emits exactly one token, so a request's preemption time is the span between its first and last token
  minus its own D - 1 iterations -- whatever the policy preempts;
* numpy: class filter + `inverted_cdf` percentiles, counts and sums on the oracle's own per-request outputs.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_18431_b200 import workloads as W
from tests.helpers import hand_cases, hand_workload, pressure_workload


@pytest.mark.parametrize("case", hand_cases(), ids=[c["name"] for c in hand_cases()])
def test_preemption_time_hand_worked(case):
    o = O.OracleSim.from_workload(hand_workload(case))
    o.run()
    n = len(case["prompt"])
    assert o.preempt_time()[0, :n].tolist() == case["expect"]["t_preempt_us"]


@pytest.mark.parametrize("policy", [W.POLICY_SRPT, W.POLICY_FCFS, W.POLICY_SJF, W.POLICY_LAS])
@pytest.mark.parametrize("preempt", [W.PRE_RECOMPUTE, W.PRE_SWAP])
def test_preemption_time_single_block_closed_form(policy, preempt):
    c0 = 1000
    for seed in range(6):
        rng = np.random.default_rng([15, seed])
        n = 14
        D = rng.integers(1, 15, n)                       # P + D <= 15 tokens: one block of 16
        P = np.ones(n, np.int64)
        a = np.sort(rng.integers(0, 40, n)) * c0
        sim = dict(kv_blocks=1, block_tokens=16, max_batch=8, chunk_tokens=64, token_budget=64, c0_us=c0,
                   c_prefill_tok_us=0, c_decode_seq_us=0, preempt_mode=preempt, swap_ns_per_block=0, swap_pool_blocks=64,
                   queue_cap=n)
        rep = W.make_replicas(1, policy=policy, guard=0, hysteresis_us=0)
        o = O.OracleSim.from_workload(W.custom(a, P, D, sim, rep))
        o.run()
        tf, tl, ne, _ = o.per_request()
        tp = o.preempt_time()[0, :n]
        assert np.array_equal(tp, (tl[0, :n] - tf[0, :n]) - (D - 1) * c0), (policy, preempt, seed)
        assert np.array_equal(tp > 0, ne[0, :n] > 0)
        if policy == W.POLICY_FCFS:
            assert not tp.any()                          # the head of the line is never displaced
        if policy == W.POLICY_SRPT:
            assert ne.sum() > 0                          # shorter newcomers do displace


def _classes(wl):
    a, P, D, n = wl.traces()
    return (P + D).astype(np.int64), a


@pytest.mark.parametrize("seed", [0, 1])
def test_class_percentiles_are_numpy_on_the_filtered_outputs(seed):
    wl = pressure_workload(seed, n=160, kv_blocks=40, preempt=W.PRE_AUTO, swap_pool_blocks=24, n_replicas=2,
                           policy=[W.POLICY_BOOST, W.POLICY_SRPT], guard=[1, 0])
    o = O.OracleSim.from_workload(wl)
    o.run()
    length, a = _classes(wl)
    tf, tl, ne, _ = o.per_request()
    tp = o.preempt_time()
    pm = [250, 500, 900, 990, 1000]
    thr = int(np.median(length[0]))
    assert tp.sum() > 0
    for r in range(2):
        tot = 0
        for lo, hi in ((0, thr), (thr + 1, 1 << 30)):
            sel = (length[0] >= lo) & (length[0] <= hi)
            tot += sel.sum()
            for which, vals in ((0, tf[r] - a[0]), (1, tl[r] - a[0]), (2, tp[r])):
                out, cnt, sm = o.class_percentiles(which, lo, hi, pm)
                v = vals[sel]
                assert cnt[r] == v.size and sm[r] == v.sum()
                want = [int(np.percentile(v, p / 10.0, method="inverted_cdf")) for p in pm]
                assert out[r].tolist() == want, (r, which, lo, hi)
                assert out[r, -1] == v.max()             # per-mille 1000 is the maximum (Table 4's "Max")
        assert tot == 160
    # the whole range reproduces the unconditional curve
    assert np.array_equal(o.class_percentiles(1, 0, 1 << 30, pm)[0], o.percentile_curve(1, pm))


def test_preemption_time_invariants():
    wl = pressure_workload(3, n=200, kv_blocks=36, preempt=W.PRE_AUTO, swap_pool_blocks=10)
    o = O.OracleSim.from_workload(wl)
    o.run()
    tf, tl, ne, _ = o.per_request()
    tp = o.preempt_time()
    a = wl.traces()[0]
    assert np.array_equal(tp[0] > 0, ne[0] > 0)          # an evicted request comes back in a later iteration
    assert np.all(tp[0] <= tl[0] - a[0])                 # and never counts more than its whole stay
    assert ne.sum() > 20


# ------------------------------------------------------------------------------------------ GPU parity

@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_2606_18431_b200 import binding
    binding.lib()
    return binding


@pytest.mark.gpu
@pytest.mark.parametrize("policy,guard", [(W.POLICY_BOOST, 1), (W.POLICY_SRPT, 0), (W.POLICY_FCFS, 0), (W.POLICY_DISTBOOST, 0)])
@pytest.mark.parametrize("preempt", [W.PRE_RECOMPUTE, W.PRE_AUTO])
def test_gpu_preemption_time_and_class_percentiles(gpu, policy, guard, preempt):
    for seed in range(2):
        wl = pressure_workload(seed, n=220, kv_blocks=40, policy=policy, guard=guard, preempt=preempt, swap_pool_blocks=20,
                               n_replicas=3)
        tr = wl.traces()
        g = gpu.Sim(wl.sim, wl.replicas, tr); o = O.OracleSim(wl.sim, wl.replicas, tr)
        g.run(); o.run()
        assert np.array_equal(g.preempt_time(), o.preempt_time())
        assert o.preempt_time().sum() > 0
        length = (tr[1] + tr[2]).astype(np.int64)[0]
        thr = int(np.median(length))
        pm = [500, 900, 990, 1000]
        for lo, hi in ((0, thr), (thr + 1, 1 << 30), (0, 1 << 30), (10 ** 6, 10 ** 7)):
            for which in (0, 1, 2):
                go, gc, gs = g.class_percentiles(which, lo, hi, pm)
                oo, oc, os_ = o.class_percentiles(which, lo, hi, pm)
                assert np.array_equal(go, oo) and np.array_equal(gc, oc) and np.array_equal(gs, os_), (which, lo, hi)
        g.close(); o.close()


@pytest.mark.gpu
def test_gpu_starvation_shape_short_vs_long(gpu):
    """The starvation experiment's shape (90 % short ~125/100, 10 % long 2000/6000, rho ~ 0.99): short- and
    long-request E2E percentiles and the long requests' preemption P99 (Tables 3-5) on the device equal the oracle's."""
    wl = W.starvation(n_seeds=4, n_requests=600)
    tr = wl.traces()
    g = gpu.Sim(wl.sim, wl.replicas, tr); o = O.OracleSim(wl.sim, wl.replicas, tr)
    g.run(); o.run()
    pm = [500, 900, 950, 990, 1000]
    for lo, hi in ((0, 1000), (1001, 1 << 30)):
        for which in (1, 2):
            a, b = g.class_percentiles(which, lo, hi, pm), o.class_percentiles(which, lo, hi, pm)
            for x, y in zip(a, b):
                assert np.array_equal(x, y)
    assert o.class_percentiles(1, 1001, 1 << 30, pm)[1].sum() > 0
    g.close(); o.close()


@pytest.mark.gpu
def test_gpu_class_percentiles_argument_checks(gpu):
    wl = pressure_workload(0, n=40)
    g = gpu.Sim(wl.sim, wl.replicas, wl.traces())
    for which, lo, hi, pm in ((3, 0, 10, [500]), (0, 10, 5, [500]), (1, 0, 10, [0]), (1, 0, 10, [1001]), (1, 0, 10, list(range(1, 18)))):
        with pytest.raises(gpu.UbError) as e:
            g.class_percentiles(which, lo, hi, pm)
        assert e.value.code == gpu.UB_EINVAL
    out, cnt, tot = g.class_percentiles(2, 0, 1 << 30, [500, 1000])      # nothing has run: empty classes
    assert not out.any() and not cnt.any() and not tot.any()
    g.close()
