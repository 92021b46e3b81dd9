"""GPU parity: the CUDA path (through the C-ABI of libuniboost.so) against the CPU oracle, element by element,
on the same seeded inputs.  Bar (north_star): the whole schedule bit-exact -- boost table, per-iteration digest,
per-request (t_first, t_last, n_evict), counters, integer-microsecond percentiles -- and the fp64 percentiles in
seconds within 1e-9 relative (they are the same integers times 1e-6, so in fact equal).
"""
import numpy as np
import pytest

from paper_2606_18431_b200 import workloads as W
from tests.helpers import hand_cases, hand_workload, pressure_workload

pytestmark = pytest.mark.gpu

INT_STATS = ("iterations", "request_steps", "n_completed", "evict_recompute", "evict_swap", "swapins",
             "tokens_lost", "tokens_emitted", "prefill_tokens", "decode_seqs", "t_end_us", "peak_active", "done",
             "swap_used", "ttft_us", "ttlt_us", "tbt_us", "sum_ttft_us", "sum_ttlt_us", "sum_tbt_num_us",
             "sum_tbt_den")
F64_STATS = ("ttft_s", "ttlt_s", "tbt_s", "mean_ttft_s", "mean_ttlt_s", "mean_tbt_s", "tokens_per_s")
REL_TOL = 1e-9


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_2606_18431_b200 import binding
    binding.lib()
    return binding


def _pair(gpu, oracle_mod, wl, ipl=1, workers=1):
    tr = wl.traces(workers=workers)
    g = gpu.Sim(wl.sim, wl.replicas, tr, iters_per_launch=ipl)
    o = oracle_mod.OracleSim(wl.sim, wl.replicas, tr)
    return g, o


def _assert_same(g, o, where=""):
    dg, do = g.digest(), o.digest()
    bad = np.nonzero(dg != do)[0]
    assert bad.size == 0, f"{where}: digest differs on replicas {bad[:8]} ({bad.size} of {len(dg)})"
    gtf, gtl, gne, gneu = g.per_request()
    otf, otl, one, oneu = o.per_request()
    assert np.array_equal(gtf, otf), f"{where}: t_first"
    assert np.array_equal(gtl, otl), f"{where}: t_last"
    assert np.array_equal(gne, one), f"{where}: n_evict"
    assert np.array_equal(gneu, oneu), f"{where}: n_evict_unforced"
    gs, os_ = g.stats(), o.stats()
    for r, (a, b) in enumerate(zip(gs, os_)):
        for k in INT_STATS:
            assert a[k] == b[k], f"{where}: replica {r} stat {k}: gpu {a[k]} oracle {b[k]}"
        for k in F64_STATS:
            av, bv = np.atleast_1d(a[k]).astype(float), np.atleast_1d(b[k]).astype(float)
            assert np.all(np.abs(av - bv) <= REL_TOL * np.maximum(1e-300, np.abs(bv))), f"{where}: replica {r} {k}"


def _assert_hist_same(g, o, reps):
    for r in reps:
        assert np.array_equal(g.tbt_hist(r), o.tbt_hist(r)), f"TBT histogram of replica {r}"


# ------------------------------------------------------------------------------------------ boost table (M4)

@pytest.mark.parametrize("gamma", [0.01, 0.05, 0.3, 1.0, 10.0, 100.0, float("inf"), 1e-7])
@pytest.mark.parametrize("quant", [W.QUANT_GEOMETRIC, W.QUANT_EXACT])
def test_boost_table_bit_exact(gpu, oracle_mod, gamma, quant):
    wl = pressure_workload(1, n=40, gamma=gamma, quant=quant)
    g, o = _pair(gpu, oracle_mod, wl)
    assert np.array_equal(g.boost_lut(0), o.boost_lut(0))


# ------------------------------------------------------------------------------------------ hand-worked schedules

@pytest.mark.parametrize("case", hand_cases(), ids=[c["name"] for c in hand_cases()])
def test_hand_worked_schedules_on_the_device(gpu, oracle_mod, case):
    """tests/golden/hand_traces.md (A-J): the CUDA path against the numbers derived by hand from Algorithm 1
     -- the PHASE signal, the AUTO swap rule, swap-time rounding, the one-token prefill tail among
    them -- iteration by iteration, and against the oracle."""
    wl = hand_workload(case)
    exp = case["expect"]
    g, o = _pair(gpu, oracle_mod, wl)
    t_prev, costs = 0, []
    for it in range(len(exp["step_costs_us"])):
        g.step(1)
        info, _ = o.step_replica(0)
        t = g.debug_state(0)["clock_us"]
        assert t == info["t_end_us"], f"iteration {it}"
        costs.append(t - info["t_start_us"])
        assert g.digest()[0] == o.digest()[0], f"iteration {it}"
    assert costs == exp["step_costs_us"]
    assert g.step(1, want_live=True) == 0
    n = len(case["prompt"])
    tf, tl, ne, neu = g.per_request()
    assert tf[0, :n].tolist() == exp["t_first_us"] and tl[0, :n].tolist() == exp["t_last_us"]
    assert ne[0, :n].tolist() == exp["n_evict"]
    if "n_evict_unforced" in exp:
        assert neu[0, :n].tolist() == exp["n_evict_unforced"]
    st = g.stats()[0]
    for k in ("iterations", "request_steps", "t_end_us", "tokens_lost", "prefill_tokens", "decode_seqs",
              "evict_recompute", "evict_swap") + (("swapins",) if "swapins" in exp else ()):
        assert st[k] == exp[k], k
    _assert_same(g, o, case["name"])


# ------------------------------------------------------------------------------------------ config 1 in full

def test_config1_full_schedule(gpu, oracle_mod):
    wl = W.config1()
    g, o = _pair(gpu, oracle_mod, wl)
    g.run(); o.run()
    _assert_same(g, o, "config1")
    _assert_hist_same(g, o, [0])
    st = g.stats()[0]
    assert st["done"] == 1 and st["n_completed"] == 256


def test_config1_step_by_step(gpu, oracle_mod):
    """Digest, clock and the active window (id, d, cached, resident) after every single iteration."""
    wl = W.config1()
    g, o = _pair(gpu, oracle_mod, wl)
    for it in range(3000):
        g.step(1)
        info, rows = o.step_replica(0)
        st = g.debug_state(0)
        assert g.digest()[0] == o.digest()[0], f"iteration {it}"
        assert st["clock_us"] == info["t_end_us"]
        live = [(r["id"], r["d_after"], r["cached_after"], r["resident_after"]) for r in rows
                if not (r["want"] > 0 and r["cached_after"] == 0 and r["resident_after"] == 0 and r["evict"] == 0)]
        got = [(int(i), int(d), int(c), int(f & 1)) for i, d, c, f in zip(st["id"], st["d"], st["cached"], st["flags"])]
        assert sorted(got) == sorted(live), f"iteration {it}"
        assert [x[0] for x in got] == [x[0] for x in live], f"iteration {it}: stored order is the priority order"


# ------------------------------------------------------------------------------------------ memory pressure

@pytest.mark.parametrize("policy", [W.POLICY_FCFS, W.POLICY_SRPT, W.POLICY_BOOST, W.POLICY_LAS, W.POLICY_SJF,
                                    W.POLICY_SPF, W.POLICY_DISTBOOST, W.POLICY_SARATHI])
@pytest.mark.parametrize("preempt", [W.PRE_RECOMPUTE, W.PRE_SWAP, W.PRE_AUTO])
def test_pressure_policies_preemption(gpu, oracle_mod, policy, preempt):
    for seed in range(4):
        wl = pressure_workload(seed, n=120, kv_blocks=40, policy=policy, preempt=preempt,
                               guard=1 if policy in (W.POLICY_BOOST, W.POLICY_DISTBOOST) else 0, swap_pool_blocks=24)
        g, o = _pair(gpu, oracle_mod, wl)
        g.run(); o.run()
        _assert_same(g, o, f"pressure seed {seed} policy {policy} preempt {preempt}")
        _assert_hist_same(g, o, [0])
        assert o.stats()[0]["evict_recompute"] + o.stats()[0]["evict_swap"] > 0, "the case must exercise eviction"


@pytest.mark.parametrize("signal,quant", [(W.SIG_UNIFIED, W.QUANT_GEOMETRIC), (W.SIG_PHASE, W.QUANT_GEOMETRIC),
                                          (W.SIG_REMAINING, W.QUANT_EXACT), (W.SIG_UNIFIED, W.QUANT_EXACT)])
@pytest.mark.parametrize("gamma", [1e-7, 0.05, 0.3, 50.0])
def test_pressure_signal_quant_gamma(gpu, oracle_mod, signal, quant, gamma):
    wl = pressure_workload(7, n=150, kv_blocks=56, gamma=gamma, signal=signal, quant=quant, preempt=W.PRE_AUTO,
                           swap_pool_blocks=30, bin_tokens=32)
    g, o = _pair(gpu, oracle_mod, wl)
    g.run(); o.run()
    _assert_same(g, o, f"signal {signal} quant {quant} gamma {gamma}")


def test_step_by_step_under_pressure(gpu, oracle_mod):
    wl = pressure_workload(3, n=200, kv_blocks=64, preempt=W.PRE_AUTO, swap_pool_blocks=20, mean_gap_us=3000)
    g, o = _pair(gpu, oracle_mod, wl)
    for it in range(2500):
        g.step(1)
        info, rows = o.step_replica(0)
        assert g.digest()[0] == o.digest()[0], f"iteration {it}"
        if not info["executed"]:
            break
        st = g.debug_state(0)
        assert st["clock_us"] == info["t_end_us"]
        kv = int(sum(-(-int(c) // 16) for c, f in zip(st["cached"], st["flags"]) if f & 1))
        assert kv == info["kv_resident_after"] <= 64


def test_many_replicas_batch_and_granularity(gpu, oracle_mod):
    """P14: a replica's result does not depend on the batch around it nor on ub_step granularity / iterations per launch."""
    rng = np.random.default_rng(5)
    n, NT = 90, 6
    P = rng.integers(1, 300, (NT, n)); D = rng.integers(1, 200, (NT, n))
    a = np.cumsum(rng.exponential(6000, (NT, n)), axis=1).astype(np.int64)
    R = 24
    rep = W.make_replicas(R, trace_id=np.arange(R) % NT, policy=np.array([0, 1, 2, 3])[np.arange(R) % 4],
                          gamma=10.0 ** rng.uniform(-2, 1, R), guard=np.arange(R) % 2,
                          hysteresis_us=rng.integers(0, 200_000, R))
    sim = dict(kv_blocks=48, queue_cap=64, preempt_mode=W.PRE_AUTO, swap_pool_blocks=16, bin_tokens=64,
               max_batch=12, chunk_tokens=48, token_budget=80)
    wl = W.custom(a, P, D, sim, rep)
    g, o = _pair(gpu, oracle_mod, wl)
    g.run(); o.run()
    _assert_same(g, o, "batch of 24")
    ref = g.digest().copy()
    g2 = gpu.Sim(wl.sim, wl.replicas, wl.traces(), iters_per_launch=7)
    for k in (1, 2, 3, 50, 1000, 100000):
        g2.step(k)
    assert g2.step(1, want_live=True) == 0
    assert np.array_equal(g2.digest(), ref)
    sub = wl.select([23, 5, 11])
    g3 = gpu.Sim(sub.sim, sub.replicas, sub.traces(), iters_per_launch=64)
    g3.run()
    assert np.array_equal(g3.digest(), ref[[23, 5, 11]])


# ------------------------------------------------------------------------------------------ edge cases

def test_edge_cases(gpu, oracle_mod):
    # one request; one token each; identical arrivals (tie-break by id); queue cap smaller than the burst
    cases = [
        (np.array([5]), np.array([1]), np.array([1]), {}),
        (np.zeros(50, np.int64), np.full(50, 3), np.full(50, 2), dict(queue_cap=7, max_batch=3)),
        (np.arange(40) * 10, np.full(40, 17), np.ones(40, int), dict(kv_blocks=4, chunk_tokens=5, token_budget=9)),
        (np.zeros(300, np.int64), np.full(300, 40), np.full(300, 30), dict(kv_blocks=30, queue_cap=300, max_batch=300)),
    ]
    for i, (a, P, D, kw) in enumerate(cases):
        sim = dict(kv_blocks=16, preempt_mode=W.PRE_RECOMPUTE)
        sim.update(kw)
        wl = W.custom(a, P, D, sim, W.make_replicas(1, trace_id=0))
        g, o = _pair(gpu, oracle_mod, wl)
        g.run(); o.run()
        _assert_same(g, o, f"edge case {i}")
    # a replica whose trace is empty is done at once
    wl = W.custom(np.array([[1, 2, 3], [4, 5, 6]]), np.full((2, 3), 4), np.full((2, 3), 2), dict(kv_blocks=8),
                  W.make_replicas(2))
    tr = list(wl.traces()); tr[3] = np.array([0, 3], np.uint32)
    g = gpu.Sim(wl.sim, wl.replicas, tr); o = oracle_mod.OracleSim(wl.sim, wl.replicas, tr)
    assert g.run() is not None
    o.run()
    _assert_same(g, o, "empty trace")


def test_full_queue_2048(gpu, oracle_mod):
    """Maximum queue size: 2048 simultaneously active requests (several sort / scan tiles and a ragged tail)."""
    n = 2300
    rng = np.random.default_rng(11)
    a = np.sort(rng.integers(0, 2000, n)).astype(np.int64)
    P = rng.integers(1, 64, n); D = rng.integers(1, 12, n)
    sim = dict(kv_blocks=600, queue_cap=2048, preempt_mode=W.PRE_AUTO, swap_pool_blocks=100, bin_tokens=16,
               max_batch=256, chunk_tokens=32, token_budget=512)
    rep = W.make_replicas(3, trace_id=0, policy=[W.POLICY_BOOST, W.POLICY_SRPT, W.POLICY_FCFS], gamma=0.5)
    wl = W.custom(a, P, D, sim, rep)
    g, o = _pair(gpu, oracle_mod, wl, ipl=16)
    g.run(); o.run()
    _assert_same(g, o, "queue 2048")
    assert max(s["peak_active"] for s in o.stats()) == 2048


def test_load_errors(gpu):
    from paper_2606_18431_b200 import binding as Bn
    wl = pressure_workload(0, n=10)
    a, p, d, n = wl.traces()

    def load(a, p, d, n):
        h = Bn.ub_create(Bn.make_config(wl.sim))
        try:
            return Bn.lib().ub_load_trace(h, np.ascontiguousarray(a, np.int64).ctypes.data,
                                          np.ascontiguousarray(p, np.int32).ctypes.data,
                                          np.ascontiguousarray(d, np.int32).ctypes.data,
                                          np.ascontiguousarray(n, np.uint32).ctypes.data, 0)
        finally:
            Bn.ub_destroy(h)

    assert load(a, p, d, n) == Bn.UB_OK
    a2 = a.copy(); a2[0, 5] = a2[0, 4] - 1
    assert load(a2, p, d, n) == Bn.UB_EUNSORTED
    p2 = p.copy(); p2[0, 3] = 0
    assert load(a, p2, d, n) == Bn.UB_EINFEASIBLE
    d2 = d.copy(); d2[0, 3] = 10 ** 6
    assert load(a, p, d2, n) == Bn.UB_EINFEASIBLE
    a3 = a.copy(); a3[0, 0] = -1
    assert load(a3, p, d, n) == Bn.UB_EINVAL
    h = Bn.ub_create(Bn.make_config(wl.sim))
    assert Bn.lib().ub_step(h, 1, None) == Bn.UB_ESTATE
    Bn.ub_destroy(h)
    bad = Bn.make_config(dict(wl.sim, queue_cap=4096))
    hh = Bn.C.c_void_p()
    assert Bn.lib().ub_create(Bn.C.byref(bad), Bn.C.byref(hh)) == Bn.UB_EINVAL


# ------------------------------------------------------------------------------------------ configs 2-5, sampled replicas

@pytest.mark.parametrize("cfg_id,kw,picks", [
    (2, dict(n_seeds=4), None),                     # 4 seeds x {FCFS, SRPT, BOOST} = 12 replicas, full run
    (3, dict(n_seeds=3), None),                     # reasoning mix, MMPP-2, swap-vs-recompute
    (4, dict(n_seeds=1, n_gamma=16), [0, 5, 9, 15]),  # shift + pressure, 4 of the 16 gamma points
    (5, dict(n_seeds=2, n_requests=8192), None),    # scale-stress shape, 2 replicas x 8192 requests
    (6, dict(n_seeds=2), None),                     # starvation shape of PAPER.md:545
])
def test_configs_sampled_full_run(gpu, oracle_mod, cfg_id, kw, picks):
    wl = W.by_id(cfg_id, **kw)
    if picks is not None:
        wl = wl.select(picks)
    g, o = _pair(gpu, oracle_mod, wl, ipl=64)
    g.run(); o.run()
    _assert_same(g, o, wl.name)
    _assert_hist_same(g, o, range(wl.R))
    assert all(s["done"] == 1 for s in g.stats())


# ------------------------------------------------------------------------------------------ full sizes, sampled replicas

def _full_size_sampled(gpu, oracle_mod, wl, picks, ipl=1):
    """Run the whole workload on the GPU in bench.py's launch configuration (one iteration per launch), then compare
    the schedule digest, the counters and the integer / fp64 percentiles of the sampled replicas with the oracle,
    which computes those replicas one by one (a replica's schedule does not depend on the batch around it, P14)."""
    import os
    tr = wl.traces(workers=max(1, min(32, os.cpu_count() or 1)))
    g = gpu.Sim(wl.sim, wl.replicas, tr, iters_per_launch=ipl)
    g.run()
    dg = g.digest()
    raw = g.stats_raw()
    sub = wl.select(picks)
    tid = wl.replicas["trace_id"][np.asarray(picks)]
    used = np.unique(tid)
    o = oracle_mod.OracleSim(sub.sim, sub.replicas, tuple(x[used] for x in tr))
    o.run()
    do, so = o.digest(), o.stats()
    for j, r in enumerate(picks):
        assert dg[r] == do[j], f"{wl.name} replica {r}: schedule digest"
        a = gpu._stats_to_dict(raw[r])
        for k in INT_STATS:
            assert a[k] == so[j][k], f"{wl.name} replica {r} stat {k}: gpu {a[k]} oracle {so[j][k]}"
        for k in F64_STATS:
            av, bv = np.atleast_1d(a[k]).astype(float), np.atleast_1d(so[j][k]).astype(float)
            assert np.all(np.abs(av - bv) <= REL_TOL * np.maximum(1e-300, np.abs(bv))), f"{wl.name} replica {r} {k}"
    assert all(raw[r].done for r in range(0, wl.R, 97))
    g.close(); o.close()


@pytest.mark.parametrize("cfg_id,picks", [
    (2, [0, 1, 2, 1535, 1536, 1537, 3069, 3070, 3071]),            # 1024 seeds x {FCFS, SRPT, BOOST}
    (3, [0, 1, 2047, 2048, 3000, 4095]),                            # 4096 replicas, MMPP-2, swap-vs-recompute
    (4, [0, 7, 15, 8191, 8192, 8200, 16368, 16383]),                # 1024 seeds x 16 gamma
])
def test_configs_full_size_sampled(gpu, oracle_mod, cfg_id, picks):
    _full_size_sampled(gpu, oracle_mod, W.by_id(cfg_id), picks)


def test_config5_full_size_sampled(gpu, oracle_mod):
    """BASELINE.json configs[4] at its full size (65536 replicas x 8192 requests; rounds split over two streams)."""
    _full_size_sampled(gpu, oracle_mod, W.config5(n_seeds=65536, n_requests=8192),
                       [0, 1, 4095, 8191, 16384, 32767, 32768, 32769, 40000, 50001, 65534, 65535])


@pytest.mark.parametrize("ipl", [1, 16])
def test_split_rounds_and_resident_mode(gpu, oracle_mod, ipl):
    """8192 replicas (rounds split over two streams, ticket-based replica distribution) with 1 and with 16 iterations
    per launch (the bench's resident-state mode): sampled replicas, both halves and their borders, against the oracle."""
    _full_size_sampled(gpu, oracle_mod, W.config5(n_seeds=8192, n_requests=640),
                       [0, 1, 2047, 4094, 4095, 4096, 4097, 6000, 8190, 8191], ipl=ipl)


@pytest.mark.parametrize("ipl", [1, 16])
def test_mixed_policies_in_parts(gpu, oracle_mod, ipl):
    """1400 seeds x {FCFS, SRPT, BOOST} = 4200 replicas: the main group runs as two parts and the SRPT replicas as the
    drift group, each from its own list from the first round on (then compacted to the unfinished ones in the tail of
    the run); sampled replicas of every policy at the borders of the parts against the oracle."""
    base = W.config2(n_seeds=1400)
    a, P, D, n = base.traces(workers=8)
    keep = 300                                                        # a short job: the first 300 requests of every trace
    wl = W.custom(a[:, :keep], P[:, :keep], D[:, :keep], dict(base.sim, max_requests=keep), base.replicas)
    _full_size_sampled(gpu, oracle_mod, wl, [0, 1, 2, 2098, 2099, 2100, 2101, 2102, 3000, 3001, 4197, 4198, 4199], ipl=ipl)


@pytest.mark.parametrize("ipl", [1, 16])
def test_specialised_and_generic_instances_agree(gpu, oracle_mod, ipl):
    """A job whose replicas are all BOOST with MemGuard runs k_stream's specialised instance (bench.py's kernel); one
    FCFS replica added to the same job forces the generic instances.  Both must give the BOOST replicas the same
    schedule, per-request times and histograms -- and the oracle's, on sampled replicas (6000 replicas: two parts)."""
    base = W.config5(n_seeds=6000, n_requests=400)
    a, P, D, n = base.traces(workers=8)
    R = base.R
    spec = gpu.Sim(base.sim, base.replicas, (a, P, D, n), iters_per_launch=ipl)
    rep2 = {k: np.concatenate([v, v[:1]]) for k, v in base.replicas.items()}
    rep2["policy"][-1] = W.POLICY_FCFS; rep2["guard"][-1] = 0
    sim2 = dict(base.sim, n_replicas=R + 1)
    gen = gpu.Sim(sim2, rep2, (a, P, D, n), iters_per_launch=ipl)
    spec.run(); gen.run()
    assert np.array_equal(spec.digest(), gen.digest()[:R])
    s1, s2 = spec.per_request(), gen.per_request()
    for x, y in zip(s1, s2):
        assert np.array_equal(x, y[:R])
    assert np.array_equal(spec.tbt_hist(5), gen.tbt_hist(5)) and np.array_equal(spec.tbt_hist(R - 1), gen.tbt_hist(R - 1))
    picks = [0, 1, 2999, 3000, 3001, 5999]
    sub = base.select(picks)
    o = oracle_mod.OracleSim(sub.sim, sub.replicas, tuple(x[np.unique(base.replicas["trace_id"][picks])] for x in (a, P, D, n)))
    o.run()
    assert np.array_equal(spec.digest()[picks], o.digest())
    spec.close(); gen.close(); o.close()


@pytest.mark.parametrize("own_stream", [False, True], ids=["default-stream", "own-stream"])
def test_run_replays_a_graph_and_survives_a_rewind(gpu, oracle_mod, own_stream):
    """ub_run replays a captured CUDA graph of 64 rounds (from a stream of the library's when the caller's is the default
    stream).  The graph holds device pointers by value: ub_set_replicas (which re-allocates the boost tables) must drop
    it.  Same digests as the oracle before and after the rewind, and after changing the replica table."""
    import torch
    wl = W.config2(n_seeds=40)
    tr = wl.traces(workers=4)
    st = torch.cuda.Stream() if own_stream else torch.cuda.current_stream()
    g = gpu.Sim(wl.sim, wl.replicas, tr, stream=st.cuda_stream)
    o = oracle_mod.OracleSim(wl.sim, wl.replicas, tr)
    o.run()
    issued = g.run()
    assert issued >= 1024                                           # (several graph replays)
    want = o.digest()
    assert np.array_equal(g.digest(), want)
    gpu._chk(gpu.lib().ub_set_replicas(g._h, gpu.make_replicas(wl.replicas, wl.R)))      # rewind
    g.run()
    assert np.array_equal(g.digest(), want)
    rep2 = {k: v.copy() for k, v in wl.replicas.items()}
    rep2["gamma"][:] = 2.0                                          # other boost tables, same shapes
    gpu._chk(gpu.lib().ub_set_replicas(g._h, gpu.make_replicas(rep2, wl.R)))
    g.run()
    o2 = oracle_mod.OracleSim(wl.sim, rep2, tr)
    o2.run()
    assert np.array_equal(g.digest(), o2.digest())
    assert not np.array_equal(o2.digest(), want)
    g.close(); o.close(); o2.close()


# ------------------------------------------------------------------------------------------ streaming kernel, randomised

@pytest.mark.parametrize("seed", range(8))
def test_stream_path_randomised(gpu, oracle_mod, seed):
    """The streaming kernel's own territory (FCFS / BOOST, paper's signal and quantiser): random batch cap, token
    budget, chunk, KV size, bin size, guard on / off, hysteresis on / off, bursty arrivals that grow windows to a
    few hundred requests (several chunks, parked-request merges, walk stops, evictions), 1 or 3 iterations per launch."""
    rng = np.random.default_rng([77, seed])
    n, NT = 700, 3
    P = rng.integers(1, 400, (NT, n)); D = rng.integers(1, 120, (NT, n))
    gaps = rng.exponential(2500, (NT, n)) * rng.choice([0.05, 1.0, 3.0], (NT, n), p=[0.3, 0.5, 0.2])
    a = np.cumsum(gaps, axis=1).astype(np.int64)
    R = 12
    rep = W.make_replicas(R, trace_id=np.arange(R) % NT, policy=rng.choice([W.POLICY_FCFS, W.POLICY_BOOST], R),
                          guard=rng.integers(0, 2, R), hysteresis_us=rng.choice([0, 100_000], R),
                          gamma=rng.choice([0.05, 0.3, 2.0, 50.0], R))
    blk = 16
    kvb = int(rng.integers(60, 400))
    D = np.minimum(D, np.maximum(1, kvb * blk - P))
    sim = dict(kv_blocks=kvb, queue_cap=int(rng.choice([400, 700])), max_batch=int(rng.choice([8, 48, 256])),
               chunk_tokens=int(rng.choice([16, 64, 512])), token_budget=int(rng.choice([64, 256, 1024])),
               bin_tokens=int(rng.choice([16, 64, 256])), preempt_mode=int(rng.integers(0, 3)),
               swap_pool_blocks=int(rng.integers(0, 200)))
    wl = W.custom(a, P, D, sim, rep)
    g, o = _pair(gpu, oracle_mod, wl, ipl=int(rng.choice([1, 3])))
    g.run(); o.run()
    _assert_same(g, o, f"randomised stream case {seed}: {sim}")
    assert max(s["peak_active"] for s in o.stats()) > 64


@pytest.mark.parametrize("seed", range(8))
def test_drift_path_randomised(gpu, oracle_mod, seed):
    """The drift instance's territory (SRPT, LAS: keys move with every token; SJF, SPF beside them), with and without
    MemGuard: windows of several hundred requests, so that its decode-run and waiting-tail phases (order checks against
    the keys written so far), the general path and evictions all occur; 1 or 3 iterations per launch."""
    rng = np.random.default_rng([78, seed])
    n, NT = 700, 3
    P = rng.integers(1, 400, (NT, n)); D = rng.integers(1, 160, (NT, n))
    gaps = rng.exponential(2500, (NT, n)) * rng.choice([0.05, 1.0, 3.0], (NT, n), p=[0.3, 0.5, 0.2])
    a = np.cumsum(gaps, axis=1).astype(np.int64)
    R = 12
    rep = W.make_replicas(R, trace_id=np.arange(R) % NT,
                          policy=rng.choice([W.POLICY_SRPT, W.POLICY_LAS, W.POLICY_SJF, W.POLICY_SPF], R, p=[0.4, 0.4, 0.1, 0.1]),
                          guard=rng.integers(0, 2, R), hysteresis_us=0)
    blk = 16
    kvb = int(rng.integers(60, 400))
    D = np.minimum(D, np.maximum(1, kvb * blk - P))
    sim = dict(kv_blocks=kvb, queue_cap=int(rng.choice([400, 700])), max_batch=int(rng.choice([8, 48, 256])),
               chunk_tokens=int(rng.choice([16, 64, 512])), token_budget=int(rng.choice([64, 256, 1024])),
               bin_tokens=int(rng.choice([16, 64, 256])), preempt_mode=int(rng.integers(0, 3)),
               swap_pool_blocks=int(rng.integers(0, 200)))
    wl = W.custom(a, P, D, sim, rep)
    g, o = _pair(gpu, oracle_mod, wl, ipl=int(rng.choice([1, 3])))
    g.run(); o.run()
    _assert_same(g, o, f"randomised drift case {seed}: {sim}")
    assert max(s["peak_active"] for s in o.stats()) > 64


# ------------------------------------------------------------------------------------------ kernel-level parity: a1 score

@pytest.mark.parametrize("policy", [W.POLICY_FCFS, W.POLICY_SRPT, W.POLICY_BOOST, W.POLICY_LAS, W.POLICY_SJF,
                                    W.POLICY_SPF, W.POLICY_DISTBOOST, W.POLICY_SARATHI])
def test_score_kernel_keys_match_oracle(gpu, oracle_mod, policy):
    """SURVEY.md Sec. 4 tier T1: before every iteration the (class, key) the device assigns to each request of the
    window (ub_debug_keys, the team kernels' own scoring function) equals what the oracle scores in that iteration."""
    wl = pressure_workload(6, n=140, kv_blocks=48, policy=policy, preempt=W.PRE_AUTO, swap_pool_blocks=20,
                           guard=1 if policy == W.POLICY_BOOST else 0, gamma=0.3, bin_tokens=32)
    g, o = _pair(gpu, oracle_mod, wl)
    checked = 0
    for it in range(1500):
        ids, kl, ky = g.debug_keys(0)
        info, rows = o.step_replica(0)
        g.step(1)
        if not info["executed"]:
            break
        want = {r["id"]: (r["klass"], r["key"]) for r in rows}
        for i, c, k in zip(ids, kl, ky):
            assert (int(c), int(k)) == want[int(i)], f"iteration {it} request {i}"
        checked += len(ids)
        assert g.digest()[0] == o.digest()[0]
    assert checked > 5000
