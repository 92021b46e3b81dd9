"""Rule M18: clusters of replicas behind a join-the-shortest-queue router (Table 9; SURVEY.md Sec. 8(f)
row 4).  CPU pins of the oracle and GPU parity.

* one replica per cluster: the router has no choice, JSQ is the plain trace;
* a burst at one instant on idle replicas: equal queue lengths, so the lowest-number tie-break deals the requests
  round robin;
* the defining property, checked after the fact on any size: for every arrival, the chosen replica had the fewest
  requests in the system at that instant (counted here from the final completion times), lowest number on a tie;
* given the assignment the replicas are independent: each one's schedule is the plain oracle on the requests it got;
* brute force on tiny cases: of all K^n assignments exactly one has that property, and it is the router's.
"""
import itertools

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_18431_b200 import workloads as W


def _cluster_sim(C, K, cap, **sim_kw):
    R = C * K
    sim = dict(W.SIM_DEFAULTS, n_replicas=R, n_traces=R, max_requests=cap, queue_cap=min(cap, 2048), kv_blocks=64,
               max_batch=16, chunk_tokens=64, token_budget=96, bin_tokens=32, preempt_mode=W.PRE_AUTO, swap_pool_blocks=24)
    sim.update(sim_kw)
    return sim


def _empty(sim):
    NT, N = sim["n_traces"], sim["max_requests"]
    return (np.zeros((NT, N), np.int64), np.ones((NT, N), np.int32), np.ones((NT, N), np.int32), np.zeros(NT, np.uint32))


def _stream(seed, C, n, gap_us=2500, pmax=300, dmax=150):
    rng = np.random.default_rng([18, seed])
    a = np.cumsum(rng.exponential(gap_us, (C, n)), axis=1).astype(np.int64)
    P = rng.integers(1, pmax + 1, (C, n)).astype(np.int32)
    D = rng.integers(1, dmax + 1, (C, n)).astype(np.int32)
    return a, P, D, np.full(C, n, np.uint32)


def _subtraces(a, P, D, assign, c, K, cap):
    """The requests each replica of cluster c got, in arrival order, as plain trace arrays."""
    out = []
    for k in range(K):
        sel = np.nonzero(assign[c] == k)[0]
        ta = np.zeros(cap, np.int64); tp = np.ones(cap, np.int32); td = np.ones(cap, np.int32)
        ta[:len(sel)], tp[:len(sel)], td[:len(sel)] = a[c, sel], P[c, sel], D[c, sel]
        out.append((ta, tp, td, len(sel), sel))
    return out


def _jsq_property_holds(a_c, assign_c, t_last_of, K):
    """For every arrival j: chosen == the lowest-numbered replica with the fewest requests assigned earlier and not
    completed by a_j."""
    for j in range(len(a_c)):
        counts = [sum(1 for i in range(j) if assign_c[i] == k and t_last_of[i] > a_c[j]) for k in range(K)]
        if assign_c[j] != int(np.argmin(counts)):
            return False
    return True


def _run_jsq(sim, rep, K, stream):
    o = O.OracleSim(sim, rep, _empty(sim))
    assign = o.jsq_run(K, *stream)
    return o, assign


@pytest.mark.parametrize("policy", [W.POLICY_BOOST, W.POLICY_SRPT])
def test_one_replica_per_cluster_is_the_plain_trace(policy):
    C, n = 3, 90
    sim = _cluster_sim(C, 1, n)
    rep = W.make_replicas(C, policy=policy, guard=1 if policy == W.POLICY_BOOST else 0)
    stream = _stream(0, C, n)
    o, assign = _run_jsq(sim, rep, 1, stream)
    assert not assign.any()
    plain = O.OracleSim(sim, rep, stream); plain.run()
    assert np.array_equal(o.digest(), plain.digest())
    for x, y in zip(o.per_request(), plain.per_request()):
        assert np.array_equal(x, y)


def test_simultaneous_burst_is_dealt_round_robin():
    C, K, n = 2, 4, 22
    sim = _cluster_sim(C, K, n)
    a, P, D, na = _stream(1, C, n)
    a[:] = 7000                                                   # everything arrives at the same instant
    o, assign = _run_jsq(sim, W.make_replicas(C * K), K, (a, P, D, na))
    for c in range(C):
        assert assign[c].tolist() == [j % K for j in range(n)]


@pytest.mark.parametrize("seed,K,policy", [(2, 2, W.POLICY_BOOST), (3, 4, W.POLICY_FCFS), (4, 3, W.POLICY_SRPT)])
def test_chosen_replica_had_the_fewest_requests_in_the_system(seed, K, policy):
    C, n = 2, 160
    sim = _cluster_sim(C, K, n)
    rep = W.make_replicas(C * K, policy=policy, guard=1 if policy == W.POLICY_BOOST else 0)
    a, P, D, na = _stream(seed, C, n, gap_us=1800)
    o, assign = _run_jsq(sim, rep, K, (a, P, D, na))
    tf, tl, ne, _ = o.per_request()
    dg = o.digest()
    used = set()
    for c in range(C):
        subs = _subtraces(a, P, D, assign, c, K, n)
        t_last_of = np.zeros(n, np.int64)
        for k, (ta, tp, td, m, sel) in enumerate(subs):
            t_last_of[sel] = tl[c * K + k, :m]
            used.add(m)
            # given the assignment the replica is independent of its neighbours: the plain oracle on what it got
            s1 = dict(sim, n_replicas=1, n_traces=1)
            r1 = {f: v[c * K + k:c * K + k + 1].copy() for f, v in rep.items()}; r1["trace_id"][:] = 0
            p1 = O.OracleSim(s1, r1, (ta[None], tp[None], td[None], np.array([m], np.uint32))); p1.run()
            assert p1.digest()[0] == dg[c * K + k]
            assert np.array_equal(p1.per_request()[1][0, :m], tl[c * K + k, :m])
        assert _jsq_property_holds(a[c], assign[c], t_last_of, K)
        assert len(set(assign[c].tolist())) == K                  # every replica is used
    assert ne.sum() > 0                                           # (the case has memory pressure)


@pytest.mark.parametrize("seed", range(6))
def test_bruteforce_only_the_routers_assignment_has_the_property(seed):
    K, n = 2, 6
    sim = _cluster_sim(1, K, n, kv_blocks=24)
    rep = W.make_replicas(K, policy=W.POLICY_SRPT, guard=0, hysteresis_us=0)
    a, P, D, na = _stream(100 + seed, 1, n, gap_us=1500, pmax=120, dmax=40)
    o, assign = _run_jsq(sim, rep, K, (a, P, D, na))
    good = []
    for cand in itertools.product(range(K), repeat=n):
        cand = np.array([cand], np.int32)
        t_last_of = np.zeros(n, np.int64)
        for k, (ta, tp, td, m, sel) in enumerate(_subtraces(a, P, D, cand, 0, K, n)):
            s1 = dict(sim, n_replicas=1, n_traces=1)
            r1 = {f: v[k:k + 1].copy() for f, v in rep.items()}; r1["trace_id"][:] = 0
            p1 = O.OracleSim(s1, r1, (ta[None], tp[None], td[None], np.array([m], np.uint32))); p1.run()
            t_last_of[sel] = p1.per_request()[1][0, :m]
        if _jsq_property_holds(a[0], cand[0], t_last_of, K):
            good.append(cand[0].tolist())
    assert good == [assign[0].tolist()]


# ------------------------------------------------------------------------------------------ GPU parity

@pytest.mark.gpu
@pytest.mark.parametrize("policy,guard,K,C", [(W.POLICY_BOOST, 1, 4, 6), (W.POLICY_FCFS, 0, 2, 5), (W.POLICY_SRPT, 0, 3, 4),
                                              (W.POLICY_DISTBOOST, 0, 4, 3), (W.POLICY_BOOST, 1, 32, 2)])
def test_gpu_jsq_router_parity(policy, guard, K, C):
    """ub_jsq_run (time-fenced runs of the step kernels + one warp per cluster for the min-reduction) against the oracle:
    the same assignment, the same schedules."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_2606_18431_b200 import binding as B
    n = 60 * K
    sim = _cluster_sim(C, K, n)
    rep = W.make_replicas(C * K, policy=policy, guard=guard, hysteresis_us=100_000 if policy == W.POLICY_BOOST else 0)
    stream = _stream(7, C, n, gap_us=max(200, 5000 // K))
    stream[3][-1] = n // 2                                        # (a cluster with a shorter stream)
    o = O.OracleSim(sim, rep, _empty(sim)); oa = o.jsq_run(K, *stream)
    g = B.Sim(sim, rep, _empty(sim)); ga = g.jsq_run(K, *stream)
    assert np.array_equal(ga, oa)
    assert np.array_equal(g.digest(), o.digest())
    for x, y in zip(g.per_request(), o.per_request()):
        assert np.array_equal(x, y)
    gs, os_ = g.stats(), o.stats()
    for x, y in zip(gs, os_):
        for kk in ("iterations", "request_steps", "n_completed", "t_end_us", "done", "ttlt_us", "evict_recompute", "evict_swap"):
            assert x[kk] == y[kk], kk
    assert sum(s["n_completed"] for s in os_) == int(stream[3].sum())
    assert sum(s["evict_recompute"] + s["evict_swap"] for s in os_) > 0 or K == 32
    g.close(); o.close()


@pytest.mark.gpu
def test_gpu_jsq_router_rejects_wrong_states():
    """ub_jsq_run wants clusters that tile the replicas, empty traces, no iteration run; a replica row that is too
    short for what the router sends it is an error, not an overrun."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_2606_18431_b200 import binding as B
    C, K, n = 2, 3, 40
    stream = _stream(9, C, n)
    sim = _cluster_sim(C, K, n)
    g = B.Sim(sim, W.make_replicas(C * K), _empty(sim))
    with pytest.raises(B.UbError) as e:                      # 4 does not divide the 6 replicas into 2 clusters
        g.jsq_run(4, *stream)
    assert e.value.code == B.UB_EINVAL
    bad = (stream[0][:, ::-1].copy(), stream[1], stream[2], stream[3])
    with pytest.raises(B.UbError) as e:                      # arrivals must be sorted, as for ub_load_trace
        g.jsq_run(K, *bad)
    assert e.value.code == B.UB_EUNSORTED
    g.jsq_run(K, *stream)                                    # fine
    with pytest.raises(B.UbError) as e:                      # ... but only once: the traces are no longer empty
        g.jsq_run(K, *stream)
    assert e.value.code == B.UB_ESTATE
    g.close()
    small = _cluster_sim(C, K, 4)                            # rows of 4 requests for 40 arrivals over 3 replicas
    g = B.Sim(small, W.make_replicas(C * K), _empty(small))
    with pytest.raises(B.UbError) as e:
        g.jsq_run(K, *stream)
    assert e.value.code == B.UB_EINVAL
    g.close()
