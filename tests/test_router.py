"""Exogenous global dispatch (the replica-independent part): round-robin
and random routers split one global arrival stream over the replicas; each replica then schedules on its own."""
import numpy as np
import pytest

from paper_2606_18431_b200 import workloads as W


@pytest.mark.parametrize("dispatch", ["round_robin", "random"])
def test_router_partitions_the_global_stream(dispatch):
    wl, tr, (arr, P, D, dest) = W.routed_cluster(n_replicas=6, n_requests_total=1000, dispatch=dispatch, seed=3)
    a, p, d, n = tr
    assert n.sum() == 1000 and a.shape[0] == 6
    got = sorted((int(a[r, i]), int(p[r, i]), int(d[r, i])) for r in range(6) for i in range(n[r]))
    assert got == sorted(zip(arr.tolist(), P.tolist(), D.tolist()))        # nothing lost, nothing invented
    for r in range(6):
        assert np.all(np.diff(a[r, :n[r]]) >= 0)                          # arrival order kept inside a replica
    if dispatch == "round_robin":
        assert np.array_equal(dest, np.arange(1000) % 6) and n.max() - n.min() <= 1
    else:
        assert n.min() > 100 and n.max() - n.min() > 1                    # uniform but not balanced


@pytest.mark.gpu
@pytest.mark.parametrize("dispatch", ["round_robin", "random"])
def test_routed_cluster_gpu_parity(oracle_mod, dispatch):
    from paper_2606_18431_b200 import binding
    from tests.test_gpu_parity import _assert_same
    wl, tr, _ = W.routed_cluster(n_replicas=8, n_requests_total=4000, dispatch=dispatch, seed=1, kv_blocks=2048)
    g = binding.Sim(wl.sim, wl.replicas, tr, iters_per_launch=4)
    o = oracle_mod.OracleSim(wl.sim, wl.replicas, tr)
    g.run(); o.run()
    _assert_same(g, o, f"routed cluster {dispatch}")
    assert sum(s["n_completed"] for s in g.stats()) == 4000
