"""GPU parity of gamma-Ada (rule M13; Eq. 9, UPDATEGAMMA PAPER.md:588-601): the CUDA path through
the C-ABI against the oracle on the same seeded inputs -- grid, per-replica (gamma_u, level, number of updates),
schedule digest, per-request results and all statistics, bit-exact."""
import numpy as np
import pytest

from paper_2606_18431_b200 import workloads as W
from tests.helpers import pressure_workload
from tests.test_gpu_parity import _assert_same, _pair, gpu  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu

ADA = dict(window=64, min_samples=8, beta_shift=2, levels=17, gamma_min=0.01, gamma_max=100.0, eps_us=1000)


def _ada_pair(gpu, oracle_mod, wl, ada, adaptive):
    g, o = _pair(gpu, oracle_mod, wl)
    g.set_gamma_ada(ada, adaptive); o.set_gamma_ada(ada, adaptive)
    assert np.array_equal(g.gamma_grid(), o.gamma_grid()), "gamma grid"
    return g, o


def _assert_gamma_same(g, o, R, where):
    for r in range(R):
        assert g.gamma_state(r) == o.gamma_state(r), f"{where}: replica {r} (gamma_u, level, n_updates)"


@pytest.mark.parametrize("seed", range(4))
@pytest.mark.parametrize("beta_shift", [0, 2, 4])
def test_pressure_adaptive(gpu, oracle_mod, seed, beta_shift):
    wl = pressure_workload(seed, n=180, kv_blocks=64, gamma=0.3, preempt=W.PRE_AUTO, swap_pool_blocks=24,
                           mean_gap_us=4000)
    ada = dict(ADA, beta_shift=beta_shift, window=max(64, int(wl.sim["max_batch"])))
    g, o = _ada_pair(gpu, oracle_mod, wl, ada, np.ones(wl.R, np.uint8))
    g.run(); o.run()
    _assert_gamma_same(g, o, wl.R, f"seed {seed}")
    _assert_same(g, o, f"adaptive pressure seed {seed} beta_shift {beta_shift}")
    assert o.gamma_state(0)[2] > 10, "the case must exercise updates"


def test_adaptive_step_by_step(gpu, oracle_mod):
    wl = pressure_workload(5, n=150, kv_blocks=56, gamma=2.0, preempt=W.PRE_AUTO, swap_pool_blocks=20, mean_gap_us=3000)
    ada = dict(ADA, window=max(64, int(wl.sim["max_batch"])))
    g, o = _ada_pair(gpu, oracle_mod, wl, ada, np.ones(wl.R, np.uint8))
    levels = set()
    for it in range(4000):
        g.step(1)
        info, _ = o.step_replica(0)
        assert g.digest()[0] == o.digest()[0], f"iteration {it}"
        if not info["executed"]:
            break
        assert g.gamma_state(0) == o.gamma_state(0), f"iteration {it}"
        levels.add(o.gamma_state(0)[1])
    assert len(levels) > 1, "the case must exercise level changes"


def test_mixed_adaptive_and_static_replicas_config4(gpu, oracle_mod):
    """Distribution shift + memory pressure (config 4 shape): gamma points of one seed, every other one adaptive."""
    wl = W.config4(n_seeds=1, n_gamma=16).select([0, 3, 6, 9, 12, 15])
    adaptive = np.array([1, 0, 1, 0, 1, 1], np.uint8)
    ada = dict(window=256, min_samples=32, beta_shift=3, levels=33, gamma_min=0.01, gamma_max=100.0, eps_us=1000)
    g, o = _ada_pair(gpu, oracle_mod, wl, ada, adaptive)
    g.run(); o.run()
    _assert_gamma_same(g, o, wl.R, "config4")
    _assert_same(g, o, "config4 adaptive")
    assert g.gamma_state(1)[1] == -1 and o.gamma_state(0)[2] > 100


def test_gamma_ada_argument_errors(gpu, oracle_mod):
    wl = pressure_workload(1, n=40, policy=W.POLICY_FCFS, guard=0)
    g, _ = _pair(gpu, oracle_mod, wl)
    with pytest.raises(gpu.UbError):
        g.set_gamma_ada(dict(ADA, window=max(64, int(wl.sim["max_batch"]))), np.ones(wl.R, np.uint8))   # not BOOST
    wl = pressure_workload(1, n=40)
    g, _ = _pair(gpu, oracle_mod, wl)
    with pytest.raises(gpu.UbError):
        g.set_gamma_ada(dict(ADA, window=4), np.ones(wl.R, np.uint8))                                  # window < max_batch
