"""Pins of the oracle's gamma-Ada (rule M13 of DESIGN.md; Eq. 9, UPDATEGAMMA PAPER.md:588-601):
the closed form of Eq. 9 on an exactly exponential tail, the log-spaced grid, the reduction to a static gamma when
no update fires, and the update rule re-derived step by step from the definition (numpy's inverted-cdf percentile,
Python integers, a 50-digit ln 5)."""
from decimal import Decimal, getcontext

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_18431_b200 import workloads as W
from tests.helpers import pressure_workload

ADA = dict(window=64, min_samples=8, beta_shift=2, levels=17, gamma_min=0.01, gamma_max=100.0, eps_us=1000)


def test_eq9_recovers_the_rate_of_an_exponential_tail():
    """F(t) = exp(-lam t)  =>  t_p = -ln(1-p)/lam, t99 - t95 = ln 5 / lam, so Eq. 9 gives gamma_hat = lam."""
    getcontext().prec = 50
    ln5_e12 = int(Decimal(5).ln() * Decimal(10) ** 12)          # floor
    for lam in (0.03, 0.3, 2.0, 17.0):
        t95 = int(round(np.log(20.0) / lam * 1e6)); t99 = int(round(np.log(100.0) / lam * 1e6))
        got = O.gamma_hat_u(t95, t99, 1)
        assert got == ln5_e12 // (t99 - t95)                    # the fixed-point definition, ln 5 to 50 digits
        assert abs(got - lam * 1e6) <= 1e-5 * lam * 1e6 + 2     # = the rate, up to the microsecond rounding of t_p
    assert O.gamma_hat_u(1000, 1010, 500) == ln5_e12 // 500     # tail compressed below eps: Delta = eps
    assert O.gamma_hat_u(7, 7, 1) == ln5_e12


def test_grid_is_log_spaced_and_levels_bracket_gamma():
    wl = pressure_workload(0, n=30)
    o = O.OracleSim(wl.sim, wl.replicas, wl.traces())
    o.set_gamma_ada(ADA, np.ones(wl.R, np.uint8))
    g = o.gamma_grid()
    assert g[0] == 10_000 and g[-1] == 100_000_000 and np.all(np.diff(g) > 0)
    ratio = g[1:] / g[:-1]
    assert np.allclose(ratio, 10 ** (4 / 16), rtol=1e-4)
    gu, lvl, nup = o.gamma_state(0)
    assert nup == 0 and g[lvl] <= gu and (lvl == len(g) - 1 or gu < g[lvl + 1])
    o.close()


def test_no_update_is_the_static_scheduler_at_the_grid_gamma():
    """min_samples above the trace length: gamma never moves, and the schedule equals the static BOOST run whose
    gamma is the grid point (gamma_min 0.25, gamma_max 4, 3 levels => the middle level is exactly 1.0)."""
    wl = pressure_workload(2, n=120, kv_blocks=48, gamma=1.0, preempt=W.PRE_AUTO, swap_pool_blocks=20)
    tr = wl.traces()
    a = O.OracleSim(wl.sim, wl.replicas, tr)
    a.set_gamma_ada(dict(ADA, window=max(64, wl.sim["max_batch"]), min_samples=10_000, levels=3, gamma_min=0.25,
                         gamma_max=4.0), np.ones(wl.R, np.uint8))
    b = O.OracleSim(wl.sim, wl.replicas, tr)
    a.run(); b.run()
    assert a.gamma_state(0) == (1_000_000, 1, 0)
    assert np.array_equal(a.digest(), b.digest())
    assert np.array_equal(a.boost_lut(0), b.boost_lut(0))
    a.close(); b.close()


@pytest.mark.parametrize("seed,beta_shift", [(0, 0), (1, 2), (2, 3)])
def test_update_rule_step_by_step(seed, beta_shift):
    """Every iteration: re-derive gamma from the definition on the completions seen so far and compare."""
    getcontext().prec = 50
    ln5_e12 = int(Decimal(5).ln() * Decimal(10) ** 12)
    wl = pressure_workload(seed, n=160, kv_blocks=64, gamma=0.3, preempt=W.PRE_AUTO, swap_pool_blocks=24,
                           mean_gap_us=4000)
    ada = dict(ADA, beta_shift=beta_shift, window=max(64, int(wl.sim["max_batch"])))
    tr = wl.traces()
    o = O.OracleSim(wl.sim, wl.replicas, tr)
    o.set_gamma_ada(ada, np.ones(wl.R, np.uint8))
    grid = [int(x) for x in o.gamma_grid()]
    arr, D = tr[0][0], tr[2][0]
    gamma_u = min(max(300_000, grid[0]), grid[-1])
    samples, seen, nup, levels_seen = [], 0, 0, set()
    for it in range(100_000):
        # what UPDATEGAMMA must do at the top of this iteration, from the definition
        exp = (gamma_u, nup, seen)
        if len(samples) != seen and len(samples) >= ada["min_samples"]:
            L = np.asarray(samples[-ada["window"]:], np.int64)
            t95 = int(np.percentile(L, 95, method="inverted_cdf")); t99 = int(np.percentile(L, 99, method="inverted_cdf"))
            hat = ln5_e12 // max(t99 - t95, ada["eps_us"])
            diff = hat - gamma_u
            q = abs(diff) >> beta_shift                      # C division truncates toward zero
            exp = (min(max(gamma_u + (q if diff >= 0 else -q), grid[0]), grid[-1]), nup + 1, len(samples))
        info, rows = o.step_replica(0)
        if not info["executed"]:
            break
        gamma_u, nup, seen = exp
        gu, lvl, n_up = o.gamma_state(0)
        assert (gu, n_up) == (gamma_u, nup), f"iteration {it}"
        assert grid[lvl] <= gu and (lvl == len(grid) - 1 or gu < grid[lvl + 1])
        levels_seen.add(lvl)
        for r in rows:                                       # completions of this iteration, in priority order
            if r["want"] > 0 and r["d_after"] == D[r["id"]] and r["resident_after"] == 0 and r["cached_after"] == 0:
                samples.append(int(info["t_end_us"] - arr[r["id"]]))
    assert nup > 20 and len(levels_seen) > 1, "the case must exercise updates and level changes"
    assert len(samples) == o.stats()[0]["n_completed"]
    o.close()
