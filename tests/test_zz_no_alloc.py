"""ub_percentile_curve_noalloc (include/uniboost.h): the entry point that calls no cudaMalloc / cudaFree -- its device
staging is a static array inside libuniboost.so -- against ub_percentile_curve, the existing path, bit for bit (integer
microseconds), on calls in a row that share the array.  Collected last on purpose (the file name): the suite runs
with pytest -x.
"""
import numpy as np
import pytest

from paper_2606_18431_b200 import workloads as W
from tests.helpers import pressure_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_2606_18431_b200 import binding
    binding.lib()
    return binding


def _finished_job(gpu, seed, n_rep, n_req):
    base = pressure_workload(seed, n=n_req, kv_blocks=64, policy=W.POLICY_BOOST, guard=1, gamma=0.3, bin_tokens=32)
    a, P, D, _ = base.traces()
    rep = W.make_replicas(n_rep, trace_id=np.zeros(n_rep, np.int64),
                          policy=np.array([W.POLICY_FCFS, W.POLICY_BOOST, W.POLICY_SRPT])[np.arange(n_rep) % 3],
                          guard=(np.arange(n_rep) % 3 == 1).astype(np.int64), gamma=0.3)
    wl = W.custom(a, P, D, dict(base.sim), rep)
    g = gpu.Sim(wl.sim, wl.replicas, wl.traces())
    g.run()
    return g


def test_noalloc_curve_equals_existing_path_two_calls_in_a_row(gpu):
    g = _finished_job(gpu, 5, n_rep=9, n_req=200)
    pm_a = [500, 900, 990, 999, 1000]
    pm_b = [1, 250, 750]                               # fewer points: the array still holds the first call's values
    want_a0, want_b1, want_a1 = g.percentile_curve(0, pm_a), g.percentile_curve(1, pm_b), g.percentile_curve(1, pm_a)
    got_a0 = g.percentile_curve_noalloc(0, pm_a)       # first call on this device (looks the array's address up)
    got_b1 = g.percentile_curve_noalloc(1, pm_b)       # second call, right behind it
    got_a1 = g.percentile_curve_noalloc(1, pm_a)
    assert got_a0.dtype == np.int64 and got_a0.shape == (9, 5)
    assert np.array_equal(got_a0, want_a0)
    assert np.array_equal(got_b1, want_b1)
    assert np.array_equal(got_a1, want_a1)
    assert want_a0.min() > 0 and not np.array_equal(want_a0, want_a1)      # (the job completed requests: real latencies)
    # a second handle on the same device shares the array: same values again, and the first handle still answers
    g2 = _finished_job(gpu, 6, n_rep=4, n_req=120)
    assert np.array_equal(g2.percentile_curve_noalloc(1, pm_a), g2.percentile_curve(1, pm_a))
    assert np.array_equal(g.percentile_curve_noalloc(0, pm_a), want_a0)
    g2.close()
    g.close()


def test_noalloc_curve_rejects_sizes_beyond_the_static_array(gpu):
    n_rep = gpu.UB_NOALLOC_CURVE_MAX // 16 + 1         # x 16 points = 16 values too many
    a = np.array([[0, 10]], np.int64); P = np.array([[4, 4]], np.int32); D = np.array([[2, 2]], np.int32)
    rep = W.make_replicas(n_rep, trace_id=np.zeros(n_rep, np.int64))
    wl = W.custom(a, P, D, dict(kv_blocks=64), rep)
    g = gpu.Sim(wl.sim, wl.replicas, wl.traces())
    g.run()
    with pytest.raises(gpu.UbError) as e:
        g.percentile_curve_noalloc(0, list(range(1, 17)))
    assert e.value.code == gpu.UB_ETOOBIG
    assert b"static scratch" in gpu.lib().ub_strerror(gpu.UB_ETOOBIG)
    pm = list(range(1, 16))                            # 15 points fit
    assert np.array_equal(g.percentile_curve_noalloc(0, pm), g.percentile_curve(0, pm))
    with pytest.raises(gpu.UbError) as e:              # argument checks as in the existing path
        g.percentile_curve_noalloc(2, [500])
    assert e.value.code == gpu.UB_EINVAL
    g.close()
