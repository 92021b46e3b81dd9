"""Rule M17, prefix / radix caching (A.5): w~ = max(w, s_pre - h) and prefill work s_pre - h.

CPU pins of the oracle: no hits == the plain schedule; the size signal every iteration is the paper's formula with w
tracked here from the per-iteration records; the prefill work executed shrinks by exactly the hit tokens; a hit is a
shorter prompt for everything the request's own KV is concerned with.  GPU parity against the oracle.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_18431_b200 import workloads as W
from tests.helpers import pressure_workload


def _wl(seed, **kw):
    kw.setdefault("kv_blocks", 64)
    wl = pressure_workload(seed, n=140, gamma=0.3, bin_tokens=32, **kw)
    tr = wl.traces()
    rng = np.random.default_rng([17, seed])
    hits = (rng.random(tr[1].shape) * tr[1] * (rng.random(tr[1].shape) < 0.6)).astype(np.int32)
    hits = np.minimum(hits, tr[1] - 1)
    return wl, tr, hits


def test_no_hits_is_the_plain_schedule():
    wl, tr, hits = _wl(0)
    o0 = O.OracleSim(wl.sim, wl.replicas, tr); o0.run()
    o1 = O.OracleSim(wl.sim, wl.replicas, tr, hits=np.zeros_like(hits)); o1.run()
    assert o0.digest()[0] == o1.digest()[0]
    assert all(np.array_equal(x, y) for x, y in zip(o0.per_request(), o1.per_request()))


@pytest.mark.parametrize("seed", [1, 2])
def test_signal_is_max_of_processed_tokens_and_uncached_prompt(seed):
    """Every iteration, every request: bin = Eq. 8 of w~ = max(w, s_pre - h), w = the tokens the request has
    processed so far without the ones a recompute eviction threw away and had redone -- tracked here from the records --
    and the key is a - b_gamma(k 2^bin) - delta [resident]."""
    wl, tr, hits = _wl(seed)
    a, P, D = tr[0][0], tr[1][0], tr[2][0]
    k, tok, delta = int(wl.sim["bin_tokens"]), int(wl.sim["tok_us"]), int(wl.replicas["hysteresis_us"][0])
    o = O.OracleSim(wl.sim, wl.replicas, tr, hits=hits)
    cached, d_of = {}, {}
    checked = 0
    for it in range(100000):
        info, rows = o.step_replica(0)
        if not info["executed"]:
            break
        for r in rows:
            i = r["id"]
            need = int(P[i] - hits[0, i])                          # s_pre - h
            w = min(cached.get(i, 0), need) if d_of.get(i, 0) == 0 else need + d_of[i]
            sig = max(w, need)
            assert r["bin"] == O.quant_bin(sig, k)
            assert r["key"] == int(a[i]) - O.boost_us(0.3, k * 2 ** r["bin"], tok) - (delta if r["resident_before"] else 0)
            checked += 1
        for r in rows:
            cached[r["id"]], d_of[r["id"]] = r["cached_after"], r["d_after"]
    assert checked > 3000 and (hits > 0).sum() > 30


def test_prefill_work_shrinks_by_the_hit_tokens():
    wl, tr, hits = _wl(3, kv_blocks=1 << 14)                       # ample KV: nothing is recomputed
    P, D = tr[1][0].astype(np.int64), tr[2][0].astype(np.int64)
    o = O.OracleSim(wl.sim, wl.replicas, tr, hits=hits); o.run()
    st = o.stats()[0]
    assert st["tokens_lost"] == 0
    assert st["prefill_tokens"] + st["decode_seqs"] == int((P - hits[0] + D - 1).sum())


@pytest.mark.parametrize("seed", [4, 5])
def test_a_hit_is_a_shorter_prompt(seed):
    """With the shared prefix's KV charged to the cache (reading G26) a request with h cached tokens is, for
    the replica, the same request with the prompt s_pre - h."""
    wl, tr, hits = _wl(seed, preempt=W.PRE_AUTO, swap_pool_blocks=20)
    o1 = O.OracleSim(wl.sim, wl.replicas, tr, hits=hits); o1.run()
    o2 = O.OracleSim(wl.sim, wl.replicas, (tr[0], tr[1] - hits, tr[2], tr[3])); o2.run()
    assert o1.digest()[0] == o2.digest()[0]
    assert o1.stats()[0]["evict_recompute"] + o1.stats()[0]["evict_swap"] > 0


def test_hits_must_leave_one_prompt_token():
    wl, tr, hits = _wl(6)
    bad = hits.copy(); bad[0, 3] = tr[1][0, 3]
    with pytest.raises(O.OracleError):
        O.OracleSim(wl.sim, wl.replicas, tr, hits=bad)


@pytest.mark.gpu
@pytest.mark.parametrize("policy,guard", [(W.POLICY_BOOST, 1), (W.POLICY_FCFS, 0), (W.POLICY_SRPT, 0)])
def test_gpu_prefix_cache_parity(policy, guard):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_2606_18431_b200 import binding as B
    for seed in (7, 8):
        wl, tr, hits = _wl(seed, policy=policy, guard=guard, preempt=W.PRE_AUTO, swap_pool_blocks=20, n_replicas=2)
        g = B.Sim(wl.sim, wl.replicas, tr, hits=hits); o = O.OracleSim(wl.sim, wl.replicas, tr, hits=hits)
        g.run(); o.run()
        assert np.array_equal(g.digest(), o.digest())
        for x, y in zip(g.per_request(), o.per_request()):
            assert np.array_equal(x, y)
        assert g.stats()[0]["prefill_tokens"] == o.stats()[0]["prefill_tokens"]
        bad = hits.copy(); bad[0, 0] = tr[1][0, 0]
        with pytest.raises(B.UbError) as e:
            B.Sim(wl.sim, wl.replicas, tr, hits=bad)
        assert e.value.code == B.UB_EINVAL
        g.close(); o.close()
