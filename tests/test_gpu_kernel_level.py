"""Kernel-level GPU parity (SURVEY.md Sec. 4 tier T1, Sec. 8(b)): single steps of the CUDA path from states that come from
the oracle, not from the device's own history.

* a1: the streaming kernel's own scorer (ub_debug_keys_stream) against the (class, key) the oracle scores.
* a3 / a4 / a5: ub_debug_set_state loads the oracle's state in front of iteration i (window in the oracle's order,
  progress, residency, MemGuard lock, clock, trace cursor, swap occupancy -- all read off the oracle's own per-step
  records, no scheduler arithmetic here), ONE ub_step runs, and the window and the clock behind it must be the
  oracle's.  Done once with every request flagged "may be out of place" (the kernels sort from scratch: the streaming
  kernel for up to 32 requests, the team kernels beyond) and once with only the requests flagged whose key inputs
  the oracle reports as changed (the streaming kernel's merge, decode-run and waiting-tail paths).
"""
import numpy as np
import pytest

from paper_2606_18431_b200 import workloads as W
from tests.helpers import pressure_workload

pytestmark = pytest.mark.gpu

F_RESIDENT, F_SWAPPED, F_EMITPREV, F_DIRTY, F_ADMITNOW, F_KLASS1, F_PREEMPTED, F_LOCK_SHIFT = 1, 2, 4, 8, 16, 32, 64, 7


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_2606_18431_b200 import binding
    binding.lib()
    return binding


@pytest.mark.parametrize("policy,guard", [(W.POLICY_FCFS, 0), (W.POLICY_BOOST, 0), (W.POLICY_BOOST, 1)])
def test_stream_scorer_keys_match_oracle(gpu, oracle_mod, policy, guard):
    """Before every iteration the (class, key) of each request from score() of ub_stream.cu -- the scorer the benchmarked
    kernel runs -- equals what the oracle scores in that iteration (pi = a - b_gamma(w_hat) - delta [resident],
    PAPER.md:429, Eq. 7, Eq. 8; MemGuard class)."""
    wl = pressure_workload(11, n=160, kv_blocks=48, policy=policy, preempt=W.PRE_AUTO, swap_pool_blocks=20,
                           guard=guard, gamma=0.3, bin_tokens=32)
    tr = wl.traces()
    g = gpu.Sim(wl.sim, wl.replicas, tr)
    o = oracle_mod.OracleSim(wl.sim, wl.replicas, tr)
    checked = 0
    for it in range(1500):
        ids, kl, ky = g.debug_keys(0, stream_scorer=True)
        ids2, kl2, ky2 = g.debug_keys(0)
        assert np.array_equal(ids, ids2) and np.array_equal(kl, kl2) and np.array_equal(ky, ky2)
        info, rows = o.step_replica(0)
        g.step(1)
        if not info["executed"]:
            break
        want = {r["id"]: (r["klass"], r["key"]) for r in rows}
        for i, c, k in zip(ids, kl, ky):
            assert (int(c), int(k)) == want[int(i)], f"iteration {it} request {i}"
        checked += len(ids)
    assert checked > 5000


def _oracle_history(oracle_mod, wl, max_steps=4000):
    """Every executed iteration of replica 0: (info, rows in priority order)."""
    o = oracle_mod.OracleSim(wl.sim, wl.replicas, wl.traces())
    hist = []
    for _ in range(max_steps):
        info, rows = o.step_replica(0)
        if not info["executed"]:
            break
        hist.append((info, rows))
    o.close()
    return hist


class _Tracker:
    """The replica's state as the oracle's per-step records report it (bookkeeping only)."""

    def __init__(self, D, blk):
        self.D, self.blk = D, blk
        self.order, self.req = [], {}       # ids in stored order; id -> dict
        self.clock, self.next = 0, 0

    def apply(self, info, rows):
        new_order = []
        for r in rows:
            i = r["id"]
            q = self.req.get(i, dict(d=0, swapped=False))
            emitted = r["d_after"] > q["d"]
            if r["evict"] == 2:
                swapped = True
            elif r["want"] > 0 or r["evict"] == 1:
                swapped = False
            else:
                swapped = q["swapped"]
            preempted = bool(r["evict"]) or (q.get("preempted", False) and r["want"] == 0)
            self.req[i] = dict(d=r["d_after"], cached=r["cached_after"], resident=bool(r["resident_after"]),
                               swapped=swapped, emitted=emitted, admitted=r["want"] > 0, klass=r["klass"], bin=r["bin"],
                               res_before=bool(r["resident_before"]), preempted=preempted)
            self.next = max(self.next, i + 1)
            if r["d_after"] < self.D[i]:
                new_order.append(i)
            else:
                del self.req[i]
        self.order = new_order
        self.clock = info["t_end_us"]

    def swap_used(self):
        return sum((q["cached"] + self.blk - 1) // self.blk for q in self.req.values() if q["swapped"])

    def arrays(self, nxt_rows, all_dirty):
        """Device records of the state as it stands; nxt_rows: the oracle's records of the NEXT iteration (by id)."""
        nxt = {r["id"]: r for r in nxt_rows}
        ids, d, cached, flags = [], [], [], []
        for i in self.order:
            q = self.req[i]
            f = 0
            if q["resident"]:
                f |= F_RESIDENT | ((q["bin"] + 1) << F_LOCK_SHIFT)
            if q["swapped"]:
                f |= F_SWAPPED
            if q["preempted"]:
                f |= F_PREEMPTED
            if q["emitted"]:
                f |= F_EMITPREV
            if q["admitted"]:
                f |= F_ADMITNOW
            if q["klass"]:
                f |= F_KLASS1
            n = nxt[i]
            changed = (bool(n["resident_before"]), n["bin"], n["klass"]) != (q["res_before"], q["bin"], q["klass"])
            if all_dirty or changed:
                f |= F_DIRTY
            ids.append(i); d.append(q["d"]); cached.append(q["cached"]); flags.append(f)
        return ids, d, cached, flags


@pytest.mark.parametrize("all_dirty", [True, False], ids=["sort-from-scratch", "merge-the-re-keyed"])
@pytest.mark.parametrize("n_req", [30, 150])
@pytest.mark.parametrize("policy,guard,preempt,seed", [
    (W.POLICY_BOOST, 1, W.PRE_AUTO, 3), (W.POLICY_BOOST, 1, W.PRE_RECOMPUTE, 4), (W.POLICY_FCFS, 0, W.PRE_SWAP, 5),
    (W.POLICY_BOOST, 0, W.PRE_AUTO, 6), (W.POLICY_SRPT, 0, W.PRE_RECOMPUTE, 7)])
def test_single_step_from_oracle_snapshots(gpu, oracle_mod, policy, guard, preempt, seed, n_req, all_dirty):
    """ub_debug_set_state + one ub_step: a3 admit, a4 victim select, a5 advance in isolation (M7-M10)."""
    if policy == W.POLICY_SRPT and not all_dirty:
        pytest.skip("SRPT keys drift every token: the team kernels verify the order themselves")
    wl = pressure_workload(seed, n=n_req, kv_blocks=40, policy=policy, guard=guard, preempt=preempt, swap_pool_blocks=16,
                           gamma=0.3, bin_tokens=32, mean_gap_us=3000, delta=100_000 if policy == W.POLICY_BOOST else 0)
    a, P, D, n = wl.traces()
    hist = _oracle_history(oracle_mod, wl, 2500)
    assert len(hist) > 300
    g = gpu.Sim(wl.sim, wl.replicas, (a, P, D, n))
    trk = _Tracker([int(x) for x in D[0]], int(wl.sim["block_tokens"]))
    tested = evictions = big = 0
    for i, (info, rows) in enumerate(hist):
        pick = i >= 1 and trk.order and (i % 5 == 0 or any(r["evict"] for r in rows)) and i < len(hist) - 2
        if pick:
            ids, d, cached, flags = trk.arrays(rows, all_dirty)
            clock, nxt, swp = trk.clock, trk.next, trk.swap_used()
        trk.apply(info, rows)                          # the oracle's state behind iteration i
        if pick:
            g.debug_set_state(0, ids, d, cached, flags, clock, nxt, swp)
            g.step(1)
            st = g.debug_state(0)
            where = f"iteration {i} ({len(ids)} requests in front of it)"
            assert st["clock_us"] == trk.clock, where
            assert st["id"].tolist() == trk.order, where
            assert st["d"].tolist() == [trk.req[j]["d"] for j in trk.order], where
            assert st["cached"].tolist() == [trk.req[j]["cached"] for j in trk.order], where
            assert [bool(f & F_RESIDENT) for f in st["flags"]] == [trk.req[j]["resident"] for j in trk.order], where
            assert [bool(f & F_SWAPPED) for f in st["flags"]] == [trk.req[j]["swapped"] for j in trk.order], where
            tested += 1
            evictions += sum(1 for r in rows if r["evict"])
            big += len(ids) > 32
    assert tested > 60 and evictions > 5 and (big > 5 if n_req > 32 else big == 0)
    g.close()


def test_set_state_rejects_inconsistent_records(gpu):
    wl = pressure_workload(1, n=40)
    g = gpu.Sim(wl.sim, wl.replicas, wl.traces())
    with pytest.raises(gpu.UbError) as e:            # request 5 has not arrived yet (cursor 3)
        g.debug_set_state(0, [0, 5], [0, 0], [0, 0], [F_KLASS1, F_KLASS1], 1000, 3)
    assert e.value.code == gpu.UB_EINVAL
    with pytest.raises(gpu.UbError) as e:            # KV held by a request that is neither resident nor swapped
        g.debug_set_state(0, [0], [0], [5], [F_KLASS1], 1000, 3)
    assert e.value.code == gpu.UB_EINVAL
    with pytest.raises(gpu.UbError) as e:            # empty window behind the last request = finished
        g.debug_set_state(0, [], [], [], [], 1000, 40)
    assert e.value.code == gpu.UB_ESTATE
    g.debug_set_state(0, [0, 1], [0, 0], [0, 0], [F_KLASS1 | F_DIRTY, F_KLASS1 | F_DIRTY], 10**9, 2)
    assert g.debug_state(0)["n_active"] == 2
    g.close()
