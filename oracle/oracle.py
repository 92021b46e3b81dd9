"""ctypes wrapper of the CPU oracle (oracle/orc_uniboost.c).

TEST INFRASTRUCTURE: imported only by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  It does not import the
CUDA package and the CUDA package does not import it.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)
sys.path.pop(0)

TBT_BINS = 4352
I64 = C.c_int64


class OrcConfig(C.Structure):
    _fields_ = [(n, I64) for n in (
        "n_replicas", "n_traces", "max_requests", "queue_cap", "kv_blocks", "block_tokens", "max_batch",
        "chunk_tokens", "token_budget", "c0_us", "c_prefill_tok_us", "c_decode_seq_us", "preempt_mode",
        "swap_ns_per_block", "swap_pool_blocks", "bin_tokens", "tok_us")]


class OrcReplica(C.Structure):
    _fields_ = [(n, I64) for n in ("trace_id", "policy", "guard", "signal_mode", "quant_mode", "hysteresis_us")] + [
        ("gamma", C.c_double)]


class OrcStats(C.Structure):
    _fields_ = [(n, I64) for n in (
        "iterations", "request_steps", "n_completed", "evict_recompute", "evict_swap", "swapins", "tokens_lost",
        "tokens_emitted", "prefill_tokens", "decode_seqs", "t_end_us", "peak_active", "done", "swap_used")] + [
        ("ttft_us", I64 * 3), ("ttlt_us", I64 * 3), ("tbt_us", I64 * 3),
        ("sum_ttft_us", I64), ("sum_ttlt_us", I64), ("sum_tbt_num_us", I64), ("sum_tbt_den", I64),
        ("ttft_s", C.c_double * 3), ("ttlt_s", C.c_double * 3), ("tbt_s", C.c_double * 3),
        ("mean_ttft_s", C.c_double), ("mean_ttlt_s", C.c_double), ("mean_tbt_s", C.c_double),
        ("tokens_per_s", C.c_double)]


class OrcGammaAda(C.Structure):
    _fields_ = [("window", I64), ("min_samples", I64), ("beta_shift", I64), ("levels", I64),
                ("gamma_min", C.c_double), ("gamma_max", C.c_double), ("eps_us", I64)]


class OrcStepEntry(C.Structure):
    _fields_ = [(n, I64) for n in ("id", "klass", "key", "bin", "resident_before", "want", "evict",
                                   "cached_after", "d_after", "resident_after")]


class OrcStepInfo(C.Structure):
    _fields_ = [(n, I64) for n in ("executed", "n_active", "t_start_us", "cost_us", "t_end_us", "claimed_blocks",
                                   "prefill_tokens", "decode_seqs", "swap_blocks", "kv_resident_after")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        P = C.POINTER
        L.orc_create.argtypes = [P(OrcConfig), P(C.c_void_p)]
        L.orc_destroy.argtypes = [C.c_void_p]; L.orc_destroy.restype = None
        L.orc_load_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_load_trace_prefix.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_set_replicas.argtypes = [C.c_void_p, P(OrcReplica)]
        L.orc_step.argtypes = [C.c_void_p, I64]
        L.orc_step_replica.argtypes = [C.c_void_p, I64, P(OrcStepInfo), P(OrcStepEntry)]
        L.orc_run.argtypes = [C.c_void_p, I64, P(I64)]
        L.orc_run_replica.argtypes = [C.c_void_p, I64, I64, P(I64)]
        L.orc_stats_get.argtypes = [C.c_void_p, P(OrcStats)]
        L.orc_per_request.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_digest.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_boost_lut.argtypes = [C.c_void_p, I64, C.c_void_p, I64, P(I64)]
        L.orc_tbt_hist.argtypes = [C.c_void_p, I64, C.c_void_p]
        L.orc_quant_bin.argtypes = [I64, I64]; L.orc_quant_bin.restype = I64
        L.orc_boost_us.argtypes = [C.c_double, I64, I64]; L.orc_boost_us.restype = I64
        L.orc_percentile_nearest_rank.argtypes = [C.c_void_p, I64, I64]; L.orc_percentile_nearest_rank.restype = I64
        L.orc_tbt_bin.argtypes = [I64]; L.orc_tbt_bin.restype = I64
        L.orc_tbt_edge.argtypes = [I64]; L.orc_tbt_edge.restype = I64
        L.orc_percentile_curve.argtypes = [C.c_void_p, I64, C.c_void_p, I64, C.c_void_p]
        L.orc_slo_attainment.argtypes = [C.c_void_p, I64, C.c_void_p, I64, C.c_void_p]
        L.orc_preempt_time.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_jsq_run.argtypes = [C.c_void_p, I64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, I64, C.c_void_p]
        L.orc_class_percentiles.argtypes = [C.c_void_p, I64, I64, I64, C.c_void_p, I64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_set_gamma_ada.argtypes = [C.c_void_p, P(OrcGammaAda), C.c_void_p]
        L.orc_gamma_state.argtypes = [C.c_void_p, I64, P(I64), P(I64), P(I64)]
        L.orc_gamma_grid.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_gamma_hat_u.argtypes = [I64, I64, I64]; L.orc_gamma_hat_u.restype = I64
        L.orc_strerror.argtypes = [C.c_int]; L.orc_strerror.restype = C.c_char_p
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code):
        self.code = code
        super().__init__(f"oracle error {code}: {lib().orc_strerror(code).decode()}")


def _chk(rc, allow=()):
    if rc != 0 and rc not in allow:
        raise OracleError(rc)
    return rc


ELIVELOCK = -7


def quant_bin(sig, k):
    return int(lib().orc_quant_bin(int(sig), int(k)))


def boost_us(gamma, w_tokens, tok_us):
    return int(lib().orc_boost_us(float(gamma), int(w_tokens), int(tok_us)))


def gamma_hat_u(t95_us, t99_us, eps_us):
    return int(lib().orc_gamma_hat_u(int(t95_us), int(t99_us), int(eps_us)))


def percentile_nearest_rank(sorted_vals, p):
    v = np.ascontiguousarray(sorted_vals, np.int64)
    return int(lib().orc_percentile_nearest_rank(v.ctypes.data, len(v), int(p)))


def tbt_bin(g):
    return int(lib().orc_tbt_bin(int(g)))


def tbt_edge(i):
    return int(lib().orc_tbt_edge(int(i)))


def _stats_to_dict(st):
    out = {}
    for name, typ in OrcStats._fields_:
        v = getattr(st, name)
        out[name] = list(v) if hasattr(v, "__len__") else v
    return out


class OracleSim:
    """Drives the oracle from a workloads.Workload-like object (sim dict, replicas dict, traces())."""

    def __init__(self, sim: dict, replicas: dict, traces, hits=None):
        L = lib()
        self.sim = dict(sim)
        cfg = OrcConfig(**{n: int(sim[n]) for n, _ in OrcConfig._fields_})
        h = C.c_void_p()
        _chk(L.orc_create(C.byref(cfg), C.byref(h)))
        self._h = h
        a, p, d, n = traces
        a = np.ascontiguousarray(a, np.int64); p = np.ascontiguousarray(p, np.int32)
        d = np.ascontiguousarray(d, np.int32); n = np.ascontiguousarray(n, np.uint32)
        assert a.shape == (sim["n_traces"], sim["max_requests"])
        if hits is None:
            _chk(L.orc_load_trace(h, a.ctypes.data, p.ctypes.data, d.ctypes.data, n.ctypes.data))
        else:                                              # prefix-cache hit tokens per request (rule M17)
            hh = np.ascontiguousarray(hits, np.int32)
            assert hh.shape == a.shape
            _chk(L.orc_load_trace_prefix(h, a.ctypes.data, p.ctypes.data, d.ctypes.data, hh.ctypes.data, n.ctypes.data))
        R = int(sim["n_replicas"])
        reps = (OrcReplica * R)()
        for r in range(R):
            for f in ("trace_id", "policy", "guard", "signal_mode", "quant_mode", "hysteresis_us"):
                setattr(reps[r], f, int(replicas[f][r]))
            reps[r].gamma = float(replicas["gamma"][r])
        _chk(L.orc_set_replicas(h, reps))
        self.R, self.N, self.Q = R, int(sim["max_requests"]), int(sim["queue_cap"])

    def percentile_curve(self, which, permille):
        pm = np.ascontiguousarray(permille, np.int64)
        out = np.zeros((self.R, len(pm)), np.int64)
        _chk(lib().orc_percentile_curve(self._h, int(which), pm.ctypes.data, len(pm), out.ctypes.data))
        return out

    def jsq_run(self, cluster_size, arrival_us, prompt_tok, decode_tok, n_arr):
        """Rule M18: route the [C][NA] global streams over clusters of `cluster_size` replicas by join-the-shortest-queue
        and run everything to completion; returns assign [C][NA] (replica number within the cluster, -1 = no arrival)."""
        a = np.ascontiguousarray(arrival_us, np.int64); p = np.ascontiguousarray(prompt_tok, np.int32)
        d = np.ascontiguousarray(decode_tok, np.int32); n = np.ascontiguousarray(n_arr, np.uint32)
        assert a.ndim == 2 and a.shape == p.shape == d.shape and n.shape == (a.shape[0],)
        out = np.full(a.shape, -1, np.int32)
        _chk(lib().orc_jsq_run(self._h, int(cluster_size), a.ctypes.data, p.ctypes.data, d.ctypes.data, n.ctypes.data,
                               a.shape[1], out.ctypes.data))
        return out

    def preempt_time(self):
        """[R][N] int64 microseconds each request spent preempted (rule M15)."""
        out = np.zeros((self.R, self.N), np.int64)
        _chk(lib().orc_preempt_time(self._h, out.ctypes.data))
        return out

    def class_percentiles(self, which, len_lo, len_hi, permille):
        """(percentiles [R][n], count [R], sum [R]) of TTFT (0) / TTLT (1) / preemption time (2) over the completed
        requests with len_lo <= P + D <= len_hi."""
        pm = np.ascontiguousarray(permille, np.int64)
        out = np.zeros((self.R, len(pm)), np.int64); cnt = np.zeros(self.R, np.int64); tot = np.zeros(self.R, np.int64)
        _chk(lib().orc_class_percentiles(self._h, int(which), int(len_lo), int(len_hi), pm.ctypes.data, len(pm),
                                         out.ctypes.data, cnt.ctypes.data, tot.ctypes.data))
        return out, cnt, tot

    def slo_attainment(self, which, threshold_us):
        thr = np.ascontiguousarray(threshold_us, np.int64)
        assert thr.ndim == 2 and thr.shape[0] == self.R
        out = np.zeros(thr.shape, np.int64)
        _chk(lib().orc_slo_attainment(self._h, int(which), thr.ctypes.data, thr.shape[1], out.ctypes.data))
        return out

    def set_gamma_ada(self, ada: dict, adaptive):
        """gamma-Ada (M13): ada = dict(window, min_samples, beta_shift, levels, gamma_min, gamma_max, eps_us)."""
        g = OrcGammaAda(**{n: (float(ada[n]) if n.startswith("gamma") else int(ada[n])) for n, _ in OrcGammaAda._fields_})
        ad = np.ascontiguousarray(adaptive, np.uint8)
        assert ad.shape == (self.R,)
        _chk(lib().orc_set_gamma_ada(self._h, C.byref(g), ad.ctypes.data))
        self._levels = int(ada["levels"])

    def gamma_state(self, r=0):
        g, l, n = I64(0), I64(0), I64(0)
        _chk(lib().orc_gamma_state(self._h, int(r), C.byref(g), C.byref(l), C.byref(n)))
        return g.value, l.value, n.value

    def gamma_grid(self):
        out = np.zeros(self._levels, np.int64)
        _chk(lib().orc_gamma_grid(self._h, out.ctypes.data))
        return out

    @classmethod
    def from_workload(cls, wl, workers: int = 1):
        return cls(wl.sim, wl.replicas, wl.traces(workers=workers))

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def step(self, n_iters=1):
        _chk(lib().orc_step(self._h, int(n_iters)))

    def step_replica(self, r=0):
        """One iteration of replica r; returns (info dict, list of entry dicts in priority order)."""
        info = OrcStepInfo()
        ents = (OrcStepEntry * self.Q)()
        _chk(lib().orc_step_replica(self._h, int(r), C.byref(info), ents))
        inf = {n: getattr(info, n) for n, _ in OrcStepInfo._fields_}
        rows = [{n: getattr(ents[j], n) for n, _ in OrcStepEntry._fields_} for j in range(inf["n_active"])]
        return inf, rows

    def run(self, max_iters=1 << 40, check=True):
        it = I64(0)
        rc = lib().orc_run(self._h, int(max_iters), C.byref(it))
        _chk(rc, allow=() if check else (ELIVELOCK,))
        return it.value

    def run_replica(self, r, max_iters=1 << 40, check=True):
        it = I64(0)
        rc = lib().orc_run_replica(self._h, int(r), int(max_iters), C.byref(it))
        _chk(rc, allow=() if check else (ELIVELOCK,))
        return it.value

    def stats(self):
        st = (OrcStats * self.R)()
        _chk(lib().orc_stats_get(self._h, st))
        return [_stats_to_dict(st[r]) for r in range(self.R)]

    def per_request(self):
        tf = np.empty((self.R, self.N), np.int64); tl = np.empty((self.R, self.N), np.int64)
        ne = np.empty((self.R, self.N), np.uint32); neu = np.empty((self.R, self.N), np.uint32)
        _chk(lib().orc_per_request(self._h, tf.ctypes.data, tl.ctypes.data, ne.ctypes.data, neu.ctypes.data))
        return tf, tl, ne, neu

    def digest(self):
        dg = np.empty(self.R, np.uint64)
        _chk(lib().orc_digest(self._h, dg.ctypes.data))
        return dg

    def boost_lut(self, r=0):
        nb = I64(0)
        _chk(lib().orc_boost_lut(self._h, int(r), None, 0, C.byref(nb)))
        lut = np.empty(nb.value, np.int64)
        _chk(lib().orc_boost_lut(self._h, int(r), lut.ctypes.data, nb.value, C.byref(nb)))
        return lut

    def tbt_hist(self, r=0):
        h = np.empty(TBT_BINS, np.uint32)
        _chk(lib().orc_tbt_hist(self._h, int(r), h.ctypes.data))
        return h
