"""Thin ctypes binding of libuniboost.so (include/uniboost.h): argument marshalling only.

Same names as the C-ABI (ub_create, ub_load_trace, ub_set_replicas, ub_step, ub_run, ub_stats, ...), plus the
`Sim` convenience class that drives them from a `workloads.Workload`.  Every step of the scheduling path runs in
the CUDA kernels; there is no CPU fallback: if the library is missing or no CUDA device is present this fails
loudly.  PyTorch is used only for the stream (and, by callers, for device buffers).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libuniboost.so")

UB_ABI_VERSION = 1
UB_MAX_QUEUE = 2048
UB_TBT_BINS = 4352
UB_OK, UB_EINVAL, UB_ENOMEM, UB_ECUDA, UB_ESTATE, UB_EUNSORTED, UB_EINFEASIBLE, UB_ELIVELOCK, UB_ETOOBIG = 0, -1, -2, -3, -4, -5, -6, -7, -8
UB_NOALLOC_CURVE_MAX = 65536

U32, I64, U64 = C.c_uint32, C.c_int64, C.c_uint64


class UbConfig(C.Structure):
    _fields_ = [(n, U32) for n in (
        "struct_size", "abi_version", "n_replicas", "n_traces", "max_requests", "queue_cap", "kv_blocks",
        "block_tokens", "max_batch", "chunk_tokens", "token_budget", "preempt_mode", "swap_ns_per_block",
        "swap_pool_blocks", "bin_tokens", "tok_us")] + [
        ("c0_us", I64), ("c_prefill_tok_us", I64), ("c_decode_seq_us", I64),
        ("iters_per_launch", U32), ("device", C.c_int32), ("stream", C.c_void_p)]


class UbReplica(C.Structure):
    _fields_ = [("trace_id", U32), ("policy", C.c_uint8), ("guard", C.c_uint8), ("signal_mode", C.c_uint8),
                ("quant_mode", C.c_uint8), ("hysteresis_us", I64), ("gamma", C.c_double)]


class UbReplicaStats(C.Structure):
    _fields_ = [(n, I64) for n in (
        "iterations", "request_steps", "n_completed", "evict_recompute", "evict_swap", "swapins", "tokens_lost",
        "tokens_emitted", "prefill_tokens", "decode_seqs", "t_end_us", "peak_active", "done", "swap_used")] + [
        ("ttft_us", I64 * 3), ("ttlt_us", I64 * 3), ("tbt_us", I64 * 3),
        ("sum_ttft_us", I64), ("sum_ttlt_us", I64), ("sum_tbt_num_us", I64), ("sum_tbt_den", I64),
        ("ttft_s", C.c_double * 3), ("ttlt_s", C.c_double * 3), ("tbt_s", C.c_double * 3),
        ("mean_ttft_s", C.c_double), ("mean_ttlt_s", C.c_double), ("mean_tbt_s", C.c_double),
        ("tokens_per_s", C.c_double)]


#: every symbol include/uniboost.h declares
class UbGammaAda(C.Structure):
    _fields_ = [("struct_size", U32), ("window", U32), ("min_samples", U32), ("beta_shift", U32), ("levels", U32),
                ("pad", U32), ("gamma_min", C.c_double), ("gamma_max", C.c_double), ("eps_us", I64)]


EXPORTS = ("ub_create", "ub_destroy", "ub_load_trace", "ub_set_replicas", "ub_step", "ub_run", "ub_stats",
           "ub_per_request", "ub_digest", "ub_boost_lut", "ub_tbt_hist", "ub_debug_get_state",
           "ub_last_step_timing", "ub_set_iters_per_launch", "ub_set_gamma_ada", "ub_gamma_state", "ub_gamma_grid",
           "ub_percentile_curve", "ub_slo_attainment", "ub_debug_keys", "ub_debug_keys_stream", "ub_debug_set_state",
           "ub_class_percentiles", "ub_preempt_time", "ub_load_trace_prefix", "ub_jsq_run", "ub_percentile_curve_noalloc",
           "ub_strerror")

_lib = None


def lib():
    """Load libuniboost.so (built by paper_2606_18431_b200/build.py).  No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2606_18431_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        P = C.POINTER
        vp = C.c_void_p
        L.ub_create.argtypes = [P(UbConfig), P(vp)]
        L.ub_destroy.argtypes = [vp]; L.ub_destroy.restype = None
        L.ub_load_trace.argtypes = [vp, vp, vp, vp, vp, C.c_int]
        L.ub_load_trace_prefix.argtypes = [vp, vp, vp, vp, vp, vp, C.c_int]
        L.ub_set_replicas.argtypes = [vp, P(UbReplica)]
        L.ub_step.argtypes = [vp, U32, P(U64)]
        L.ub_run.argtypes = [vp, U64, P(U64)]
        L.ub_stats.argtypes = [vp, P(UbReplicaStats)]
        L.ub_per_request.argtypes = [vp, vp, vp, vp, vp, C.c_int]
        L.ub_digest.argtypes = [vp, vp]
        L.ub_boost_lut.argtypes = [vp, U32, vp, U32, P(U32)]
        L.ub_tbt_hist.argtypes = [vp, U32, vp]
        L.ub_debug_get_state.argtypes = [vp, U32, P(U32), vp, vp, vp, vp, P(I64)]
        L.ub_last_step_timing.argtypes = [vp, P(C.c_float), P(U32)]
        L.ub_set_iters_per_launch.argtypes = [vp, U32]
        L.ub_debug_keys.argtypes = [vp, U32, P(U32), vp, vp, vp]
        L.ub_debug_keys_stream.argtypes = [vp, U32, P(U32), vp, vp, vp]
        L.ub_debug_set_state.argtypes = [vp, U32, U32, vp, vp, vp, vp, I64, U32, U32]
        L.ub_percentile_curve.argtypes = [vp, U32, vp, U32, vp]
        L.ub_percentile_curve_noalloc.argtypes = [vp, U32, vp, U32, vp]
        L.ub_slo_attainment.argtypes = [vp, U32, vp, U32, vp]
        L.ub_class_percentiles.argtypes = [vp, U32, U32, U32, vp, U32, vp, vp, vp]
        L.ub_preempt_time.argtypes = [vp, vp, C.c_int]
        L.ub_jsq_run.argtypes = [vp, U32, U32, U32, vp, vp, vp, vp, vp]
        L.ub_set_gamma_ada.argtypes = [vp, P(UbGammaAda), vp]
        L.ub_gamma_state.argtypes = [vp, U32, P(I64), P(C.c_int32), P(U64)]
        L.ub_gamma_grid.argtypes = [vp, vp]
        L.ub_strerror.argtypes = [C.c_int]; L.ub_strerror.restype = C.c_char_p
        _lib = L
    return _lib


class UbError(RuntimeError):
    def __init__(self, code):
        self.code = code
        super().__init__(f"uniboost error {code}: {lib().ub_strerror(code).decode()}")


def _chk(rc, allow=()):
    if rc != 0 and rc not in allow:
        raise UbError(rc)
    return rc


# ---- the C-ABI calls under their own names (thin) -------------------------------------------------------

def ub_create(cfg: UbConfig) -> C.c_void_p:
    h = C.c_void_p()
    _chk(lib().ub_create(C.byref(cfg), C.byref(h)))
    return h


def ub_destroy(h):
    lib().ub_destroy(h)


def ub_load_trace(h, arrival_us, prompt_tok, decode_tok, n_req, ptrs_on_device=False):
    """numpy arrays (host) or integer device pointers (ptrs_on_device=True)."""
    if ptrs_on_device:
        args = [C.c_void_p(int(x)) for x in (arrival_us, prompt_tok, decode_tok, n_req)]
        return _chk(lib().ub_load_trace(h, *args, 1))
    a = np.ascontiguousarray(arrival_us, np.int64); p = np.ascontiguousarray(prompt_tok, np.int32)
    d = np.ascontiguousarray(decode_tok, np.int32); n = np.ascontiguousarray(n_req, np.uint32)
    return _chk(lib().ub_load_trace(h, a.ctypes.data, p.ctypes.data, d.ctypes.data, n.ctypes.data, 0))


def ub_load_trace_prefix(h, arrival_us, prompt_tok, decode_tok, hit_tok, n_req):
    """As ub_load_trace (host numpy arrays) plus the prefix-cache hit tokens per request (rule M17)."""
    a = np.ascontiguousarray(arrival_us, np.int64); p = np.ascontiguousarray(prompt_tok, np.int32)
    d = np.ascontiguousarray(decode_tok, np.int32); hh = np.ascontiguousarray(hit_tok, np.int32)
    n = np.ascontiguousarray(n_req, np.uint32)
    return _chk(lib().ub_load_trace_prefix(h, a.ctypes.data, p.ctypes.data, d.ctypes.data, hh.ctypes.data, n.ctypes.data, 0))


def ub_set_replicas(h, reps):
    return _chk(lib().ub_set_replicas(h, reps))


def ub_set_gamma_ada(h, ada: dict, adaptive):
    """ada = dict(window, min_samples, beta_shift, levels, gamma_min, gamma_max, eps_us); adaptive: [R] of 0/1."""
    g = UbGammaAda()
    g.struct_size = C.sizeof(UbGammaAda)
    for k in ("window", "min_samples", "beta_shift", "levels", "eps_us"):
        setattr(g, k, int(ada[k]))
    g.gamma_min, g.gamma_max = float(ada["gamma_min"]), float(ada["gamma_max"])
    ad = np.ascontiguousarray(adaptive, np.uint8)
    _chk(lib().ub_set_gamma_ada(h, C.byref(g), ad.ctypes.data))


def ub_gamma_state(h, r):
    g, l, n = I64(0), C.c_int32(0), U64(0)
    _chk(lib().ub_gamma_state(h, int(r), C.byref(g), C.byref(l), C.byref(n)))
    return g.value, l.value, n.value


def ub_gamma_grid(h, levels):
    out = np.zeros(int(levels), np.int64)
    _chk(lib().ub_gamma_grid(h, out.ctypes.data))
    return out


def ub_set_iters_per_launch(h, iters_per_launch):
    _chk(lib().ub_set_iters_per_launch(h, int(iters_per_launch)))


def ub_step(h, n_iters, want_live=False):
    if want_live:
        live = U64(0)
        _chk(lib().ub_step(h, int(n_iters), C.byref(live)))
        return live.value
    _chk(lib().ub_step(h, int(n_iters), None))
    return None


def ub_run(h, max_iters=1 << 40, check=True):
    it = U64(0)
    _chk(lib().ub_run(h, int(max_iters), C.byref(it)), allow=() if check else (UB_ELIVELOCK,))
    return it.value


def ub_last_step_timing(h):
    ms = C.c_float(0); nl = U32(0)
    _chk(lib().ub_last_step_timing(h, C.byref(ms), C.byref(nl)))
    return ms.value, nl.value


def _stats_to_dict(st):
    out = {}
    for name, _ in UbReplicaStats._fields_:
        v = getattr(st, name)
        out[name] = list(v) if hasattr(v, "__len__") else v
    return out


def make_config(sim: dict, iters_per_launch: int = 1, device: int = 0, stream: int = 0) -> UbConfig:
    cfg = UbConfig()
    cfg.struct_size = C.sizeof(UbConfig); cfg.abi_version = UB_ABI_VERSION
    for name, _ in UbConfig._fields_:
        if name in sim:
            setattr(cfg, name, int(sim[name]))
    cfg.iters_per_launch = int(iters_per_launch); cfg.device = int(device)
    cfg.stream = C.c_void_p(int(stream) if stream else None)
    return cfg


def make_replicas(replicas: dict, R: int):
    reps = (UbReplica * R)()
    for r in range(R):
        for f in ("trace_id", "policy", "guard", "signal_mode", "quant_mode", "hysteresis_us"):
            setattr(reps[r], f, int(replicas[f][r]))
        reps[r].gamma = float(replicas["gamma"][r])
    return reps


class Sim:
    """Drives libuniboost.so from a workloads.Workload-like description (sim dict, replica table, traces)."""

    def __init__(self, sim: dict, replicas: dict, traces, iters_per_launch: int = 1, device: int = 0,
                 stream: int | None = None, hits=None):
        import torch  # plumbing only: the current CUDA stream
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_18431_b200 needs a CUDA device (B200, sm_100a); there is no CPU fallback")
        if stream is None:
            with torch.cuda.device(device):
                stream = torch.cuda.current_stream().cuda_stream
        self.sim = dict(sim)
        self.R, self.N, self.Q = int(sim["n_replicas"]), int(sim["max_requests"]), int(sim["queue_cap"])
        self._h = ub_create(make_config(sim, iters_per_launch, device, stream))
        a, p, d, n = traces
        assert np.shape(a) == (sim["n_traces"], sim["max_requests"])
        if hits is None:
            ub_load_trace(self._h, a, p, d, n)
        else:
            ub_load_trace_prefix(self._h, a, p, d, hits, n)
        ub_set_replicas(self._h, make_replicas(replicas, self.R))

    @classmethod
    def from_workload(cls, wl, workers: int = 1, **kw):
        return cls(wl.sim, wl.replicas, wl.traces(workers=workers), **kw)

    def close(self):
        if getattr(self, "_h", None):
            ub_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def step(self, n_iters=1, want_live=False):
        return ub_step(self._h, n_iters, want_live)

    def run(self, max_iters=1 << 40, check=True):
        return ub_run(self._h, max_iters, check)

    def debug_keys(self, r=0, stream_scorer=False):
        """(id, klass, key) arrays of replica r's window as the next iteration would score it (stored order);
        stream_scorer: through the streaming kernel's own scorer (ub_debug_keys_stream)."""
        n = U32(0)
        ids = np.zeros(self.Q, np.uint32); kl = np.zeros(self.Q, np.uint32); ky = np.zeros(self.Q, np.int64)
        fn = lib().ub_debug_keys_stream if stream_scorer else lib().ub_debug_keys
        _chk(fn(self._h, int(r), C.byref(n), ids.ctypes.data, kl.ctypes.data, ky.ctypes.data))
        return ids[:n.value], kl[:n.value], ky[:n.value]

    def debug_set_state(self, r, ids, d, cached, flags, clock_us, next_request, swap_used_blocks=0):
        """ub_debug_set_state: overwrite replica r's window (stored order), clock, trace cursor and swap occupancy."""
        a = [np.ascontiguousarray(x, np.uint32) for x in (ids, d, cached, flags)]
        n = len(a[0])
        assert all(len(x) == n for x in a)
        _chk(lib().ub_debug_set_state(self._h, int(r), n, *[x.ctypes.data for x in a], int(clock_us), int(next_request),
                                      int(swap_used_blocks)))

    def percentile_curve(self, which, permille):
        """[R][n] int64 microseconds: nearest-rank percentiles of TTFT (which=0) / TTLT (1) at per-mille points."""
        pm = np.ascontiguousarray(permille, np.uint32)
        out = np.zeros((self.R, len(pm)), np.int64)
        _chk(lib().ub_percentile_curve(self._h, int(which), pm.ctypes.data, len(pm), out.ctypes.data))
        return out

    def percentile_curve_noalloc(self, which, permille):
        """percentile_curve through the entry point that allocates nothing on the device (static scratch in the library;
        UB_ETOOBIG when R x n exceeds UB_NOALLOC_CURVE_MAX)."""
        pm = np.ascontiguousarray(permille, np.uint32)
        out = np.zeros((self.R, len(pm)), np.int64)
        _chk(lib().ub_percentile_curve_noalloc(self._h, int(which), pm.ctypes.data, len(pm), out.ctypes.data))
        return out

    def slo_attainment(self, which, threshold_us):
        """[R][n] uint32: completed requests with latency <= threshold_us[r][k]."""
        thr = np.ascontiguousarray(threshold_us, np.int64)
        assert thr.ndim == 2 and thr.shape[0] == self.R
        out = np.zeros(thr.shape, np.uint32)
        _chk(lib().ub_slo_attainment(self._h, int(which), thr.ctypes.data, thr.shape[1], out.ctypes.data))
        return out

    def class_percentiles(self, which, len_lo, len_hi, permille):
        """(percentiles [R][n] int64 us, count [R], sum [R]) of TTFT (0) / TTLT (1) / preemption time (2) over the completed
        requests with len_lo <= P + D <= len_hi (ub_class_percentiles)."""
        pm = np.ascontiguousarray(permille, np.uint32)
        out = np.zeros((self.R, len(pm)), np.int64); cnt = np.zeros(self.R, np.uint32); tot = np.zeros(self.R, np.int64)
        hi = min(int(len_hi), 0xFFFFFFFF)
        _chk(lib().ub_class_percentiles(self._h, int(which), int(len_lo), hi, pm.ctypes.data, len(pm), out.ctypes.data,
                                        cnt.ctypes.data, tot.ctypes.data))
        return out, cnt.astype(np.int64), tot

    def jsq_run(self, cluster_size, arrival_us, prompt_tok, decode_tok, n_arr):
        """ub_jsq_run: route the [C][NA] global streams over clusters of `cluster_size` replicas by join-the-shortest-queue
        and run everything to completion; returns assign [C][NA] (replica number within the cluster, -1 = no arrival)."""
        a = np.ascontiguousarray(arrival_us, np.int64); p = np.ascontiguousarray(prompt_tok, np.int32)
        d = np.ascontiguousarray(decode_tok, np.int32); n = np.ascontiguousarray(n_arr, np.uint32)
        assert a.ndim == 2 and a.shape == p.shape == d.shape and n.shape == (a.shape[0],)
        out = np.full(a.shape, -1, np.int32)
        _chk(lib().ub_jsq_run(self._h, int(cluster_size), a.shape[0], a.shape[1], a.ctypes.data, p.ctypes.data,
                              d.ctypes.data, n.ctypes.data, out.ctypes.data))
        return out

    def preempt_time(self):
        """[R][N] int64 microseconds each request spent preempted (rule M15)."""
        out = np.zeros((self.R, self.N), np.int64)
        _chk(lib().ub_preempt_time(self._h, out.ctypes.data, 0))
        return out

    def set_gamma_ada(self, ada: dict, adaptive):
        assert len(adaptive) == self.R
        ub_set_gamma_ada(self._h, ada, adaptive)
        self._levels = int(ada["levels"])

    def gamma_state(self, r=0):
        return ub_gamma_state(self._h, r)

    def gamma_grid(self):
        return ub_gamma_grid(self._h, self._levels)

    def last_step_timing(self):
        return ub_last_step_timing(self._h)

    def stats(self):
        st = (UbReplicaStats * self.R)()
        _chk(lib().ub_stats(self._h, st))
        return [_stats_to_dict(st[r]) for r in range(self.R)]

    def stats_raw(self):
        st = (UbReplicaStats * self.R)()
        _chk(lib().ub_stats(self._h, st))
        return st

    def per_request(self):
        tf = np.empty((self.R, self.N), np.int64); tl = np.empty((self.R, self.N), np.int64)
        ne = np.empty((self.R, self.N), np.uint32); neu = np.empty((self.R, self.N), np.uint32)
        _chk(lib().ub_per_request(self._h, tf.ctypes.data, tl.ctypes.data, ne.ctypes.data, neu.ctypes.data, 0))
        return tf, tl, ne, neu

    def digest(self):
        dg = np.empty(self.R, np.uint64)
        _chk(lib().ub_digest(self._h, dg.ctypes.data))
        return dg

    def boost_lut(self, r=0):
        nb = U32(0)
        _chk(lib().ub_boost_lut(self._h, int(r), None, 0, C.byref(nb)))
        lut = np.empty(nb.value, np.int64)
        _chk(lib().ub_boost_lut(self._h, int(r), lut.ctypes.data, nb.value, C.byref(nb)))
        return lut

    def tbt_hist(self, r=0):
        h = np.empty(UB_TBT_BINS, np.uint32)
        _chk(lib().ub_tbt_hist(self._h, int(r), h.ctypes.data))
        return h

    def debug_state(self, r=0):
        n = U32(0); t = I64(0)
        ids = np.zeros(self.Q, np.uint32); d = np.zeros(self.Q, np.uint32)
        cached = np.zeros(self.Q, np.uint32); flags = np.zeros(self.Q, np.uint32)
        _chk(lib().ub_debug_get_state(self._h, int(r), C.byref(n), ids.ctypes.data, d.ctypes.data,
                                      cached.ctypes.data, flags.ctypes.data, C.byref(t)))
        k = n.value
        return dict(n_active=k, clock_us=t.value, id=ids[:k], d=d[:k], cached=cached[:k], flags=flags[:k])
