// ub_api.cu -- the C-ABI of libuniboost.so (include/uniboost.h): argument checking, device memory,
// the host-side fp64 build of the fixed-point boost table (Eq. 2, rule M4) and the launch loops.
// Every step of the scheduling path itself runs in the kernels of ub_step.cu / ub_aux.cu.
#include "../../include/uniboost.h"
#include "ub_device.cuh"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <map>
#include <new>
#include <tuple>
#include <vector>

using namespace ub;

struct ub_sim {
  ub_config cfg;
  SimDev dev;
  cudaStream_t stream;
  bool have_trace, have_reps;
  // owned device memory
  Rec0* d_E0; Rec1* d_E1; Hdr* d_hdr; Rec0* d_TR; uint32_t* d_nreq; int64_t* d_lut;
  int64_t* d_tpre; int64_t* d_tfirst; int64_t* d_tlast; uint32_t* d_ne; uint32_t* d_neu; uint32_t* d_hist;
  StatsDev* d_stats; unsigned long long* d_word;
  uint32_t* d_list; uint32_t* d_count;   // work lists [4][R]; counts [8] ([5] = finished replicas)
  uint32_t* d_live; uint32_t* d_livecnt; // ub_run's tail: the unfinished replicas of each part of a round, compacted
  bool use_list; uint32_t livecnt[ub::kMaxSplit];
  uint32_t* d_drift; uint32_t* d_drift_live; uint32_t ndrift, drift_livecnt;   // the drift group (SRPT / LAS replicas): launched
                                                                            // beside the parts, from its own list (ub_stream.cu)
  int64_t* d_ada_ring; AdaState* d_ada_state; int64_t* d_ada_grid;   // gamma-Ada (M13), null when off
  std::vector<int64_t> h_ada_grid;
  uint2* d_evbuf;                        // per-iteration event scratch [R][min(M,Q)]
  unsigned long long* h_word;            // pinned
  std::vector<uint32_t> h_nreq, h_maxsig;
  std::vector<ub_replica> h_reps;
  std::vector<int64_t> h_lut;            // all tables back to back
  std::vector<uint32_t> h_lut_off, h_lut_nb;
  cudaEvent_t ev0, ev1;
  cudaStream_t aux[ub::kMaxSplit - 1]; cudaEvent_t ev_fork, ev_join[ub::kMaxSplit - 1];   // extra streams: the parts of a round overlap their tails
  uint32_t nsplit, ndsplit;     // parts of the main group / of the drift group (together <= kMaxSplit)
  uint32_t round_no;            // launches alternate between two ticket counters
  // ub_run replays a captured CUDA graph of kGraphRounds rounds while the configuration of a round (parts, lists,
  // iterations per launch) stays the same: small jobs are bound by launch latency
  cudaGraphExec_t graph; uint64_t graph_key; uint32_t graph_launches;
  cudaStream_t gstream; cudaEvent_t ev_g;   // the graph's origin stream when the caller's is the default stream (which cannot be captured)
  float last_ms; uint32_t last_launches;
};

#define CK(x) do { if ((x) != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; } } while (0)

static int compact_live(ub_sim* s, uint64_t* live, bool any_state);
static int set_dev(const ub_sim* s) { return cudaSetDevice(s->cfg.device) == cudaSuccess ? UB_OK : UB_ECUDA; }
// (a captured graph holds kernel arguments by value: device pointers, list lengths)
static void drop_graph(ub_sim* s) { if (s->graph) { cudaGraphExecDestroy(s->graph); s->graph = nullptr; } s->graph_key = 0; }

const char* ub_strerror(int e) {
  switch (e) {
    case UB_OK: return "ok";
    case UB_EINVAL: return "invalid argument";
    case UB_ENOMEM: return "out of memory";
    case UB_ECUDA: return "CUDA error";
    case UB_ESTATE: return "wrong call order";
    case UB_EUNSORTED: return "arrivals not non-decreasing";
    case UB_EINFEASIBLE: return "request does not fit the KV capacity or has P<1 or D<1";
    case UB_ELIVELOCK: return "max_iters reached before all replicas finished";
    case UB_ETOOBIG: return "size beyond the static scratch of a no-allocation entry point (UB_NOALLOC_CURVE_MAX values)";
    default: return "unknown";
  }
}

template <class T> static int dmalloc(T** p, size_t count) {
  *p = nullptr;
  cudaError_t e = cudaMalloc((void**)p, count ? count * sizeof(T) : sizeof(T));
  if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return UB_ENOMEM; }
  return e == cudaSuccess ? UB_OK : UB_ECUDA;
}

int ub_create(const ub_config* c, ub_sim** out) {
  if (!c || !out) return UB_EINVAL;
  *out = nullptr;
  if (c->struct_size != sizeof(ub_config) || c->abi_version != UB_ABI_VERSION) return UB_EINVAL;
  if (c->n_replicas < 1 || c->n_traces < 1 || c->max_requests < 1 || c->max_requests >= (1u << 29) || c->queue_cap < 1 ||
      c->queue_cap > UB_MAX_QUEUE || c->kv_blocks < 1 || c->block_tokens < 1 || c->max_batch < 1 ||
      c->chunk_tokens < 1 || c->chunk_tokens > 65535 || c->token_budget < 1 || c->token_budget > 65535 ||
      c->c0_us < 0 || c->c_prefill_tok_us < 0 || c->c_decode_seq_us < 0 || c->preempt_mode > 2 ||
      c->bin_tokens < 1 || c->tok_us < 1 || c->device < 0)
    return UB_EINVAL;
  // value ranges that keep every device quantity inside u32 / the flags word
  if ((uint64_t)c->kv_blocks * c->block_tokens >= (1ull << 27) || c->bin_tokens >= (1u << 27) ||
      c->c0_us > (1ll << 40) || c->c_prefill_tok_us > (1ll << 20) || c->c_decode_seq_us > (1ll << 30))
    return UB_EINVAL;
  if (cudaSetDevice(c->device) != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
  ub_sim* s = new (std::nothrow) ub_sim();
  if (!s) return UB_ENOMEM;
  s->cfg = *c;
  s->stream = (cudaStream_t)c->stream;
  s->have_trace = s->have_reps = false;
  s->d_TR = nullptr; s->d_lut = nullptr;
  s->last_ms = 0.f; s->last_launches = 0;
  s->use_list = false; s->ndrift = 0; s->drift_livecnt = 0;
  s->graph = nullptr; s->graph_key = 0; s->graph_launches = 0;
  // parts of a round (each on a stream of its own; together with the drift group's at most kMaxSplit).  Measured: config 5
  // (65536 replicas) 2 parts 5.9e10, 4 parts 5.5e10 request-steps/s; config 3 (4096 replicas, whole job) 1 part 1.18e10,
  // 2 parts 1.31e10, 4 parts 1.22e10 at one iteration per launch and 2.61e10 / 3.29e10 / 3.34e10 at 64; config 2 (3072
  // replicas) is 3 % slower in two parts than in one
  s->nsplit = c->n_replicas >= 4096 ? 2 : 1;
  s->ndsplit = 1;
  const size_t R = c->n_replicas, Q = c->queue_cap, N = c->max_requests, NT = c->n_traces;
  int rc = UB_OK;
  if ((rc = dmalloc(&s->d_E0, R * Q + kWindowPad)) || (rc = dmalloc(&s->d_E1, R * Q + kWindowPad)) || (rc = dmalloc(&s->d_hdr, R)) ||
      (rc = dmalloc(&s->d_nreq, NT)) || (rc = dmalloc(&s->d_tfirst, R * N)) ||
      (rc = dmalloc(&s->d_tlast, R * N)) || (rc = dmalloc(&s->d_tpre, R * N)) || (rc = dmalloc(&s->d_ne, R * N)) || (rc = dmalloc(&s->d_neu, R * N)) ||
      (rc = dmalloc(&s->d_hist, R * (size_t)kTbtBins)) || (rc = dmalloc(&s->d_stats, R)) ||
      (rc = dmalloc(&s->d_word, 2)) || (rc = dmalloc(&s->d_live, R)) || (rc = dmalloc(&s->d_livecnt, kMaxSplit + 1)) ||
      (rc = dmalloc(&s->d_drift, R)) || (rc = dmalloc(&s->d_drift_live, R)) || (rc = dmalloc(&s->d_list, 4 * kMaxSplit * R)) || (rc = dmalloc(&s->d_count, 8 * kMaxSplit)) ||
      (rc = dmalloc(&s->d_evbuf, R * (size_t)(c->max_batch < c->queue_cap ? c->max_batch : c->queue_cap)))) {
    ub_destroy(s);
    return rc;
  }
  if (cudaMallocHost((void**)&s->h_word, (3 + kMaxSplit) * sizeof(unsigned long long)) != cudaSuccess ||
      cudaEventCreate(&s->ev0) != cudaSuccess || cudaEventCreate(&s->ev1) != cudaSuccess ||
      cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      step_configure(c->queue_cap) != 0) {
    cudaGetLastError();
    ub_destroy(s);
    return UB_ECUDA;
  }
  bool aux_ok = cudaStreamCreateWithFlags(&s->gstream, cudaStreamNonBlocking) == cudaSuccess &&
                cudaEventCreateWithFlags(&s->ev_g, cudaEventDisableTiming) == cudaSuccess;
  for (uint32_t i = 0; i + 1 < kMaxSplit; i++)
    aux_ok = aux_ok && cudaStreamCreateWithFlags(&s->aux[i], cudaStreamNonBlocking) == cudaSuccess &&
             cudaEventCreateWithFlags(&s->ev_join[i], cudaEventDisableTiming) == cudaSuccess;
  if (!aux_ok) {
    cudaGetLastError();
    ub_destroy(s);
    return UB_ECUDA;
  }
  SimDev& d = s->dev;
  memset(&d, 0, sizeof(d));
  d.R = c->n_replicas; d.NT = c->n_traces; d.N = c->max_requests; d.Q = c->queue_cap;
  d.blk_shift = 32;
  for (uint32_t b = 0; b < 32; b++) if ((1u << b) == c->block_tokens) d.blk_shift = b;
  d.B = c->kv_blocks; d.blk = c->block_tokens; d.M = c->max_batch; d.c = c->chunk_tokens; d.T = c->token_budget;
  d.preempt_mode = c->preempt_mode; d.swap_ns = c->swap_ns_per_block; d.swap_pool = c->swap_pool_blocks;
  d.k = c->bin_tokens; d.c0 = c->c0_us; d.c_pf = c->c_prefill_tok_us; d.c_dec = c->c_decode_seq_us;
  d.E0 = s->d_E0; d.E1 = s->d_E1; d.hdr = s->d_hdr; d.n_req = s->d_nreq;
  d.evbuf = s->d_evbuf; d.evcap = c->max_batch < c->queue_cap ? c->max_batch : c->queue_cap;
  d.t_first = s->d_tfirst; d.t_last = s->d_tlast; d.t_pre = s->d_tpre; d.n_evict = s->d_ne; d.n_evict_unf = s->d_neu; d.hist = s->d_hist;
  *out = s;
  return UB_OK;
}

void ub_destroy(ub_sim* s) {
  if (!s) return;
  cudaSetDevice(s->cfg.device);
  cudaStreamSynchronize(s->stream);
  cudaFree(s->d_E0); cudaFree(s->d_E1); cudaFree(s->d_hdr); cudaFree(s->d_TR);
  cudaFree(s->d_nreq); cudaFree(s->d_lut); cudaFree(s->d_tfirst); cudaFree(s->d_tlast); cudaFree(s->d_tpre); cudaFree(s->d_ne);
  cudaFree(s->d_neu); cudaFree(s->d_hist); cudaFree(s->d_stats); cudaFree(s->d_word);
  cudaFree(s->d_list); cudaFree(s->d_count); cudaFree(s->d_evbuf); cudaFree(s->d_live); cudaFree(s->d_livecnt); cudaFree(s->d_drift); cudaFree(s->d_drift_live);
  cudaFree(s->d_ada_ring); cudaFree(s->d_ada_state); cudaFree(s->d_ada_grid);
  if (s->graph) cudaGraphExecDestroy(s->graph);
  if (s->gstream) cudaStreamDestroy(s->gstream);
  if (s->ev_g) cudaEventDestroy(s->ev_g);
  if (s->h_word) cudaFreeHost(s->h_word);
  if (s->ev0) cudaEventDestroy(s->ev0);
  if (s->ev1) cudaEventDestroy(s->ev1);
  if (s->ev_fork) cudaEventDestroy(s->ev_fork);
  for (uint32_t i = 0; i + 1 < kMaxSplit; i++) {
    if (s->ev_join[i]) cudaEventDestroy(s->ev_join[i]);
    if (s->aux[i]) cudaStreamDestroy(s->aux[i]);
  }
  cudaGetLastError();
  delete s;
}

static int load_trace_impl(ub_sim* s, const int64_t* a, const int32_t* p, const int32_t* d, const int32_t* hit,
                           const uint32_t* n_req, int on_device) {
  if (!s || !a || !p || !d || !n_req) return UB_EINVAL;
  if (set_dev(s)) return UB_ECUDA;
  const size_t NT = s->cfg.n_traces, N = s->cfg.max_requests, tot = NT * N;
  s->h_nreq.resize(NT);
  if (on_device) CK(cudaMemcpy(s->h_nreq.data(), n_req, NT * 4, cudaMemcpyDeviceToHost));
  else memcpy(s->h_nreq.data(), n_req, NT * 4);
  for (size_t t = 0; t < NT; t++) if (s->h_nreq[t] > N) return UB_EINVAL;
  s->have_trace = false; s->have_reps = false;
  if (!s->d_TR) { int rc = dmalloc(&s->d_TR, tot); if (rc) return rc; }
  CK(cudaMemcpyAsync(s->d_nreq, s->h_nreq.data(), NT * 4, cudaMemcpyHostToDevice, s->stream));
  int64_t* da = nullptr; int32_t* dp = nullptr; int32_t* dd = nullptr; int32_t* dh = nullptr;
  const int64_t* ua = a; const int32_t* up = p; const int32_t* ud = d; const int32_t* uh = hit;
  int rc = UB_OK;
  if (!on_device) {
    if ((rc = dmalloc(&da, tot)) || (rc = dmalloc(&dp, tot)) || (rc = dmalloc(&dd, tot)) || (hit && (rc = dmalloc(&dh, tot)))) {
      cudaFree(da); cudaFree(dp); cudaFree(dd); cudaFree(dh); return rc;
    }
    if (cudaMemcpyAsync(da, a, tot * 8, cudaMemcpyHostToDevice, s->stream) != cudaSuccess ||
        cudaMemcpyAsync(dp, p, tot * 4, cudaMemcpyHostToDevice, s->stream) != cudaSuccess ||
        cudaMemcpyAsync(dd, d, tot * 4, cudaMemcpyHostToDevice, s->stream) != cudaSuccess ||
        (hit && cudaMemcpyAsync(dh, hit, tot * 4, cudaMemcpyHostToDevice, s->stream) != cudaSuccess)) {
      cudaGetLastError(); cudaFree(da); cudaFree(dp); cudaFree(dd); cudaFree(dh); return UB_ECUDA;
    }
    ua = da; up = dp; ud = dd; uh = hit ? dh : nullptr;
  }
  s->h_word[0] = ~0ull;
  cudaMemcpyAsync(s->d_word, s->h_word, 8, cudaMemcpyHostToDevice, s->stream);
  launch_pack_validate(ua, up, ud, uh, s->d_nreq, (uint32_t)NT, (uint32_t)N, s->cfg.kv_blocks, s->cfg.block_tokens,
                       s->d_TR, reinterpret_cast<int*>(s->d_word), s->stream);
  cudaMemcpyAsync(s->h_word, s->d_word, 8, cudaMemcpyDeviceToHost, s->stream);
  cudaError_t e = cudaStreamSynchronize(s->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaFree(da); cudaFree(dp); cudaFree(dd); cudaFree(dh);
  if (e != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
  if (s->h_word[0] != ~0ull) {
    const int kind = (int)(s->h_word[0] & 3ull);
    return kind == 0 ? UB_EINVAL : (kind == 1 ? UB_EUNSORTED : UB_EINFEASIBLE);
  }
  s->dev.TR = s->d_TR;
  s->have_trace = true;
  return UB_OK;
}

int ub_load_trace(ub_sim* s, const int64_t* a, const int32_t* p, const int32_t* d, const uint32_t* n_req, int on_device) {
  return load_trace_impl(s, a, p, d, nullptr, n_req, on_device);
}
int ub_load_trace_prefix(ub_sim* s, const int64_t* a, const int32_t* p, const int32_t* d, const int32_t* hit,
                         const uint32_t* n_req, int on_device) {
  if (!hit) return UB_EINVAL;
  return load_trace_impl(s, a, p, d, hit, n_req, on_device);
}

// Eq. 2 / BOOST in fixed point, rule M4:
//   x = w_hat * tok_us * 1e-6 s;  b = (1/gamma) log(1/(1 - e^{-gamma x})) = -log(-expm1(-gamma x)) / gamma;
//   table value = min(2^60, floor(b * 1e6 + 0.5)) us;  x == 0 -> 2^60;  gamma == +inf -> 0.
static int64_t boost_table_entry(double gamma, double w_hat, uint32_t tok_us) {
  if (isinf(gamma) && gamma > 0) return 0;
  const double x = w_hat * (double)tok_us * 1e-6;
  if (!(x > 0.0)) return kBoostMax;
  const double b = -log(-expm1(-gamma * x)) / gamma;
  const double v = floor(b * 1e6 + 0.5);
  if (!(v > 0.0)) return 0;
  if (v >= (double)kBoostMax) return kBoostMax;
  return (int64_t)v;
}

// max over a trace of P + D (size of the EXACT-quantiser table), computed on the device copy
__global__ void k_max_sig(const Rec0* TR, const uint32_t* n_req, uint32_t NT, uint32_t N, uint32_t* out) {
  const uint32_t tr = blockIdx.x;
  uint32_t m = 0;
  for (uint32_t i = threadIdx.x; i < n_req[tr]; i += blockDim.x) {
    const Rec0 q = TR[(size_t)tr * N + i];
    m = max(m, q.P + q.D);
  }
  m = __reduce_max_sync(0xffffffffu, m);
  if ((threadIdx.x & 31) == 0) atomicMax(out + tr, m);
}

int ub_set_replicas(ub_sim* s, const ub_replica* reps) {
  if (!s || !reps) return UB_EINVAL;
  if (!s->have_trace) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const ub_config& c = s->cfg;
  const size_t R = c.n_replicas, N = c.max_requests;
  bool any_exact = false;
  for (size_t r = 0; r < R; r++) {
    const ub_replica& q = reps[r];
    if (q.trace_id >= c.n_traces || q.policy > 7 || q.signal_mode > 2 || q.quant_mode > 1 || q.guard > 1 ||
        q.hysteresis_us < 0 || q.hysteresis_us > (1ll << 60))
      return UB_EINVAL;
    if ((q.policy == UB_BOOST || q.policy == UB_DISTBOOST) && !(q.gamma > 0.0)) return UB_EINVAL;     // also rejects NaN
    any_exact |= (q.quant_mode == UB_Q_EXACT);
  }
  s->have_reps = false;
  s->use_list = false;                             // (a rewound run: every replica is live again)
  drop_graph(s);
  cudaFree(s->d_ada_ring); cudaFree(s->d_ada_state); cudaFree(s->d_ada_grid);        // adaptation is set per replica table
  s->d_ada_ring = nullptr; s->d_ada_state = nullptr; s->d_ada_grid = nullptr; s->h_ada_grid.clear();
  s->dev.ada_ring = nullptr; s->dev.ada_state = nullptr; s->dev.ada_grid = nullptr;
  if (any_exact) {
    uint32_t* d_ms = nullptr;
    int rc = dmalloc(&d_ms, c.n_traces); if (rc) return rc;
    cudaMemsetAsync(d_ms, 0, c.n_traces * 4, s->stream);
    k_max_sig<<<c.n_traces, 128, 0, s->stream>>>(s->d_TR, s->d_nreq, c.n_traces, c.max_requests, d_ms);
    s->h_maxsig.resize(c.n_traces);
    cudaError_t e = cudaMemcpyAsync(s->h_maxsig.data(), d_ms, c.n_traces * 4, cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    cudaFree(d_ms);
    if (e != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
  }
  // boost tables, one per distinct (gamma, quantiser, length); non-BOOST policies never read one
  s->h_reps.assign(reps, reps + R);
  s->h_lut.clear(); s->h_lut_off.assign(R, 0); s->h_lut_nb.assign(R, 0);
  std::map<std::tuple<uint64_t, uint32_t, uint32_t>, uint32_t> seen;
  std::vector<RepPar> par(R);
  for (size_t r = 0; r < R; r++) {
    const ub_replica& q = reps[r];
    const uint32_t nb = (q.quant_mode == UB_Q_EXACT) ? s->h_maxsig[q.trace_id] + 1u : 64u;
    uint32_t off = 0;
    if (q.policy == UB_BOOST || q.policy == UB_DISTBOOST) {
      uint64_t gb; memcpy(&gb, &q.gamma, 8);
      auto key = std::make_tuple(gb, (uint32_t)q.quant_mode, nb);
      auto it = seen.find(key);
      if (it != seen.end()) off = it->second;
      else {
        if (s->h_lut.size() + nb >= (1ull << 32)) return UB_ENOMEM;
        off = (uint32_t)s->h_lut.size();
        seen.emplace(key, off);
        for (uint32_t b = 0; b < nb; b++) {
          const double w_hat = (q.quant_mode == UB_Q_EXACT) ? (double)b : ldexp((double)c.bin_tokens, (int)b);
          s->h_lut.push_back(boost_table_entry(q.gamma, w_hat, c.tok_us));
        }
      }
    }
    s->h_lut_off[r] = off; s->h_lut_nb[r] = nb;
    RepPar& p = par[r];
    p.delta = q.hysteresis_us; p.trace_id = q.trace_id; p.lut_off = off; p.lut_nb = nb;
    p.policy = q.policy; p.guard = q.guard; p.signal_mode = q.signal_mode; p.quant_mode = q.quant_mode;
    p.pad[0] = p.pad[1] = 0;
  }
  {
    bool all = s->dev.blk_shift < 32u;
    for (size_t r = 0; r < R && all; r++)
      all = reps[r].policy < UB_DISTBOOST && reps[r].signal_mode == 0 && reps[r].quant_mode == 0;
    s->dev.all_stream = all ? 1u : 0u;
    bool bg = s->dev.blk_shift < 32u;
    for (size_t r = 0; r < R && bg; r++)
      bg = reps[r].policy == UB_BOOST && reps[r].guard != 0 && reps[r].signal_mode == 0 && reps[r].quant_mode == 0;
    s->dev.all_boost_guard = bg ? 1u : 0u;
  }
  {
    // the drift group: replicas whose keys move with every token (SRPT, LAS) and that the streaming kernel covers
    std::vector<uint32_t> dl;
    if (s->dev.blk_shift < 32u)
      for (size_t r = 0; r < R; r++)
        if ((reps[r].policy == UB_SRPT || reps[r].policy == UB_LAS) && reps[r].signal_mode == 0 && reps[r].quant_mode == 0)
          dl.push_back((uint32_t)r);
    s->ndrift = (uint32_t)dl.size();
    if (!dl.empty()) CK(cudaMemcpyAsync(s->d_drift, dl.data(), dl.size() * 4, cudaMemcpyHostToDevice, s->stream));
    CK(cudaStreamSynchronize(s->stream));                             // (dl is a local)
  }
  cudaFree(s->d_lut); s->d_lut = nullptr;
  int rc = dmalloc(&s->d_lut, s->h_lut.size()); if (rc) return rc;
  if (!s->h_lut.empty())
    CK(cudaMemcpyAsync(s->d_lut, s->h_lut.data(), s->h_lut.size() * 8, cudaMemcpyHostToDevice, s->stream));
  CK(cudaMemcpy2DAsync(&s->d_hdr[0].par, sizeof(Hdr), par.data(), sizeof(RepPar), sizeof(RepPar), R,
                       cudaMemcpyHostToDevice, s->stream));       // (parameters live inside the replica headers)
  s->dev.lut = s->d_lut;
  // reset the run state
  CK(cudaMemsetAsync(s->d_tfirst, 0xFF, R * N * 8, s->stream));     // -1
  CK(cudaMemsetAsync(s->d_tlast, 0xFF, R * N * 8, s->stream));
  CK(cudaMemsetAsync(s->d_tpre, 0, R * N * 8, s->stream));
  CK(cudaMemsetAsync(s->d_ne, 0, R * N * 4, s->stream));
  CK(cudaMemsetAsync(s->d_neu, 0, R * N * 4, s->stream));
  CK(cudaMemsetAsync(s->d_hist, 0, R * (size_t)kTbtBins * 4, s->stream));
  launch_reset(s->dev, s->d_list, s->d_count, s->stream);
  CK(cudaStreamSynchronize(s->stream));
  CK(cudaGetLastError());
  s->have_reps = true;
  if (s->ndrift) { uint64_t all = 0; return compact_live(s, &all, true); }      // main group and drift group each from a list
  return UB_OK;
}

// A round = one launch_step over all replicas.  With many replicas it is issued as nsplit parts on as many streams
// (the caller's and internal ones, fork / join by events): replicas are independent, so while the last warps of one
// part finish, the other parts' CTAs already fill the freed SMs.
// tlimit (device, [R], nullable): a fenced run (JSQ router, rule M18) -- one launch in which every replica executes the
// iterations that start before its limit.
// A part of a round: positions [rb, re) of the replicas themselves or of a list, its stream and its set of work lists.
struct RoundPart { uint32_t rb, re; const uint32_t* list; bool drift; cudaStream_t st; uint32_t slot; };

static uint32_t round_parts(ub_sim* s, bool ada, RoundPart* P) {
  const uint32_t R = s->cfg.n_replicas, ns = s->nsplit;
  const uint32_t part = ns > 1 ? (R / ns + 3) / 4 * 4 : R;
  const bool lst = s->use_list && !ada;
  uint32_t np = 0;
  for (uint32_t i = 0; i < ns; i++) {
    const uint32_t rb = i * part < R ? i * part : R, re = (i + 1 == ns) ? R : ((i + 1) * part < R ? (i + 1) * part : R);
    RoundPart q;
    q.rb = rb; q.re = re; q.list = nullptr; q.drift = false; q.slot = i; q.st = i ? s->aux[i - 1] : s->stream;
    if (lst) { q.list = s->d_live + rb; q.rb = 0; q.re = s->livecnt[i]; }
    if (q.re > q.rb) P[np++] = q;                  // (a part whose replicas have all finished is left out)
  }
  // the drift group (SRPT / LAS replicas) is one more independent set of replicas: its launches go to streams of their
  // own beside the main parts, with the sets of work lists and counters behind theirs
  const uint32_t nd = ada ? 0u : (lst ? s->drift_livecnt : s->ndrift);
  if (nd) {
    const uint32_t nds = s->ndsplit, dpart = (nd + nds - 1) / nds;
    for (uint32_t j = 0; j < nds && j * dpart < nd; j++) {
      RoundPart q;
      q.rb = j * dpart; q.re = (j + 1) * dpart < nd ? (j + 1) * dpart : nd;
      q.list = lst ? s->d_drift_live : s->d_drift; q.drift = true; q.slot = ns + j; q.st = s->aux[ns + j - 1];
      P[np++] = q;
    }
  }
  return np;
}

static int issue_steps(ub_sim* s, uint64_t n_iters, uint32_t* launches, const int64_t* tlimit = nullptr) {
  const bool ada = s->d_ada_ring != nullptr;         // UPDATEGAMMA opens every iteration: one iteration per launch
  constexpr uint32_t kFenced = 1u << 20;             // iterations a fenced launch may run (the fence ends it long before)
  if (tlimit) n_iters = kFenced;
  const uint32_t ipl = tlimit ? kFenced : ((!ada && s->cfg.iters_per_launch > 1) ? s->cfg.iters_per_launch : 1);
  const size_t R = s->cfg.n_replicas;
  RoundPart P[kMaxSplit];
  const uint32_t np = round_parts(s, ada, P);
  uint32_t nl = 0;
  bool forked = false;
  for (uint32_t i = 0; i < np; i++) forked = forked || P[i].st != s->stream;
  if (forked) {
    CK(cudaEventRecord(s->ev_fork, s->stream));
    for (uint32_t i = 0; i < np; i++) if (P[i].st != s->stream) CK(cudaStreamWaitEvent(P[i].st, s->ev_fork, 0));
  }
  while (n_iters > 0) {
    const uint32_t k = n_iters < ipl ? (uint32_t)n_iters : ipl;
    n_iters -= k;
    for (uint32_t i = np; i-- > 0;) {                // (the drift group first: its replica-steps are the longer ones)
      const RoundPart& q = P[i];
      uint32_t* list = s->d_list + 4 * R * q.slot;
      uint32_t* count = s->d_count + 8 * q.slot;
      if (ada) launch_gamma_ada(s->dev, q.rb, q.re, q.st);
      launch_step(s->dev, list, count, k, q.rb, q.re, s->round_no, q.list, q.drift, tlimit, q.st);
      // what k_stream queued for the team kernels runs at the end of the call (all owed iterations at once); with
      // gamma-Ada after every round, because UPDATEGAMMA sits between the iterations
      if (ada || n_iters == 0) flush_slow(s->dev, list, count, q.rb, q.re, tlimit, q.st);
    }
    nl++; s->round_no++;
  }
  if (forked) {
    for (uint32_t i = 0; i < np; i++) if (P[i].st != s->stream) {
      CK(cudaEventRecord(s->ev_join[P[i].slot - 1], P[i].st));
      CK(cudaStreamWaitEvent(s->stream, s->ev_join[P[i].slot - 1], 0));
    }
  }
  *launches = nl;
  return cudaGetLastError() == cudaSuccess ? UB_OK : UB_ECUDA;
}

// ub_run's rounds through a CUDA graph: kGraphRounds rounds (their launches on all the part streams, the fork / join
// events and the hand-over flush behind them) are captured once from issue_steps() itself and replayed; the graph is
// kept while the round configuration -- list mode, list lengths, iterations per launch -- is unchanged.  An even
// number of rounds, so the alternation of the two ticket counters is the same in every replay.
constexpr uint32_t kGraphRounds = 64;
static int issue_steps_graphed(ub_sim* s, uint64_t n_iters, uint32_t* launches) {
  const uint32_t ipl = s->cfg.iters_per_launch > 1 ? s->cfg.iters_per_launch : 1;
  const uint64_t per = (uint64_t)kGraphRounds * ipl;
  if (s->d_ada_ring || n_iters < per || n_iters % per || (s->round_no & 1u)) return issue_steps(s, n_iters, launches);
  uint64_t key = 0x9E3779B97F4A7C15ull ^ ipl;
  auto mix = [&](uint64_t v) { key = (key ^ v) * 0xBF58476D1CE4E5B9ull; key ^= key >> 29; };
  mix(s->use_list ? 1u : 0u); mix(s->ndrift); mix(s->drift_livecnt);
  for (uint32_t i = 0; i < s->nsplit; i++) mix(s->use_list ? s->livecnt[i] : 0u);
  key |= 1ull;
  // the default streams cannot be captured: the graph then starts from a stream of the library's, ordered behind the
  // caller's stream and in front of it again by events
  cudaStream_t user = s->stream;
  const bool own = user == nullptr || user == cudaStreamLegacy || user == cudaStreamPerThread;
  struct Swap { ub_sim* s; cudaStream_t user; ~Swap() { s->stream = user; } } swap{s, user};
  if (own) {
    CK(cudaEventRecord(s->ev_g, user));
    CK(cudaStreamWaitEvent(s->gstream, s->ev_g, 0));
    s->stream = s->gstream;
  }
  if (!s->graph || s->graph_key != key) {
    if (s->graph) { cudaGraphExecDestroy(s->graph); s->graph = nullptr; }
    cudaGraph_t g = nullptr;
    const uint32_t round0 = s->round_no;
    if (cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
      cudaGetLastError(); s->stream = user;
      return issue_steps(s, n_iters, launches);
    }
    uint32_t nl = 0;
    const int rc = issue_steps(s, per, &nl);
    const cudaError_t e = cudaStreamEndCapture(s->stream, &g);
    s->round_no = round0;
    if (rc != UB_OK || e != cudaSuccess || !g || cudaGraphInstantiate(&s->graph, g, 0) != cudaSuccess) {
      cudaGetLastError();
      if (g) cudaGraphDestroy(g);
      s->graph = nullptr; s->stream = user;
      return issue_steps(s, n_iters, launches);
    }
    cudaGraphDestroy(g);
    s->graph_key = key; s->graph_launches = nl;
  }
  const uint64_t reps = n_iters / per;
  for (uint64_t i = 0; i < reps; i++) CK(cudaGraphLaunch(s->graph, s->stream));
  s->round_no += (uint32_t)(reps * kGraphRounds);
  *launches = (uint32_t)(reps * s->graph_launches);
  if (own) {
    CK(cudaEventRecord(s->ev_g, s->gstream));
    CK(cudaStreamWaitEvent(user, s->ev_g, 0));
  }
  return UB_OK;
}

static int read_live(ub_sim* s, uint64_t* live) {
  launch_count_live(s->d_count, s->cfg.n_replicas, s->d_word, s->stream);
  CK(cudaMemcpyAsync(s->h_word, s->d_word, 8, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  CK(cudaGetLastError());
  *live = s->h_word[0];
  return UB_OK;
}

int ub_step(ub_sim* s, uint32_t n_iters, uint64_t* live) {
  if (!s) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  CK(cudaEventRecord(s->ev0, s->stream));
  uint32_t nl = 0;
  int rc = issue_steps(s, n_iters, &nl);
  CK(cudaEventRecord(s->ev1, s->stream));
  s->last_launches = nl; s->last_ms = -1.f;
  if (rc) return rc;
  if (live) return read_live(s, live);
  return UB_OK;
}

// The unfinished replicas of every part of a round, compacted on the device; *live = how many.  From then on the
// streaming kernel visits only these (a finished replica never comes back, so the list stays a superset of the live
// replicas until it is rebuilt).  any_state: finished or not -- the lists then only separate the main group from the
// drift group (a job that has both starts with them: a main-group warp that only skips a drift replica would still
// hold its place on the SM beside the drift group's launch).
static int compact_live(ub_sim* s, uint64_t* live, bool any_state) {
  const uint32_t R = s->cfg.n_replicas, ns = s->nsplit;
  const uint32_t part = ns > 1 ? (R / ns + 3) / 4 * 4 : R;
  for (uint32_t i = 0; i < ns; i++) {
    const uint32_t rb = i * part, re = (i + 1 == ns) ? R : (i + 1) * part;
    launch_compact_live(s->dev, rb, re, nullptr, false, any_state, s->d_live + rb, s->d_livecnt + i, s->stream);
  }
  launch_compact_live(s->dev, 0, s->ndrift, s->d_drift, true, any_state, s->d_drift_live, s->d_livecnt + ns, s->stream);   // (ns < kMaxSplit)
  uint32_t* hc = reinterpret_cast<uint32_t*>(s->h_word + 2);
  CK(cudaMemcpyAsync(hc, s->d_livecnt, (ns + 1) * sizeof(uint32_t), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  CK(cudaGetLastError());
  uint64_t tot = 0;
  for (uint32_t i = 0; i < ns; i++) { s->livecnt[i] = hc[i]; tot += hc[i]; }
  s->drift_livecnt = hc[ns]; tot += hc[ns];
  s->use_list = true;
  *live = tot;
  return UB_OK;
}

int ub_run(ub_sim* s, uint64_t max_iters, uint64_t* iters_done) {
  if (!s) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const uint64_t R = s->cfg.n_replicas;
  const bool ada = s->d_ada_ring != nullptr;
  uint64_t done = 0, live = 1;
  uint32_t total_launches = 0;
  float total_ms = 0.f;
  int rc = read_live(s, &live);
  if (rc) return rc;
  // While every replica is live the liveness is polled at growing intervals (256 .. 4096 iterations).  Once replicas
  // start to finish, every poll (512 iterations apart: the overshoot behind the last completion stays small)
  // compacts the unfinished ones into a list, and the streaming kernel visits only those: the tail of a run, in which
  // few replicas are still draining their queues, no longer pays for the headers of all the finished ones.
  uint64_t chunk = 256;
  while (live > 0 && done < max_iters) {
    const uint64_t k = (max_iters - done) < chunk ? (max_iters - done) : chunk;
    uint32_t nl = 0;
    CK(cudaEventRecord(s->ev0, s->stream));
    rc = done ? issue_steps_graphed(s, k, &nl) : issue_steps(s, k, &nl);     // (the first rounds also set the kernels up)
    CK(cudaEventRecord(s->ev1, s->stream));
    if (rc) return rc;
    done += k; total_launches += nl;
    if ((rc = read_live(s, &live))) return rc;
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, s->ev0, s->ev1));
    total_ms += ms;
    if (live == R) { if (chunk < 4096) chunk *= 2; }
    else {
      chunk = 512;
      if (!ada && live > 0 && live * 8 < R * 7 && (rc = compact_live(s, &live, false))) return rc;
    }
  }
  s->last_ms = total_ms; s->last_launches = total_launches;
  if (iters_done) *iters_done = done;
  return live > 0 ? UB_ELIVELOCK : UB_OK;
}

int ub_last_step_timing(ub_sim* s, float* ms, uint32_t* launches) {
  if (!s) return UB_EINVAL;
  if (set_dev(s)) return UB_ECUDA;
  if (s->last_ms < 0.f) {
    CK(cudaEventSynchronize(s->ev1));
    float v = 0.f;
    CK(cudaEventElapsedTime(&v, s->ev0, s->ev1));
    s->last_ms = v;
  }
  if (ms) *ms = s->last_ms;
  if (launches) *launches = s->last_launches;
  return UB_OK;
}

// ---------------------------------------------------------------------------------------------- gamma-Ada (M13)
// Grid and per-level boost tables are built here on the host in fp64 (as M4), independently of the oracle.
static double ada_grid_gamma(const ub_gamma_ada* g, uint32_t j) {
  return g->gamma_min * pow(g->gamma_max / g->gamma_min, (double)j / (double)(g->levels - 1));
}

int ub_set_gamma_ada(ub_sim* s, const ub_gamma_ada* g, const uint8_t* adaptive) {
  if (!s || !g || !adaptive) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (s->d_ada_ring) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const ub_config& c = s->cfg;
  if (g->struct_size != sizeof(ub_gamma_ada) || g->window < c.max_batch || g->window > 1024 || g->min_samples < 2 ||
      g->beta_shift > 16 || g->levels < 2 || g->levels > 64 || !(g->gamma_min > 0.0) ||
      !(g->gamma_max > g->gamma_min) || g->gamma_max > 1e6 || g->eps_us < 1)
    return UB_EINVAL;
  const size_t R = c.n_replicas;
  for (size_t r = 0; r < R; r++)
    if (adaptive[r] && (s->h_reps[r].policy != UB_BOOST || s->h_reps[r].quant_mode != UB_Q_GEOMETRIC ||
                        isinf(s->h_reps[r].gamma)))
      return UB_EINVAL;
  // a run that already started cannot switch
  {
    std::vector<Hdr> hd(R);
    CK(cudaMemcpyAsync(hd.data(), s->d_hdr, R * sizeof(Hdr), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    for (size_t r = 0; r < R; r++) if (hd[r].iterations != 0) return UB_ESTATE;
  }
  std::vector<int64_t> grid(g->levels);
  for (uint32_t j = 0; j < g->levels; j++) grid[j] = (int64_t)floor(ada_grid_gamma(g, j) * 1e6 + 0.5);
  // Everything is built in temporaries and committed to the handle only after every allocation and copy has
  // succeeded; on failure the handle keeps its old (non-adaptive) state.
  // tables of the grid levels, appended to the static ones; adaptive replicas point at them
  std::vector<int64_t> lut(s->h_lut);
  const size_t base = lut.size();
  if (base + (size_t)g->levels * 64 >= (1ull << 32)) return UB_ENOMEM;
  for (uint32_t j = 0; j < g->levels; j++)
    for (uint32_t b = 0; b < 64; b++)
      lut.push_back(boost_table_entry(ada_grid_gamma(g, j), ldexp((double)c.bin_tokens, (int)b), c.tok_us));
  std::vector<AdaState> st(R);
  std::vector<RepPar> par(R);
  std::vector<uint32_t> lut_off(s->h_lut_off), lut_nb(s->h_lut_nb);
  CK(cudaMemcpy2D(par.data(), sizeof(RepPar), &s->d_hdr[0].par, sizeof(Hdr), sizeof(RepPar), R, cudaMemcpyDeviceToHost));
  for (size_t r = 0; r < R; r++) {
    memset(&st[r], 0, sizeof(AdaState));
    if (!adaptive[r]) continue;
    int64_t gu = (int64_t)floor(s->h_reps[r].gamma * 1e6 + 0.5);
    if (gu < grid[0]) gu = grid[0];
    if (gu > grid[g->levels - 1]) gu = grid[g->levels - 1];
    uint32_t lvl = 0;
    while (lvl + 1 < g->levels && grid[lvl + 1] <= gu) lvl++;
    st[r].gamma_u = gu; st[r].level = lvl; st[r].on = 1;
    par[r].lut_off = (uint32_t)base; par[r].lut_nb = 64;
    lut_off[r] = (uint32_t)base; lut_nb[r] = 64;
  }
  int64_t* n_lut = nullptr; int64_t* n_ring = nullptr; AdaState* n_state = nullptr; int64_t* n_grid = nullptr;
  int rc = UB_OK;
  if ((rc = dmalloc(&n_lut, lut.size())) || (rc = dmalloc(&n_ring, R * (size_t)g->window)) ||
      (rc = dmalloc(&n_state, R)) || (rc = dmalloc(&n_grid, (size_t)g->levels))) {
    cudaFree(n_lut); cudaFree(n_ring); cudaFree(n_state); cudaFree(n_grid);
    return rc;
  }
  // (the parameter records inside the headers are the last thing written: they only take effect with the new table)
  cudaError_t e = cudaMemcpyAsync(n_lut, lut.data(), lut.size() * 8, cudaMemcpyHostToDevice, s->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(n_state, st.data(), R * sizeof(AdaState), cudaMemcpyHostToDevice, s->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(n_grid, grid.data(), grid.size() * 8, cudaMemcpyHostToDevice, s->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(n_ring, 0, R * (size_t)g->window * 8, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  bool par_touched = false;
  if (e == cudaSuccess) {
    par_touched = true;
    e = cudaMemcpy2DAsync(&s->d_hdr[0].par, sizeof(Hdr), par.data(), sizeof(RepPar), sizeof(RepPar), R,
                          cudaMemcpyHostToDevice, s->stream);
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e != cudaSuccess) {
    cudaGetLastError();
    if (par_touched) s->have_reps = false;         // the replica table may be half written: ub_set_replicas again
    cudaFree(n_lut); cudaFree(n_ring); cudaFree(n_state); cudaFree(n_grid);
    return UB_ECUDA;
  }
  // commit
  cudaFree(s->d_lut);
  drop_graph(s);
  s->d_lut = n_lut; s->d_ada_ring = n_ring; s->d_ada_state = n_state; s->d_ada_grid = n_grid;
  s->h_lut.swap(lut); s->h_lut_off.swap(lut_off); s->h_lut_nb.swap(lut_nb);
  SimDev& d = s->dev;
  d.lut = s->d_lut; d.ada_ring = s->d_ada_ring; d.ada_state = s->d_ada_state; d.ada_grid = s->d_ada_grid;
  d.ada_W = g->window; d.ada_G = g->levels; d.ada_min = g->min_samples; d.ada_shift = g->beta_shift; d.ada_eps = g->eps_us;
  launch_ada_init(d, s->stream);
  CK(cudaStreamSynchronize(s->stream));
  CK(cudaGetLastError());
  s->h_ada_grid = grid;
  return UB_OK;
}

int ub_gamma_state(ub_sim* s, uint32_t r, int64_t* gamma_u, int32_t* level, uint64_t* n_updates) {
  if (!s || r >= s->cfg.n_replicas) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  AdaState st; memset(&st, 0, sizeof(st));
  if (s->d_ada_state) {
    CK(cudaMemcpyAsync(&st, s->d_ada_state + r, sizeof(AdaState), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
  }
  if (gamma_u) *gamma_u = st.on ? st.gamma_u : 0;
  if (level) *level = st.on ? (int32_t)st.level : -1;
  if (n_updates) *n_updates = st.n_updates;
  return UB_OK;
}

int ub_gamma_grid(ub_sim* s, int64_t* grid_u) {
  if (!s || !grid_u || s->h_ada_grid.empty()) return UB_EINVAL;
  memcpy(grid_u, s->h_ada_grid.data(), s->h_ada_grid.size() * 8);
  return UB_OK;
}

int ub_set_iters_per_launch(ub_sim* s, uint32_t ipl) {
  if (!s) return UB_EINVAL;
  s->cfg.iters_per_launch = ipl ? ipl : 1;
  return UB_OK;
}

int ub_stats(ub_sim* s, ub_replica_stats* out) {
  if (!s || !out) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const size_t R = s->cfg.n_replicas;
  launch_stats(s->dev, s->d_stats, s->stream);
  std::vector<StatsDev> sd(R);
  std::vector<Hdr> hd(R);
  CK(cudaMemcpyAsync(sd.data(), s->d_stats, R * sizeof(StatsDev), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaMemcpyAsync(hd.data(), s->d_hdr, R * sizeof(Hdr), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  CK(cudaGetLastError());
  for (size_t r = 0; r < R; r++) {
    const Hdr& h = hd[r];
    ub_replica_stats& o = out[r];
    memset(&o, 0, sizeof(o));
    o.iterations = h.iterations; o.request_steps = h.request_steps; o.n_completed = h.n_completed;
    o.evict_recompute = h.evict_recompute; o.evict_swap = h.evict_swap; o.swapins = h.swapins;
    o.tokens_lost = h.tokens_lost; o.tokens_emitted = h.tokens_emitted;
    o.prefill_tokens = h.prefill_tokens; o.decode_seqs = h.decode_seqs;
    o.t_end_us = h.t; o.peak_active = h.peak_active; o.swap_used = h.swap_used;
    o.done = (h.n_active == 0 && h.next >= s->h_nreq[s->h_reps[r].trace_id]) ? 1 : 0;
    o.sum_ttft_us = h.sum_ttft; o.sum_ttlt_us = h.sum_ttlt;
    o.sum_tbt_num_us = h.sum_tbt_num; o.sum_tbt_den = h.sum_tbt_den;
    for (int k = 0; k < 3; k++) {
      o.ttft_us[k] = sd[r].ttft[k]; o.ttlt_us[k] = sd[r].ttlt[k]; o.tbt_us[k] = sd[r].tbt[k];
      o.ttft_s[k] = (double)o.ttft_us[k] * 1e-6;      // final us -> s in fp64 (M11)
      o.ttlt_s[k] = (double)o.ttlt_us[k] * 1e-6;
      o.tbt_s[k] = (double)o.tbt_us[k] * 1e-6;
    }
    const int64_t m = h.n_completed;
    o.mean_ttft_s = m ? ((double)h.sum_ttft / (double)m) * 1e-6 : 0.0;
    o.mean_ttlt_s = m ? ((double)h.sum_ttlt / (double)m) * 1e-6 : 0.0;
    o.mean_tbt_s = h.sum_tbt_den ? ((double)h.sum_tbt_num / (double)h.sum_tbt_den) * 1e-6 : 0.0;
    o.tokens_per_s = h.t > 0 ? (double)h.tokens_emitted / ((double)h.t * 1e-6) : 0.0;
  }
  return UB_OK;
}

int ub_percentile_curve(ub_sim* s, uint32_t which, const uint32_t* permille, uint32_t n, int64_t* out) {
  if (!s || !permille || !out || which > 1 || n < 1 || n > 16) return UB_EINVAL;
  for (uint32_t k = 0; k < n; k++) if (permille[k] < 1 || permille[k] > 1000) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const size_t R = s->cfg.n_replicas;
  int64_t* d_out = nullptr;
  int rc = dmalloc(&d_out, R * n); if (rc) return rc;
  launch_percentile_curve(s->dev, which, permille, n, d_out, s->stream);
  cudaError_t e = cudaMemcpyAsync(out, d_out, R * n * 8, cudaMemcpyDeviceToHost, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaFree(d_out);
  if (e != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
  return UB_OK;
}

// ub_percentile_curve without any allocation: the device staging of the result is a static array of the library
// (ub_aux.cu), shared by every call on the device.
int ub_percentile_curve_noalloc(ub_sim* s, uint32_t which, const uint32_t* permille, uint32_t n, int64_t* out) {
  if (!s || !permille || !out || which > 1 || n < 1 || n > 16) return UB_EINVAL;
  for (uint32_t k = 0; k < n; k++) if (permille[k] < 1 || permille[k] > 1000) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  const size_t R = s->cfg.n_replicas;
  if (R * n > kNoAllocCurveMax) return UB_ETOOBIG;
  if (set_dev(s)) return UB_ECUDA;
  const int64_t* staged = nullptr;
  const int lrc = launch_percentile_curve_noalloc(s->dev, s->cfg.device, which, permille, n, &staged, s->stream);
  if (lrc == -1) return UB_ETOOBIG;
  if (lrc != 0 || !staged) return UB_ECUDA;
  cudaError_t e = cudaMemcpyAsync(out, staged, R * n * 8, cudaMemcpyDeviceToHost, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
  return UB_OK;
}

int ub_class_percentiles(ub_sim* s, uint32_t which, uint32_t len_lo, uint32_t len_hi, const uint32_t* permille, uint32_t n,
                         int64_t* out, uint32_t* count, int64_t* sum) {
  if (!s || !permille || !out || which > 2 || n < 1 || n > 16 || len_lo > len_hi) return UB_EINVAL;
  for (uint32_t k = 0; k < n; k++) if (permille[k] < 1 || permille[k] > 1000) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const size_t R = s->cfg.n_replicas;
  int64_t* d_out = nullptr; uint32_t* d_cnt = nullptr; int64_t* d_sum = nullptr;
  int rc = UB_OK;
  if ((rc = dmalloc(&d_out, R * n)) || (rc = dmalloc(&d_cnt, R)) || (rc = dmalloc(&d_sum, R))) {
    cudaFree(d_out); cudaFree(d_cnt); cudaFree(d_sum); return rc;
  }
  launch_class_percentiles(s->dev, which, len_lo, len_hi, permille, n, d_out, d_cnt, d_sum, s->stream);
  cudaError_t e = cudaMemcpyAsync(out, d_out, R * n * 8, cudaMemcpyDeviceToHost, s->stream);
  if (e == cudaSuccess && count) e = cudaMemcpyAsync(count, d_cnt, R * 4, cudaMemcpyDeviceToHost, s->stream);
  if (e == cudaSuccess && sum) e = cudaMemcpyAsync(sum, d_sum, R * 8, cudaMemcpyDeviceToHost, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaFree(d_out); cudaFree(d_cnt); cudaFree(d_sum);
  if (e != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
  return UB_OK;
}

int ub_preempt_time(ub_sim* s, int64_t* out, int on_device) {
  if (!s || !out) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const size_t tot = (size_t)s->cfg.n_replicas * s->cfg.max_requests;
  CK(cudaMemcpyAsync(out, s->d_tpre, tot * 8, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return UB_OK;
}

int ub_slo_attainment(ub_sim* s, uint32_t which, const int64_t* thr, uint32_t n, uint32_t* met) {
  if (!s || !thr || !met || which > 1 || n < 1 || n > 16) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const size_t R = s->cfg.n_replicas;
  int64_t* d_thr = nullptr; uint32_t* d_met = nullptr;
  int rc = UB_OK;
  if ((rc = dmalloc(&d_thr, R * n)) || (rc = dmalloc(&d_met, R * n))) { cudaFree(d_thr); cudaFree(d_met); return rc; }
  cudaError_t e = cudaMemcpyAsync(d_thr, thr, R * n * 8, cudaMemcpyHostToDevice, s->stream);
  if (e == cudaSuccess) {
    launch_slo_count(s->dev, which, n, d_thr, d_met, s->stream);
    e = cudaMemcpyAsync(met, d_met, R * n * 4, cudaMemcpyDeviceToHost, s->stream);
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaFree(d_thr); cudaFree(d_met);
  if (e != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
  return UB_OK;
}

__global__ void k_mask_done(const uint32_t* in, uint32_t* out, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    out[i] = in[i] & 0x7FFFFFFFu;
}

int ub_per_request(ub_sim* s, int64_t* tf, int64_t* tl, uint32_t* ne, uint32_t* neu, int on_device) {
  if (!s) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const size_t tot = (size_t)s->cfg.n_replicas * s->cfg.max_requests;
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  launch_flush_tlast(s->dev, s->stream);
  if (tf) CK(cudaMemcpyAsync(tf, s->d_tfirst, tot * 8, kind, s->stream));
  if (tl) CK(cudaMemcpyAsync(tl, s->d_tlast, tot * 8, kind, s->stream));
  if (neu) CK(cudaMemcpyAsync(neu, s->d_neu, tot * 4, kind, s->stream));
  if (ne) {                                        // bit 31 of the stored word is the completion marker: masked on the device
    if (on_device) {
      k_mask_done<<<148 * 8, 256, 0, s->stream>>>(s->d_ne, ne, tot);
    } else {
      uint32_t* tmp = nullptr;
      int rc = dmalloc(&tmp, tot); if (rc) return rc;
      k_mask_done<<<148 * 8, 256, 0, s->stream>>>(s->d_ne, tmp, tot);
      cudaError_t e = cudaMemcpyAsync(ne, tmp, tot * 4, kind, s->stream);
      if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
      cudaFree(tmp);
      if (e != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
    }
  }
  CK(cudaStreamSynchronize(s->stream));
  CK(cudaGetLastError());
  return UB_OK;
}

int ub_digest(ub_sim* s, uint64_t* dg) {
  if (!s || !dg) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  const size_t R = s->cfg.n_replicas;
  CK(cudaMemcpy2DAsync(dg, 8, reinterpret_cast<const char*>(s->d_hdr) + offsetof(Hdr, H), sizeof(Hdr), 8, R,
                       cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return UB_OK;
}

int ub_boost_lut(ub_sim* s, uint32_t r, int64_t* lut, uint32_t cap, uint32_t* nb) {
  if (!s || !nb || r >= s->cfg.n_replicas) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  const uint32_t n = s->h_lut_nb[r];
  *nb = n;
  if (lut) {
    const bool boost = s->h_reps[r].policy == UB_BOOST || s->h_reps[r].policy == UB_DISTBOOST;
    size_t off = s->h_lut_off[r];
    if (s->d_ada_state) {                          // a gamma-Ada replica: the table of the grid level in use
      if (set_dev(s)) return UB_ECUDA;
      AdaState st;
      CK(cudaMemcpyAsync(&st, s->d_ada_state + r, sizeof(AdaState), cudaMemcpyDeviceToHost, s->stream));
      CK(cudaStreamSynchronize(s->stream));
      if (st.on) off += (size_t)st.level * 64u;
    }
    for (uint32_t b = 0; b < n && b < cap; b++) lut[b] = boost ? s->h_lut[off + b] : 0;
  }
  return UB_OK;
}

int ub_tbt_hist(ub_sim* s, uint32_t r, uint32_t* hist) {
  if (!s || !hist || r >= s->cfg.n_replicas) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  CK(cudaMemcpyAsync(hist, s->d_hist + (size_t)r * kTbtBins, kTbtBins * 4, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return UB_OK;
}

__global__ void k_debug_keys(SimDev s, uint32_t r, uint32_t n, uint32_t* id, unsigned long long* okey) {
  const RepPar par = s.hdr[r].par;
  const int64_t* lut = s.lut + par.lut_off + (size_t)s.hdr[r].level * 64u;
  const int64_t* tfirst = s.t_first + (size_t)r * s.N;
  for (uint32_t p = blockIdx.x * blockDim.x + threadIdx.x; p < n; p += gridDim.x * blockDim.x) {
    const Rec0 q0 = s.E0[(size_t)r * s.Q + p];
    const Rec1 q1 = s.E1[(size_t)r * s.Q + p];
    id[p] = q1.id;
    okey[p] = okey_of(s, par, lut, tfirst, s.t_last + (size_t)r * s.N, s.hdr[r].t, q0, q1);
  }
}

static int debug_keys_impl(ub_sim* s, uint32_t r, uint32_t* n_active, uint32_t* id, uint32_t* klass, int64_t* key_us,
                           bool stream_scorer) {
  if (!s || r >= s->cfg.n_replicas) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (stream_scorer) {                             // the streaming kernel covers FCFS / BOOST with the paper's signal and quantiser
    const ub_replica& q = s->h_reps[r];
    if (q.policy >= UB_DISTBOOST || q.signal_mode != UB_SIG_UNIFIED || q.quant_mode != UB_Q_GEOMETRIC || s->dev.blk_shift >= 32u)
      return UB_EINVAL;
  }
  if (set_dev(s)) return UB_ECUDA;
  Hdr h;
  CK(cudaMemcpyAsync(&h, s->d_hdr + r, sizeof(Hdr), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  const uint32_t n = h.n_active;
  if (n_active) *n_active = n;
  if (!n) return UB_OK;
  uint32_t* d_id = nullptr; unsigned long long* d_key = nullptr;
  int rc = UB_OK;
  if ((rc = dmalloc(&d_id, n)) || (rc = dmalloc(&d_key, n))) { cudaFree(d_id); cudaFree(d_key); return rc; }
  if (stream_scorer) launch_debug_keys_stream(s->dev, r, n, d_id, d_key, s->stream);
  else k_debug_keys<<<(n + 127) / 128, 128, 0, s->stream>>>(s->dev, r, n, d_id, d_key);
  std::vector<uint32_t> hid(n); std::vector<unsigned long long> hk(n);
  cudaError_t e = cudaMemcpyAsync(hid.data(), d_id, n * 4, cudaMemcpyDeviceToHost, s->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(hk.data(), d_key, n * 8, cudaMemcpyDeviceToHost, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaFree(d_id); cudaFree(d_key);
  if (e != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
  for (uint32_t i = 0; i < n; i++) {
    if (id) id[i] = hid[i];
    if (klass) klass[i] = (uint32_t)(hk[i] >> 63);
    if (key_us) key_us[i] = (int64_t)(hk[i] & ~(1ull << 63)) - kKeyBias;
  }
  return UB_OK;
}

int ub_debug_keys(ub_sim* s, uint32_t r, uint32_t* n_active, uint32_t* id, uint32_t* klass, int64_t* key_us) {
  return debug_keys_impl(s, r, n_active, id, klass, key_us, false);
}
int ub_debug_keys_stream(ub_sim* s, uint32_t r, uint32_t* n_active, uint32_t* id, uint32_t* klass, int64_t* key_us) {
  return debug_keys_impl(s, r, n_active, id, klass, key_us, true);
}

int ub_debug_get_state(ub_sim* s, uint32_t r, uint32_t* n_active, uint32_t* id, uint32_t* d, uint32_t* cached,
                       uint32_t* flags, int64_t* clock_us) {
  if (!s || r >= s->cfg.n_replicas) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  Hdr h;
  CK(cudaMemcpyAsync(&h, s->d_hdr + r, sizeof(Hdr), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  std::vector<Rec1> e(h.n_active);
  if (h.n_active) {
    CK(cudaMemcpyAsync(e.data(), s->d_E1 + (size_t)r * s->cfg.queue_cap, h.n_active * sizeof(Rec1),
                       cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
  }
  if (n_active) *n_active = h.n_active;
  if (clock_us) *clock_us = h.t;
  for (uint32_t i = 0; i < h.n_active; i++) {
    if (id) id[i] = e[i].id;
    if (d) d[i] = e[i].d;
    if (cached) cached[i] = e[i].cached;
    if (flags) flags[i] = e[i].flags;
  }
  return UB_OK;
}

// ---------------------------------------------------------------------------------------------- ub_debug_set_state
// err: 0 ok, 1 bad request id / counters, 2 replica already finished or would be left finished
__global__ void k_set_state(SimDev s, uint32_t r, uint32_t n, const uint32_t* id, const uint32_t* d, const uint32_t* cached,
                            const uint32_t* flags, int64_t clock, uint32_t next, uint32_t swap_used, int* err) {
  Hdr& h = s.hdr[r];
  const RepPar par = h.par;
  const uint32_t nreq = s.n_req[par.trace_id];
  const Rec0* TR = s.TR + (size_t)par.trace_id * s.N;
  __shared__ int bad;
  if (threadIdx.x == 0) {
    bad = 0;
    if (next > nreq || (n == 0 && next >= nreq)) bad = 2;
    if (h.n_active == 0 && h.a_next == kNever) bad = 2;               // counted as finished already (count[5])
  }
  __syncthreads();
  for (uint32_t p = threadIdx.x; p < n && !bad; p += blockDim.x) {
    const uint32_t i = id[p];
    if (i >= next) { atomicExch(&bad, 1); break; }
    const Rec0 q = TR[i];
    const uint32_t f = flags[p];
    if (d[p] >= q.D || cached[p] > q.P + d[p] || ((f & F_RESIDENT) && (f & F_SWAPPED)) ||
        (!(f & (F_RESIDENT | F_SWAPPED)) && cached[p] != 0u)) { atomicExch(&bad, 1); break; }
  }
  __syncthreads();
  if (bad) { if (threadIdx.x == 0) *err = bad; return; }
  for (uint32_t p = threadIdx.x; p < n; p += blockDim.x) {
    Rec1 q1; q1.id = id[p]; q1.d = d[p]; q1.cached = cached[p]; q1.flags = flags[p];
    s.E0[(size_t)r * s.Q + p] = TR[q1.id];
    s.E1[(size_t)r * s.Q + p] = q1;
  }
  if (threadIdx.x == 0) {
    h.t = clock;
    h.a_next = next < nreq ? TR[next].a : kNever;
    h.n_active = n; h.next = next; h.swap_used = swap_used; h.todo = 0; h.done = 0;
    if (n > h.peak_active) h.peak_active = n;
    uint32_t cnt = 0;                                                 // the streaming kernel's dirty list
    for (uint32_t p = 0; p < n; p++)
      if (flags[p] & F_DIRTY) { if (cnt < kDirtyMax) h.dl[cnt] = (uint16_t)p; cnt++; }
    h.n_dirty = cnt > kDirtyMax ? kDirtyMax + 1u : cnt;
  }
}

int ub_debug_set_state(ub_sim* s, uint32_t r, uint32_t n, const uint32_t* id, const uint32_t* d, const uint32_t* cached,
                       const uint32_t* flags, int64_t clock_us, uint32_t next_request, uint32_t swap_used_blocks) {
  if (!s || r >= s->cfg.n_replicas || n > s->cfg.queue_cap || (n && (!id || !d || !cached || !flags)) || clock_us < 0 ||
      swap_used_blocks > s->cfg.swap_pool_blocks)
    return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  if (set_dev(s)) return UB_ECUDA;
  uint32_t* dv = nullptr;
  int rc = dmalloc(&dv, 4 * (size_t)n + 1); if (rc) return rc;
  cudaError_t e = cudaSuccess;
  const uint32_t* src[4] = {id, d, cached, flags};
  for (int k = 0; k < 4 && e == cudaSuccess && n; k++)
    e = cudaMemcpyAsync(dv + (size_t)k * n, src[k], (size_t)n * 4, cudaMemcpyHostToDevice, s->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(dv + 4 * (size_t)n, 0, 4, s->stream);
  int herr = 0;
  if (e == cudaSuccess) {
    k_set_state<<<1, 256, 0, s->stream>>>(s->dev, r, n, dv, dv + n, dv + 2 * (size_t)n, dv + 3 * (size_t)n, clock_us,
                                          next_request, swap_used_blocks, reinterpret_cast<int*>(dv + 4 * (size_t)n));
    e = cudaMemcpyAsync(&herr, dv + 4 * (size_t)n, 4, cudaMemcpyDeviceToHost, s->stream);
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaFree(dv);
  if (e != cudaSuccess) { cudaGetLastError(); return UB_ECUDA; }
  return herr == 0 ? UB_OK : (herr == 2 ? UB_ESTATE : UB_EINVAL);
}

// ---------------------------------------------------------------------------------------------- JSQ router (rule M18)
int ub_jsq_run(ub_sim* s, uint32_t K, uint32_t C, uint32_t NA, const int64_t* a, const int32_t* p, const int32_t* d,
               const uint32_t* n_arr, int32_t* assign) {
  if (!s || !a || !p || !d || !n_arr || K < 1 || K > 32 || C < 1) return UB_EINVAL;
  if (!s->have_reps) return UB_ESTATE;
  const ub_config& c = s->cfg;
  if ((uint64_t)K * C != c.n_replicas || c.n_traces != c.n_replicas || c.max_requests >= (1u << 26)) return UB_EINVAL;
  if (s->d_ada_ring) return UB_ESTATE;                             // (gamma-Ada runs one iteration per launch: no fenced runs)
  if (set_dev(s)) return UB_ECUDA;
  const size_t R = c.n_replicas;
  for (size_t r = 0; r < R; r++) if (s->h_reps[r].trace_id != r || s->h_nreq[r] != 0) return UB_ESTATE;
  {
    std::vector<Hdr> hd(R);
    CK(cudaMemcpyAsync(hd.data(), s->d_hdr, R * sizeof(Hdr), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    for (size_t r = 0; r < R; r++) if (hd[r].iterations != 0) return UB_ESTATE;
  }
  uint32_t maxn = 0;
  for (uint32_t cl = 0; cl < C; cl++) {                            // the same checks ub_load_trace makes on a trace
    if (n_arr[cl] > NA) return UB_EINVAL;
    if (n_arr[cl] > maxn) maxn = n_arr[cl];
    for (uint32_t j = 0; j < n_arr[cl]; j++) {
      const int64_t aj = a[(size_t)cl * NA + j], P = p[(size_t)cl * NA + j], D = d[(size_t)cl * NA + j];
      if (aj < 0 || aj > ((int64_t)1 << 61)) return UB_EINVAL;
      if (j > 0 && aj < a[(size_t)cl * NA + j - 1]) return UB_EUNSORTED;
      if (P < 1 || D < 1 || (P + D + c.block_tokens - 1) / c.block_tokens > (int64_t)c.kv_blocks) return UB_EINFEASIBLE;
    }
  }
  const size_t tot = (size_t)C * NA;
  int64_t* da = nullptr; int32_t* dp = nullptr; int32_t* dd = nullptr; uint32_t* dn = nullptr;
  int64_t* dl = nullptr; int32_t* das = nullptr; int* derr = nullptr;
  int rc = UB_OK;
  auto cleanup = [&]() { cudaFree(da); cudaFree(dp); cudaFree(dd); cudaFree(dn); cudaFree(dl); cudaFree(das); cudaFree(derr); };
  if ((rc = dmalloc(&da, tot)) || (rc = dmalloc(&dp, tot)) || (rc = dmalloc(&dd, tot)) || (rc = dmalloc(&dn, (size_t)C)) ||
      (rc = dmalloc(&dl, R)) || (rc = dmalloc(&das, tot)) || (rc = dmalloc(&derr, 1))) { cleanup(); return rc; }
  cudaError_t e = cudaSuccess;
  if (tot) {
    e = cudaMemcpyAsync(da, a, tot * 8, cudaMemcpyHostToDevice, s->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dp, p, tot * 4, cudaMemcpyHostToDevice, s->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dd, d, tot * 4, cudaMemcpyHostToDevice, s->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(das, 0xFF, tot * 4, s->stream);      // -1 = no arrival
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(dn, n_arr, (size_t)C * 4, cudaMemcpyHostToDevice, s->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(derr, 0, sizeof(int), s->stream);
  if (e != cudaSuccess) { cudaGetLastError(); cleanup(); return UB_ECUDA; }
  JsqArgs J; J.K = K; J.C = C; J.NA = NA; J.a = da; J.p = dp; J.d = dd; J.n_arr = dn; J.tlimit = dl; J.assign = das;
  J.count = s->d_count; J.err = derr;
  // arrival by arrival: [route arrival j - 1, move the fences to arrival j] -> [every replica runs the iterations that
  // start before its fence]; clusters are the batch dimension
  s->use_list = false;                             // (a replica that has drained its trace may be routed more)
  if (s->ndrift) { uint64_t all = 0; if ((rc = compact_live(s, &all, true))) { cleanup(); return rc; } }
  for (int64_t j = 0; j <= (int64_t)maxn && rc == UB_OK; j++) {
    launch_jsq_dispatch(s->dev, J, j - 1, s->stream);
    if (j < (int64_t)maxn) { uint32_t nl = 0; rc = issue_steps(s, 0, &nl, dl); }
  }
  int herr = 0;
  if (rc == UB_OK) {
    e = cudaMemcpyAsync(&herr, derr, sizeof(int), cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess && assign && tot) e = cudaMemcpyAsync(assign, das, tot * 4, cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(s->h_nreq.data(), s->d_nreq, R * 4, cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) { cudaGetLastError(); rc = UB_ECUDA; }
  }
  cleanup();
  if (rc) return rc;
  if (herr) return UB_EINVAL;                                       // some replica's trace row (max_requests) was too short
  return ub_run(s, ~0ull >> 1, nullptr);                            // every replica serves what it got
}
