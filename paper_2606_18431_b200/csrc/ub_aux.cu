// ub_aux.cu -- the kernels around the scheduling step: trace validation + packing, reset, live count,
// t_last flush, and the device-resident percentile reduction a6 (M11; t_p of PAPER.md:225).
#include <mutex>
#include "ub_internal.cuh"

namespace ub {

// ------------------------------------------------------------------ trace validation + packing (ub_load_trace)
// err: first offending (trace, request) in row-major scan order, encoded (linear index << 2 | kind),
// kind 0 = arrival outside [0, 2^61] (UB_EINVAL), 1 = arrivals decrease (UB_EUNSORTED), 2 = infeasible request.
// hit (nullable): prefix-cache hit tokens per request (rule M17): the record carries the effective
// prefill work s_pre - h, which is also what the size signal w~ = max(w, s_pre - h) starts from.
__global__ void k_pack_validate(const int64_t* __restrict__ a, const int32_t* __restrict__ p,
                                const int32_t* __restrict__ d, const int32_t* __restrict__ hit,
                                const uint32_t* __restrict__ n_req,
                                uint32_t NT, uint32_t N, uint32_t B, uint32_t blk, Rec0* __restrict__ out,
                                unsigned long long* err) {
  const size_t total = (size_t)NT * N;
  for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (size_t)gridDim.x * blockDim.x) {
    const uint32_t tr = (uint32_t)(g / N), i = (uint32_t)(g % N);
    const int64_t h = hit ? (int64_t)hit[g] : 0;
    Rec0 rec; rec.a = a[g]; rec.P = (uint32_t)((int64_t)p[g] - h); rec.D = (uint32_t)d[g];
    out[g] = rec;
    if (i >= n_req[tr]) continue;
    const int64_t ai = rec.a;
    const int64_t P = p[g], D = d[g];
    int kind = -1;
    if (ai < 0 || ai > ((int64_t)1 << 61) || h < 0 || (P >= 1 && h >= P)) kind = 0;
    else if (i > 0 && ai < a[g - 1]) kind = 1;
    else if (P < 1 || D < 1 || (P + D + blk - 1) / blk > (int64_t)B) kind = 2;
    if (kind >= 0) atomicMin(err, ((unsigned long long)g << 2) | (unsigned long long)kind);
  }
}

void launch_pack_validate(const int64_t* a, const int32_t* p, const int32_t* d, const int32_t* hit, const uint32_t* n_req,
                          uint32_t NT, uint32_t N, uint32_t B, uint32_t blk, Rec0* out, int* err, cudaStream_t st) {
  const size_t total = (size_t)NT * N;
  int blocks = (int)((total + 255) / 256);
  if (blocks > 148 * 16) blocks = 148 * 16;
  if (blocks < 1) blocks = 1;
  k_pack_validate<<<blocks, 256, 0, st>>>(a, p, d, hit, n_req, NT, N, B, blk, out,
                                          reinterpret_cast<unsigned long long*>(err));
}

// ------------------------------------------------------------------ reset (ub_set_replicas)
// count[0..3] = work lists of the current round, count[4] = k_stream's ticket counter, count[5] = replicas that have finished their trace
__global__ void k_reset(SimDev s, uint32_t* count) {
  const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= s.R) return;
  Hdr h = s.hdr[r];                                 // (keeps the parameters ub_set_replicas wrote)
  memset(&h, 0, offsetof(Hdr, par));
  const uint32_t tr = h.par.trace_id;
  const bool empty = s.n_req[tr] == 0;
  h.a_next = empty ? kNever : s.TR[(size_t)tr * s.N].a;
  s.hdr[r] = h;
  if (empty) atomicAdd(count + 5, 1u);
}
void launch_reset(const SimDev& s, uint32_t* list, uint32_t* count, cudaStream_t st) {
  (void)list;
  cudaMemsetAsync(count, 0, 8 * kMaxSplit * sizeof(uint32_t), st);
  k_reset<<<(s.R + 127) / 128, 128, 0, st>>>(s, count);
}

// ------------------------------------------------------------------ gamma-Ada (M13; Eq. 9, UPDATEGAMMA PAPER.md:588-601)
// Launched in front of every scheduler round while adaptation is on ("gamma <- UPDATEGAMMA(S)" opens the loop of
// Algorithm 1).  One warp per replica; it leaves at once unless the replica adapts, is not finished, and
// a request completed since the last update.  Then: window of the last min(W, n_completed) end-to-end latencies ->
// shared memory, nearest-rank t95 / t99 by selection, the fixed-point update, the grid level.  A level change
// switches the boost table (Hdr::level) and re-keys every request: n_dirty is set to overflow, so this round's
// ordering is rebuilt from scratch by the team kernel.
constexpr int kAdaThreads = 128;                   // 4 warps, one replica each
constexpr long long kLn5e12 = 1609437912434LL;     // floor(ln 5 * 1e12)

// One WARP per replica.  Only two order statistics near the top are wanted (nearest-rank t95 and t99 of the last
// m <= W <= 1024 latencies), so the window is not sorted: the largest value is taken out m - r95 + 1 times (each lane
// keeps the largest of its own strided share; a round is one 64-bit warp maximum and a re-scan by the winning lane).
__global__ void __launch_bounds__(kAdaThreads) k_gamma_ada(SimDev s, uint32_t rbeg, uint32_t rend) {
  __shared__ long long vs[kAdaThreads / 32][1024];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  const uint32_t r = rbeg + blockIdx.x * (kAdaThreads / 32) + warp;
  if (r >= rend) return;
  AdaState* st = s.ada_state + r;
  if (!st->on) return;
  Hdr* h = s.hdr + r;
  const uint32_t nc = h->n_completed;
  if ((h->n_active == 0 && h->a_next == kNever) || nc == st->seen || nc < s.ada_min) return;
  const uint32_t m = nc < s.ada_W ? nc : s.ada_W;
  long long* v = vs[warp];
  const int64_t* ring = s.ada_ring + (size_t)r * s.ada_W;
  // (latencies are >= 0: INT64_MIN marks a value that was taken out)
  long long best = INT64_MIN; uint32_t besti = 0;
  for (uint32_t i = lane; i < m; i += 32u) {
    const long long x = (long long)ring[i];
    v[i] = x;
    if (x > best) { best = x; besti = i; }
  }
  uint32_t r95 = (95u * m + 99u) / 100u, r99 = (99u * m + 99u) / 100u;        // nearest rank (t_p of PAPER.md:225)
  if (r95 < 1) r95 = 1; if (r99 < 1) r99 = 1;
  const uint32_t k99 = m - r99 + 1u, k95 = m - r95 + 1u;                      // the k-th largest has rank m - k + 1
  long long t99 = 0, t95 = 0;
  for (uint32_t kk = 1; kk <= k95; kk++) {
    // 64-bit maximum over the lanes: high words (signed), then low words (unsigned) among the lanes that hold it
    const int hi = (int)(best >> 32);
    const int mhi = __reduce_max_sync(0xffffffffu, hi);
    const uint32_t lo = hi == mhi ? (uint32_t)best : 0u;
    const uint32_t mlo = __reduce_max_sync(0xffffffffu, lo);
    const uint32_t who = __ballot_sync(0xffffffffu, hi == mhi && (uint32_t)best == mlo);
    const long long top = ((long long)mhi << 32) | (long long)mlo;
    if (kk == k99) t99 = top;
    if (kk == k95) t95 = top;
    if (lane == (uint32_t)__ffs(who) - 1u && kk < k95) {                      // take one instance out, find my next largest
      v[besti] = INT64_MIN;
      best = INT64_MIN; besti = 0;
      for (uint32_t i = lane; i < m; i += 32u) { const long long x = v[i]; if (x > best) { best = x; besti = i; } }
    }
  }
  if (lane == 0) {
    long long delta = t99 - t95;
    if (delta < s.ada_eps) delta = s.ada_eps;
    const long long hat = kLn5e12 / delta;                                     // Eq. 9 in micro units
    long long g = st->gamma_u;
    g += (hat - g) / (1ll << s.ada_shift);                                     // (1 - beta) gamma + beta gamma_hat
    if (g < s.ada_grid[0]) g = s.ada_grid[0];                                  // clip
    if (g > s.ada_grid[s.ada_G - 1]) g = s.ada_grid[s.ada_G - 1];
    uint32_t lvl = 0;
    while (lvl + 1 < s.ada_G && s.ada_grid[lvl + 1] <= g) lvl++;
    st->gamma_u = g; st->seen = nc; st->n_updates++;
    if (lvl != st->level) { st->level = lvl; h->level = lvl; h->n_dirty = kDirtyMax + 1u; }
  }
}
void launch_gamma_ada(const SimDev& s, uint32_t rbeg, uint32_t rend, cudaStream_t st) {
  constexpr uint32_t per = kAdaThreads / 32;
  if (rend > rbeg) k_gamma_ada<<<(rend - rbeg + per - 1) / per, kAdaThreads, 0, st>>>(s, rbeg, rend);
}

__global__ void k_ada_init(SimDev s) {
  const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r < s.R && s.ada_state[r].on) s.hdr[r].level = s.ada_state[r].level;
}
void launch_ada_init(const SimDev& s, cudaStream_t st) { k_ada_init<<<(s.R + 127) / 128, 128, 0, st>>>(s); }

// ------------------------------------------------------------------ live replicas (ub_step / ub_run)
__global__ void k_count_live(const uint32_t* count, uint32_t R, unsigned long long* live) {
  uint32_t fin = 0;
  for (uint32_t i = 0; i < kMaxSplit; i++) fin += count[8 * i + 5];   // (one set of counters per part of a round)
  *live = (unsigned long long)(R - fin);
}
void launch_count_live(const uint32_t* count, uint32_t R, unsigned long long* live, cudaStream_t st) {
  k_count_live<<<1, 1, 0, st>>>(count, R, live);
}

// The unfinished replicas among positions [rbeg, rend) -- of the list `in`, else the replica numbers themselves --
// that belong to the drift group (SRPT / LAS) or to the main one, compacted (ub_run's tail: the streaming kernel then
// visits only these).  A replica is finished when its trace is exhausted and nothing is active (M6); finished
// replicas never come back.
__global__ void k_compact_live(SimDev s, uint32_t rbeg, uint32_t rend, const uint32_t* in, uint32_t drift_group, uint32_t any_state,
                               uint32_t* out, uint32_t* cnt) {
  const uint32_t lane = threadIdx.x & 31u;
  for (uint32_t base = rbeg + (blockIdx.x * blockDim.x + threadIdx.x - lane); base < rend; base += gridDim.x * blockDim.x) {
    const uint32_t i = base + lane;
    bool alive = false;
    uint32_t r = 0;
    if (i < rend) {
      r = in ? in[i] : i;
      const Hdr* h = s.hdr + r;
      const RepPar& q = h->par;
      const uint32_t dg = (!s.ada_ring && (q.policy == 1u || q.policy == 3u) && q.signal_mode == 0u && q.quant_mode == 0u &&
                           s.blk_shift < 32u) ? 1u : 0u;
      alive = (any_state || !(h->n_active == 0u && h->a_next == kNever)) && dg == drift_group;
    }
    const uint32_t m = __ballot_sync(0xffffffffu, alive);
    uint32_t off = 0;
    if (lane == 0 && m) off = atomicAdd(cnt, (uint32_t)__popc(m));
    off = __shfl_sync(0xffffffffu, off, 0);
    if (alive) out[off + __popc(m & ((1u << lane) - 1u))] = r;
  }
}
void launch_compact_live(const SimDev& s, uint32_t rbeg, uint32_t rend, const uint32_t* in, bool drift_group, bool any_state,
                         uint32_t* out, uint32_t* cnt, cudaStream_t st) {
  cudaMemsetAsync(cnt, 0, sizeof(uint32_t), st);
  if (rend > rbeg) k_compact_live<<<148, 256, 0, st>>>(s, rbeg, rend, in, drift_group ? 1u : 0u, any_state ? 1u : 0u, out, cnt);
}

// ------------------------------------------------------------------ JSQ router (rule M18; Table 9)
// One warp per cluster of K <= 32 replicas (lane k = replica c K + k).  Called between two fenced runs: every replica of
// the cluster has executed every iteration that starts before arrival j of its cluster's stream.  The arrival goes to
// the replica with the fewest requests in the system at that instant -- assigned to it and not completed by then: the
// completions of the replica's last iteration count only if that iteration has ended by the arrival time --, lowest
// replica number on a tie; it is appended to that replica's trace.  Then the fence of the cluster moves to arrival j + 1
// (INT64_MIN when the stream is exhausted: the replicas wait for the final free run).  j = -1: only the first fence.
__global__ void k_jsq_dispatch(SimDev s, JsqArgs J, long long j) {
  const uint32_t c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), k = threadIdx.x & 31u;
  if (c >= J.C) return;
  const uint32_t na = J.n_arr[c];
  if (j >= 0 && (uint64_t)j < na) {
    const int64_t a = J.a[(size_t)c * J.NA + j];
    const uint32_t r = c * J.K + k;
    uint32_t load = 0xFFFFFFFFu;
    Hdr* h = nullptr;
    uint32_t* nreq = const_cast<uint32_t*>(s.n_req);
    if (k < J.K) {
      h = s.hdr + r;
      const uint32_t gone = h->n_completed - ((h->t > a) ? h->last_done : 0u);
      load = nreq[r] - gone;
    }
    const uint32_t best = __reduce_min_sync(0xffffffffu, load >= (1u << 26) ? 0xFFFFFFFFu : ((load << 5) | k));
    if (k == (best & 31u) && k < J.K) {
      const uint32_t at = nreq[r];
      if (at >= s.N) atomicExch(J.err, 1);                          // the replica's row is full
      else {
        Rec0 q; q.a = a; q.P = (uint32_t)J.p[(size_t)c * J.NA + j]; q.D = (uint32_t)J.d[(size_t)c * J.NA + j];
        const_cast<Rec0*>(s.TR)[(size_t)r * s.N + at] = q;
        nreq[r] = at + 1u;
        if (h->a_next == kNever) {                                  // its trace was exhausted: it has a next arrival again,
          h->a_next = a;
          if (h->n_active == 0u) atomicSub(J.count + 5, 1u);        // and, if it was idle, it is no longer finished
        }
        J.assign[(size_t)c * J.NA + j] = (int32_t)k;
      }
    }
  }
  if (k < J.K) J.tlimit[c * J.K + k] = ((uint64_t)(j + 1) < na) ? J.a[(size_t)c * J.NA + (j + 1)] : INT64_MIN;
}
void launch_jsq_dispatch(const SimDev& s, const JsqArgs& J, int64_t j, cudaStream_t st) {
  k_jsq_dispatch<<<(J.C + 3) / 4, 128, 0, st>>>(s, J, (long long)j);
}

// ------------------------------------------------------------------ t_last flush (ub_per_request)
// A request that emitted in the last executed iteration carries its t_last implicitly (== replica clock).
__global__ void k_flush_tlast(SimDev s) {
  const uint32_t r = blockIdx.x;
  const Hdr* h = s.hdr + r;
  const uint32_t n = h->n_active;
  const int64_t t = h->t;
  const Rec1* e1 = s.E1 + (size_t)r * s.Q;
  for (uint32_t p = threadIdx.x; p < n; p += blockDim.x) {
    const Rec1 r1 = e1[p];
    if (r1.flags & F_EMITPREV) s.t_last[(size_t)r * s.N + r1.id] = t;
  }
}
void launch_flush_tlast(const SimDev& s, cudaStream_t st) { k_flush_tlast<<<s.R, 128, 0, st>>>(s); }

// ------------------------------------------------------------------ a6: percentile reduction (M11)
// Nearest rank: the ceil(p m / 100)-th smallest of the m completed requests' TTFT_i = t_first - a_i and
// TTLT_i = t_last - a_i, found exactly by an MSD radix select (8 passes of 8 bits) over values recomputed
// on the fly from HBM (L2-resident after the first pass); TBT from the pooled log-linear histogram.
constexpr int kStatThreads = 256;
constexpr uint32_t kDoneBit = 0x80000000u;      // n_evict bit 31 marks a completed request

__device__ __forceinline__ int64_t tbt_edge(uint32_t idx) {
  int sft = (int)(idx / 128) - 1; if (sft < 0) sft = 0;
  return (int64_t)(idx - 128u * (uint32_t)sft) << sft;
}

struct SelectSmem { uint32_t hist[256]; uint32_t wtot[kStatThreads / 32]; unsigned long long prefix; uint32_t rank; };

// The rank0-th smallest (0-based) of { src[i] - TR[i].a : request i completed }: MSD radix select, whole CTA.
__device__ int64_t radix_select(SelectSmem& sm, const int64_t* src, const Rec0* TR, const uint32_t* ne, uint32_t nreq,
                                uint32_t rank0) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) { sm.prefix = 0ull; sm.rank = rank0; }
  for (int pass = 7; pass >= 0; pass--) {
    sm.hist[tid] = 0;
    __syncthreads();
    const unsigned long long prefix = sm.prefix;
    const int sh_hi = 8 * (pass + 1);
    for (uint32_t i = tid; i < nreq; i += kStatThreads) {
      if (!(ne[i] & kDoneBit)) continue;
      const unsigned long long v = (unsigned long long)(src[i] - TR[i].a);
      const bool match = (pass == 7) || ((v >> sh_hi) == (prefix >> sh_hi));
      if (match) atomicAdd(&sm.hist[(v >> (8 * pass)) & 0xFF], 1u);
    }
    __syncthreads();
    // bucket holding the rank-th (0-based) matching value: thread b owns bucket b
    const uint32_t cntb = sm.hist[tid];
    uint32_t inc = cntb;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t x = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += x; }
    if (lane == 31) sm.wtot[warp] = inc;
    __syncthreads();
    uint32_t off = 0;
    for (int w = 0; w < warp; w++) off += sm.wtot[w];
    inc += off;
    const uint32_t exc = inc - cntb, want = sm.rank;
    __syncthreads();
    if (want >= exc && want < inc) {
      sm.prefix = prefix | ((unsigned long long)tid << (8 * pass));
      sm.rank = want - exc;
    }
    __syncthreads();
  }
  const int64_t result = (int64_t)sm.prefix;
  __syncthreads();
  return result;
}

// The same select over m values staged in shared memory (k_stats: a replica's latencies are read from HBM once and the
// 3 x 8 passes run on chip; the first version re-read them from HBM / L2 in every pass: 466 GB of DRAM reads at
// config 5, profiles/r02_stats.md).
__device__ int64_t radix_select_smem(SelectSmem& sm, const unsigned long long* vals, uint32_t m, uint32_t rank0) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) { sm.prefix = 0ull; sm.rank = rank0; }
  for (int pass = 7; pass >= 0; pass--) {
    sm.hist[tid] = 0;
    __syncthreads();
    const unsigned long long prefix = sm.prefix;
    const int sh_hi = 8 * (pass + 1);
    for (uint32_t i = tid; i < m; i += kStatThreads) {
      const unsigned long long v = vals[i];
      if (pass == 7 || (v >> sh_hi) == (prefix >> sh_hi)) atomicAdd(&sm.hist[(v >> (8 * pass)) & 0xFF], 1u);
    }
    __syncthreads();
    const uint32_t cntb = sm.hist[tid];
    uint32_t inc = cntb;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t x = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += x; }
    if (lane == 31) sm.wtot[warp] = inc;
    __syncthreads();
    uint32_t off = 0;
    for (int w = 0; w < warp; w++) off += sm.wtot[w];
    inc += off;
    const uint32_t exc = inc - cntb, want = sm.rank;
    __syncthreads();
    if (want >= exc && want < inc) {
      sm.prefix = prefix | ((unsigned long long)tid << (8 * pass));
      sm.rank = want - exc;
    }
    __syncthreads();
  }
  const int64_t result = (int64_t)sm.prefix;
  __syncthreads();
  return result;
}

constexpr uint32_t kStatSmemVals = 16384;        // latencies of one replica staged in shared memory (128 KB); longer rows use HBM

__global__ void __launch_bounds__(kStatThreads) k_stats(SimDev s, StatsDev* out, uint32_t cap) {
  __shared__ SelectSmem sm;
  __shared__ uint32_t wtot[kStatThreads / 32];
  __shared__ uint32_t fill;
  extern __shared__ __align__(16) unsigned long long vals[];    // [cap]
  const uint32_t r = blockIdx.x;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t tr = s.hdr[r].par.trace_id, nreq = s.n_req[tr];
  const Rec0* TR = s.TR + (size_t)tr * s.N;
  const int64_t* tf = s.t_first + (size_t)r * s.N;
  const int64_t* tl = s.t_last + (size_t)r * s.N;
  const uint32_t* ne = s.n_evict + (size_t)r * s.N;
  const uint32_t m = s.hdr[r].n_completed;
  const int pct[3] = {50, 90, 99};

  for (int which = 0; which < 2; which++) {
    const int64_t* src = which == 0 ? tf : tl;
    const bool staged = m <= cap;
    if (staged && m > 0) {                       // the completed requests' latencies -> shared memory, once (any order)
      if (tid == 0) fill = 0u;
      __syncthreads();
      for (uint32_t base = 0; base < nreq; base += kStatThreads) {
        const uint32_t i = base + tid;
        const bool done = i < nreq && (ne[i] & kDoneBit);
        const uint32_t bm = __ballot_sync(0xffffffffu, done);
        uint32_t off = 0;
        if (lane == 0 && bm) off = atomicAdd(&fill, (uint32_t)__popc(bm));
        off = __shfl_sync(0xffffffffu, off, 0);
        if (done) vals[off + __popc(bm & ((1u << lane) - 1u))] = (unsigned long long)(src[i] - TR[i].a);
      }
      __syncthreads();
    }
    for (int k = 0; k < 3; k++) {
      int64_t result = 0;
      if (m > 0) {
        uint64_t rank = ((uint64_t)pct[k] * m + 99) / 100;
        if (rank < 1) rank = 1;
        if (rank > m) rank = m;
        result = staged ? radix_select_smem(sm, vals, m, (uint32_t)(rank - 1))
                        : radix_select(sm, src, TR, ne, nreq, (uint32_t)(rank - 1));
      }
      if (tid == 0) { if (which == 0) out[r].ttft[k] = result; else out[r].ttlt[k] = result; }
    }
  }

  // TBT: thread i owns bins [17 i, 17 i + 17)
  {
    const uint32_t* gh = s.hist + (size_t)r * kTbtBins;
    constexpr int per = kTbtBins / kStatThreads;      // 17
    uint32_t loc[per];
    uint32_t sum = 0;
#pragma unroll
    for (int b = 0; b < per; b++) { loc[b] = gh[tid * per + b]; sum += loc[b]; }
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t x = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += x; }
    if (lane == 31) wtot[warp] = inc;
    __syncthreads();
    uint64_t off = 0, total = 0;
    for (int w = 0; w < kStatThreads / 32; w++) { if (w < warp) off += wtot[w]; total += wtot[w]; }
    const uint64_t incl = off + inc, excl = incl - sum;
    for (int k = 0; k < 3; k++) {
      if (total == 0) { if (tid == 0) out[r].tbt[k] = 0; continue; }
      uint64_t rank = ((uint64_t)pct[k] * total + 99) / 100;
      if (rank < 1) rank = 1;
      if (rank > excl && rank <= incl) {
        uint64_t cum = excl;
#pragma unroll
        for (int b = 0; b < per; b++) {
          cum += loc[b];
          if (cum >= rank) { out[r].tbt[k] = tbt_edge((uint32_t)(tid * per + b)); break; }
        }
      }
    }
  }
}

void launch_stats(const SimDev& s, StatsDev* out, cudaStream_t st) {
  const uint32_t cap = s.N < kStatSmemVals ? s.N : kStatSmemVals;
  const size_t bytes = (size_t)cap * sizeof(unsigned long long);
  static size_t configured = 0;
  if (bytes > configured) {
    cudaFuncSetAttribute(k_stats, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    configured = bytes;
  }
  k_stats<<<s.R, kStatThreads, bytes, st>>>(s, out, cap);
}

// ------------------------------------------------------------------ richer reductions
// Percentile curves (Fig. 6): nearest-rank percentiles at arbitrary per-mille points, rank =
// ceil(p m / 1000) (t_p of PAPER.md:225), of TTFT (which = 0) or TTLT (which = 1) over a replica's completed requests.
struct CurveArgs { uint32_t which, n; uint32_t permille[16]; };
__global__ void __launch_bounds__(kStatThreads) k_percentile_curve(SimDev s, CurveArgs c, int64_t* out) {
  __shared__ SelectSmem sm;
  const uint32_t r = blockIdx.x;
  const uint32_t tr = s.hdr[r].par.trace_id, nreq = s.n_req[tr];
  const Rec0* TR = s.TR + (size_t)tr * s.N;
  const int64_t* src = (c.which == 0 ? s.t_first : s.t_last) + (size_t)r * s.N;
  const uint32_t* ne = s.n_evict + (size_t)r * s.N;
  const uint32_t m = s.hdr[r].n_completed;
  for (uint32_t k = 0; k < c.n; k++) {
    int64_t result = 0;
    if (m > 0) {
      uint64_t rank = ((uint64_t)c.permille[k] * m + 999) / 1000;
      if (rank < 1) rank = 1;
      if (rank > m) rank = m;
      result = radix_select(sm, src, TR, ne, nreq, (uint32_t)(rank - 1));
    }
    if (threadIdx.x == 0) out[(size_t)r * c.n + k] = result;
  }
}
void launch_percentile_curve(const SimDev& s, uint32_t which, const uint32_t* permille, uint32_t n, int64_t* out,
                             cudaStream_t st) {
  CurveArgs c; c.which = which; c.n = n;
  for (uint32_t k = 0; k < 16; k++) c.permille[k] = k < n ? permille[k] : 0;
  k_percentile_curve<<<s.R, kStatThreads, 0, st>>>(s, c, out);
}

// ub_percentile_curve_noalloc: the same kernel with its result staged in a file-scope device array instead of a
// cudaMalloc'ed buffer (callers that cannot allocate).  Every GPU that loads the library holds the array (512 KB)
// until exit; every call on a device shares it, so calls that overlap on the GPU race.  The kernel writes every
// one of the R x n values it is asked for (0 for a replica without completed requests): nothing has to start at zero.
// In host code `g_curve_scratch` is only a stand-in for the symbol: the device address comes from
// cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) long long g_curve_scratch[kNoAllocCurveMax];
int launch_percentile_curve_noalloc(const SimDev& s, int device, uint32_t which, const uint32_t* permille, uint32_t n,
                                    const int64_t** staged, cudaStream_t st) {
  constexpr int kMaxDev = 64;
  static std::mutex mu;
  static long long* addr[kMaxDev] = {};
  if (device < 0 || device >= kMaxDev || (size_t)s.R * n > kNoAllocCurveMax) return -1;
  long long* ptr = nullptr;
  {
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {                              // set-up, once per device (the caller made `device` current)
      void* p = nullptr;
      if (cudaGetSymbolAddress(&p, g_curve_scratch) != cudaSuccess || !p) { cudaGetLastError(); return -2; }
      addr[device] = static_cast<long long*>(p);
    }
    ptr = addr[device];
  }
  launch_percentile_curve(s, which, permille, n, reinterpret_cast<int64_t*>(ptr), st);
  *staged = reinterpret_cast<const int64_t*>(ptr);
  return 0;
}

// Per-class reductions (Tables 3-5): over the completed requests of a replica whose total
// length P + D lies in [len_lo, len_hi] -- the paper's short / long split -- nearest-rank percentiles of TTFT (which 0),
// TTLT (1) or preemption time (2, rule M15), their number and their sum.  The same MSD radix select as a6, with the
// class filter and the value folded into the scan.
struct ClassArgs { uint32_t which, n, len_lo, len_hi; uint32_t permille[16]; };
__global__ void __launch_bounds__(kStatThreads) k_class_percentiles(SimDev s, ClassArgs c, int64_t* out, uint32_t* count,
                                                                    int64_t* sum) {
  __shared__ SelectSmem sm;
  __shared__ unsigned long long tot_sum;
  __shared__ uint32_t tot_cnt;
  const uint32_t r = blockIdx.x;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t tr = s.hdr[r].par.trace_id, nreq = s.n_req[tr];
  const Rec0* TR = s.TR + (size_t)tr * s.N;
  const int64_t* src = (c.which == 0 ? s.t_first : (c.which == 1 ? s.t_last : s.t_pre)) + (size_t)r * s.N;
  const uint32_t* ne = s.n_evict + (size_t)r * s.N;
  // value of request i if it belongs to the class
  auto value = [&](uint32_t i, unsigned long long& v) -> bool {
    if (!(ne[i] & kDoneBit)) return false;
    const Rec0 q = TR[i];
    const uint32_t len = q.P + q.D;
    if (len < c.len_lo || len > c.len_hi) return false;
    v = (unsigned long long)(c.which == 2 ? src[i] : src[i] - q.a);
    return true;
  };
  if (tid == 0) { tot_sum = 0ull; tot_cnt = 0u; }
  __syncthreads();
  {
    unsigned long long ls = 0; uint32_t lc = 0;
    for (uint32_t i = tid; i < nreq; i += kStatThreads) { unsigned long long v; if (value(i, v)) { ls += v; lc++; } }
    for (int o = 16; o > 0; o >>= 1) { ls += __shfl_xor_sync(0xffffffffu, ls, o); lc += __shfl_xor_sync(0xffffffffu, lc, o); }
    if (lane == 0) { atomicAdd(&tot_sum, ls); atomicAdd(&tot_cnt, lc); }
  }
  __syncthreads();
  const uint32_t m = tot_cnt;
  if (tid == 0) { if (count) count[r] = m; if (sum) sum[r] = (int64_t)tot_sum; }
  for (uint32_t k = 0; k < c.n; k++) {
    int64_t result = 0;
    if (m > 0) {
      uint64_t rank = ((uint64_t)c.permille[k] * m + 999) / 1000;
      if (rank < 1) rank = 1;
      if (rank > m) rank = m;
      // MSD radix select of the (rank-1)-th smallest class value, 8 passes of 8 bits
      if (tid == 0) { sm.prefix = 0ull; sm.rank = (uint32_t)(rank - 1); }
      for (int pass = 7; pass >= 0; pass--) {
        sm.hist[tid] = 0;
        __syncthreads();
        const unsigned long long prefix = sm.prefix;
        const int sh_hi = 8 * (pass + 1);
        for (uint32_t i = tid; i < nreq; i += kStatThreads) {
          unsigned long long v;
          if (!value(i, v)) continue;
          if (pass == 7 || (v >> sh_hi) == (prefix >> sh_hi)) atomicAdd(&sm.hist[(v >> (8 * pass)) & 0xFF], 1u);
        }
        __syncthreads();
        const uint32_t cntb = sm.hist[tid];
        uint32_t inc = cntb;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t x = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += x; }
        if (lane == 31) sm.wtot[warp] = inc;
        __syncthreads();
        uint32_t off = 0;
        for (int w = 0; w < warp; w++) off += sm.wtot[w];
        inc += off;
        const uint32_t exc = inc - cntb, want = sm.rank;
        __syncthreads();
        if (want >= exc && want < inc) { sm.prefix = prefix | ((unsigned long long)tid << (8 * pass)); sm.rank = want - exc; }
        __syncthreads();
      }
      result = (int64_t)sm.prefix;
      __syncthreads();
    }
    if (tid == 0) out[(size_t)r * c.n + k] = result;
  }
}
void launch_class_percentiles(const SimDev& s, uint32_t which, uint32_t len_lo, uint32_t len_hi, const uint32_t* permille,
                              uint32_t n, int64_t* out, uint32_t* count, int64_t* sum, cudaStream_t st) {
  ClassArgs c; c.which = which; c.n = n; c.len_lo = len_lo; c.len_hi = len_hi;
  for (uint32_t k = 0; k < 16; k++) c.permille[k] = k < n ? permille[k] : 0;
  k_class_percentiles<<<s.R, kStatThreads, 0, st>>>(s, c, out, count, sum);
}

// SLO attainment (Fig. 8): per replica and threshold, the number of completed requests whose
// latency is <= the threshold (the caller forms thresholds = SLO scale x base latency).  thr: [R][n] device.
__global__ void __launch_bounds__(kStatThreads) k_slo_count(SimDev s, uint32_t which, uint32_t n, const int64_t* thr,
                                                            uint32_t* out) {
  __shared__ uint32_t cnt[16];
  const uint32_t r = blockIdx.x;
  const uint32_t tr = s.hdr[r].par.trace_id, nreq = s.n_req[tr];
  const Rec0* TR = s.TR + (size_t)tr * s.N;
  const int64_t* src = (which == 0 ? s.t_first : s.t_last) + (size_t)r * s.N;
  const uint32_t* ne = s.n_evict + (size_t)r * s.N;
  if (threadIdx.x < 16) cnt[threadIdx.x] = 0;
  __syncthreads();
  uint32_t loc[16];
#pragma unroll
  for (int k = 0; k < 16; k++) loc[k] = 0;
  for (uint32_t i = threadIdx.x; i < nreq; i += kStatThreads) {
    if (!(ne[i] & kDoneBit)) continue;
    const int64_t v = src[i] - TR[i].a;
#pragma unroll
    for (int k = 0; k < 16; k++) if ((uint32_t)k < n && v <= thr[(size_t)r * n + k]) loc[k]++;
  }
#pragma unroll
  for (int k = 0; k < 16; k++) {
    const uint32_t t = __reduce_add_sync(0xffffffffu, loc[k]);
    if ((threadIdx.x & 31) == 0 && t) atomicAdd(&cnt[k], t);
  }
  __syncthreads();
  if (threadIdx.x < n) out[(size_t)r * n + threadIdx.x] = cnt[threadIdx.x];
}
void launch_slo_count(const SimDev& s, uint32_t which, uint32_t n, const int64_t* thr, uint32_t* out, cudaStream_t st) {
  k_slo_count<<<s.R, kStatThreads, 0, st>>>(s, which, n, thr, out);
}


}  // namespace ub
