// ub_step.cu -- the scheduling-step kernel of libuniboost.so (sm_100a).
//
// One CTA advances one replica by one (or `iters`) scheduler iterations of Algorithm 1
// under the model rules M1..M12 of DESIGN.md Sec. 3:
//   a0 ingest / idle jump      (M6,  PAPER.md:117-123, 419)
//   a1 score                   (M3-M5, Eq. 2 PAPER.md:136 via the host-built table, Eq. 8, Eq. 7)
//   a2 order by (class,key,id)
//   a3 admission prefix scans  (M7,  PAPER.md:434-456)
//   a4 victim select           (M8,  PAPER.md:457-462)
//   a5 advance                 (M9-M10, M12; cost model of BASELINE.json)
// The replica's active window is streamed HBM -> shared memory -> HBM once per iteration; everything in
// between (keys, order, scans) stays on chip.  Integer arithmetic only.
#include "ub_internal.cuh"

namespace ub {

constexpr int kThreads = 128;
constexpr int kWarps = kThreads / 32;

// ---------------------------------------------------------------------------------------------- helpers

__device__ __forceinline__ uint32_t ceil_div_u32(uint32_t x, uint32_t y) { return (x + y - 1) / y; }

__device__ __forceinline__ uint64_t splitmix64(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull;
  uint64_t z = x;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// M12 event hash; events are summed (wrapping) inside an iteration, so the reduction order is free.
enum { EV_ADMIT = 1, EV_EVICT_RECOMPUTE = 2, EV_EVICT_SWAP = 3, EV_SWAPIN = 4, EV_EMIT_FIRST = 5, EV_COMPLETE = 6 };
__device__ __forceinline__ uint64_t event_hash(uint32_t type, uint32_t id, uint32_t payload) {
  uint32_t h = ((id + 1u) * 0x9E3779B1u) ^ (type * 0x85EBCA6Bu);
  return (uint64_t)h * (uint64_t)(2u * payload + 1u);
}

// M11 log-linear bin of a TBT gap (7 sub-bits).
__device__ __forceinline__ uint32_t tbt_bin(int64_t g) {
  if (g < 0) g = 0;
  if (g >= ((int64_t)1 << 40)) g = ((int64_t)1 << 40) - 1;
  int lg = (g > 0) ? 63 - __clzll((long long)g) : 0;
  int shift = lg - 7; if (shift < 0) shift = 0;
  return (uint32_t)(128 * shift + (g >> shift));
}

// Eq. 8 exponent: floor(log2(max(sig,k)/k)) == largest b with k 2^b <= max(sig,k)  (sig, k < 2^31)
__device__ __forceinline__ uint32_t geo_bin(uint32_t sig, uint32_t k) {
  uint32_t s = sig > k ? sig : k;
  int b = __clz(k) - __clz(s);
  if (((uint64_t)k << b) > (uint64_t)s) b--;
  return (uint32_t)b;
}

struct Shared {
  Hdr hdr;
  uint32_t scan[2][kWarps];      // double-buffered warp totals for the block scans
  uint32_t red32[8][kWarps];     // block reductions
  uint64_t red64[kWarps];
  unsigned long long acc64[6];   // rare-event accumulators (smem atomics)
  uint32_t acc32[4];
  uint32_t misc[8];
};

__device__ __forceinline__ uint32_t warp_scan_incl(uint32_t v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += n;
  }
  return v;
}

// Inclusive block scan of one u32 per thread; one barrier; `buf` alternates between calls.
__device__ __forceinline__ uint32_t block_scan_incl(uint32_t v, uint32_t& total, uint32_t* buf, int lane, int warp) {
  uint32_t w = warp_scan_incl(v, lane);
  if (lane == 31) buf[warp] = w;
  __syncthreads();
  uint32_t off = 0, tot = 0;
#pragma unroll
  for (int i = 0; i < kWarps; i++) {
    uint32_t x = buf[i];
    if (i < warp) off += x;
    tot += x;
  }
  total = tot;
  return w + off;
}

__device__ __forceinline__ uint64_t warp_sum_u64(uint64_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// (class,key,id) order on slots: okey first, id breaks ties (ids are unique)
__device__ __forceinline__ bool slot_less(const uint64_t* key, const Rec1* r1, uint32_t sa, uint32_t sb) {
  uint64_t ka = key[sa], kb = key[sb];
  if (ka != kb) return ka < kb;
  return r1[sa].id < r1[sb].id;
}

// ---------------------------------------------------------------------------------------------- the kernel

__global__ void __launch_bounds__(kThreads) k_step(const SimDev s, const uint32_t iters) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t Q = s.Q;
  uint32_t Qpad = 1; while (Qpad < Q) Qpad <<= 1;
  Rec0* s_r0 = reinterpret_cast<Rec0*>(smem_raw);
  Rec1* s_r1 = reinterpret_cast<Rec1*>(s_r0 + Q);
  uint64_t* s_key = reinterpret_cast<uint64_t*>(s_r1 + Q);
  uint32_t* s_bin = reinterpret_cast<uint32_t*>(s_key + Q);
  uint16_t* s_perm = reinterpret_cast<uint16_t*>(s_bin + Q);
  uint16_t* s_want = s_perm + Qpad;
  uint16_t* s_evl = s_want + Q;
  uint8_t* s_ev = reinterpret_cast<uint8_t*>(s_evl + Q);
  Shared* sh = reinterpret_cast<Shared*>(smem_raw + (((size_t)Q * 49 + (size_t)Qpad * 2 + 15) & ~(size_t)15));

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t r = blockIdx.x;
  if (r >= s.R) return;

  {  // header -> smem (40 words)
    const uint32_t* g = reinterpret_cast<const uint32_t*>(s.hdr + r);
    uint32_t* d = reinterpret_cast<uint32_t*>(&sh->hdr);
    if (tid < (int)(sizeof(Hdr) / 4)) d[tid] = __ldcg(g + tid);
  }
  __syncthreads();
  const RepPar par = s.par[r];
  const uint32_t nreq = s.n_req[par.trace_id];
  if (sh->hdr.n_active == 0 && sh->hdr.next >= nreq) return;     // replica finished: no-op
  const Rec0* TR = s.TR + (size_t)par.trace_id * s.N;
  Rec0* gE0 = s.E0 + (size_t)r * Q;
  Rec1* gE1 = s.E1 + (size_t)r * Q;
  const int64_t* lut = s.lut + par.lut_off;
  int64_t* g_tfirst = s.t_first + (size_t)r * s.N;
  int64_t* g_tlast = s.t_last + (size_t)r * s.N;
  uint32_t* g_hist = s.hist + (size_t)r * kTbtBins;
  uint32_t* g_ne = s.n_evict + (size_t)r * s.N;          // bit 31 = completed marker (read by the stats kernel)
  uint32_t* g_neu = s.n_evict_unf + (size_t)r * s.N;
  const uint32_t B = s.B, blk = s.blk, M = s.M, c = s.c, Tb = s.T;

  for (uint32_t it = 0; it < iters; it++) {
    uint32_t n = sh->hdr.n_active, next = sh->hdr.next;
    int64_t t = sh->hdr.t, a_next = sh->hdr.a_next;

    // ---------------- a0: idle jump + ingest (M6)
    if (n == 0) {
      if (next >= nreq) break;                  // done: this and all later iterations are no-ops
      if (a_next > t) t = a_next;
    }
    for (uint32_t p = tid; p < n; p += kThreads) {      // window HBM -> smem (stored = last priority order)
      int4 v0 = __ldcg(reinterpret_cast<const int4*>(gE0 + p));
      int4 v1 = __ldcg(reinterpret_cast<const int4*>(gE1 + p));
      *reinterpret_cast<int4*>(s_r0 + p) = v0;
      *reinterpret_cast<int4*>(s_r1 + p) = v1;
    }
    while (a_next <= t && n < Q && next < nreq) {
      const uint32_t i = next + tid, pos = n + tid;
      const bool ok = (i < nreq) && (pos < Q);
      Rec0 rec; rec.a = kNever; rec.P = 0; rec.D = 0;
      if (ok) *reinterpret_cast<int4*>(&rec) = __ldg(reinterpret_cast<const int4*>(TR + i));
      const bool take = ok && rec.a <= t;       // arrivals are sorted => `take` is a prefix over tid
      const uint32_t cnt = (uint32_t)__syncthreads_count(take);
      if (take) {
        s_r0[pos] = rec;
        Rec1 z; z.id = i; z.d = 0; z.cached = 0; z.flags = F_DIRTY;
        s_r1[pos] = z;
      }
      next += cnt; n += cnt;
      a_next = (next < nreq) ? __ldg(&TR[next].a) : kNever;
      if (cnt < (uint32_t)kThreads) break;
    }
    __syncthreads();

    // ---------------- a1: score (M3-M5).  okey = class<<63 | (key + 2^62); class 0 = MemGuard-locked resident
    for (uint32_t p = tid; p < n; p += kThreads) {
      const Rec0 r0 = s_r0[p];
      const Rec1 r1 = s_r1[p];
      uint32_t sig;
      if (par.signal_mode == 0) sig = r0.P + r1.d;                       // w~ = max(w, s_pre)
      else if (par.signal_mode == 1) sig = (r1.d == 0) ? r0.P : r1.d;    // SIGNAL
      else sig = r0.D - r1.d;                                            // remaining (tests: SRPT limit)
      const uint32_t bin = (par.quant_mode == 0) ? geo_bin(sig, s.k) : sig;   // QUANTIZE, Eq. 8
      int64_t key;
      if (par.policy == 0) key = r0.a;
      else if (par.policy == 1) key = (int64_t)(r0.D - r1.d);
      else if (par.policy == 3) key = (int64_t)sig;
      else key = r0.a - __ldg(lut + (bin < par.lut_nb ? bin : par.lut_nb - 1));   // pi = a - b
      const bool res = (r1.flags & F_RESIDENT) != 0;
      if (res && (par.policy == 0 || par.policy == 2)) key -= par.delta;  // Eq. 7 as a bias
      const uint32_t lockp1 = r1.flags >> F_LOCK_SHIFT;
      const uint64_t klass = (par.guard && res && lockp1 == bin + 1u) ? 0ull : 1ull;
      s_key[p] = (klass << 63) | (uint64_t)(key + kKeyBias);
      s_bin[p] = bin;
      s_perm[p] = (uint16_t)p;
      s_want[p] = 0;
      s_ev[p] = 0;
    }
    if (tid < 6) sh->acc64[tid] = 0ull;
    if (tid < 4) sh->acc32[tid] = 0u;
    if (tid < 2) sh->misc[tid] = 0xFFFFFFFFu;
    __syncthreads();

    // ---------------- a2: order.  The stored order is last iteration's priority order; if it is still sorted
    // (the common case: MemGuard keeps keys piecewise constant) nothing moves, else bitonic sort.
    {
      int viol = 0;
      for (uint32_t p = tid + 1; p < n; p += kThreads) viol |= slot_less(s_key, s_r1, p, p - 1) ? 1 : 0;
      if (__syncthreads_or(viol)) {
        uint32_t npad = 1; while (npad < n) npad <<= 1;
        for (uint32_t p = n + tid; p < npad; p += kThreads) s_perm[p] = 0xFFFFu;     // +inf sentinels
        __syncthreads();
        for (uint32_t kk = 2; kk <= npad; kk <<= 1) {
          for (uint32_t j = kk >> 1; j > 0; j >>= 1) {
            for (uint32_t i = tid; i < npad; i += kThreads) {
              const uint32_t l = i ^ j;
              if (l > i) {
                const uint32_t pa = s_perm[i], pb = s_perm[l];
                const bool asc = (i & kk) == 0;
                bool b_lt_a;                                     // is perm[l] < perm[i] ?
                if (pb == 0xFFFFu) b_lt_a = false;
                else if (pa == 0xFFFFu) b_lt_a = true;
                else b_lt_a = slot_less(s_key, s_r1, pb, pa);
                if (b_lt_a == asc) { s_perm[i] = (uint16_t)pb; s_perm[l] = (uint16_t)pa; }
              }
            }
            __syncthreads();
          }
        }
      }
    }

    // ---------------- a3: admission walk as prefix scans (M7; Algorithm 1 "while |B| < M ... U + dU <= B").
    // Round 0 walks everybody up to the first entry that does not fit; if that entry is a non-resident that failed
    // on KV only ("newblocked"), round 1 continues over the residents behind it.  Both rounds are the same scans:
    //   W = incl. scan of min(c, rem);  tok_before = min(T, W - w);  want = min(T, W) - tok_before;
    //   foot = ceil((cached + want)/blk);  Cf = incl. scan of foot;  ok = cnt_before < M & tok_before < T & Cf <= B.
    // ok is monotone along the walk, so the admitted set is a prefix of the walked entries.
    uint32_t C = 0, tok = 0, cnt = 0;
    {
      uint32_t start = 0;
      bool only_res = false;
      for (int round = 0; round < 2; round++) {
        uint32_t carryW = tok, carryC = C, carryN = cnt;
        bool failed = false;
        for (uint32_t base = start; base < n; base += kThreads) {
          const uint32_t j = base + tid;
          const bool in = j < n;
          const uint32_t slot = in ? s_perm[j] : 0u;
          Rec0 r0; Rec1 r1;
          r0.a = 0; r0.P = 0; r0.D = 0; r1.id = 0; r1.d = 0; r1.cached = 0; r1.flags = 0;
          if (in) { r0 = s_r0[slot]; r1 = s_r1[slot]; }
          const bool res = (r1.flags & F_RESIDENT) != 0;
          const bool valid = in && (!only_res || res);
          const uint32_t rem = r0.P + r1.d - r1.cached;
          const uint32_t w = valid ? (rem < c ? rem : c) : 0u;
          uint32_t wtot, ctot, vtot;
          const uint32_t W = carryW + block_scan_incl(w, wtot, sh->scan[0], lane, warp);
          const uint32_t tok_before = (W - w) < Tb ? (W - w) : Tb;
          const uint32_t tok_after = W < Tb ? W : Tb;
          const uint32_t want = tok_after - tok_before;
          const uint32_t foot = valid ? ceil_div_u32(r1.cached + want, blk) : 0u;
          const uint32_t Cf = carryC + block_scan_incl(foot, ctot, sh->scan[1], lane, warp);
          uint32_t cnt_before;
          if (only_res) {
            cnt_before = carryN + block_scan_incl(valid ? 1u : 0u, vtot, sh->scan[0], lane, warp) - (valid ? 1u : 0u);
          } else {
            cnt_before = carryN + (j - base);
            vtot = (n - base) < (uint32_t)kThreads ? (n - base) : (uint32_t)kThreads;
          }
          const bool ok = valid && cnt_before < M && tok_before < Tb && Cf <= B;
          const bool fail = valid && !ok;
          if (ok) s_want[slot] = (uint16_t)want;
          if (__syncthreads_or(fail)) {
            if (fail) atomicMin(&sh->misc[round], j);
            __syncthreads();
            if (fail && j == sh->misc[round]) {                 // the first entry that did not fit
              sh->misc[2] = Cf - foot;                           // walk state in front of it
              sh->misc[3] = tok_before;
              sh->misc[4] = cnt_before;
              sh->misc[5] = (cnt_before < M && tok_before < Tb) ? 1u : 0u;   // failed on KV only
              sh->misc[6] = res ? 1u : 0u;
            }
            __syncthreads();
            failed = true;
            break;
          }
          carryW += wtot; carryC += ctot; carryN += vtot;
        }
        if (!failed) { C = carryC; tok = carryW < Tb ? carryW : Tb; cnt = carryN; break; }
        C = sh->misc[2]; tok = sh->misc[3]; cnt = sh->misc[4];
        const bool kv_only = sh->misc[5] != 0, fail_res = sh->misc[6] != 0;
        const uint32_t fp = sh->misc[round];
        if (round == 0 && kv_only && !fail_res) { start = fp + 1; only_res = true; __syncthreads(); continue; }
        break;
      }
    }
    __syncthreads();

    // ---------------- a4: batch totals (M9) and victim select (M8; SELECTVICTIM / SWAPOUT)
    uint32_t pf_tot, dec_tot, swin_blocks, swin_cnt, kres_tot;
    uint64_t ev_tot;
    {
      uint32_t pf = 0, dec = 0, swb = 0, swc = 0, kres = 0;
      uint64_t evh = 0;
      for (uint32_t p = tid; p < n; p += kThreads) {
        const Rec0 r0 = s_r0[p];
        const Rec1 r1 = s_r1[p];
        const uint32_t want = s_want[p];
        if (want) {
          const uint32_t rem = r0.P + r1.d - r1.cached;
          if (r1.d >= 1 && rem == 1) dec++; else pf += want;        // decode sequence vs prefill tokens
          evh += event_hash(EV_ADMIT, r1.id, want);
          if (r1.flags & F_SWAPPED) {                                 // swap-in on admission
            const uint32_t blocks = ceil_div_u32(r1.cached, blk);
            swb += blocks; swc++;
            evh += event_hash(EV_SWAPIN, r1.id, blocks);
          }
        } else if (r1.flags & F_RESIDENT) {
          kres += ceil_div_u32(r1.cached, blk);                       // non-admitted resident keeps its blocks
        }
      }
      pf = __reduce_add_sync(0xffffffffu, pf); dec = __reduce_add_sync(0xffffffffu, dec);
      swb = __reduce_add_sync(0xffffffffu, swb); swc = __reduce_add_sync(0xffffffffu, swc);
      kres = __reduce_add_sync(0xffffffffu, kres);
      evh = warp_sum_u64(evh);
      if (lane == 0) {
        sh->red32[0][warp] = pf; sh->red32[1][warp] = dec; sh->red32[2][warp] = swb;
        sh->red32[3][warp] = swc; sh->red32[4][warp] = kres; sh->red64[warp] = evh;
      }
      __syncthreads();
      pf_tot = dec_tot = swin_blocks = swin_cnt = kres_tot = 0; ev_tot = 0;
#pragma unroll
      for (int i = 0; i < kWarps; i++) {
        pf_tot += sh->red32[0][i]; dec_tot += sh->red32[1][i]; swin_blocks += sh->red32[2][i];
        swin_cnt += sh->red32[3][i]; kres_tot += sh->red32[4][i]; ev_tot += sh->red64[i];
      }
    }
    uint32_t swap_used = sh->hdr.swap_used - swin_blocks;
    uint32_t swout_blocks = 0;
    if (kres_tot > B - C) {                      // block-uniform; rare
      // victims = the suffix of the non-admitted residents (in priority order) whose prefix sum exceeds B - C
      const uint32_t thr = B - C;
      uint32_t carry = 0, ecarry = 0;
      for (uint32_t base = 0; base < n; base += kThreads) {
        const uint32_t j = base + tid;
        const bool in = j < n;
        const uint32_t slot = in ? s_perm[j] : 0u;
        uint32_t v = 0;
        if (in && s_want[slot] == 0) {
          const Rec1 r1 = s_r1[slot];
          if (r1.flags & F_RESIDENT) v = ceil_div_u32(r1.cached, blk);
        }
        // a resident always holds >= 1 block?  cached can be 0 only for non-residents, so v > 0 <=> member of K
        uint32_t tot, etot;
        const uint32_t ps = carry + block_scan_incl(v, tot, sh->scan[0], lane, warp);
        const bool evict = (v > 0) && ps > thr;
        const uint32_t ei = ecarry + block_scan_incl(evict ? 1u : 0u, etot, sh->scan[1], lane, warp);
        if (evict) s_evl[ei - 1] = (uint16_t)slot;
        carry += tot; ecarry += etot;
      }
      __syncthreads();
      if (tid == 0) {                            // lowest priority first; swap pool is a sequential resource
        uint32_t n_sw = 0, n_rc = 0; uint64_t evh = 0; int64_t lost = 0;
        for (int e = (int)ecarry - 1; e >= 0; e--) {
          const uint32_t slot = s_evl[e];
          const Rec1 r1 = s_r1[slot];
          const uint32_t resb = ceil_div_u32(r1.cached, blk);
          bool do_swap = false;
          if (s.preempt_mode == 1) do_swap = (swap_used + resb <= s.swap_pool);
          else if (s.preempt_mode == 2)
            do_swap = (swap_used + resb <= s.swap_pool) &&
                      (2ll * resb * (int64_t)s.swap_ns < 1000ll * s.c_pf * (int64_t)r1.cached);
          if (do_swap) {
            swap_used += resb; swout_blocks += resb; n_sw++;
            evh += event_hash(EV_EVICT_SWAP, r1.id, resb);
            s_ev[slot] = 2;
          } else {
            lost += r1.cached; n_rc++;
            evh += event_hash(EV_EVICT_RECOMPUTE, r1.id, r1.cached);
            s_ev[slot] = 1;
          }
          g_ne[r1.id] = __ldcg(g_ne + r1.id) + 1u;
          if (s_key[slot] >> 63) g_neu[r1.id] = __ldcg(g_neu + r1.id) + 1u;   // victim was not MemGuard-locked
        }
        sh->hdr.evict_swap += n_sw; sh->hdr.evict_recompute += n_rc; sh->hdr.tokens_lost += lost;
        sh->acc64[0] += evh;
        sh->misc[7] = swout_blocks;
        sh->misc[2] = swap_used;
      }
      __syncthreads();
      swout_blocks = sh->misc[7];
      swap_used = sh->misc[2];
    }

    // ---------------- a5: execute one step with the stated cost model (M9), apply (M10)
    const int64_t cost = s.c0 + s.c_pf * (int64_t)pf_tot + s.c_dec * (int64_t)dec_tot +
                         (int64_t)(((uint64_t)(swin_blocks + swout_blocks) * s.swap_ns + 500u) / 1000u);
    const int64_t t_end = t + cost;
    uint32_t n_emit = 0, n_agg = 0;
    for (uint32_t p = tid; p < n; p += kThreads) {
      const Rec0 r0 = s_r0[p];
      Rec1 r1 = s_r1[p];
      const uint32_t want = s_want[p];
      const uint32_t evm = s_ev[p];
      uint32_t nf = r1.flags & (F_RESIDENT | F_SWAPPED | F_EMITPREV);
      if (want) {
        nf = (nf | F_RESIDENT) & ~F_SWAPPED;
        r1.cached += want;
        if (r1.cached == r0.P + r1.d) {                       // KV caught up => one token out (M2)
          r1.d += 1; n_emit++;
          if (r1.d == 1) {
            g_tfirst[r1.id] = t_end;
            atomicAdd(&sh->acc64[0], (unsigned long long)event_hash(EV_EMIT_FIRST, r1.id, 0));
          } else if (nf & F_EMITPREV) {
            n_agg++;                                          // gap == this iteration's cost
          } else {
            const int64_t tl = __ldcg(g_tlast + r1.id);
            atomicAdd(&g_hist[tbt_bin(t_end - tl)], 1u);
          }
          nf |= F_EMITPREV;
          if (r1.d == r0.D) {                                 // complete: KV freed at once
            g_tlast[r1.id] = t_end;
            const int64_t tf = (r1.d == 1) ? t_end : __ldcg(g_tfirst + r1.id);
            atomicAdd(&sh->acc64[1], (unsigned long long)(tf - r0.a));
            atomicAdd(&sh->acc64[2], (unsigned long long)(t_end - r0.a));
            atomicAdd(&sh->acc64[3], (unsigned long long)(t_end - tf));
            atomicAdd(&sh->acc64[4], (unsigned long long)(r0.D - 1));
            atomicAdd(&sh->acc64[0], (unsigned long long)event_hash(EV_COMPLETE, r1.id, 0));
            atomicAdd(&sh->acc32[0], 1u);
            g_ne[r1.id] = __ldcg(g_ne + r1.id) | 0x80000000u;
            s_ev[p] = 3;
          }
        } else if (nf & F_EMITPREV) {
          g_tlast[r1.id] = t; nf &= ~F_EMITPREV;
        }
      } else {
        if (nf & F_EMITPREV) { g_tlast[r1.id] = t; nf &= ~F_EMITPREV; }   // persist t_last when the streak ends
        if (evm == 1) { r1.cached = 0; nf &= ~F_RESIDENT; }
        else if (evm == 2) { nf = (nf | F_SWAPPED) & ~F_RESIDENT; }
      }
      if (nf & F_RESIDENT) nf |= (s_bin[p] + 1u) << F_LOCK_SHIFT;   // re-lock at this iteration's bin (M10, G6)
      r1.flags = nf;
      s_r1[p] = r1;
    }
    n_emit = __reduce_add_sync(0xffffffffu, n_emit);
    n_agg = __reduce_add_sync(0xffffffffu, n_agg);
    if (lane == 0) { sh->red32[5][warp] = n_emit; sh->red32[6][warp] = n_agg; }
    __syncthreads();

    // ---------------- write back in priority order, dropping completed requests
    uint32_t n_new = 0;
    for (uint32_t base = 0; base < n; base += kThreads) {
      const uint32_t j = base + tid;
      const bool in = j < n;
      const uint32_t slot = in ? s_perm[j] : 0u;
      const bool keep = in && s_ev[slot] != 3;
      uint32_t tot;
      const uint32_t pos = n_new + block_scan_incl(keep ? 1u : 0u, tot, sh->scan[(base / kThreads) & 1], lane, warp) - 1u;
      if (keep) {
        *reinterpret_cast<int4*>(gE0 + pos) = *reinterpret_cast<const int4*>(s_r0 + slot);
        *reinterpret_cast<int4*>(gE1 + pos) = *reinterpret_cast<const int4*>(s_r1 + slot);
      }
      n_new += tot;
    }
    if (tid == 0) {
      Hdr& h = sh->hdr;
      uint32_t emitted = 0, agg = 0;
      for (int i = 0; i < kWarps; i++) { emitted += sh->red32[5][i]; agg += sh->red32[6][i]; }
      if (agg) atomicAdd(&g_hist[tbt_bin(cost)], agg);
      h.t = t_end;
      h.H = splitmix64(h.H ^ (ev_tot + sh->acc64[0]) ^ splitmix64((uint64_t)t_end));
      h.a_next = a_next; h.next = next;
      h.request_steps += n; h.iterations += 1;
      h.tokens_emitted += emitted; h.prefill_tokens += pf_tot; h.decode_seqs += dec_tot;
      h.sum_ttft += (int64_t)sh->acc64[1]; h.sum_ttlt += (int64_t)sh->acc64[2];
      h.sum_tbt_num += (int64_t)sh->acc64[3]; h.sum_tbt_den += (int64_t)sh->acc64[4];
      h.n_completed += sh->acc32[0];
      h.swapins += swin_cnt; h.swap_used = swap_used;
      if (n > h.peak_active) h.peak_active = n;
      h.n_active = n_new;
    }
    __syncthreads();
  }

  {  // header -> HBM
    uint32_t* g = reinterpret_cast<uint32_t*>(s.hdr + r);
    const uint32_t* d = reinterpret_cast<const uint32_t*>(&sh->hdr);
    if (tid < (int)(sizeof(Hdr) / 4)) g[tid] = d[tid];
  }
}

size_t step_smem_bytes(uint32_t Q) {
  uint32_t Qpad = 1; while (Qpad < Q) Qpad <<= 1;
  size_t arrays = ((size_t)Q * 49 + (size_t)Qpad * 2 + 15) & ~(size_t)15;
  return arrays + sizeof(Shared);
}

int step_configure(uint32_t Q) {
  return (int)cudaFuncSetAttribute(k_step, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)step_smem_bytes(Q));
}

void launch_step(const SimDev& s, uint32_t iters, cudaStream_t st) {
  k_step<<<s.R, kThreads, step_smem_bytes(s.Q), st>>>(s, iters);
}

}  // namespace ub
