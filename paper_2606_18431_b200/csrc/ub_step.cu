// ub_step.cu -- the scheduling-step kernels of libuniboost.so (sm_100a).
//
// One TEAM (1, 4 or 8 warps) advances one replica by one (or `iters`) scheduler iterations of Algorithm 1
// under the model rules M1..M12 of DESIGN.md Sec. 3:
//   a0 ingest / idle jump      (M6,  PAPER.md:117-123, 419)
//   a1 score                   (M3-M5, Eq. 2 PAPER.md:136 via the host-built table, Eq. 8, Eq. 7)
//   a2 order by (class,key,id)
//   a3 admission prefix scans  (M7,  PAPER.md:434-456)
//   a4 victim select           (M8,  PAPER.md:457-462)
//   a5 advance                 (M9-M10, M12; cost model of BASELINE.json)
// The replica's active window is streamed HBM -> registers -> HBM once per iteration (E requests per thread,
// the request at priority position j lives in thread j % TEAM, register slot j / TEAM); shared memory is only
// the exchange buffer of the ordering step.  Replicas are binned by window size into three work lists
// (S: one warp per replica, M: 4 warps, L: 8 warps) that the kernels of iteration i build for iteration i+1.
// Integer arithmetic only.
#include "ub_device.cuh"

namespace ub {

// ---------------------------------------------------------------------------------------------- helpers

__device__ __forceinline__ uint64_t warp_sum_u64(uint64_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ordering record in the exchange buffer: (okey, id) is the total order; aux carries the dirty hint
struct __align__(16) KeyRec { uint64_t okey; uint32_t id; uint32_t aux; };

// ---------------------------------------------------------------------------------------------- team primitives
// WARPS == 1: a team is a warp, everything is shuffles.  WARPS > 1: the team is the whole CTA.

struct TeamScratch {            // per team, in shared memory
  uint32_t scan[2][8];
  uint32_t red[8][8];
  unsigned long long red64[8];
  uint32_t bc[16];              // broadcast words
  unsigned long long bc64[8];
  unsigned long long acc64[6];  // rare-event accumulators
  uint32_t acc32[4];
  uint32_t ndirty;             // next iteration's dirty-list length
  unsigned long long smax[2][8]; // exchange buffer of the prefix maximum
};

template <int WARPS> struct Team {
  static constexpr int THREADS = 32 * WARPS;
  TeamScratch* ts;
  int tid, lane, warp;          // within the team
  uint32_t phase;               // alternates the scan buffer

  __device__ __forceinline__ void sync() const {
    if constexpr (WARPS == 1) __syncwarp(); else __syncthreads();
  }
  // inclusive scan over the team in thread order, and the team total
  __device__ __forceinline__ uint32_t scan_incl(uint32_t v, uint32_t& total) {
    uint32_t w = warp_scan_incl(v, lane);
    if constexpr (WARPS == 1) {
      total = __shfl_sync(0xffffffffu, w, 31);
      return w;
    } else {
      uint32_t* buf = ts->scan[phase & 1]; phase++;
      if (lane == 31) buf[warp] = w;
      __syncthreads();
      uint32_t off = 0, tot = 0;
#pragma unroll
      for (int i = 0; i < WARPS; i++) { uint32_t x = buf[i]; if (i < warp) off += x; tot += x; }
      total = tot;
      return w + off;
    }
  }
  // exclusive prefix maximum over the team in thread order (0 in front of the first thread), and the team maximum
  __device__ __forceinline__ uint64_t scanmax_excl(uint64_t v, uint64_t& total) {
    uint64_t w = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint64_t t = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o && t > w) w = t;
    }
    uint64_t ex = __shfl_up_sync(0xffffffffu, w, 1);
    if (lane == 0) ex = 0ull;
    if constexpr (WARPS == 1) {
      total = __shfl_sync(0xffffffffu, w, 31);
      return ex;
    } else {
      unsigned long long* buf = ts->smax[phase & 1]; phase++;
      if (lane == 31) buf[warp] = w;
      __syncthreads();
      uint64_t off = 0, tot = 0;
#pragma unroll
      for (int i = 0; i < WARPS; i++) { const uint64_t x = buf[i]; if (i < warp && x > off) off = x; if (x > tot) tot = x; }
      total = tot;
      return ex > off ? ex : off;
    }
  }
  __device__ __forceinline__ bool any(bool p) const {
    if constexpr (WARPS == 1) return __any_sync(0xffffffffu, p); else return __syncthreads_or(p) != 0;
  }
  // K team-wide sums of u32 (all threads get all K results)
  template <int K> __device__ __forceinline__ void sum32(uint32_t (&v)[K]) {
#pragma unroll
    for (int k = 0; k < K; k++) v[k] = __reduce_add_sync(0xffffffffu, v[k]);
    if constexpr (WARPS > 1) {
      if (lane == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) ts->red[k][warp] = v[k];
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < K; k++) {
        uint32_t a = 0;
#pragma unroll
        for (int i = 0; i < WARPS; i++) a += ts->red[k][i];
        v[k] = a;
      }
      __syncthreads();
    }
  }
  __device__ __forceinline__ uint64_t sum64(uint64_t v) {
    v = warp_sum_u64(v);
    if constexpr (WARPS > 1) {
      if (lane == 0) ts->red64[warp] = v;
      __syncthreads();
      uint64_t a = 0;
#pragma unroll
      for (int i = 0; i < WARPS; i++) a += ts->red64[i];
      v = a;
      __syncthreads();
    }
    return v;
  }
};

// ---------------------------------------------------------------------------------------------- one replica, `iters` iterations

template <int WARPS, int E>
__device__ __forceinline__ void team_step(Team<WARPS>& tm, const StepArgs& A, const uint32_t r, unsigned char* xbuf) {
  constexpr int TH = 32 * WARPS, CAP = TH * E;
  const SimDev& s = A.s;
  const int tid = tm.tid, lane = tm.lane, warp = tm.warp;
  TeamScratch* ts = tm.ts;
  KeyRec* x_key = reinterpret_cast<KeyRec*>(xbuf);
  Rec0* x_r0 = reinterpret_cast<Rec0*>(xbuf);
  Rec1* x_r1 = reinterpret_cast<Rec1*>(xbuf + (size_t)CAP * 16);
  uint4* x_ev = reinterpret_cast<uint4*>(xbuf);                       // a4: {id, cached, class, pos}
  uint8_t* x_mode = reinterpret_cast<uint8_t*>(xbuf + (size_t)CAP * 16);
  uint16_t* x_idx = reinterpret_cast<uint16_t*>(xbuf + (size_t)CAP * 32);
  uint16_t* x_dl = x_idx + CAP;
  uint32_t* x_cnt = reinterpret_cast<uint32_t*>(x_dl + 32);

  const RepPar par = s.hdr[r].par;
  const uint32_t nreq = s.n_req[par.trace_id];
  const Rec0* TR = s.TR + (size_t)par.trace_id * s.N;
  Rec0* gE0 = s.E0 + (size_t)r * s.Q;
  Rec1* gE1 = s.E1 + (size_t)r * s.Q;
  // (a gamma-Ada replica owns one table per grid level, Hdr::level selects; 0 for a static replica)
  const int64_t* lut = s.lut + par.lut_off + (size_t)s.hdr[r].level * 64u;
  const uint32_t ncomp0 = s.ada_ring ? s.hdr[r].n_completed : 0u;     // (gamma-Ada runs one iteration per launch)
  int64_t* g_tfirst = s.t_first + (size_t)r * s.N;
  int64_t* g_tlast = s.t_last + (size_t)r * s.N;
  int64_t* g_tpre = s.t_pre + (size_t)r * s.N;
  uint32_t* g_hist = s.hist + (size_t)r * kTbtBins;
  uint32_t* g_ne = s.n_evict + (size_t)r * s.N;          // bit 31 = completed marker (read by the stats kernel)
  uint32_t* g_neu = s.n_evict_unf + (size_t)r * s.N;
  const uint32_t B = s.B, M = s.M, cc = s.c, Tb = s.T, Q = s.Q;

  // ---- header: thread i < 20 of warp 0 holds 64-bit word i of Hdr
  uint64_t* ghdr = reinterpret_cast<uint64_t*>(s.hdr + r);
  uint64_t hv = 0;
  if (warp == 0 && lane < 20) hv = __ldcg(ghdr + lane);
  int64_t t, a_next; uint32_t n, next, swap_used, todo;
  if constexpr (WARPS == 1) {
    t = (int64_t)__shfl_sync(0xffffffffu, hv, 0);
    a_next = (int64_t)__shfl_sync(0xffffffffu, hv, 2);
    const uint64_t w13 = __shfl_sync(0xffffffffu, hv, 13), w14 = __shfl_sync(0xffffffffu, hv, 14);
    const uint64_t w17 = __shfl_sync(0xffffffffu, hv, 17);
    n = (uint32_t)w13; next = (uint32_t)(w13 >> 32); swap_used = (uint32_t)w14; todo = (uint32_t)(w17 >> 32);
  } else {
    if (warp == 0) {
      if (lane == 0) ts->bc64[0] = hv;
      if (lane == 2) ts->bc64[1] = hv;
      if (lane == 13) ts->bc64[2] = hv;
      if (lane == 14) ts->bc64[3] = hv;
      if (lane == 17) ts->bc64[4] = hv;
    }
    __syncthreads();
    t = (int64_t)ts->bc64[0]; a_next = (int64_t)ts->bc64[1];
    n = (uint32_t)ts->bc64[2]; next = (uint32_t)(ts->bc64[2] >> 32);
    swap_used = (uint32_t)ts->bc64[3]; todo = (uint32_t)(ts->bc64[4] >> 32);
    __syncthreads();
  }
  const uint32_t iters = todo ? todo : A.iters;
  bool handed_over = false, ran = false;

  for (uint32_t it = 0; it < iters; it++) {
    // time fence (JSQ router, rule M18): only iterations that start before the replica's limit run
    if (A.tlimit && (n != 0 || next < nreq) && (n == 0 && a_next > t ? a_next : t) >= A.tlimit[r]) break;
    // ---------------- a0: idle jump + ingest (M6)
    if (n == 0) {
      if (next >= nreq) break;                  // done: this and all later iterations are no-ops
      if (a_next > t) t = a_next;
    }
    uint32_t cnt = 0;
    if (a_next <= t && n < Q && next < nreq) {
      const uint32_t avail = (Q - n) < (nreq - next) ? (Q - n) : (nreq - next);
      for (uint32_t base = 0; base < avail; base += TH) {
        const uint32_t i = base + tid;
        const bool take = i < avail && __ldg(&TR[next + i].a) <= t;     // arrivals sorted => a prefix
        uint32_t c_;
        if constexpr (WARPS == 1) c_ = __popc(__ballot_sync(0xffffffffu, take));
        else c_ = (uint32_t)__syncthreads_count(take);
        cnt += c_;
        if (c_ < (uint32_t)TH) break;
      }
    }
    if (n + cnt > (uint32_t)CAP) {              // window outgrew this team: hand the replica to the L kernel
      todo = iters - it;
      handed_over = true;
      break;
    }

    // window HBM -> registers (stored order = last priority order), arrivals appended behind it
    Rec0 r0[E]; Rec1 r1[E];
#pragma unroll
    for (int c = 0; c < E; c++) {
      const uint32_t pos = c * TH + tid;
      int4 v0 = make_int4(0, 0, 0, 0), v1 = make_int4(0, 0, 0, 0);
      if (pos < n) {
        v0 = __ldcg(reinterpret_cast<const int4*>(gE0 + pos));
        v1 = __ldcg(reinterpret_cast<const int4*>(gE1 + pos));
      } else if (pos < n + cnt) {
        const uint32_t i = next + (pos - n);
        v0 = __ldg(reinterpret_cast<const int4*>(TR + i));
        v1 = make_int4((int)i, 0, 0, (int)F_DIRTY);
      }
      r0[c] = *reinterpret_cast<Rec0*>(&v0);
      r1[c] = *reinterpret_cast<Rec1*>(&v1);
    }
    next += cnt; n += cnt;
    if (cnt) a_next = (next < nreq) ? __ldg(&TR[next].a) : kNever;

    // ---------------- a1: score (M3-M5).  okey = class<<63 | (key + 2^62); class 0 = MemGuard-locked resident
    uint64_t key[E];
    uint32_t n_dirty = 0;
#pragma unroll
    for (int c = 0; c < E; c++) {
      const uint32_t pos = c * TH + tid;
      key[c] = ~0ull;
      if (pos < n) {
        key[c] = okey_of(s, par, lut, g_tfirst, g_tlast, t, r0[c], r1[c]);
        const uint64_t klass = key[c] >> 63;
        const uint32_t dirty = (r1[c].flags & F_DIRTY) ? 1u : 0u;
        n_dirty += dirty;
        KeyRec kr; kr.okey = key[c]; kr.id = r1[c].id; kr.aux = dirty;
        x_key[pos] = kr;
        // from here on bit 3 of flags carries the class bit of this iteration
        r1[c].flags = (r1[c].flags & ~F_DIRTY) | (klass ? F_DIRTY : 0u);
      }
    }
    if (tid < 6) ts->acc64[tid] = 0ull;
    if (tid < 4) ts->acc32[tid] = 0u;
    if (tid == 0) { ts->bc[0] = 0xFFFFFFFFu; ts->ndirty = 0u; }
    tm.sync();

    // ---------------- a2: order.  The stored order is last iteration's priority order (MemGuard keeps keys
    // piecewise constant).  L0: still sorted -> nothing moves.  L1: few "dirty" requests (arrivals,
    // residency / bin / lock changes) -> rank them against the still-sorted rest.  L2: bitonic sort.
    {
      bool viol = false;
#pragma unroll
      for (int c = 0; c < E; c++) {
        const uint32_t pos = c * TH + tid;
        if (pos > 0 && pos < n) {
          const KeyRec pr = x_key[pos - 1];
          viol |= key_less(key[c], r1[c].id, pr.okey, pr.id);
        }
      }
      if (tm.any(viol)) {
        uint32_t newpos[E];
        uint32_t nd[1] = {n_dirty};
        tm.template sum32<1>(nd);
        const uint32_t m = nd[0];
        bool merged = false;
        if (m <= 16u) {
          // the non-dirty requests must still be sorted among themselves, else fall through to L2
          bool bad = false;
          uint32_t di[E];                       // dirty requests in front of me
          uint32_t carry = 0;
#pragma unroll
          for (int c = 0; c < E; c++) {
            const uint32_t pos = c * TH + tid;
            const bool in = pos < n;
            const uint32_t dirty = in ? x_key[pos].aux : 0u;
            uint32_t tot;
            di[c] = carry + tm.scan_incl(dirty, tot) - dirty;
            carry += tot;
            if (in && !dirty) {
              int p = (int)pos - 1;
              while (p >= 0 && x_key[p].aux) p--;
              if (p >= 0) { const KeyRec pr = x_key[p]; bad |= key_less(key[c], r1[c].id, pr.okey, pr.id); }
            } else if (in) {
              x_dl[di[c]] = (uint16_t)pos;
            }
          }
          if (tid < 16) x_cnt[tid] = 0u;
          if (!tm.any(bad)) {
            tm.sync();                          // publish x_dl / x_cnt
            uint32_t dlt[E];                    // dirty requests that sort before me
#pragma unroll
            for (int c = 0; c < E; c++) dlt[c] = 0;
            for (uint32_t x = 0; x < m; x++) {
              const KeyRec kx = x_key[x_dl[x]];
              uint32_t before = 0;              // requests (clean or dirty) that sort before x
#pragma unroll
              for (int c = 0; c < E; c++) {
                const uint32_t pos = c * TH + tid;
                if (pos < n) {
                  const bool lt = key_less(key[c], r1[c].id, kx.okey, kx.id);
                  before += lt ? 1u : 0u;
                  dlt[c] += lt ? 0u : 1u;         // x sorts before me (used by clean requests only)
                }
              }
              before = __reduce_add_sync(0xffffffffu, before);
              if (lane == 0) {
                if constexpr (WARPS == 1) x_cnt[x] = before; else atomicAdd(&x_cnt[x], before);
              }
            }
            tm.sync();
#pragma unroll
            for (int c = 0; c < E; c++) {
              const uint32_t pos = c * TH + tid;
              if (pos < n) {
                const bool dirty = x_key[pos].aux != 0;
                newpos[c] = dirty ? x_cnt[di[c]] : (pos - di[c]) + dlt[c];
              }
            }
            merged = true;
          }
        }
        if (!merged) {
          uint32_t npad = 1; while (npad < n) npad <<= 1;
          for (uint32_t p = tid; p < npad; p += TH) x_idx[p] = (p < n) ? (uint16_t)p : (uint16_t)0xFFFFu;
          tm.sync();
          for (uint32_t kk = 2; kk <= npad; kk <<= 1) {
            for (uint32_t j = kk >> 1; j > 0; j >>= 1) {
              for (uint32_t i = tid; i < npad; i += TH) {
                const uint32_t l = i ^ j;
                if (l > i) {
                  const uint32_t pa = x_idx[i], pb = x_idx[l];
                  const bool asc = (i & kk) == 0;
                  bool b_lt_a;
                  if (pb == 0xFFFFu) b_lt_a = false;
                  else if (pa == 0xFFFFu) b_lt_a = true;
                  else { const KeyRec ka = x_key[pa], kb = x_key[pb]; b_lt_a = key_less(kb.okey, kb.id, ka.okey, ka.id); }
                  if (b_lt_a == asc) { x_idx[i] = (uint16_t)pb; x_idx[l] = (uint16_t)pa; }
                }
              }
              tm.sync();
            }
          }
          for (uint32_t p = tid; p < n; p += TH) x_key[x_idx[p]].aux = p;     // inverse permutation
          tm.sync();
#pragma unroll
          for (int c = 0; c < E; c++) {
            const uint32_t pos = c * TH + tid;
            if (pos < n) newpos[c] = x_key[pos].aux;
          }
        }
        tm.sync();                              // everybody is done with the key records: reuse the buffer
#pragma unroll
        for (int c = 0; c < E; c++) {
          const uint32_t pos = c * TH + tid;
          if (pos < n) { x_r0[newpos[c]] = r0[c]; x_r1[newpos[c]] = r1[c]; }
        }
        tm.sync();
#pragma unroll
        for (int c = 0; c < E; c++) {
          const uint32_t pos = c * TH + tid;
          if (pos < n) { r0[c] = x_r0[pos]; r1[c] = x_r1[pos]; }
        }
      }
    }

    // ---------------- a3: admission walk as prefix scans (M7; Algorithm 1 "while |B| < M ... U + dU <= B").
    // Round 0 walks everybody up to the first entry that does not fit; if that entry is a non-resident that failed
    // on KV only ("newblocked"), round 1 continues over the residents behind it.  Both rounds are the same scans:
    //   W = incl. scan of min(c, rem);  tok_before = min(T, W - w);  want = min(T, W) - tok_before;
    //   foot = ceil((cached + want)/blk);  Cf = incl. scan of foot;  ok = cnt_before < M & tok_before < T & Cf <= B.
    // ok is monotone along the walk, so the admitted set is a prefix of the walked entries.
    uint32_t want[E];
#pragma unroll
    for (int c = 0; c < E; c++) want[c] = 0;
    uint32_t C = 0, tok = 0, cntb = 0;
    {
      uint32_t start = 0;
      bool only_res = false;
      for (int round = 0; round < 2; round++) {
        uint32_t carryW = tok, carryC = C, carryN = cntb;
        bool failed = false;
        uint32_t f_C = 0, f_tok = 0, f_cnt = 0, f_kv = 0, f_res = 0, f_pos = 0;
#pragma unroll
        for (int c = 0; c < E; c++) {
          const uint32_t base = c * TH;
          if (failed || base >= n || base + TH <= start) continue;     // team-uniform
          const uint32_t pos = base + tid;
          const bool res = (r1[c].flags & F_RESIDENT) != 0;
          const bool valid = pos < n && pos >= start && (!only_res || res);
          const uint32_t rem = r0[c].P + r1[c].d - r1[c].cached;
          const uint32_t w = valid ? (rem < cc ? rem : cc) : 0u;
          uint32_t wtot, ctot, vtot;
          const uint32_t W = carryW + tm.scan_incl(w, wtot);
          const uint32_t tok_before = (W - w) < Tb ? (W - w) : Tb;
          const uint32_t tok_after = W < Tb ? W : Tb;
          const uint32_t wnt = tok_after - tok_before;
          const uint32_t foot = valid ? blocks_of(s, r1[c].cached + wnt) : 0u;
          const uint32_t Cf = carryC + tm.scan_incl(foot, ctot);
          uint32_t cnt_before;
          if (only_res) {
            cnt_before = carryN + tm.scan_incl(valid ? 1u : 0u, vtot) - (valid ? 1u : 0u);
          } else {                                                     // round 0 walks everybody: rank == position
            cnt_before = carryN + (uint32_t)tid;
            vtot = (n - base) < (uint32_t)TH ? (n - base) : (uint32_t)TH;
          }
          const bool ok = valid && cnt_before < M && tok_before < Tb && Cf <= B;
          const bool fail = valid && !ok;
          if (ok) want[c] = wnt;
          if (tm.any(fail)) {
            // the first entry that did not fit, and the walk state in front of it
            if constexpr (WARPS == 1) {
              const uint32_t fm = __ballot_sync(0xffffffffu, fail);
              const int fl = __ffs(fm) - 1;
              f_C = __shfl_sync(0xffffffffu, Cf - foot, fl);
              f_tok = __shfl_sync(0xffffffffu, tok_before, fl);
              f_cnt = __shfl_sync(0xffffffffu, cnt_before, fl);
              f_res = __shfl_sync(0xffffffffu, res ? 1u : 0u, fl);
              f_pos = base + fl;
            } else {
              if (fail) atomicMin(&ts->bc[0], (uint32_t)tid);
              __syncthreads();
              if ((uint32_t)tid == ts->bc[0]) {
                ts->bc[1] = Cf - foot; ts->bc[2] = tok_before; ts->bc[3] = cnt_before; ts->bc[4] = res ? 1u : 0u;
              }
              __syncthreads();
              f_C = ts->bc[1]; f_tok = ts->bc[2]; f_cnt = ts->bc[3]; f_res = ts->bc[4];
              f_pos = base + ts->bc[0];
              __syncthreads();
              if (tid == 0) ts->bc[0] = 0xFFFFFFFFu;
            }
            f_kv = (f_cnt < M && f_tok < Tb) ? 1u : 0u;                // failed on KV only
            failed = true;
          } else {
            carryW += wtot; carryC += ctot; carryN += vtot;
          }
        }
        if (!failed) { C = carryC; tok = carryW < Tb ? carryW : Tb; cntb = carryN; break; }
        C = f_C; tok = f_tok; cntb = f_cnt;
        if (round == 0 && f_kv && !f_res) { start = f_pos + 1; only_res = true; continue; }
        break;
      }
    }

    // ---------------- a4: batch totals (M9) and victim select (M8; SELECTVICTIM / SWAPOUT)
    uint32_t tot5[5] = {0, 0, 0, 0, 0};          // prefill tokens, decode seqs, swap-in blocks, swap-ins, K blocks
    uint32_t evl = 0, evu = 0;                   // M12: low / high halves of the event hashes, summed mod 2^32
#pragma unroll
    for (int c = 0; c < E; c++) {
      const uint32_t pos = c * TH + tid;
      if (pos < n) {
        if (want[c]) {
          const uint32_t rem = r0[c].P + r1[c].d - r1[c].cached;
          if (r1[c].d >= 1 && rem == 1) tot5[1]++; else tot5[0] += want[c];       // decode sequence vs prefill tokens
          ev_add(evl, evu, EV_ADMIT, r1[c].id, want[c]);
          if (r1[c].flags & F_SWAPPED) {                                          // swap-in on admission
            const uint32_t blocks = blocks_of(s, r1[c].cached);
            tot5[2] += blocks; tot5[3]++;
            ev_add(evl, evu, EV_SWAPIN, r1[c].id, blocks);
          }
        } else if (r1[c].flags & F_RESIDENT) {
          tot5[4] += blocks_of(s, r1[c].cached);                             // non-admitted resident keeps its blocks
        }
      }
    }
    tm.template sum32<5>(tot5);
    uint32_t ev2[2] = {evl, evu};
    tm.template sum32<2>(ev2);
    const uint32_t pf_tot = tot5[0], dec_tot = tot5[1], swin_blocks = tot5[2], swin_cnt = tot5[3], kres_tot = tot5[4];
    swap_used -= swin_blocks;
    uint32_t swout_blocks = 0, ev_nsw = 0, ev_nrc = 0;
    uint64_t ev_lost = 0;
    uint32_t evm[E];
#pragma unroll
    for (int c = 0; c < E; c++) evm[c] = 0;
    if (kres_tot > B - C) {                      // team-uniform; rare
      // victims = the suffix of the non-admitted residents (in priority order) whose prefix sum exceeds B - C
      const uint32_t thr = B - C;
      uint32_t carry = 0, ecarry = 0;
      bool mine[E];
#pragma unroll
      for (int c = 0; c < E; c++) {
        const uint32_t pos = c * TH + tid;
        uint32_t v = 0;
        if (pos < n && want[c] == 0 && (r1[c].flags & F_RESIDENT)) v = blocks_of(s, r1[c].cached);
        uint32_t tot, etot;
        const uint32_t ps = carry + tm.scan_incl(v, tot);
        mine[c] = (v > 0) && ps > thr;           // a resident holds >= 1 block, so v > 0 <=> member of K
        const uint32_t ei = ecarry + tm.scan_incl(mine[c] ? 1u : 0u, etot);
        if (mine[c]) x_ev[ei - 1] = make_uint4(r1[c].id, r1[c].cached, (r1[c].flags & F_DIRTY) ? 1u : 0u, pos);
        carry += tot; ecarry += etot;
      }
      tm.sync();
      if (tid == 0) {                            // lowest priority first; the swap pool is a sequential resource
        uint32_t su = swap_used, swo = 0, n_sw = 0, n_rc = 0, ehl = 0, ehu = 0; uint64_t lost = 0;
        for (int e = (int)ecarry - 1; e >= 0; e--) {
          const uint4 q = x_ev[e];
          const uint32_t resb = blocks_of(s, q.y);
          bool do_swap = false;
          if (s.preempt_mode == 1) do_swap = (su + resb <= s.swap_pool);
          else if (s.preempt_mode == 2)
            do_swap = (su + resb <= s.swap_pool) && (2ll * resb * (int64_t)s.swap_ns < 1000ll * s.c_pf * (int64_t)q.y);
          if (do_swap) { su += resb; swo += resb; n_sw++; ev_add(ehl, ehu, EV_EVICT_SWAP, q.x, resb); x_mode[q.w] = 2; }
          else { lost += q.y; n_rc++; ev_add(ehl, ehu, EV_EVICT_RECOMPUTE, q.x, q.y); x_mode[q.w] = 1; }
          g_ne[q.x] = __ldcg(g_ne + q.x) + 1u;
          if (q.z) g_neu[q.x] = __ldcg(g_neu + q.x) + 1u;      // victim was not MemGuard-locked
        }
        ts->bc[8] = su; ts->bc[9] = swo; ts->bc[10] = n_sw; ts->bc[11] = n_rc;
        ts->bc[12] = ehl; ts->bc[13] = ehu; ts->bc64[6] = lost;
      }
      tm.sync();
      swap_used = ts->bc[8]; swout_blocks = ts->bc[9]; ev_nsw = ts->bc[10]; ev_nrc = ts->bc[11];
      ev2[0] += ts->bc[12]; ev2[1] += ts->bc[13]; ev_lost = ts->bc64[6];
#pragma unroll
      for (int c = 0; c < E; c++) if (mine[c]) evm[c] = x_mode[c * TH + tid];
      tm.sync();
    }

    // ---------------- a5: execute one step with the stated cost model (M9), apply (M10)
    const int64_t cost = s.c0 + s.c_pf * (int64_t)pf_tot + s.c_dec * (int64_t)dec_tot +
                         (int64_t)(((uint64_t)(swin_blocks + swout_blocks) * s.swap_ns + 500u) / 1000u);
    const int64_t t_end = t + cost;
    uint32_t tot2[2] = {0, 0};                   // tokens emitted; gaps equal to this iteration's cost
    bool gone[E];
#pragma unroll
    for (int c = 0; c < E; c++) {
      const uint32_t pos = c * TH + tid;
      gone[c] = false;
      if (pos < n) {
        const uint32_t of = r1[c].flags;
        const uint32_t klass = (of & F_DIRTY) ? 1u : 0u;
        const uint32_t d_old = r1[c].d;
        uint32_t nf = of & (F_RESIDENT | F_SWAPPED | F_EMITPREV | F_PREEMPTED);
        const uint32_t id = r1[c].id;
        if (want[c]) {
          if (nf & F_PREEMPTED) g_tpre[id] = __ldcg(g_tpre + id) + t;           // M15: the preemption ends where this iteration starts
          nf = (nf | F_RESIDENT) & ~(F_SWAPPED | F_PREEMPTED);
          r1[c].cached += want[c];
          if (r1[c].cached == r0[c].P + d_old) {               // KV caught up => one token out (M2)
            r1[c].d = d_old + 1; tot2[0]++;
            if (d_old == 0) {
              g_tfirst[id] = t_end;
              { uint32_t l_ = 0, u_ = 0; ev_add(l_, u_, EV_EMIT_FIRST, id, 0); atomicAdd(&ts->acc32[2], l_); atomicAdd(&ts->acc32[3], u_); }
            } else if (nf & F_EMITPREV) {
              tot2[1]++;                                        // gap == this iteration's cost
            } else {
              const int64_t tl = __ldcg(g_tlast + id);
              atomicAdd(&g_hist[tbt_bin(t_end - tl)], 1u);
            }
            nf |= F_EMITPREV;
            if (r1[c].d == r0[c].D) {                           // complete: KV freed at once
              g_tlast[id] = t_end;
              const int64_t tf = (d_old == 0) ? t_end : __ldcg(g_tfirst + id);
              atomicAdd(&ts->acc64[1], (unsigned long long)(tf - r0[c].a));
              atomicAdd(&ts->acc64[2], (unsigned long long)(t_end - r0[c].a));
              atomicAdd(&ts->acc64[3], (unsigned long long)(t_end - tf));
              atomicAdd(&ts->acc64[4], (unsigned long long)(r0[c].D - 1));
              { uint32_t l_ = 0, u_ = 0; ev_add(l_, u_, EV_COMPLETE, id, 0); atomicAdd(&ts->acc32[2], l_); atomicAdd(&ts->acc32[3], u_); }
              atomicAdd(&ts->acc32[0], 1u);
              g_ne[id] = __ldcg(g_ne + id) | 0x80000000u;
              gone[c] = true;
            }
          } else if (nf & F_EMITPREV) {
            g_tlast[id] = t; nf &= ~F_EMITPREV;
          }
        } else {
          if (nf & F_EMITPREV) { g_tlast[id] = t; nf &= ~F_EMITPREV; }   // persist t_last when the streak ends
          if (evm[c] == 1) { r1[c].cached = 0; nf = (nf | F_PREEMPTED) & ~F_RESIDENT; }
          else if (evm[c] == 2) { nf = (nf | F_SWAPPED | F_PREEMPTED) & ~F_RESIDENT; }
          if (evm[c]) g_tpre[id] = __ldcg(g_tpre + id) - t;                     // M15: preempted from the start of this iteration on
        }
        // re-lock at this iteration's bin (M10, G6) and leave the dirty hint for the next iteration's ordering:
        // set when (resident, bin, class) -- the inputs of a BOOST / FCFS key -- change.  SRPT / LAS keys move by
        // one per emitted token for every running request alike, which rarely reorders: not hinted, the ordering
        // step verifies.
        const uint32_t bin = bin_of(par, s.k, signal_of(par, r0[c].P, r0[c].D, d_old));
        uint32_t bin2 = bin;
        if (r1[c].d != d_old) bin2 = bin_of(par, s.k, signal_of(par, r0[c].P, r0[c].D, r1[c].d));
        const bool res2 = (nf & F_RESIDENT) != 0;
        uint32_t klass2 = (par.guard && res2 && bin2 == bin) ? 0u : 1u;
        if (par.policy == 6 || par.policy == 7) klass2 = r1[c].d >= 1u ? 0u : 1u;      // DistBoost, Sarathi: phase = class
        const bool bin_matters = par.policy == 2;
        const bool dirty = (((nf ^ of) & F_RESIDENT) != 0) || (bin_matters && bin2 != bin) || (klass2 != klass);
        if (res2) nf |= (bin + 1u) << F_LOCK_SHIFT;
        if (dirty) nf |= F_DIRTY;
        r1[c].flags = nf;
      }
    }
    tm.template sum32<2>(tot2);                   // (for WARPS > 1 its barriers also publish the smem accumulators)
    if constexpr (WARPS == 1) __syncwarp();
    if (s.ada_ring) {
      // gamma-Ada (M13): the end-to-end latencies of this iteration's completions go to the replica's window in
      // priority order (slot = completion number mod W)
      uint32_t carry = ncomp0;
#pragma unroll
      for (int c = 0; c < E; c++) {
        uint32_t tot;
        const uint32_t inc = tm.scan_incl(gone[c] ? 1u : 0u, tot);
        if (gone[c]) s.ada_ring[(size_t)r * s.ada_W + (carry + inc - 1u) % s.ada_W] = t_end - r0[c].a;
        carry += tot;
      }
    }

    // SRPT / LAS keys drift with every emitted token.  The streaming kernel trusts the dirty hints, so they must cover
    // the drift too: a request whose next (class, key, id) sorts in front of one that is written before it is hinted
    // (the same rule as in ub_stream.cu process()).
    if (par.policy == 1 || par.policy == 3) {
      uint64_t carry = 0;
#pragma unroll
      for (int c = 0; c < E; c++) {
        const uint32_t base = c * TH;
        if (base < n) {
          const uint32_t pos = base + tid;
          const bool keep = pos < n && !gone[c];
          uint64_t comp = 0;
          if (keep) {
            const uint32_t f = r1[c].flags;
            const uint32_t bin2 = bin_of(par, s.k, signal_of(par, r0[c].P, r0[c].D, r1[c].d));
            const uint32_t klass2 = (par.guard && (f & F_RESIDENT) && (f >> F_LOCK_SHIFT) == bin2 + 1u) ? 0u : 1u;
            const uint32_t key2 = par.policy == 1 ? r0[c].D - r1[c].d : signal_of(par, r0[c].P, r0[c].D, r1[c].d);
            comp = ((uint64_t)klass2 << 63) | ((uint64_t)key2 << 32) | (uint64_t)r1[c].id;
          }
          uint64_t tot;
          uint64_t before = tm.scanmax_excl(comp, tot);
          if (carry > before) before = carry;
          if (keep && comp < before) r1[c].flags |= F_DIRTY;
          if (tot > carry) carry = tot;
        }
      }
    }

    // ---------------- write back in priority order, dropping completed requests
    uint32_t n_new = 0;
#pragma unroll
    for (int c = 0; c < E; c++) {
      const uint32_t base = c * TH;
      if (base < n) {
        const uint32_t pos = base + tid;
        const bool keep = pos < n && !gone[c];
        uint32_t tot;
        const uint32_t np = n_new + tm.scan_incl(keep ? 1u : 0u, tot) - 1u;
        if (keep) {
          *reinterpret_cast<int4*>(gE0 + np) = *reinterpret_cast<const int4*>(&r0[c]);
          *reinterpret_cast<int4*>(gE1 + np) = *reinterpret_cast<const int4*>(&r1[c]);
          if (r1[c].flags & F_DIRTY) {                       // the streaming kernel's dirty list (ub_stream.cu)
            const uint32_t slot = atomicAdd(&ts->ndirty, 1u);
            if (slot < kDirtyMax) s.hdr[r].dl[slot] = (uint16_t)np;
          }
        }
        n_new += tot;
      }
    }

    // ---------------- header words (thread i of warp 0 owns word i)
    if (tid == 0 && tot2[1]) atomicAdd(&g_hist[tbt_bin(cost)], tot2[1]);
    tm.sync();                                   // ts->ndirty complete
    {
      const uint32_t evs_lo = ev2[0] + ts->acc32[2], evs_hi = ev2[1] + ts->acc32[3];
      const uint32_t n_done = ts->acc32[0];
      if (warp == 0) {
        switch (lane) {
          case 0: hv = (uint64_t)t_end; break;
          case 1: hv = digest_fold(hv, evs_lo, evs_hi, t_end); break;
          case 2: hv = (uint64_t)a_next; break;
          case 3: hv += n; break;
          case 4: hv += tot2[0]; break;
          case 5: hv += pf_tot; break;
          case 6: hv += dec_tot; break;
          case 7: hv += ev_lost; break;
          case 8: hv += ts->acc64[1]; break;
          case 9: hv += ts->acc64[2]; break;
          case 10: hv += ts->acc64[3]; break;
          case 11: hv += ts->acc64[4]; break;
          case 12: hv += 1; break;
          case 13: hv = (uint64_t)n_new | ((uint64_t)next << 32); break;
          case 14: { uint32_t pk = (uint32_t)(hv >> 32); if (n > pk) pk = n; hv = (uint64_t)swap_used | ((uint64_t)pk << 32); } break;
          case 15: hv += (uint64_t)n_done + ((uint64_t)ev_nrc << 32); break;
          case 16: hv += (uint64_t)ev_nsw + ((uint64_t)swin_cnt << 32); break;
          case 19: hv = (hv & 0xFFFFFFFF00000000ull) | (uint64_t)n_done; break;           // Hdr::last_done
          case 18: { const uint32_t q = ts->ndirty; hv = (hv & 0xFFFFFFFF00000000ull) | (q > kDirtyMax ? kDirtyMax + 1u : q); } break;
          default: break;
        }
      }
    }
    t = t_end; n = n_new; ran = true;
    tm.sync();                                   // window stores / smem accumulators before the next iteration
  }

  // ---------------- header -> HBM; a window that outgrew this team goes to the overflow list of this round
  if (warp == 0) {
    if (lane == 17) hv = (hv & 0xFFFFFFFFull) | ((uint64_t)(handed_over ? todo : 0u) << 32);
    if (lane < 20) ghdr[lane] = hv;
  }
  if (tid == 0) {
    if (handed_over) push_list(A, 3, r);
    else if (ran && n == 0 && next >= nreq) atomicAdd(A.count + 5, 1u);      // finished its trace in this call
  }
}

// ---------------------------------------------------------------------------------------------- kernels

template <int WARPS, int E> struct TeamSmem {
  static constexpr int CAP = 32 * WARPS * E;
  static constexpr size_t XB = (size_t)CAP * 34 + 128;                       // exchange buffer + x_idx + x_dl + x_cnt
  static constexpr size_t BYTES = ((XB + sizeof(TeamScratch) + 15) / 16) * 16;
};

// Teams stride over one work list (and then, for the L kernel, over a second one).
template <int WARPS, int E, int TEAMS>
__global__ void __launch_bounds__(32 * WARPS * TEAMS) k_step(const StepArgs A, const uint32_t slot0, const uint32_t slot1) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int TH = 32 * WARPS;
  const int tix = threadIdx.x / TH;
  unsigned char* base = smem_raw + (size_t)tix * TeamSmem<WARPS, E>::BYTES;
  Team<WARPS> tm;
  tm.ts = reinterpret_cast<TeamScratch*>(base + TeamSmem<WARPS, E>::XB);
  tm.tid = threadIdx.x % TH; tm.lane = threadIdx.x & 31; tm.warp = tm.tid >> 5; tm.phase = 0;
  const uint32_t g = blockIdx.x * TEAMS + tix, nteams = gridDim.x * TEAMS;
  for (int pass = 0; pass < 2; pass++) {
    const uint32_t slot = pass == 0 ? slot0 : slot1;
    if (slot == 0xFFFFFFFFu) continue;
    const uint32_t count = __ldcg(A.count + slot);
    const uint32_t* list = A.list + (size_t)slot * A.s.R;
    for (uint32_t i = g; i < count; i += nteams) team_step<WARPS, E>(tm, A, __ldcg(list + i), base);
  }
}

constexpr int kES = 4, kEM = 4, kEL = 8;         // requests per thread: S 1 warp x 4 = 128, M 4 x 4 = 512, L 8 x 8 = 2048
constexpr int kTeamsS = 4;

int step_configure(uint32_t) {
  cudaError_t e = cudaFuncSetAttribute(k_step<8, kEL, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)TeamSmem<8, kEL>::BYTES);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(k_step<4, kEM, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TeamSmem<4, kEM>::BYTES);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(k_step<1, kES, kTeamsS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(kTeamsS * TeamSmem<1, kES>::BYTES));
  return (int)e;
}

// One scheduler round (`iters` iterations of every live replica) is ONE launch: the streaming kernel (ub_stream.cu)
// visits every replica.  What it does not handle itself (SRPT / LAS / SJF / SPF / DistBoost keys, test-only modes,
// re-key bursts) it queues ONCE for the team kernels and from then on only counts the iterations that replica owes
// (Hdr::todo); replicas are independent, so the owed iterations are run later, all at once, by flush_slow(): L list,
// M list, S list, then the overflow list.  (The 8-warp L kernel needs a whole SM per CTA; launched after every round
// it stalled the stream of k_stream launches by 14 % although its list is empty in config 5.)
static void make_args(StepArgs& A, const SimDev& s, uint32_t* list, uint32_t* count, uint32_t iters, uint32_t rbeg,
                      uint32_t rend) {
  A.s = s; A.list = list; A.count = count; A.iters = iters; A.rbeg = rbeg; A.rend = rend; A.nstat = A.dynbase = A.tick = 0;
  A.live = nullptr; A.drift = 0; A.tlimit = nullptr;
  const uint32_t capS = 32 * kES, capM = 128 * kEM;
  A.thrS = s.Q <= capS ? s.Q : capS - 16;
  A.thrM = s.Q <= capM ? s.Q : capM - 16;
  if (s.all_stream) A.thrS = A.thrM = 0;                                        // (windows are never empty when queued)
}

void launch_step(const SimDev& s, uint32_t* list, uint32_t* count, uint32_t iters, uint32_t rbeg, uint32_t rend,
                 uint32_t tick, const uint32_t* live, bool drift, const int64_t* tlimit, cudaStream_t st) {
  StepArgs A;
  make_args(A, s, list, count, iters, rbeg, rend);
  A.tick = tick & 1u;
  A.drift = drift ? 1u : 0u;
  A.tlimit = tlimit;
  A.live = live;                                                // list mode: positions [rbeg, rend) of the list
  launch_stream(A, st);
}

// Runs the iterations owed by the queued replicas and empties the lists.
void flush_slow(const SimDev& s, uint32_t* list, uint32_t* count, uint32_t rbeg, uint32_t rend, const int64_t* tlimit,
                cudaStream_t st) {
  StepArgs A;
  make_args(A, s, list, count, 1, rbeg, rend);
  A.tlimit = tlimit;
  const uint32_t R = rend - rbeg;
  const uint32_t gL = R < 148u * 2 ? R : 148u * 2, gM = R < 148u * 8 ? R : 148u * 8;
  const uint32_t nS = (R + kTeamsS - 1) / kTeamsS, gS = nS < 148u * 10 ? nS : 148u * 10;
  k_step<8, kEL, 1><<<gL, 256, TeamSmem<8, kEL>::BYTES, st>>>(A, 2u, 0xFFFFFFFFu);
  if (!s.all_stream) {                           // (else nothing can be queued for the smaller teams)
    k_step<4, kEM, 1><<<gM, 128, TeamSmem<4, kEM>::BYTES, st>>>(A, 1u, 0xFFFFFFFFu);
    k_step<1, kES, kTeamsS><<<gS, 32 * kTeamsS, kTeamsS * TeamSmem<1, kES>::BYTES, st>>>(A, 0u, 0xFFFFFFFFu);
    k_step<8, kEL, 1><<<gL, 256, TeamSmem<8, kEL>::BYTES, st>>>(A, 3u, 0xFFFFFFFFu);
  }
  cudaMemsetAsync(count, 0, 4 * sizeof(uint32_t), st);                          // the lists are empty again
}

}  // namespace ub
