// ub_fast.cu -- the lean scheduling-step kernels of libuniboost.so (sm_100a): ONE WARP advances one replica by one
// (or `iters`) scheduler iterations of Algorithm 1 under the model rules M1..M12 of DESIGN.md Sec. 3.
//
// The replica's active window (kept in HBM in the priority order of the last iteration) is streamed
// HBM -> registers -> HBM once per iteration, one 16-byte record of each array per lane and chunk of 32 requests:
//   a0 ingest / idle jump  (M6)   arrivals are read from the packed trace and appended behind the window
//   a1 score               (M3-M5) boost table held in registers (lane b holds LUT[b]), looked up by shuffle
//   a2 order               the stored order is verified with one neighbour compare; the few re-keyed ("dirty")
//                          requests -- arrivals, residency / bin / lock changes -- are ranked against the rest by
//                          ballots and the records are permuted through shared memory, then verified again
//   a3 admit               (M7) two warp scans per chunk (tokens, KV blocks) + ballot for the first misfit
//   a5 advance             (M9-M10, M12) counters by redux.sync + RED, compaction by ballot / popc
// The common path is straight-line predicated code; everything rare sits behind one warp vote.  Two instances:
// k_fast<2> visits every replica (windows up to 64 requests), k_fast<4> takes the list of windows up to 128.
// Anything else -- larger windows, an eviction (a4, M8), more than 8 dirty requests, an order that the insertion
// cannot restore, the SRPT / LAS keys (they drift every token) and the test-only signal / quantiser modes -- is
// decided BEFORE any global write and handed to the general team kernels of ub_step.cu through the work lists of
// the same round; all kernels share the HBM state, so a replica may change path in any iteration.  Integers only.
#include "ub_device.cuh"

namespace ub {

constexpr int kFWarps = 4;                 // warps (= replicas) per CTA
constexpr int kFCapMax = 128;
constexpr uint32_t kMaxMerge = 8;          // dirty requests inserted in-warp; more => team kernel
constexpr uint32_t kFull = 0xffffffffu;

// inclusive warp scan, one SHFL + one predicated add per step (the shuffle's own "source lane in range" predicate)
__device__ __forceinline__ uint32_t scan32(uint32_t v) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    asm volatile("{ .reg .u32 t; .reg .pred p; shfl.sync.up.b32 t|p, %0, %1, 0x0, 0xffffffff; @p add.u32 %0, %0, t; }"
                 : "+r"(v) : "r"(o));
  }
  return v;
}

template <int E> struct __align__(16) FastSmem {      // per warp: exchange buffer of the in-warp permutation
  uint4 r0[32 * E];
  uint4 r1[32 * E];
  uint4 kb[32 * E];                                   // {key lo, key hi, bin, -}
};

template <int E, bool LIST>
__global__ void __launch_bounds__(32 * kFWarps) k_fast(const StepArgs A) {
  __shared__ FastSmem<E> sm[kFWarps];
  constexpr uint32_t CAP = 32 * E;
  const SimDev& s = A.s;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  uint32_t r = blockIdx.x * kFWarps + wib;
  if (LIST) {
    if (r >= __ldcg(A.count + 4)) return;
    r = __ldcg(A.list + (size_t)4 * s.R + r);
  } else if (r >= s.R) return;
  const uint32_t ltmask = (1u << lane) - 1u;
  FastSmem<E>& X = sm[wib];

  // ---- header words (Hdr, ub_internal.cuh): uniform loads, no shuffles
  unsigned long long* h64 = reinterpret_cast<unsigned long long*>(s.hdr + r);
  int64_t t = (int64_t)__ldcg(h64 + 0);
  uint64_t H = __ldcg(h64 + 1);
  int64_t a_next = (int64_t)__ldcg(h64 + 2);
  const unsigned long long w13 = __ldcg(h64 + 13), w14 = __ldcg(h64 + 14);
  uint32_t n = (uint32_t)w13, next = (uint32_t)(w13 >> 32);
  uint32_t swap_used = (uint32_t)w14, peak = (uint32_t)(w14 >> 32);
  if (n == 0 && a_next == kNever) return;                           // finished its trace
  uint32_t iters = A.iters;
  if (LIST) {                                                       // iterations the first instance left to do
    const uint32_t todo = (uint32_t)(__ldcg(h64 + 17) >> 32);
    if (todo) { iters = todo; reinterpret_cast<uint32_t*>(h64 + 17)[1] = 0u; }
  }

  const RepPar par = s.par[r];
  const Rec0* TR = s.TR + (size_t)par.trace_id * s.N;
  Rec0* gE0 = s.E0 + (size_t)r * s.Q;
  Rec1* gE1 = s.E1 + (size_t)r * s.Q;
  const uint32_t B = s.B, M = s.M, cc = s.c, Tb = s.T, Q = s.Q, k = s.k;
  const uint32_t blk_m1 = s.blk - 1u, blk_sh = s.blk_shift;
  const bool isboost = par.policy == 2;
  const int64_t delta = par.delta;
  const bool guard = par.guard != 0;

  // boost table in registers: lane b holds LUT[b] (Eq. 2 in fixed point, built on the host, M4); FCFS: all 0
  uint32_t it = 0;
  uint32_t wsize = n;                                               // window size seen when leaving (list class)
  // the lean path covers arrival-keyed policies with the paper's signal and quantiser and a power-of-two block
  bool slow = !(par.policy == 0 || par.policy == 2) || par.signal_mode != 0 || par.quant_mode != 0 || blk_sh >= 32u;
  int64_t lutv = 0;
  if (isboost && !slow) lutv = __ldg(s.lut + par.lut_off + lane);   // geometric tables have 64 entries, bins < 32
  bool grow = false;                                                // window too large for this instance only

  for (; !slow && it < iters; it++) {
    // ---------------- a0: idle jump + ingest (M6)
    if (n == 0) {
      if (a_next == kNever) break;
      if (a_next > t) t = a_next;
    }
    uint32_t cnt = 0, nreq = 0;
    if (a_next <= t && n < Q) {                                     // a_next != kNever => next < nreq
      nreq = __ldg(s.n_req + par.trace_id);
      const uint32_t avail = (Q - n) < (nreq - next) ? (Q - n) : (nreq - next);
      const bool take = (uint32_t)lane < avail && __ldg(&TR[next + lane].a) <= t;   // arrivals sorted => a prefix
      cnt = __popc(__ballot_sync(kFull, take));
      if (cnt == 32u && avail > 32u) cnt = 2 * kFCapMax;            // maybe more: not for this kernel
    }
    wsize = n + cnt;
    if (wsize > CAP) { slow = true; grow = wsize <= (uint32_t)kFCapMax && CAP < (uint32_t)kFCapMax; break; }

    // window HBM -> registers (stored order = last priority order), arrivals appended behind it
    const uint32_t n_old = n;
    n += cnt;
    Rec0 r0[E]; Rec1 r1[E];
#pragma unroll
    for (int c = 0; c < E; c++) {
      const uint32_t pos = c * 32 + lane;
      int4 v0 = make_int4(0, 0, 0, 0), v1 = make_int4(0, 0, 0, 0);
      if (pos < n_old) {
        v0 = __ldcg(reinterpret_cast<const int4*>(gE0 + pos));
        v1 = __ldcg(reinterpret_cast<const int4*>(gE1 + pos));
      }
      r0[c] = *reinterpret_cast<Rec0*>(&v0);
      r1[c] = *reinterpret_cast<Rec1*>(&v1);
    }
    if (cnt) {
#pragma unroll
      for (int c = 0; c < E; c++) {
        const uint32_t pos = c * 32 + lane;
        if (pos >= n_old && pos < n) {
          const uint32_t i = next + (pos - n_old);
          const int4 v0 = __ldg(reinterpret_cast<const int4*>(TR + i));
          r0[c] = *reinterpret_cast<const Rec0*>(&v0);
          r1[c].id = i; r1[c].flags = F_DIRTY;
        }
      }
      next += cnt;
      a_next = (next < nreq) ? __ldg(&TR[next].a) : kNever;
    }

    // ---------------- a1: score (M3-M5).  sig = P + d; bin = Eq. 8 exponent; pi = a - b_gamma(w_hat)
    // - delta if resident (Eq. 7); key = class<<63 | (pi + 2^62); class 0 = MemGuard-locked resident
    uint64_t key[E]; uint32_t bin[E];
#pragma unroll
    for (int c = 0; c < E; c++) {
      const uint32_t sig = r0[c].P + r1[c].d;
      const uint32_t sg = sig > k ? sig : k;
      uint32_t b = (uint32_t)(__clz(k) - __clz(sg));
      b -= ((k << b) > sg) ? 1u : 0u;
      const uint32_t lo = __shfl_sync(kFull, (uint32_t)lutv, (int)b);
      const uint32_t hi = __shfl_sync(kFull, (uint32_t)((uint64_t)lutv >> 32), (int)b);
      const bool res = (r1[c].flags & F_RESIDENT) != 0;
      const int64_t kv = r0[c].a - (int64_t)(((uint64_t)hi << 32) | lo) - (res ? delta : 0ll);
      const bool locked = guard && res && (r1[c].flags >> F_LOCK_SHIFT) == b + 1u;
      const uint64_t kk = (uint64_t)(kv + kKeyBias) | (locked ? 0ull : (1ull << 63));
      key[c] = (uint32_t)(c * 32 + lane) < n ? kk : ~0ull;
      bin[c] = b;
    }

    // ---------------- a2: order.  MemGuard keeps keys piecewise constant: the stored order is still
    // the priority order unless a request was re-keyed.  Verify; if violated, insert the dirty requests by rank.
    auto out_of_order = [&]() -> bool {
      bool viol = false;
#pragma unroll
      for (int c = 0; c < E; c++) {
        uint64_t pk = __shfl_up_sync(kFull, key[c], 1);
        uint32_t pi = __shfl_up_sync(kFull, r1[c].id, 1);
        if (c > 0) {
          const uint64_t qk = __shfl_sync(kFull, key[c > 0 ? c - 1 : 0], 31);
          const uint32_t qi = __shfl_sync(kFull, r1[c > 0 ? c - 1 : 0].id, 31);
          if (lane == 0) { pk = qk; pi = qi; }
        }
        const uint32_t pos = c * 32 + lane;
        viol |= pos > 0 && pos < n && key_less(key[c], r1[c].id, pk, pi);
      }
      return __any_sync(kFull, viol);
    };
    bool permuted = false;
    if (out_of_order()) {
      uint32_t dm[E]; uint32_t m = 0;
#pragma unroll
      for (int c = 0; c < E; c++) {
        dm[c] = __ballot_sync(kFull, (uint32_t)(c * 32 + lane) < n && (r1[c].flags & F_DIRTY));
        m += __popc(dm[c]);
      }
      if (m == 0u || m > kMaxMerge) { slow = true; break; }
      uint32_t dlt[E], myrank[E];
#pragma unroll
      for (int c = 0; c < E; c++) { dlt[c] = 0; myrank[c] = 0; }
#pragma unroll
      for (int cx = 0; cx < E; cx++) {
        uint32_t mm = dm[cx];
        while (mm) {                                                // warp-uniform: one dirty request x at a time
          const int lx = __ffs(mm) - 1; mm &= mm - 1u;
          const uint64_t kx = __shfl_sync(kFull, key[cx], lx);
          const uint32_t ix = __shfl_sync(kFull, r1[cx].id, lx);
          uint32_t before = 0;                                      // requests (clean or dirty) that sort before x
#pragma unroll
          for (int c = 0; c < E; c++) {
            const bool in = (uint32_t)(c * 32 + lane) < n;
            const bool lt = in && key_less(key[c], r1[c].id, kx, ix);
            before += __popc(__ballot_sync(kFull, lt));
            dlt[c] += (in && !lt) ? 1u : 0u;                        // x sorts before me (used by clean requests)
          }
          if (lane == lx) myrank[cx] = before;
        }
      }
      uint32_t dcarry = 0;
      bool clash = false;
      uint32_t newpos[E];
#pragma unroll
      for (int c = 0; c < E; c++) {
        const uint32_t pos = c * 32 + lane;
        const bool isd = (dm[c] >> lane) & 1u;
        const uint32_t di = dcarry + __popc(dm[c] & ltmask);        // dirty requests stored in front of me
        dcarry += __popc(dm[c]);
        newpos[c] = isd ? myrank[c] : (pos - di) + dlt[c];
        if (pos < n) {
          X.r0[newpos[c]] = *reinterpret_cast<const uint4*>(&r0[c]);
          X.r1[newpos[c]] = *reinterpret_cast<const uint4*>(&r1[c]);
          X.kb[newpos[c]] = make_uint4((uint32_t)key[c], (uint32_t)(key[c] >> 32), bin[c], 0u);
        }
      }
      __syncwarp();
      // the ranks are a permutation iff every request still finds its own record (the clean ones were sorted)
#pragma unroll
      for (int c = 0; c < E; c++)
        if ((uint32_t)(c * 32 + lane) < n) clash |= X.r1[newpos[c]].x != r1[c].id;
      if (__any_sync(kFull, clash)) { slow = true; break; }
#pragma unroll
      for (int c = 0; c < E; c++) {
        const uint32_t pos = c * 32 + lane;
        if (pos < n) {
          const uint4 a0 = X.r0[pos], a1 = X.r1[pos], ak = X.kb[pos];
          r0[c] = *reinterpret_cast<const Rec0*>(&a0);
          r1[c] = *reinterpret_cast<const Rec1*>(&a1);
          key[c] = (uint64_t)ak.x | ((uint64_t)ak.y << 32); bin[c] = ak.z;
        }
      }
      __syncwarp();
      if (out_of_order()) { slow = true; break; }
      permuted = true;
    }
    uint32_t resm[E];                                               // residents of each chunk (ballot)
#pragma unroll
    for (int c = 0; c < E; c++) resm[c] = __ballot_sync(kFull, (r1[c].flags & F_RESIDENT) != 0);

    // ---------------- a3: admission walk as prefix scans (M7; Algorithm 1 "while |B| < M ... U + dU <= B").
    // Round 0 walks everybody; per chunk
    //   W = incl. scan of min(c, rem);  tok_before = min(T, W - w);  want = min(T, W) - tok_before;
    //   foot = ceil((cached + want)/blk);  Cf = incl. scan of foot;  ok = pos < M & tok_before < T & Cf <= B.
    // ok is monotone along the walk, so the admitted set is the prefix in front of the first misfit.  If that one is
    // a non-resident that failed on KV only ("newblocked") and residents follow it, round 1 continues over them.
    uint32_t want[E];
    uint32_t C, tok;
    {
      uint32_t carryW = 0, carryC = 0;
      bool failed = false;
      uint32_t f_C = 0, f_tok = 0, f_pos = 0, f_res = 0;
#pragma unroll
      for (int c = 0; c < E; c++) {
        const uint32_t pos = c * 32 + lane;
        const bool in = pos < n;
        const uint32_t rem = r0[c].P + r1[c].d - r1[c].cached;
        const uint32_t w = in ? (rem < cc ? rem : cc) : 0u;
        const uint32_t W = carryW + scan32(w);
        const uint32_t tok_before = (W - w) < Tb ? (W - w) : Tb;
        const uint32_t tok_after = W < Tb ? W : Tb;
        const uint32_t wnt = tok_after - tok_before;
        const uint32_t foot = in ? (r1[c].cached + wnt + blk_m1) >> blk_sh : 0u;
        const uint32_t Cf = carryC + scan32(foot);
        const bool ok = in && pos < M && tok_before < Tb && Cf <= B;
        want[c] = ok ? wnt : 0u;
        const uint32_t fm = __ballot_sync(kFull, in && !ok);
        if (fm && !failed) {                                        // the first request that did not fit
          const int fl = __ffs(fm) - 1;
          f_C = __shfl_sync(kFull, Cf - foot, fl);
          f_tok = __shfl_sync(kFull, tok_before, fl);
          f_res = (resm[c] >> fl) & 1u;
          f_pos = c * 32 + fl;
          failed = true;
        }
        carryW = __shfl_sync(kFull, W, 31);
        carryC = __shfl_sync(kFull, Cf, 31);
      }
      C = carryC; tok = carryW < Tb ? carryW : Tb;
      if (failed) {
        C = f_C; tok = f_tok;
        bool behind = false;                                        // residents behind the blocked newcomer?
#pragma unroll
        for (int c = 0; c < E; c++) {
          const int sh = (int)f_pos + 1 - c * 32;
          const uint32_t msk = sh <= 0 ? kFull : (sh >= 32 ? 0u : (kFull << sh));
          behind |= (resm[c] & msk) != 0u;
        }
        if (f_pos < M && f_tok < Tb && !f_res && behind) {          // round 1: residents only, from f_pos + 1
          uint32_t cW = f_tok, cC = f_C, cN = f_pos;
          bool stop = false;
#pragma unroll
          for (int c = 0; c < E; c++) {
            if (stop || (uint32_t)(c * 32 + 32) <= f_pos + 1u) continue;       // warp-uniform
            const uint32_t pos = c * 32 + lane;
            const bool valid = pos < n && pos > f_pos && ((resm[c] >> lane) & 1u);
            const uint32_t rem = r0[c].P + r1[c].d - r1[c].cached;
            const uint32_t w = valid ? (rem < cc ? rem : cc) : 0u;
            const uint32_t W = cW + scan32(w);
            const uint32_t tok_before = (W - w) < Tb ? (W - w) : Tb;
            const uint32_t tok_after = W < Tb ? W : Tb;
            const uint32_t wnt = tok_after - tok_before;
            const uint32_t foot = valid ? (r1[c].cached + wnt + blk_m1) >> blk_sh : 0u;
            const uint32_t Cf = cC + scan32(foot);
            const uint32_t vm = __ballot_sync(kFull, valid);
            const uint32_t cnt_before = cN + __popc(vm & ltmask);
            const bool ok = valid && cnt_before < M && tok_before < Tb && Cf <= B;
            if (ok) want[c] = wnt;
            const uint32_t fm = __ballot_sync(kFull, valid && !ok);
            if (fm) {
              const int fl = __ffs(fm) - 1;
              C = __shfl_sync(kFull, Cf - foot, fl);
              stop = true;
            } else {
              cW = __shfl_sync(kFull, W, 31);
              cC = __shfl_sync(kFull, Cf, 31);
              cN += __popc(vm);
              C = cC;
            }
          }
        }
      }
    }

    // ---------------- batch totals (M9).  Stalled residents must still fit behind the claims (M8): if they do not,
    // victims have to be selected -> team kernel (nothing has been written yet).
    uint32_t pf = 0, dec = 0, kres = 0, evl = 0, evu = 0;
    bool swp = false;
#pragma unroll
    for (int c = 0; c < E; c++) {
      const bool adm = want[c] != 0u;
      const uint32_t rem = r0[c].P + r1[c].d - r1[c].cached;
      const bool isdec = adm && r1[c].d >= 1u && rem == 1u;         // decode sequence vs prefill tokens
      dec += isdec ? 1u : 0u;
      pf += isdec ? 0u : want[c];
      const uint32_t m32 = ((r1[c].id + 1u) * 0x9E3779B1u) ^ ((uint32_t)EV_ADMIT * 0x85EBCA6Bu);
      const uint64_t h = (uint64_t)m32 * (uint64_t)(2u * want[c] + 1u);
      evl += adm ? (uint32_t)h : 0u;
      evu += adm ? (uint32_t)(h >> 32) : 0u;
      swp |= adm && (r1[c].flags & F_SWAPPED);
      const bool stalled = !adm && ((resm[c] >> lane) & 1u);
      kres += stalled ? (r1[c].cached + blk_m1) >> blk_sh : 0u;
    }
    pf = __reduce_add_sync(kFull, pf);
    dec = __reduce_add_sync(kFull, dec);
    kres = __reduce_add_sync(kFull, kres);
    if (kres > B - C) { slow = true; break; }
    uint32_t swin_blocks = 0, swin_cnt = 0;
    if (__any_sync(kFull, swp)) {                                   // swap-in on admission (rare)
#pragma unroll
      for (int c = 0; c < E; c++) {
        if (want[c] && (r1[c].flags & F_SWAPPED)) {
          const uint32_t blocks = (r1[c].cached + blk_m1) >> blk_sh;
          swin_blocks += blocks; swin_cnt++;
          ev_add(evl, evu, EV_SWAPIN, r1[c].id, blocks);
        }
      }
      swin_blocks = __reduce_add_sync(kFull, swin_blocks);
      swin_cnt = __reduce_add_sync(kFull, swin_cnt);
      swap_used -= swin_blocks;
    }

    // ---------------- a5: execute one step with the stated cost model (M9), apply (M10)
    const int64_t cost = s.c0 + s.c_pf * (int64_t)pf + s.c_dec * (int64_t)dec +
                         (int64_t)(((uint64_t)swin_blocks * s.swap_ns + 500u) / 1000u);
    const int64_t t_end = t + cost;
    uint32_t emit = 0, same = 0;
    uint32_t gonem[E], nflags[E];
#pragma unroll
    for (int c = 0; c < E; c++) {
      const bool in = (uint32_t)(c * 32 + lane) < n;
      const bool adm = want[c] != 0u;
      const uint32_t of = r1[c].flags;
      const uint32_t d_old = r1[c].d;
      const uint32_t sig = r0[c].P + d_old;
      r1[c].cached += want[c];
      const bool emitted = adm && r1[c].cached == sig;              // KV caught up => one token out (M2)
      const bool ep_old = (of & F_EMITPREV) != 0;
      r1[c].d = d_old + (emitted ? 1u : 0u);
      emit += emitted ? 1u : 0u;
      same += (emitted && d_old != 0u && ep_old) ? 1u : 0u;         // gap == this iteration's cost
      const bool gone = emitted && r1[c].d == r0[c].D;              // complete: KV freed at once
      uint32_t nf = of & (F_RESIDENT | F_SWAPPED);
      if (adm) nf = F_RESIDENT;
      if (emitted) nf |= F_EMITPREV;
      // re-lock at this iteration's bin (M10, G6); dirty hint for the next iteration's ordering: set when
      // (resident, bin, class) -- the inputs of the key -- change
      const uint32_t b = bin[c];
      const uint32_t b2 = b + ((emitted && sig + 1u == (k << (b + 1u))) ? 1u : 0u);
      const bool res2 = (nf & F_RESIDENT) != 0;
      const uint32_t klass = (uint32_t)(key[c] >> 63);
      const uint32_t klass2 = (guard && res2 && b2 == b) ? 0u : 1u;
      const bool dirty = (((nf ^ of) & F_RESIDENT) != 0) || (isboost && b2 != b) || (klass2 != klass);
      if (res2) nf |= (b + 1u) << F_LOCK_SHIFT;
      if (dirty) nf |= F_DIRTY;
      nflags[c] = nf;
      gonem[c] = __ballot_sync(kFull, gone);
      // everything that touches the per-request outputs is rare: first token, a gap after a stall, completion,
      // the end of an emission streak (t_last is implicit while a request emits every iteration)
      const bool rare = in && (emitted ? (d_old == 0u || !ep_old || gone) : ep_old);
      if (__any_sync(kFull, rare)) {
        if (rare) {
          const uint32_t id = r1[c].id;
          int64_t* g_tfirst = s.t_first + (size_t)r * s.N;
          int64_t* g_tlast = s.t_last + (size_t)r * s.N;
          if (emitted) {
            if (d_old == 0u) {
              g_tfirst[id] = t_end;
              ev_add(evl, evu, EV_EMIT_FIRST, id, 0u);
            } else if (!ep_old) {
              const int64_t tl = __ldcg(g_tlast + id);
              atomicAdd(s.hist + (size_t)r * kTbtBins + tbt_bin(t_end - tl), 1u);
            }
            if (gone) {
              g_tlast[id] = t_end;
              const int64_t tf = (d_old == 0u) ? t_end : __ldcg(g_tfirst + id);
              atomicAdd(h64 + 8, (unsigned long long)(tf - r0[c].a));
              atomicAdd(h64 + 9, (unsigned long long)(t_end - r0[c].a));
              atomicAdd(h64 + 10, (unsigned long long)(t_end - tf));
              atomicAdd(h64 + 11, (unsigned long long)(r0[c].D - 1u));
              ev_add(evl, evu, EV_COMPLETE, id, 0u);
              uint32_t* g_ne = s.n_evict + (size_t)r * s.N;
              g_ne[id] = __ldcg(g_ne + id) | 0x80000000u;           // completion marker read by the stats kernel
            }
          } else {
            g_tlast[id] = t;                                        // persist t_last when the streak ends
          }
        }
      }
    }
    emit = __reduce_add_sync(kFull, emit);
    same = __reduce_add_sync(kFull, same);
    evl = __reduce_add_sync(kFull, evl);
    evu = __reduce_add_sync(kFull, evu);

    // ---------------- write back in priority order, dropping completed requests; untouched records stay put
    uint32_t n_new = 0, n_done = 0;
#pragma unroll
    for (int c = 0; c < E; c++) {
      const uint32_t pos = c * 32 + lane;
      const bool keep = pos < n && !((gonem[c] >> lane) & 1u);
      const uint32_t km = __ballot_sync(kFull, keep);
      const uint32_t np = n_new + __popc(km & ltmask);
      const bool moved = permuted || np != pos || pos >= n_old;
      const bool changed = want[c] != 0u || nflags[c] != r1[c].flags;
      r1[c].flags = nflags[c];
      if (keep && moved) __stcg(reinterpret_cast<int4*>(gE0 + np), *reinterpret_cast<const int4*>(&r0[c]));
      if (keep && (moved || changed)) __stcg(reinterpret_cast<int4*>(gE1 + np), *reinterpret_cast<const int4*>(&r1[c]));
      n_new += __popc(km);
      n_done += __popc(gonem[c]);
    }

    // ---------------- header: clock, digest (M12), cursors; counters by RED (no read needed)
    H = digest_fold(H, evl, evu, t_end);
    if (lane == 0) {
      if (same) atomicAdd(s.hist + (size_t)r * kTbtBins + tbt_bin(cost), same);
      __stcg(h64 + 0, (unsigned long long)t_end);
      __stcg(h64 + 1, (unsigned long long)H);
      if (cnt) __stcg(h64 + 2, (unsigned long long)a_next);
      __stcg(h64 + 13, (unsigned long long)n_new | ((unsigned long long)next << 32));
      if (n > peak || swin_blocks)
        __stcg(h64 + 14, (unsigned long long)swap_used | ((unsigned long long)(n > peak ? n : peak) << 32));
      atomicAdd(h64 + 3, (unsigned long long)n);                    // request-steps
      atomicAdd(h64 + 4, (unsigned long long)emit);
      if (pf) atomicAdd(h64 + 5, (unsigned long long)pf);
      atomicAdd(h64 + 6, (unsigned long long)dec);
      atomicAdd(h64 + 12, 1ull);                                    // iterations
      if (n_done) atomicAdd(reinterpret_cast<uint32_t*>(h64 + 15), n_done);
      if (swin_cnt) atomicAdd(reinterpret_cast<uint32_t*>(h64 + 16) + 1, swin_cnt);
    }
    if (n > peak) peak = n;
    t = t_end; n = n_new; wsize = n_new;
    if (n == 0 && a_next == kNever) {                               // finished its trace in this call
      if (lane == 0) atomicAdd(A.count + 5, 1u);
      it++;
      break;
    }
    __syncwarp();                                                   // window stores before the next iteration's loads
  }

  // ---------------- not handled here: queue the replica for the next kernel of this round
  if (slow && lane == 0) {
    if (it > 0 || (LIST && iters != A.iters)) reinterpret_cast<uint32_t*>(h64 + 17)[1] = iters - it;   // still to do
    const uint32_t cls = grow ? 4u : (wsize <= A.thrS ? 0u : (wsize <= A.thrM ? 1u : 2u));
    push_list(A, cls, r);
  }
}

int fast_configure() { return 0; }

// k_fast<2> visits every replica; k_fast<4> takes list 4 (windows of 65..128 requests)
void launch_fast(const StepArgs& A, cudaStream_t st) {
  const uint32_t grid = (A.s.R + kFWarps - 1) / kFWarps;
  k_fast<2, false><<<grid, 32 * kFWarps, 0, st>>>(A);
  k_fast<4, true><<<grid, 32 * kFWarps, 0, st>>>(A);
}

}  // namespace ub
