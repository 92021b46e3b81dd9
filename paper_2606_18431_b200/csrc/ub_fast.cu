// ub_fast.cu -- the lean scheduling-step kernel of libuniboost.so (sm_100a): ONE WARP advances one replica by one
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
// Anything else -- a window above 128 requests, an eviction (a4, M8), more than 8 dirty requests, an order that the
// insertion cannot restore (SRPT / LAS keys drift every token) -- is decided BEFORE any global write and handed to
// the general team kernels of ub_step.cu through the work lists of the same round; both kernels share the HBM
// state, so a replica may change path in any iteration.  Integer arithmetic only.
#include "ub_device.cuh"

namespace ub {

constexpr int kFE = 4;                     // chunks of 32 requests a warp holds: windows up to 128 requests
constexpr int kFWarps = 4;                 // warps (= replicas) per CTA
constexpr int kFCap = 32 * kFE;
constexpr uint32_t kMaxMerge = 8;          // dirty requests inserted in-warp; more => team kernel
constexpr uint32_t kFull = 0xffffffffu;

struct __align__(16) FastSmem {            // per warp: exchange buffer of the in-warp permutation
  uint4 r0[kFCap];
  uint4 r1[kFCap];
  uint4 kb[kFCap];                         // {key lo, key hi, bin, -}
};

__device__ __forceinline__ uint32_t scan32(uint32_t v, int lane) { return warp_scan_incl(v, lane); }

template <int E>
__global__ void __launch_bounds__(32 * kFWarps) k_fast(const StepArgs A) {
  __shared__ FastSmem sm[kFWarps];
  const SimDev& s = A.s;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const uint32_t r = blockIdx.x * kFWarps + wib;
  if (r >= s.R) return;
  const uint32_t ltmask = (1u << lane) - 1u;
  FastSmem& X = sm[wib];

  // ---- header words (Hdr, ub_internal.cuh): uniform loads, no shuffles
  unsigned long long* h64 = reinterpret_cast<unsigned long long*>(s.hdr + r);
  int64_t t = (int64_t)__ldcg(h64 + 0);
  uint64_t H = __ldcg(h64 + 1);
  int64_t a_next = (int64_t)__ldcg(h64 + 2);
  const unsigned long long w13 = __ldcg(h64 + 13), w14 = __ldcg(h64 + 14);
  uint32_t n = (uint32_t)w13, next = (uint32_t)(w13 >> 32);
  uint32_t swap_used = (uint32_t)w14, peak = (uint32_t)(w14 >> 32);
  if (n == 0 && a_next == kNever) return;                           // finished its trace

  const RepPar par = s.par[r];
  const Rec0* TR = s.TR + (size_t)par.trace_id * s.N;
  Rec0* gE0 = s.E0 + (size_t)r * s.Q;
  Rec1* gE1 = s.E1 + (size_t)r * s.Q;
  const int64_t* lut = s.lut + par.lut_off;
  const uint32_t B = s.B, M = s.M, cc = s.c, Tb = s.T, Q = s.Q;

  // boost table in registers: lane b holds LUT[b] (Eq. 2 in fixed point, built on the host, M4)
  int64_t lutv = 0;
  if (par.policy == 2) lutv = __ldg(lut + ((uint32_t)lane < par.lut_nb ? (uint32_t)lane : par.lut_nb - 1u));

  uint32_t it = 0;
  bool slow = n > (uint32_t)kFCap;
  uint32_t wsize = n;                                               // window size seen when leaving (list class)

  for (; !slow && it < A.iters; it++) {
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
      if (cnt == 32u && avail > 32u) { wsize = n + 64u; slow = true; break; }
    }
    wsize = n + cnt;
    if (n + cnt > (uint32_t)kFCap) { slow = true; break; }

    // window HBM -> registers (stored order = last priority order), arrivals appended behind it
    Rec0 r0[E]; Rec1 r1[E];
#pragma unroll
    for (int c = 0; c < E; c++) {
      const uint32_t pos = c * 32 + lane;
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
    const uint32_t n_old = n;
    next += cnt; n += cnt;
    if (cnt) a_next = (next < nreq) ? __ldg(&TR[next].a) : kNever;

    // ---------------- a1: score (M3-M5).  key = class<<63 | (pi + 2^62); class 0 = MemGuard-locked resident
    uint64_t key[E]; uint32_t bin[E];
#pragma unroll
    for (int c = 0; c < E; c++) {
      key[c] = ~0ull; bin[c] = 0;
      if (c * 32 < (int)n) {
        const uint32_t sig = signal_of(par, r0[c].P, r0[c].D, r1[c].d);
        const uint32_t b = bin_of(par, s.k, sig);
        int64_t kv;
        if (par.policy == 0) kv = r0[c].a;
        else if (par.policy == 1) kv = (int64_t)(r0[c].D - r1[c].d);
        else if (par.policy == 3) kv = (int64_t)sig;
        else {                                                      // pi = a - b_gamma(w_hat)
          const uint32_t bi = b < par.lut_nb ? b : par.lut_nb - 1u;
          int64_t bv = __shfl_sync(kFull, lutv, (int)(bi & 31u));
          if (__any_sync(kFull, bi >= 32u)) { if (bi >= 32u) bv = __ldg(lut + bi); }
          kv = r0[c].a - bv;
        }
        const bool res = (r1[c].flags & F_RESIDENT) != 0;
        if (res && (par.policy == 0 || par.policy == 2)) kv -= par.delta;           // Eq. 7 as a bias
        const uint32_t lockp1 = r1[c].flags >> F_LOCK_SHIFT;
        const uint64_t klass = (par.guard && res && lockp1 == b + 1u) ? 0ull : 1ull;
        if (c * 32 + lane < (int)n) { key[c] = (klass << 63) | (uint64_t)(kv + kKeyBias); bin[c] = b; }
      }
    }

    // ---------------- a2: order.  MemGuard keeps keys piecewise constant: the stored order is still
    // the priority order unless a request was re-keyed.  Verify; if violated, insert the dirty requests by rank.
    auto out_of_order = [&]() -> bool {
      bool viol = false;
#pragma unroll
      for (int c = 0; c < E; c++) {
        if (c * 32 < (int)n) {
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
    // Round 0 walks everybody up to the first request that does not fit; if that one is a non-resident that failed on
    // KV only ("newblocked"), round 1 continues over the residents behind it.  Per chunk:
    //   W = incl. scan of min(c, rem);  tok_before = min(T, W - w);  want = min(T, W) - tok_before;
    //   foot = ceil((cached + want)/blk);  Cf = incl. scan of foot;  ok = cnt_before < M & tok_before < T & Cf <= B.
    uint32_t want[E];
#pragma unroll
    for (int c = 0; c < E; c++) want[c] = 0;
    uint32_t C = 0, tok = 0, cntb = 0;
    {
      uint32_t start = 0;
      bool only_res = false;
#pragma unroll 1
      for (int round = 0; round < 2; round++) {
        uint32_t carryW = tok, carryC = C, carryN = cntb;
        bool failed = false;
        uint32_t f_C = 0, f_tok = 0, f_cnt = 0, f_res = 0, f_pos = 0;
#pragma unroll
        for (int c = 0; c < E; c++) {
          const uint32_t base = c * 32;
          if (failed || base >= n || base + 32u <= start) continue;            // warp-uniform
          const uint32_t pos = base + lane;
          const bool res = (resm[c] >> lane) & 1u;
          const bool valid = pos < n && pos >= start && (!only_res || res);
          const uint32_t rem = r0[c].P + r1[c].d - r1[c].cached;
          const uint32_t w = valid ? (rem < cc ? rem : cc) : 0u;
          const uint32_t W = carryW + scan32(w, lane);
          const uint32_t tok_before = (W - w) < Tb ? (W - w) : Tb;
          const uint32_t tok_after = W < Tb ? W : Tb;
          const uint32_t wnt = tok_after - tok_before;
          const uint32_t foot = valid ? blocks_of(s, r1[c].cached + wnt) : 0u;
          const uint32_t Cf = carryC + scan32(foot, lane);
          const uint32_t vm = __ballot_sync(kFull, valid);
          const uint32_t cnt_before = carryN + __popc(vm & ltmask);
          const bool ok = valid && cnt_before < M && tok_before < Tb && Cf <= B;
          if (ok) want[c] = wnt;
          const uint32_t fm = __ballot_sync(kFull, valid && !ok);
          if (fm) {                                                            // the first request that did not fit
            const int fl = __ffs(fm) - 1;
            f_C = __shfl_sync(kFull, Cf - foot, fl);
            f_tok = __shfl_sync(kFull, tok_before, fl);
            f_cnt = __shfl_sync(kFull, cnt_before, fl);
            f_res = (resm[c] >> fl) & 1u;
            f_pos = base + fl;
            failed = true;
          } else {
            carryW = __shfl_sync(kFull, W, 31);
            carryC = __shfl_sync(kFull, Cf, 31);
            carryN += __popc(vm);
          }
        }
        if (!failed) { C = carryC; tok = carryW < Tb ? carryW : Tb; cntb = carryN; break; }
        C = f_C; tok = f_tok; cntb = f_cnt;
        const bool f_kv = f_cnt < M && f_tok < Tb;                             // failed on KV only
        if (round == 0 && f_kv && !f_res) { start = f_pos + 1; only_res = true; continue; }
        break;
      }
    }

    // ---------------- batch totals (M9).  Non-admitted residents must still fit behind the claims (M8): if they do
    // not, victims have to be selected -> team kernel (nothing has been written yet).
    uint32_t pf = 0, dec = 0, kres = 0, evl = 0, evu = 0;
    bool swp = false;
#pragma unroll
    for (int c = 0; c < E; c++) {
      if ((uint32_t)(c * 32 + lane) < n) {
        if (want[c]) {
          const uint32_t rem = r0[c].P + r1[c].d - r1[c].cached;
          if (r1[c].d >= 1u && rem == 1u) dec++; else pf += want[c];           // decode sequence vs prefill tokens
          ev_add(evl, evu, EV_ADMIT, r1[c].id, want[c]);
          swp |= (r1[c].flags & F_SWAPPED) != 0;
        } else if ((resm[c] >> lane) & 1u) {
          kres += blocks_of(s, r1[c].cached);                                  // stalled resident keeps its blocks
        }
      }
    }
    pf = __reduce_add_sync(kFull, pf);
    dec = __reduce_add_sync(kFull, dec);
    kres = __reduce_add_sync(kFull, kres);
    if (kres > B - C) { slow = true; break; }
    uint32_t swin_blocks = 0, swin_cnt = 0;
    if (__any_sync(kFull, swp)) {                                              // swap-in on admission (rare)
#pragma unroll
      for (int c = 0; c < E; c++) {
        if ((uint32_t)(c * 32 + lane) < n && want[c] && (r1[c].flags & F_SWAPPED)) {
          const uint32_t blocks = blocks_of(s, r1[c].cached);
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
    int64_t* g_tfirst = s.t_first + (size_t)r * s.N;
    int64_t* g_tlast = s.t_last + (size_t)r * s.N;
    uint32_t* g_hist = s.hist + (size_t)r * kTbtBins;
    uint32_t emit = 0, same = 0;
    uint32_t gonem[E], nflags[E];
#pragma unroll
    for (int c = 0; c < E; c++) {
      bool gone = false;
      nflags[c] = 0;
      if ((uint32_t)(c * 32 + lane) < n) {
        const uint32_t of = r1[c].flags;
        const uint32_t klass = (uint32_t)(key[c] >> 63);
        const uint32_t d_old = r1[c].d;
        const uint32_t id = r1[c].id;
        uint32_t nf = of & (F_RESIDENT | F_SWAPPED | F_EMITPREV);
        if (want[c]) {
          nf = (nf | F_RESIDENT) & ~F_SWAPPED;
          r1[c].cached += want[c];
          if (r1[c].cached == r0[c].P + d_old) {                    // KV caught up => one token out (M2)
            r1[c].d = d_old + 1u; emit++;
            if (d_old == 0u) {
              g_tfirst[id] = t_end;
              ev_add(evl, evu, EV_EMIT_FIRST, id, 0u);
            } else if (nf & F_EMITPREV) {
              same++;                                               // gap == this iteration's cost
            } else {
              const int64_t tl = __ldcg(g_tlast + id);
              atomicAdd(&g_hist[tbt_bin(t_end - tl)], 1u);
            }
            nf |= F_EMITPREV;
            if (r1[c].d == r0[c].D) {                               // complete: KV freed at once
              g_tlast[id] = t_end;
              const int64_t tf = (d_old == 0u) ? t_end : __ldcg(g_tfirst + id);
              atomicAdd(h64 + 8, (unsigned long long)(tf - r0[c].a));
              atomicAdd(h64 + 9, (unsigned long long)(t_end - r0[c].a));
              atomicAdd(h64 + 10, (unsigned long long)(t_end - tf));
              atomicAdd(h64 + 11, (unsigned long long)(r0[c].D - 1u));
              ev_add(evl, evu, EV_COMPLETE, id, 0u);
              uint32_t* g_ne = s.n_evict + (size_t)r * s.N;
              g_ne[id] = __ldcg(g_ne + id) | 0x80000000u;           // completion marker read by the stats kernel
              gone = true;
            }
          } else if (nf & F_EMITPREV) {
            g_tlast[id] = t; nf &= ~F_EMITPREV;                     // persist t_last when the streak ends
          }
        } else if (nf & F_EMITPREV) {
          g_tlast[id] = t; nf &= ~F_EMITPREV;
        }
        // re-lock at this iteration's bin (M10, G6); dirty hint for the next iteration's ordering: set when
        // (resident, bin, class) -- the inputs of a BOOST / FCFS key -- change
        const uint32_t b = bin[c];
        uint32_t b2 = b;
        if (r1[c].d != d_old) b2 = bin_of(par, s.k, signal_of(par, r0[c].P, r0[c].D, r1[c].d));
        const bool res2 = (nf & F_RESIDENT) != 0;
        const uint32_t klass2 = (par.guard && res2 && b2 == b) ? 0u : 1u;
        const bool dirty = (((nf ^ of) & F_RESIDENT) != 0) || (par.policy == 2 && b2 != b) || (klass2 != klass);
        if (res2) nf |= (b + 1u) << F_LOCK_SHIFT;
        if (dirty) nf |= F_DIRTY;
        nflags[c] = nf;
      }
      gonem[c] = __ballot_sync(kFull, gone);
    }
    emit = __reduce_add_sync(kFull, emit);
    same = __reduce_add_sync(kFull, same);
    evl = __reduce_add_sync(kFull, evl);
    evu = __reduce_add_sync(kFull, evu);

    // ---------------- write back in priority order, dropping completed requests; untouched records stay put
    uint32_t n_new = 0, n_done = 0;
#pragma unroll
    for (int c = 0; c < E; c++) {
      if (c * 32 < (int)n) {
        const uint32_t pos = c * 32 + lane;
        const bool in = pos < n;
        const bool keep = in && !((gonem[c] >> lane) & 1u);
        const uint32_t km = __ballot_sync(kFull, keep);
        const uint32_t np = n_new + __popc(km & ltmask);
        if (keep) {
          const bool moved = permuted || np != pos || pos >= n_old;
          const bool changed = want[c] != 0u || nflags[c] != r1[c].flags;
          r1[c].flags = nflags[c];
          if (moved) __stcg(reinterpret_cast<int4*>(gE0 + np), *reinterpret_cast<const int4*>(&r0[c]));
          if (moved || changed) __stcg(reinterpret_cast<int4*>(gE1 + np), *reinterpret_cast<const int4*>(&r1[c]));
        }
        n_new += __popc(km);
        n_done += __popc(gonem[c]);
      }
    }

    // ---------------- header: clock, digest (M12), cursors; counters by RED (no read needed)
    H = digest_fold(H, evl, evu, t_end);
    if (lane == 0) {
      if (same) atomicAdd(&g_hist[tbt_bin(cost)], same);
      __stcg(h64 + 0, (unsigned long long)t_end);
      __stcg(h64 + 1, (unsigned long long)H);
      if (cnt) __stcg(h64 + 2, (unsigned long long)a_next);
      __stcg(h64 + 13, (unsigned long long)n_new | ((unsigned long long)next << 32));
      if (n > peak || swin_blocks) {
        if (n > peak) peak = n;
        __stcg(h64 + 14, (unsigned long long)swap_used | ((unsigned long long)peak << 32));
      }
      atomicAdd(h64 + 3, (unsigned long long)n);                    // request-steps
      if (emit) atomicAdd(h64 + 4, (unsigned long long)emit);
      if (pf) atomicAdd(h64 + 5, (unsigned long long)pf);
      if (dec) atomicAdd(h64 + 6, (unsigned long long)dec);
      atomicAdd(h64 + 12, 1ull);                                    // iterations
      if (n_done) atomicAdd(reinterpret_cast<uint32_t*>(h64 + 15), n_done);
      if (swin_cnt) atomicAdd(reinterpret_cast<uint32_t*>(h64 + 16) + 1, swin_cnt);
    }
    if (n > peak) peak = n;
    t = t_end; n = n_new; wsize = n_new;
    if (n == 0 && a_next == kNever) {                               // finished its trace in this call
      if (lane == 0) atomicAdd(A.count + 4, 1u);
      it++;
      break;
    }
    __syncwarp();                                                   // window stores before the next iteration's loads
  }

  // ---------------- not handled here: queue the replica for the team kernels of this round
  if (slow && lane == 0) {
    if (it > 0) reinterpret_cast<uint32_t*>(h64 + 17)[1] = A.iters - it;     // iterations still to do in this round
    const uint32_t cls = wsize <= A.thrS ? 0u : (wsize <= A.thrM ? 1u : 2u);
    push_list(A, cls, r);
  }
}

int fast_configure() { return 0; }

void launch_fast(const StepArgs& A, cudaStream_t st) {
  const uint32_t grid = (A.s.R + kFWarps - 1) / kFWarps;
  k_fast<kFE><<<grid, 32 * kFWarps, 0, st>>>(A);
}

}  // namespace ub
