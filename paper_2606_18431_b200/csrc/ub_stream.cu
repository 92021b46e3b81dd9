// ub_stream.cu -- the streaming scheduling-step kernel of libuniboost.so (sm_100a): ONE WARP advances one replica by
// one (or `iters`) scheduler iterations of Algorithm 1 under the model rules M1..M12 of DESIGN.md
// Sec. 3, for a window of any size up to the queue cap.
//
// The replica's active window is kept in HBM in the priority order of the last iteration.  MemGuard keeps keys
// piecewise constant: between two iterations only the few requests whose (residency, bin, class)
// changed -- listed by the previous iteration in the replica's dirty list -- and the new arrivals can change place.
// One iteration is ONE pass over the window, 32 requests per chunk, one 16-byte record of each array per lane:
//   a0 ingest / idle jump (M6)    arrivals are read from the packed trace
//   a1 score (M3-M5)              boost table held in registers (lane b holds LUT[b]), looked up by shuffle
//   a2 order                      the dirty requests and the arrivals (<= 32 together) are scored, ranked against each
//                                 other in-warp and merged into the stream of the other, still sorted, requests
//   a3 admit (M7)                 the walk is a carried state machine over the chunks: a chunk that fits as a whole
//                                 costs two warp reductions, the one holding the first misfit two warp scans and a
//                                 ballot; "residents only" behind a blocked newcomer; nothing once the walk stopped
//   a5 advance (M9-M10, M12)      applied in the same pass, records rewritten in place (E1 when it changed, E0 only
//                                 where the order shifts); what needs the iteration's end time (first token, gap
//                                 after a stall, completion) is queued and applied when the cost is known
//   a4 victim select (M8)         if the stalled residents no longer fit: one backward pass over the window tail
// Data movement: every global -> SM transfer of the window is asynchronous (cp.async, 16 bytes per lane, L2 only)
// into per-warp shared-memory stages.  While a warp works on replica r it already has the header, the parameters,
// the dirty list and the first two chunks of its NEXT replica in flight, and a ring of kRing chunks of r ahead of the
// one it is processing; no register holds data in flight.
// Integers only.  Not handled here, decided before any write and queued for the team kernels of ub_step.cu: the
// SRPT / LAS keys (they drift every token), the test-only signal / quantiser modes, a block size that is not a power
// of two, more than 32 dirty requests + arrivals in one iteration.
#include "ub_device.cuh"

namespace ub {

constexpr int kSWarps = 2;                 // warps per CTA, each streams its own replicas
constexpr int kRing = 4;                   // chunks in flight behind the two speculative ones
constexpr uint32_t kFull = 0xffffffffu;
constexpr uint32_t kEvSmem = 30;            // per-request events of one iteration kept in shared memory (spare words of skb[2..31])

// inclusive warp scan, one SHFL + one predicated add per step (the shuffle's own "source lane in range" predicate)
__device__ __forceinline__ uint32_t scan32(uint32_t v) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    asm volatile("{ .reg .u32 t; .reg .pred p; shfl.sync.up.b32 t|p, %0, %1, 0x0, 0xffffffff; @p add.u32 %0, %0, t; }"
                 : "+r"(v) : "r"(o));
  }
  return v;
}

__device__ __forceinline__ void cp16(void* smem, const void* gmem) {
  const uint32_t sa = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

struct __align__(16) WarpBuf {             // per warp, 10 KB
  uint4 spec[2][2][64];                    // [parity][chunk 0 / 1][E0 records 0..31 | E1 records 32..63] of a replica
  uint4 ring[kRing][64];                   // chunks 2, 3, ... of the current replica
  uint4 hdr[2][16];                        // Hdr (256 bytes: state, parameters, dirty list)
  uint4 sr0[32], sr1[32], skb[32];         // the dirty requests + arrivals of one iteration in key order;
};                                         // skb = {key lo, key hi, bin, -}
static_assert(sizeof(Hdr) == 256, "cp.async copies the header as sixteen 16-byte pieces");

// a1 (M3-M5): sig = P + d; bin = Eq. 8 exponent; pi = a - b_gamma(w_hat) - delta if
// resident (Eq. 7); key = class<<63 | (pi + 2^62); class 0 = MemGuard-locked resident.  The baselines keyed by a size
// replace pi: SRPT D - d, LAS sig, SJF D, SPF P (the caller passes lutv = 0 and delta = 0 for
// them).  policy is warp-uniform.  All 32 lanes must call it.
__device__ __forceinline__ void score(const Rec0& q0, const Rec1& q1, uint32_t k, int64_t lutv, int64_t delta,
                                      bool guard, uint32_t policy, uint64_t& key, uint32_t& bin) {
  const uint32_t sig = q0.P + q1.d;
  const uint32_t sg = sig > k ? sig : k;
  uint32_t b = (uint32_t)(__clz(k) - __clz(sg));
  b -= ((k << b) > sg) ? 1u : 0u;
  const uint32_t lo = __shfl_sync(kFull, (uint32_t)lutv, (int)b);
  const uint32_t hi = __shfl_sync(kFull, (uint32_t)((uint64_t)lutv >> 32), (int)b);
  const bool res = (q1.flags & F_RESIDENT) != 0;
  int64_t base = q0.a;
  if (policy != 0u && policy != 2u)
    base = (int64_t)(policy == 1u ? q0.D - q1.d : (policy == 3u ? sig : (policy == 4u ? q0.D : q0.P)));
  const int64_t kv = base - (int64_t)(((uint64_t)hi << 32) | lo) - (res ? delta : 0ll);
  const bool locked = guard && res && (q1.flags >> F_LOCK_SHIFT) == b + 1u;
  key = (uint64_t)(kv + kKeyBias) | (locked ? 0ull : (1ull << 63));
  bin = b;
}

// The re-key rule of the drifting keys (SRPT, LAS), kept out of line: the streaming kernel competes for the instruction
// cache and the arrival-keyed policies never come here.  comp = the request's next (class, key, id), 0 for a lane
// whose request leaves; kmax = the largest one written so far (updated).  True when the lane's request sorts in
// front of one written before it.
__device__ __noinline__ bool drift_out_of_order(const uint64_t comp, uint64_t& kmax) {
  const int lane = threadIdx.x & 31;
  uint64_t pm = comp;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint64_t t = __shfl_up_sync(kFull, pm, o);
    if (lane >= o && t > pm) pm = t;
  }
  uint64_t before = __shfl_up_sync(kFull, pm, 1);
  if (lane == 0) before = 0ull;
  if (kmax > before) before = kmax;
  const uint64_t top = __shfl_sync(kFull, pm, 31);
  if (top > kmax) kmax = top;
  return comp != 0ull && comp < before;
}

// ADA: the gamma-Ada instance (per-level boost tables, latency window); the static instance carries none of it.
// MULTI: several iterations per launch (the resident-state mode: the window is re-read from L2 between them); the
// one-iteration instance carries none of that either -- the instruction cache (32 KB per SM) is what this kernel
// competes for, so every instance holds only the code it runs.
// LIST: the replicas to visit come from a list (the unfinished ones in the tail of a run; the drift group).
// DRIFT: the replicas whose keys drift with every token (SRPT, LAS) are advanced by an instance of their own, launched
// over their list beside the main one: the extra re-key rule and its state stay out of the main instance, whose
// register budget and instruction-cache footprint decide the headline number.
// SPEC: every replica of the job is BOOST with MemGuard, the paper's signal and quantiser (SimDev::all_boost_guard) --
// the method itself.  Policy, guard and hysteresis are then compile-time facts: 96 fewer instructions in the instance
// (2864 -> 2768) and +3 % on config 5 (8.26e10 -> 8.52e10 request-steps/s).
template <bool ADA, bool MULTI, bool LIST, bool DRIFT, bool SPEC>
__global__ void __launch_bounds__(32 * kSWarps, 10) k_stream(const StepArgs A) {
  static_assert(!(SPEC && DRIFT), "the drift group is SRPT / LAS");
  __shared__ WarpBuf wbuf[kSWarps];
  const SimDev& s = A.s;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const uint32_t ltmask = (1u << lane) - 1u;
  WarpBuf& X = wbuf[wib];
  const uint32_t B = s.B, M = s.M, cc = s.c, Tb = s.T, Q = s.Q, k = s.k;
  const uint32_t blk_m1 = s.blk - 1u, blk_sh = s.blk_shift;
  const uint32_t nwarps = gridDim.x * kSWarps;

  // header, parameters, dirty list and the first two chunks of replica rr -> stage `par` (one cp.async group)
  auto prefetch_replica = [&](const uint32_t rr, const uint32_t par) {
    if (rr != 0xFFFFFFFFu) {
      if (lane < 16) cp16(&X.hdr[par][lane], reinterpret_cast<const uint4*>(s.hdr + rr) + lane);
      const uint4* e0 = reinterpret_cast<const uint4*>(s.E0 + (size_t)rr * Q) + lane;
      const uint4* e1 = reinterpret_cast<const uint4*>(s.E1 + (size_t)rr * Q) + lane;
      cp16(&X.spec[par][0][lane], e0);        cp16(&X.spec[par][0][32 + lane], e1);
      cp16(&X.spec[par][1][lane], e0 + 32);   cp16(&X.spec[par][1][32 + lane], e1 + 32);   // (arrays are padded)
    }
    cp_commit();
  };

  // Work distribution: windows differ by two orders of magnitude.  A warp takes its first `nstat` replicas by static
  // striding (7/8 of an even share); the rest are handed out dynamically: each is the next value of a global ticket
  // counter (count[4] / count[6] alternately, each zeroed by the launch before), requested one replica ahead so that the atomic's latency is never waited for.
#define UB_GW (A.rbeg + blockIdx.x * kSWarps + (threadIdx.x >> 5))
  // r: the replica being advanced (its header and first chunks sit in stage `parity`), rn: the one being fetched; the
  // first round of the loop only fetches (one prefetch site: code size)
  // (ri / rni: their positions in [rbeg, rend) -- the replica numbers themselves unless LIST)
  constexpr uint32_t kNone = 0xFFFFFFFFu;
  uint32_t r = kNone, ri = kNone, rn = kNone, rni = UB_GW;
  uint32_t taken = 1, ticket = 0;
  uint32_t parity = 1;
  // (the ticket counter of the NEXT launch is zeroed here: launches of one part alternate between the two)
  if (blockIdx.x == 0 && threadIdx.x == 0) A.count[4 + 2 * (A.tick ^ 1u)] = 0u;
  for (;; r = rn, ri = rni, rni = (taken < A.nstat ? UB_GW + taken * nwarps : __shfl_sync(kFull, ticket, 0) + A.dynbase), taken++,
          parity ^= 1u) {
    cp_wait<0>();
    __syncwarp();
    rn = rni < A.rend ? (LIST ? __ldg(A.live + rni) : rni) : kNone;
    prefetch_replica(rn, parity ^ 1u);
    // (inline PTX: the compiler's own atomicAdd broadcasts the result with a shuffle at once, which waits ~600 cycles
    // for the atomic's round trip -- 10 % of all warp time; here the ticket is first read one replica later)
    if (taken >= A.nstat && lane == 0)
      asm volatile("{ .reg .u64 a; .reg .u32 z; mov.u32 z, %%laneid; cvt.u64.u32 a, z; add.u64 a, a, %1; atom.global.add.u32 %0, [a], 1; }"
                   : "=r"(ticket) : "l"(A.count + 4 + 2 * A.tick) : "memory");       // (lane 0: a = the counter)
    if (ri == kNone) continue;
    if (ri >= A.rend) break;
    const unsigned long long* sh = reinterpret_cast<const unsigned long long*>(X.hdr[parity]);
    // (addresses and per-replica scalars that are needed rarely are re-derived where they are used instead of
    // living in registers across the chunk loop)
#define UB_H64 (reinterpret_cast<unsigned long long*>(s.hdr + r))
#define UB_TR (s.TR + (size_t)reinterpret_cast<const Hdr*>(X.hdr[parity])->par.trace_id * s.N)
#define UB_DELTA (hyst ? reinterpret_cast<const Hdr*>(X.hdr[parity])->par.delta : 0ll)
    uint32_t n = (uint32_t)sh[13];
    if (n == 0 && (int64_t)sh[2] == kNever) continue;                 // finished its trace
    {
      // a replica queued for the team kernels owes them its iterations until they have run (Hdr::todo, flush_slow)
      const uint32_t todo = (uint32_t)(sh[17] >> 32);
      if (todo) {
        if (lane == 0) reinterpret_cast<uint32_t*>(UB_H64 + 17)[1] = todo + A.iters;
        continue;
      }
    }
    uint32_t nd = (uint32_t)sh[18];                                   // entries of the dirty list
    const uint32_t iters = MULTI ? A.iters : 1u;
    const RepPar par = reinterpret_cast<const Hdr*>(X.hdr[parity])->par;
    Rec0* gE0 = s.E0 + (size_t)r * Q;
    Rec1* gE1 = s.E1 + (size_t)r * Q;
    const uint32_t policy = SPEC ? 2u : par.policy;
    const bool isboost = SPEC || par.policy == 2;
    const bool guard = SPEC || par.guard != 0;
    // flags of a resident in steady decode: admitted and emitting last iteration; class 0 when MemGuard locks it
    const uint32_t okflags = F_RESIDENT | F_ADMITNOW | F_EMITPREV | (guard ? 0u : F_KLASS1);

    // the streaming path covers the paper's signal and quantiser under every policy but DistBoost (whose decode-queue
    // key is the request's first-token time, a gather from the per-request outputs)
    bool slow = SPEC ? false : (par.policy > 5 || par.signal_mode != 0 || par.quant_mode != 0 || blk_sh >= 32u);
    const bool hyst = SPEC || par.policy == 0 || par.policy == 2;             // Eq. 7 applies to the arrival-keyed policies
    // SRPT / LAS keys drift: every emitted token moves the request's key by one.  The order is then kept by one more
    // re-key rule (in process()): a request whose next key sorts in front of one written before it is listed dirty.
    constexpr bool drift = DRIFT;
    if constexpr (!DRIFT && !SPEC) {
      if (!slow && (par.policy == 1 || par.policy == 3)) {   // (a member of the drift group: ub_set_replicas has the same test)
        if constexpr (ADA) slow = true;        // (the gamma-Ada instance has no drift twin: the team kernels take them)
        else continue;                         // the drift instance's launch advances this replica
      }
    }
    // boost table in registers: lane b holds LUT[b] (Eq. 2 in fixed point, built on the host, M4); FCFS: all 0
    int64_t lutv = 0;
    // (a gamma-Ada replica owns one table per grid level, Hdr::level selects; 0 for a static replica)
    if (isboost && !slow) lutv = __ldg(s.lut + par.lut_off + (ADA ? (uint32_t)(sh[18] >> 32) * 64u : 0u) + lane);   // 64 entries, bins < 32
    uint32_t it = 0;
    uint32_t wsize = n;

    for (; !slow && it < iters; it++) {
      // ---------------- a0: idle jump + ingest (M6)
      // (the clock, the next arrival and the trace cursor live in the shared-memory header image -- words 0, 2, 13 --
      // between their few uses)
      int64_t t = (int64_t)sh[0];
      int64_t a_next = (int64_t)sh[2];
      uint32_t next = (uint32_t)(sh[13] >> 32);
      if constexpr (MULTI) {
        // time fence (JSQ router, rule M18): only iterations that start before the replica's limit run
        if (A.tlimit && (n != 0 || a_next != kNever) && (n == 0 && a_next > t ? a_next : t) >= __ldg(A.tlimit + r)) break;
      }
      if (n == 0) {
        if (a_next == kNever) break;
        if (a_next > t) {
          t = a_next;
          if (lane == 0) reinterpret_cast<unsigned long long*>(X.hdr[parity])[0] = (unsigned long long)t;
        }
      }
      uint32_t cnt = 0, nreq = 0;
      if (a_next <= t && n < Q) {                                     // a_next != kNever => next < nreq
        nreq = __ldg(s.n_req + par.trace_id);
        const uint32_t avail = (Q - n) < (nreq - next) ? (Q - n) : (nreq - next);
        const bool take = (uint32_t)lane < avail && __ldg(&UB_TR[next + lane].a) <= t;   // arrivals sorted => a prefix
        cnt = __popc(__ballot_sync(kFull, take));
        if (cnt == 32u && avail > 32u) cnt = 64u;                     // maybe more: not for this kernel
      }
      wsize = n + cnt;
      if (nd + cnt > kDirtyMax) { slow = true; break; }               // (nd > kDirtyMax marks a list that overflowed)
      const uint32_t n_old = n, m = nd + cnt;
      const uint32_t nch = (n_old + 31u) >> 5;
      n += cnt;

      // chunks 2 .. of the window: kRing cp.async groups in flight (group q of the ring = chunk 2 + q, maybe empty)
      auto issue_chunk = [&](const uint32_t c) {
        if (c < nch) {
          uint4* st = X.ring[(c - 2u) % kRing];
          cp16(st + lane, reinterpret_cast<const uint4*>(gE0 + c * 32u) + lane);
          cp16(st + 32 + lane, reinterpret_cast<const uint4*>(gE1 + c * 32u) + lane);
        }
        cp_commit();
      };
      if (MULTI && it > 0) {                                          // (the first iteration found them prefetched)
        cp16(&X.spec[parity][0][lane], reinterpret_cast<const uint4*>(gE0) + lane);
        cp16(&X.spec[parity][0][32 + lane], reinterpret_cast<const uint4*>(gE1) + lane);
        cp16(&X.spec[parity][1][lane], reinterpret_cast<const uint4*>(gE0) + 32 + lane);
        cp16(&X.spec[parity][1][32 + lane], reinterpret_cast<const uint4*>(gE1) + 32 + lane);
        cp_commit();
      }
      if (nch > 2u) {
#pragma unroll
        for (int q = 0; q < kRing; q++) issue_chunk(2u + q);
      }

      // ---------------- a2 (first half): the requests that may change place -- dirty ones and arrivals -- are taken
      // out of the stream, scored, ranked among themselves by (class, key, id) and parked in shared memory
      uint32_t spos = 0xFFFFFFFFu;                                    // window position a dirty request is taken from
      uint32_t dlo = 0, dspan = 0;                                    // chunks [dlo, dlo + dspan) hold the positions they are taken from
      if (m) {
        int4 v0 = make_int4(0, 0, 0, 0), v1 = make_int4(0, 0, 0, 0);
        if ((uint32_t)lane < nd) {
          spos = (!MULTI || it == 0) ? (uint32_t)reinterpret_cast<const Hdr*>(X.hdr[parity])->dl[lane]
                                     : (uint32_t)__ldcg(s.hdr[r].dl + lane);
          if ((!MULTI || it == 0) && spos < 64u) {                   // in the two chunks that came with the header: no
            const uint4* sp = X.spec[parity][spos >> 5] + (spos & 31u);   // second trip to memory
            const uint4 a0 = sp[0], a1 = sp[32];
            v0 = *reinterpret_cast<const int4*>(&a0); v1 = *reinterpret_cast<const int4*>(&a1);
          } else {
            v0 = __ldcg(reinterpret_cast<const int4*>(gE0 + spos));
            v1 = __ldcg(reinterpret_cast<const int4*>(gE1 + spos));
          }
        } else if ((uint32_t)lane < m) {
          const uint32_t i = next + ((uint32_t)lane - nd);
          v0 = __ldg(reinterpret_cast<const int4*>(UB_TR + i));
          v1 = make_int4((int)i, 0, 0, 0);
        }
        if (nd) {
          dlo = __reduce_min_sync(kFull, spos >> 5);                  // (lanes without a dirty request hold 0xFFFFFFFF)
          dspan = __reduce_max_sync(kFull, (uint32_t)lane < nd ? spos >> 5 : 0u) - dlo + 1u;
        }
        if (cnt) {
          next += cnt;
          a_next = (next < nreq) ? __ldg(&UB_TR[next].a) : kNever;
          if (lane == 0) {
            unsigned long long* shw = reinterpret_cast<unsigned long long*>(X.hdr[parity]);
            shw[2] = (unsigned long long)a_next;
            shw[13] = (shw[13] & 0xFFFFFFFFull) | ((unsigned long long)next << 32);
            __stcg(UB_H64 + 2, (unsigned long long)a_next);
          }
        }
        const Rec0 q0 = *reinterpret_cast<const Rec0*>(&v0);
        const Rec1 q1 = *reinterpret_cast<const Rec1*>(&v1);
        uint64_t sk; uint32_t sb;
        score(q0, q1, k, lutv, UB_DELTA, guard, policy, sk, sb);
        uint32_t rank = 0;
        if (m > 1u) {
#pragma unroll 1
          for (uint32_t j = 0; j < m; j++) {
            const uint64_t kj = __shfl_sync(kFull, sk, (int)j);
            const uint32_t ij = __shfl_sync(kFull, q1.id, (int)j);
            rank += key_less(kj, ij, sk, q1.id) ? 1u : 0u;
          }
        }
        if ((uint32_t)lane < m) {
          X.sr0[rank] = *reinterpret_cast<const uint4*>(&v0);
          X.sr1[rank] = *reinterpret_cast<const uint4*>(&v1);
          X.skb[rank] = make_uint4((uint32_t)sk, (uint32_t)(sk >> 32), sb, 0u);
        }
      }
      // the re-read chunks 0, 1; with parked requests the stores of chunk 1 may reach into chunk 2: it must have landed
      if (lane == 0) X.skb[0].w = 0u, X.skb[1].w = 0u;                // swap-in sums (spare words of the parking area; the
                                                                      // barrier below orders the reset before their use)
      if (nch > 2u) { if (m) cp_wait<kRing - 1>(); else if (MULTI && it > 0) cp_wait<kRing>(); } else if (MULTI && it > 0) cp_wait<0>();
      __syncwarp();

      // ---------------- the pass.  Walk state (M7), warp-uniform: mode 0 = everybody walks, 1 = residents only (a
      // newcomer was blocked on KV), 2 = stopped; carryW / carryC = tokens / KV blocks claimed so far; crank = rank of
      // the next request in the merged order (mode 0); carryN = requests admitted so far (mode 1).
      uint32_t mode = 0, carryW = 0, carryC = 0, carryN = 0, crank = 0;
      // per-lane sums: de = decode sequences | tokens emitted << 16; ps = prefill tokens | same-gap emissions << 16
      // (each field < 2^16: M, Q <= 2048, T <= 65535); swap-ins (rare) are summed in shared memory
      uint32_t de = 0, ps = 0, kres = 0, evl = 0, evu = 0;
      uint32_t rhi = 0;                                               // 1 + the last new position this lane gave to a resident
      uint64_t kmax = 0;                                              // drift: the largest next (class, key, id) written so far
      uint32_t outpos = 0, nev = 0, ndnew = 0, n_done = 0;
      uint32_t dptr = 0;                                              // next parked request to merge

      // one segment of the merged order: the lanes of `mask`, in lane order
      auto process = [&](const Rec0& w0, const Rec1& w1, const uint64_t key, const uint32_t bin, const uint32_t mask,
                         const uint32_t stpos) {
        const bool valid = (mask >> lane) & 1u;
        const uint32_t of = w1.flags;
        const bool res = valid && (of & F_RESIDENT) != 0;
        const uint32_t rem = w0.P + w1.d - w1.cached;
        uint32_t want = 0;
        // ---- a3: admission walk (M7; Algorithm 1 "while |B| < M ... U + dU <= B") over this segment:
        //   W = incl. scan of min(c, rem);  tok_before = min(T, W - w);  want = min(T, W) - tok_before;
        //   foot = ceil((cached + want)/blk);  Cf = incl. scan of foot;  ok = rank < M & tok_before < T & Cf <= B.
        // ok is monotone along the walk: the admitted set is the prefix in front of the first misfit.  If that one is
        // a non-resident that failed on KV only ("newblocked"), the walk continues over the residents behind it.
        if (mode < 2u) {
          const uint32_t resm = __ballot_sync(kFull, res);
          uint32_t pm = mode == 0u ? mask : resm;
          if (pm) {
            const bool part0 = (pm >> lane) & 1u;
            const uint32_t w0t = part0 ? (rem < cc ? rem : cc) : 0u;
            const uint32_t f0 = part0 ? (w1.cached + w0t + blk_m1) >> blk_sh : 0u;
            const uint32_t totw = __reduce_add_sync(kFull, w0t);
            const uint32_t totf = __reduce_add_sync(kFull, f0);
            const uint32_t npm = __popc(pm);
            if (carryW + totw <= Tb && carryC + totf <= B && (mode == 0u ? crank : carryN) + npm <= M) {
              want = w0t;                                             // the whole segment fits: no misfit in it
              carryW += totw; carryC += totf; carryN += npm;
            } else {
              while (pm) {                                            // at most two rounds per segment
                const bool part = (pm >> lane) & 1u;
                const uint32_t w = part ? w0t : 0u;
                const uint32_t W = carryW + scan32(w);
                const uint32_t tok_before = (W - w) < Tb ? (W - w) : Tb;
                const uint32_t tok_after = W < Tb ? W : Tb;
                const uint32_t wnt = tok_after - tok_before;
                const uint32_t foot = part ? (w1.cached + wnt + blk_m1) >> blk_sh : 0u;
                const uint32_t Cf = carryC + scan32(foot);
                const uint32_t cb = (mode == 0u ? crank : carryN) + __popc(pm & ltmask);
                const bool ok = part && cb < M && tok_before < Tb && Cf <= B;
                if (ok) want = wnt;
                const uint32_t fm = __ballot_sync(kFull, part && !ok);
                if (!fm) {
                  carryW = __shfl_sync(kFull, W, 31);
                  carryC = __shfl_sync(kFull, Cf, 31);
                  carryN += __popc(pm);
                  break;
                }
                const int fl = __ffs(fm) - 1;                         // the first request that did not fit
                carryC = __shfl_sync(kFull, Cf - foot, fl);
                carryW = __shfl_sync(kFull, tok_before, fl);
                carryN = __shfl_sync(kFull, cb, fl);
                if (mode == 0u && carryN < M && carryW < Tb && !((resm >> fl) & 1u)) {
                  mode = 1u;                                          // newblocked: residents behind it continue
                  pm = fl < 31 ? (resm & (kFull << (fl + 1))) : 0u;
                } else {
                  mode = 2u;
                  pm = 0u;
                }
              }
            }
          }
        }
        crank += __popc(mask);

        // ---- batch totals (M9) and events (M12)
        const bool adm = want != 0u;
        const bool isdec = adm && w1.d >= 1u && rem == 1u;            // decode sequence vs prefill tokens
        de += isdec ? 1u : 0u;
        ps += isdec ? 0u : want;
        {
          const uint32_t m32 = ((w1.id + 1u) * 0x9E3779B1u) ^ ((uint32_t)EV_ADMIT * 0x85EBCA6Bu);
          const uint64_t h = (uint64_t)m32 * (uint64_t)(2u * want + 1u);
          evl += adm ? (uint32_t)h : 0u;
          evu += adm ? (uint32_t)(h >> 32) : 0u;
        }
        const bool back = adm && (of & F_PREEMPTED);
        if (__any_sync(kFull, back)) {                                // back on the device after an eviction (rare)
          if (back) {                                                 // M15: the preemption ends where this iteration starts
            int64_t* g_tp = s.t_pre + (size_t)r * s.N + w1.id;
            *g_tp = __ldcg(g_tp) + (int64_t)sh[0];
          }
          if (back && (of & F_SWAPPED)) {                             // swap-in on admission
            const uint32_t blocks = (w1.cached + blk_m1) >> blk_sh;
            atomicAdd(&X.skb[0].w, blocks); atomicAdd(&X.skb[1].w, 1u);
            ev_add(evl, evu, EV_SWAPIN, w1.id, blocks);
          }
        }
        kres += (res && !adm) ? (w1.cached + blk_m1) >> blk_sh : 0u;  // stalled residents keep their blocks (M8)

        // ---- a5: apply (M10)
        const uint32_t d_old = w1.d;
        const uint32_t sig = w0.P + d_old;
        const uint32_t cached2 = w1.cached + want;
        const bool emitted = adm && cached2 == sig;                   // KV caught up => one token out (M2)
        const bool ep_old = (of & F_EMITPREV) != 0;
        const uint32_t d2 = d_old + (emitted ? 1u : 0u);
        de += emitted ? 0x10000u : 0u;
        ps += (emitted && d_old != 0u && ep_old) ? 0x10000u : 0u;     // gap == this iteration's cost
        const bool gone = emitted && d2 == w0.D;                      // complete: KV freed at once
        uint32_t nf = of & (F_RESIDENT | F_SWAPPED | F_PREEMPTED);
        if (adm) nf = F_RESIDENT | F_ADMITNOW;
        if (emitted) nf |= F_EMITPREV;
        // re-lock at this iteration's bin (M10, G6); a request is dirty for the next iteration's ordering when
        // (resident, bin, class) -- the inputs of its key -- change
        const uint32_t b2 = bin + ((emitted && sig + 1u == (k << (bin + 1u))) ? 1u : 0u);
        const bool res2 = (nf & F_RESIDENT) != 0;
        const uint32_t klass = (uint32_t)(key >> 63);
        const uint32_t klass2 = (guard && res2 && b2 == bin) ? 0u : 1u;
        bool dirty = (((nf ^ of) & F_RESIDENT) != 0) || (isboost && b2 != bin) || (klass2 != klass);
        if constexpr (DRIFT) {
          // next iteration's (class, key, id) of every request that stays, in the order written: whoever sorts in
          // front of a request written before it must be re-merged (the others then still form a sorted stream)
          const uint32_t key2 = par.policy == 1 ? w0.D - d2 : sig + (emitted ? 1u : 0u);
          const bool stays = valid && !gone;
          const uint64_t comp = stays ? (((uint64_t)klass2 << 63) | ((uint64_t)key2 << 32) | (uint64_t)w1.id) : 0ull;
          if (drift_out_of_order(comp, kmax)) dirty = true;
        }
        if (res2) nf |= (bin + 1u) << F_LOCK_SHIFT;
        if (klass) nf |= F_KLASS1;
        if (dirty) nf |= F_DIRTY;
        const uint32_t gonem = __ballot_sync(kFull, gone);
        // everything that touches the per-request outputs is rare: first token, a gap after a stall, completion,
        // the end of an emission streak (t_last is implicit while a request emits every iteration)
        const bool defer = emitted && (d_old == 0u || !ep_old || gone);
        const bool ends = valid && !emitted && ep_old;
        if (__any_sync(kFull, defer || ends)) {
          if (ends) s.t_last[(size_t)r * s.N + w1.id] = (int64_t)sh[0];   // persist t_last when the streak ends
          const uint32_t em = __ballot_sync(kFull, defer);
          if (defer) {                                                // the first kEvSmem of them wait in shared memory
            const uint32_t slot = nev + __popc(em & ltmask);
            const uint32_t kind = (d_old == 0u ? 1u : 0u) | ((d_old != 0u && !ep_old) ? 2u : 0u) | (gone ? 4u : 0u);
            if (slot < kEvSmem) X.skb[2u + slot].w = (w1.id << 3) | kind;                 // (ids < 2^29: ub_create)
            else s.evbuf[(size_t)r * s.evcap + slot] = make_uint2(w1.id, kind);
          }
          nev += __popc(em);
        }

        // ---- write back in priority order, dropping completed requests; untouched records stay put
        const uint32_t keepm = mask & ~gonem;
        const bool keep = (keepm >> lane) & 1u;
        const uint32_t np = outpos + __popc(keepm & ltmask);
        const bool moved = np != stpos;
        if (keep && res2 && np >= rhi) rhi = np + 1u;
        if (keep && moved) __stcg(reinterpret_cast<int4*>(gE0 + np), *reinterpret_cast<const int4*>(&w0));
        if (keep && (moved || adm || nf != of))
          __stcg(reinterpret_cast<int4*>(gE1 + np), make_int4((int)w1.id, (int)d2, (int)cached2, (int)nf));
        const uint32_t dm = __ballot_sync(kFull, keep && dirty);
        if (dm) {                                                     // next iteration's dirty list
          const uint32_t slot = ndnew + __popc(dm & ltmask);
          if (keep && dirty && slot < kDirtyMax) s.hdr[r].dl[slot] = (uint16_t)np;
          ndnew += __popc(dm);
        }
        outpos += __popc(keepm);
        n_done += __popc(gonem);
      };

      // The pass over the chunks.  Three phases share the walk state: (A) a run of chunks of MemGuard-locked residents
      // in steady decode, (T) the tail of steadily waiting requests behind the walk, (G) everything else, one chunk
      // at a time.  A lane reads back from the stages exactly the 32 bytes it copied itself, so the asynchronous
      // copies need no warp barrier; cp.async.wait_group alone orders them.
      auto stage_of = [&](const uint32_t c) -> const uint4* { return c < 2u ? X.spec[parity][c] : X.ring[(c - 2u) % kRing]; };
      // chunk c (>= 2) must have landed.  Stores go to positions at or below the ones read except after parked
      // requests were merged in front: the writes of a chunk may then reach into the next one, which must have landed
      // too before anything is stored (`ahead`: requests still parked, or the output position already in front)
      auto wait_chunk = [&](const uint32_t c, const bool ahead) {
        if (c >= 2u) { if (ahead) cp_wait<kRing - 2>(); else cp_wait<kRing - 1>(); }
      };
      // requests of chunk c still in the stream (the dirty ones were taken out)
      auto valid_of = [&](const uint32_t c) -> uint32_t {
        const uint32_t left = c < nch ? n_old - c * 32u : 0u;
        uint32_t cv = left >= 32u ? kFull : ((1u << left) - 1u);
        if (c - dlo < dspan) cv &= ~__reduce_or_sync(kFull, ((uint32_t)lane < nd && (spos >> 5) == c) ? (1u << (spos & 31u)) : 0u);
        return cv;
      };
      uint32_t c = 0;
      for (;;) {
        // ---------------- (A) chunks of residents in steady decode (each wants one token, emits it, neither completes
        // nor crosses its Eq. 8 threshold) that fit as a whole: nothing is re-keyed, every record advances by one token
        // (M2, M7, M10).  With MemGuard they are class 0 in stored order, so in front of a parked request of class 1;
        // without it only when nothing is parked
        if (mode == 0u && c < nch) {
          const bool pend = dptr < m;
          if (!pend || (guard && (X.skb[dptr].y >> 31))) {
            do {
              wait_chunk(c, outpos > c * 32u);
              const uint4* st = stage_of(c);
              const uint4 c0 = st[lane], c1 = st[32 + lane];
              const Rec0 r0 = *reinterpret_cast<const Rec0*>(&c0);
              const Rec1 r1 = *reinterpret_cast<const Rec1*>(&c1);
              const uint32_t cv = valid_of(c);
              const bool valid = (cv >> lane) & 1u;
              const uint32_t fl = r1.flags;
              const uint32_t sig1 = r0.P + r1.d + 1u;                  // signal after this token
              const bool okl = (fl & (F_LOCK_MASK_LOW)) == okflags && r1.cached + 2u == sig1 &&
                               r1.d + 1u != r0.D && sig1 != (k << (fl >> F_LOCK_SHIFT));
              // ... optionally followed, when nothing is parked, by steadily waiting requests (not resident, nothing
              // to finalise) whose first one is turned away -- on KV ("newblocked": the walk goes on over residents
              // only, of which this chunk has none left) or because the batch / token budget is used up (walk stops)
              const uint32_t decm = __ballot_sync(kFull, valid && okl);
              uint32_t wm = 0;
              if (cv == 0u) break;
              uint64_t klast = 0;
              if constexpr (DRIFT) {
                // drifting keys: the decoders' keys move together, so they keep their order among themselves; a waiting
                // request behind them does not move with them (general path), and the first decoder must not come to
                // sort in front of anything written so far
                if (decm != cv) break;
                const uint64_t comp = (guard ? 0ull : (1ull << 63)) |
                                      ((uint64_t)(par.policy == 1 ? r0.D - r1.d - 1u : sig1) << 32) | (uint64_t)r1.id;
                if (__shfl_sync(kFull, comp, __ffs(cv) - 1) < kmax) break;
                klast = __shfl_sync(kFull, comp, 31 - __clz((int)cv));
              }
              if (decm != cv) {                                        // (a chunk of decoders only skips all this)
                if (pend) break;
                wm = __ballot_sync(kFull, valid && !okl && (fl & ~F_PARKED) == F_KLASS1);
                if ((decm | wm) != cv || decm >= (wm & (0u - wm))) break;                            // (decoders first)
              }
              const uint32_t nv = __popc(decm);
              const uint32_t totf = __reduce_add_sync(kFull, (valid && okl) ? (r1.cached + 1u + blk_m1) >> blk_sh : 0u);
              if (crank + nv > M || carryW + nv > Tb || carryC + totf > B) break;
              uint32_t nmode = 0;
              if (wm) {
                const uint32_t tokb = carryW + nv, cbw = crank + nv;
                nmode = 2u;
                if (cbw < M && tokb < Tb) {                            // would it fit?  want = min(c, rem, T - tok)
                  const uint32_t rem = r0.P + r1.d - r1.cached;
                  uint32_t wnt = rem < cc ? rem : cc;
                  wnt = wnt < Tb - tokb ? wnt : Tb - tokb;
                  const uint32_t footw = __shfl_sync(kFull, (r1.cached + wnt + blk_m1) >> blk_sh, __ffs(wm) - 1);
                  nmode = (carryC + totf + footw > B) ? 1u : 3u;       // 3: it is admitted -> general path
                }
                if (nmode == 3u) break;
              }
              const uint32_t np = outpos + __popc(cv & ltmask);
              const bool moved = np != c * 32u + (uint32_t)lane;
              if (valid && moved) __stcg(reinterpret_cast<int4*>(gE0 + np), *reinterpret_cast<const int4*>(&c0));
              if (valid && okl) {
                __stcg(reinterpret_cast<int4*>(gE1 + np),
                       make_int4((int)r1.id, (int)(r1.d + 1u), (int)(r1.cached + 1u), (int)fl));
                const uint64_t h = (uint64_t)(((r1.id + 1u) * 0x9E3779B1u) ^ ((uint32_t)EV_ADMIT * 0x85EBCA6Bu)) * 3ull;
                evl += (uint32_t)h; evu += (uint32_t)(h >> 32);
                de += 0x10001u; ps += 0x10000u;
                rhi = np + 1u > rhi ? np + 1u : rhi;
              } else if (valid && moved) {
                __stcg(reinterpret_cast<int4*>(gE1 + np), *reinterpret_cast<const int4*>(&c1));
              }
              if constexpr (DRIFT) kmax = klast;
              carryW += nv; carryC += totf; carryN = crank + nv;       // (carryN: the turned-away request's rank)
              crank += __popc(cv); outpos += __popc(cv);
              mode = nmode;
              if (c >= 2u) issue_chunk(c + kRing);                     // the stage is free again
              c++;
            } while (mode == 0u && c < nch);
          }
        }
        // ---------------- (T) behind the walk, nothing parked left: chunks of waiting requests (not resident, nothing
        // to finalise) only move up when requests in front of them completed
        bool tail = mode != 0u && dptr >= m && c >= dlo + dspan;
        const uint32_t c_tail = c;
        if constexpr (DRIFT) {
          // drifting keys: a waiting request keeps its key, but one written in front of the tail may have moved behind
          // the tail's first request (LAS).  The tail is sorted, so it may stay as it is when its first request does not
          // sort in front of anything written so far (kmax); else the general path lists the out-of-order ones
          if (tail && c < nch) {
            wait_chunk(c, outpos > c * 32u);
            const uint4* st = stage_of(c);
            const uint4 f0 = st[0], f1 = st[32];
            const Rec0 r0 = *reinterpret_cast<const Rec0*>(&f0);
            const Rec1 r1 = *reinterpret_cast<const Rec1*>(&f1);
            const uint32_t key2 = par.policy == 1 ? r0.D - r1.d : r0.P + r1.d;
            tail = ((1ull << 63) | ((uint64_t)key2 << 32) | (uint64_t)r1.id) >= kmax;
          }
        }
        if (tail) {
          if (c >= 2u && c < nch && outpos == c * 32u) {
            // the usual case, written tight: nothing in front of the tail moved, so it stays where it is and only its
            // flags are looked at (one 4-byte read per lane and chunk); running pointers for the chunks issued ahead
            const char* g0 = reinterpret_cast<const char*>(reinterpret_cast<const uint4*>(gE0 + (c + kRing) * 32u) + lane);
            const ptrdiff_t dE = reinterpret_cast<const char*>(s.E1) - reinterpret_cast<const char*>(s.E0);
            uint32_t left = n_old - c * 32u;
            for (;;) {
              cp_wait<kRing - 1>();
              uint4* stg = X.ring[(c - 2u) % kRing];
              const uint32_t fl = reinterpret_cast<const uint32_t*>(stg + 32 + lane)[3];
              if (!__all_sync(kFull, (fl & ~F_PARKED) == F_KLASS1 || (uint32_t)lane >= left)) break;
              if (c + kRing < nch) { cp16(stg + lane, g0); cp16(stg + 32 + lane, g0 + dE); }
              cp_commit();
              g0 += 512;
              outpos += left < 32u ? left : 32u;
              c++;
              if (c >= nch) break;
              left -= 32u;
            }
          }
          while (c < nch) {
            wait_chunk(c, outpos > c * 32u);
            const uint4* st = stage_of(c);
            const uint32_t fl = reinterpret_cast<const uint32_t*>(st + 32 + lane)[3];
            const uint32_t left = n_old - c * 32u;
            const bool valid = (uint32_t)lane < left;
            if (!__all_sync(kFull, (fl & ~F_PARKED) == F_KLASS1 || !valid)) break;
            const uint32_t np = outpos + (uint32_t)lane;
            if (outpos != c * 32u && valid) {
              const uint4 c0 = st[lane], c1 = st[32 + lane];
              __stcg(reinterpret_cast<int4*>(gE0 + np), *reinterpret_cast<const int4*>(&c0));
              __stcg(reinterpret_cast<int4*>(gE1 + np), *reinterpret_cast<const int4*>(&c1));
            }
            outpos += left < 32u ? left : 32u;
            if (c >= 2u) issue_chunk(c + kRing);
            c++;
          }
          if constexpr (DRIFT) {
            if (c > c_tail && c < nch) {                              // more follows: the tail's last request is the largest so far
              __syncwarp();
              const int4 v0 = __ldcg(reinterpret_cast<const int4*>(gE0 + outpos - 1u));
              const int4 v1 = __ldcg(reinterpret_cast<const int4*>(gE1 + outpos - 1u));
              const Rec0 r0 = *reinterpret_cast<const Rec0*>(&v0);
              const Rec1 r1 = *reinterpret_cast<const Rec1*>(&v1);
              const uint32_t key2 = par.policy == 1 ? r0.D - r1.d : r0.P + r1.d;
              const uint64_t comp = (1ull << 63) | ((uint64_t)key2 << 32) | (uint64_t)r1.id;
              if (comp > kmax) kmax = comp;
            }
          }
        }
        if (c > nch || (c == nch && dptr >= m)) break;                // (chunk nch is empty: the parked tail)

        // ---------------- (G) one chunk on the general path
        wait_chunk(c, dptr < m || outpos > c * 32u);
        const uint4* st = stage_of(c);
        const uint4 c0 = st[lane], c1 = st[32 + lane];
        if (c >= 2u) issue_chunk(c + kRing);                          // the stage is free again
        const Rec0 r0 = *reinterpret_cast<const Rec0*>(&c0);
        const Rec1 r1 = *reinterpret_cast<const Rec1*>(&c1);
        const uint32_t cv = valid_of(c);
        uint64_t key; uint32_t bin;
        score(r0, r1, k, lutv, UB_DELTA, guard, policy, key, bin);
        if (mode != 0u && cv != 0u && !drift) {
          // ---- behind the walk: a chunk of waiting requests (not resident, nothing to finalise) that sorts in front
          // of the next parked request, if any, only moves up
          const bool steady = (r1.flags & ~F_PARKED) == F_KLASS1;
          if (__all_sync(kFull, steady || !((cv >> lane) & 1u))) {
            bool before = true;
            if (dptr < m) {
              const uint4 dk = X.skb[dptr];
              const uint32_t pk_id = X.sr1[dptr].x;
              const int last = 31 - __clz((int)cv);
              const uint64_t lk = __shfl_sync(kFull, key, last);
              const uint32_t li = __shfl_sync(kFull, r1.id, last);
              before = key_less(lk, li, (uint64_t)dk.x | ((uint64_t)dk.y << 32), pk_id);
            }
            if (before) {
              const uint32_t np = outpos + __popc(cv & ltmask);
              if (np != c * 32u + (uint32_t)lane && ((cv >> lane) & 1u)) {
                __stcg(reinterpret_cast<int4*>(gE0 + np), *reinterpret_cast<const int4*>(&c0));
                __stcg(reinterpret_cast<int4*>(gE1 + np), *reinterpret_cast<const int4*>(&c1));
              }
              outpos += __popc(cv);
              c++;
              continue;
            }
          }
        }
        // the merged order of this chunk: alternately a run of its clean requests (up to the first one that sorts
        // behind the next parked request) and the parked requests that sort in front of that one
        uint32_t lo = 0, fl = 32;
        bool turn = false;                                            // false: clean run, true: parked run
#pragma unroll 1
        for (;;) {
          Rec0 w0 = r0; Rec1 w1 = r1; uint64_t wk = key; uint32_t wb = bin, wmask, wst = c * 32u + (uint32_t)lane;
          uint32_t j = 0;
          if (!turn) {
            fl = 32;
            if (dptr < m) {                                           // clean requests that sort behind the next parked one
              const uint4 dk = X.skb[dptr];
              const uint32_t di = X.sr1[dptr].x;
              const uint32_t after = __ballot_sync(kFull, ((cv >> lane) & 1u) && (uint32_t)lane >= lo &&
                                                   key_less((uint64_t)dk.x | ((uint64_t)dk.y << 32), di, key, r1.id));
              if (after) fl = (uint32_t)__ffs(after) - 1u;
            }
            wmask = cv & (fl < 32u ? ((1u << fl) - 1u) : kFull) & (lo < 32u ? (kFull << lo) : 0u);
          } else {
            j = m - dptr;                                             // parked requests in front of clean lane fl
            if (fl < 32u) {
              const uint64_t ck = __shfl_sync(kFull, key, (int)fl);
              const uint32_t ci = __shfl_sync(kFull, r1.id, (int)fl);
              const uint4 kb = X.skb[lane];
              j = __popc(__ballot_sync(kFull, (uint32_t)lane >= dptr && (uint32_t)lane < m &&
                                       key_less((uint64_t)kb.x | ((uint64_t)kb.y << 32), X.sr1[lane].x, ck, ci)));
            }
            const uint32_t src = dptr + (uint32_t)lane < 32u ? dptr + (uint32_t)lane : 31u;
            const uint4 a0 = X.sr0[src], a1 = X.sr1[src], ak = X.skb[src];
            w0 = *reinterpret_cast<const Rec0*>(&a0); w1 = *reinterpret_cast<const Rec1*>(&a1);
            wk = (uint64_t)ak.x | ((uint64_t)ak.y << 32); wb = ak.z;
            wmask = j < 32u ? ((1u << j) - 1u) : kFull; wst = 0xFFFFFFFFu;
          }
          if (wmask) process(w0, w1, wk, wb, wmask, wst);
          if (!turn) {
            lo = fl;
            if ((fl == 32u && c < nch) || dptr >= m) break;
          } else {
            dptr += j;
          }
          turn = !turn;
        }
        c++;
      }
      __syncwarp();

      // ---------------- batch totals, victim select, cost
      de = __reduce_add_sync(kFull, de);
      ps = __reduce_add_sync(kFull, ps);
      const uint32_t dec = de & 0xFFFFu, emit = de >> 16, pf = ps & 0xFFFFu, same = ps >> 16;
      kres = __reduce_add_sync(kFull, kres);
      const unsigned long long w14 = reinterpret_cast<const unsigned long long*>(X.hdr[parity])[14];
      uint32_t swap_used = (uint32_t)w14;
      const uint32_t peak = (uint32_t)(w14 >> 32);
      uint32_t swin_blocks = 0, swin_cnt = 0;
      if (X.skb[1].w) {
        swin_blocks = X.skb[0].w;
        swin_cnt = X.skb[1].w;
        swap_used -= swin_blocks;
      }
      const uint32_t C = carryC;
      const uint32_t n_new = outpos;
      uint32_t swout_blocks = 0, ev_nsw = 0, ev_nrc = 0;
      uint64_t ev_lost = 0;
      if (kres > B - C) {
        // ---- a4 (M8; SELECTVICTIM / SWAPOUT): the stalled residents (resident, not admitted) no
        // longer fit behind the claims.  Victims = the suffix of them, in priority order, whose inclusive prefix sum
        // of blocks exceeds B - C; lowest priority first, the swap pool being a sequential resource.
        const uint32_t thr = B - C;
        uint32_t behind = 0;                                          // blocks of stalled residents behind this chunk
        // (behind the last resident there is nothing to look at)
        for (int c = (int)((__reduce_max_sync(kFull, rhi) - 1u) >> 5); c >= 0; c--) {
          const uint32_t pos = (uint32_t)c * 32u + (uint32_t)lane;
          int4 v1 = make_int4(0, 0, 0, 0);
          if (pos < n_new) v1 = __ldcg(reinterpret_cast<const int4*>(gE1 + pos));
          Rec1 q = *reinterpret_cast<Rec1*>(&v1);
          const bool st = pos < n_new && (q.flags & F_RESIDENT) && !(q.flags & F_ADMITNOW);
          const uint32_t v = st ? (q.cached + blk_m1) >> blk_sh : 0u;
          const uint32_t inc = scan32(v);
          const uint32_t tot = __shfl_sync(kFull, inc, 31);
          const uint32_t prefix = kres - behind - (tot - inc);        // blocks of stalled residents up to and with me
          const bool victim = st && prefix > thr;
          uint32_t vm = __ballot_sync(kFull, victim);
          const uint32_t allvm = vm;
          const uint32_t of = q.flags;
          while (vm) {
            const int l = 31 - __clz((int)vm); vm &= ~(1u << l);
            const uint32_t cached_l = __shfl_sync(kFull, q.cached, l);
            const uint32_t id_l = __shfl_sync(kFull, q.id, l);
            const uint32_t resb = (cached_l + blk_m1) >> blk_sh;
            bool do_swap = false;
            if (s.preempt_mode == 1) do_swap = (swap_used + resb <= s.swap_pool);
            else if (s.preempt_mode == 2)
              do_swap = (swap_used + resb <= s.swap_pool) &&
                        (2ll * resb * (int64_t)s.swap_ns < 1000ll * s.c_pf * (int64_t)cached_l);
            if (do_swap) {
              swap_used += resb; swout_blocks += resb; ev_nsw++;
              if (lane == 0) ev_add(evl, evu, EV_EVICT_SWAP, id_l, resb);
              if (lane == l) q.flags = F_SWAPPED | F_PREEMPTED | F_DIRTY;
            } else {
              ev_lost += cached_l; ev_nrc++;
              if (lane == 0) ev_add(evl, evu, EV_EVICT_RECOMPUTE, id_l, cached_l);
              if (lane == l) { q.cached = 0; q.flags = F_PREEMPTED | F_DIRTY; }
            }
          }
          if (victim) {
            uint32_t* g_ne = s.n_evict + (size_t)r * s.N;
            g_ne[q.id] = __ldcg(g_ne + q.id) + 1u;
            int64_t* g_tp = s.t_pre + (size_t)r * s.N + q.id;         // M15: preempted from the start of this iteration on
            *g_tp = __ldcg(g_tp) - (int64_t)sh[0];
            if (of & F_KLASS1) {                                      // victim was not MemGuard-locked
              uint32_t* g_neu = s.n_evict_unf + (size_t)r * s.N;
              g_neu[q.id] = __ldcg(g_neu + q.id) + 1u;
            }
            __stcg(reinterpret_cast<int4*>(gE1 + pos), *reinterpret_cast<const int4*>(&q));
          }
          const uint32_t dm = __ballot_sync(kFull, victim && !(of & F_DIRTY));      // residency changed => dirty
          if (dm) {
            const uint32_t slot = ndnew + __popc(dm & ltmask);
            if (victim && !(of & F_DIRTY) && slot < kDirtyMax) s.hdr[r].dl[slot] = (uint16_t)pos;
            ndnew += __popc(dm);
          }
          behind += tot;
          if (__ballot_sync(kFull, st) != allvm) break;               // a stalled resident that stays: so do all before it
        }
      }
      int64_t cost = s.c0 + s.c_pf * (int64_t)pf + s.c_dec * (int64_t)dec;
      if (swin_blocks + swout_blocks) cost += (int64_t)(((uint64_t)(swin_blocks + swout_blocks) * s.swap_ns + 500u) / 1000u);
      const int64_t t_end = (int64_t)sh[0] + cost;

      // ---------------- the queued per-request events, now that t_end is known (M10, M11)
      if (nev) {
        const uint2* gev = s.evbuf + (size_t)r * s.evcap;
        int64_t* g_tfirst = s.t_first + (size_t)r * s.N;
        int64_t* g_tlast = s.t_last + (size_t)r * s.N;
        uint32_t cseq = ADA ? (uint32_t)reinterpret_cast<const unsigned long long*>(X.hdr[parity])[15] : 0u;   // completions so far
#pragma unroll 1
        for (uint32_t e0 = 0; e0 < nev; e0 += 32u) {
          const uint32_t e = e0 + (uint32_t)lane;
          uint32_t cm = 0;
          uint2 ev = make_uint2(0u, 0u);
          if (e < nev) {
            if (e < kEvSmem) { const uint32_t w = X.skb[2u + e].w; ev = make_uint2(w >> 3, w & 7u); }
            else ev = __ldcg(gev + e);
          }
          if constexpr (ADA) cm = __ballot_sync(kFull, (ev.y & 4u) != 0u);   // completions of this batch, in priority order
          if (e < nev) {
            const uint32_t id = ev.x;
            if (ev.y & 1u) {
              g_tfirst[id] = t_end;
              ev_add(evl, evu, EV_EMIT_FIRST, id, 0u);
            }
            if (ev.y & 2u) {
              const int64_t tl = __ldcg(g_tlast + id);
              atomicAdd(s.hist + (size_t)r * kTbtBins + tbt_bin(t_end - tl), 1u);
            }
            if (ev.y & 4u) {
              g_tlast[id] = t_end;
              const int64_t tf = (ev.y & 1u) ? t_end : __ldcg(g_tfirst + id);
              const int4 tv = __ldg(reinterpret_cast<const int4*>(UB_TR + id));
              const Rec0 q0 = *reinterpret_cast<const Rec0*>(&tv);
              if constexpr (ADA)                                      // gamma-Ada: end-to-end latency sample (M13)
                s.ada_ring[(size_t)r * s.ada_W + (cseq + __popc(cm & ltmask)) % s.ada_W] = t_end - q0.a;
              atomicAdd(UB_H64 + 8, (unsigned long long)(tf - q0.a));
              atomicAdd(UB_H64 + 9, (unsigned long long)(t_end - q0.a));
              atomicAdd(UB_H64 + 10, (unsigned long long)(t_end - tf));
              atomicAdd(UB_H64 + 11, (unsigned long long)(q0.D - 1u));
              ev_add(evl, evu, EV_COMPLETE, id, 0u);
              uint32_t* g_ne = s.n_evict + (size_t)r * s.N;
              g_ne[id] = __ldcg(g_ne + id) | 0x80000000u;             // completion marker read by the stats kernel
            }
          }
          cseq += __popc(cm);
        }
      }
      evl = __reduce_add_sync(kFull, evl);
      evu = __reduce_add_sync(kFull, evu);

      // ---------------- header: clock, digest (M12), cursors; counters by RED (no read needed)
      if (ndnew > kDirtyMax) ndnew = kDirtyMax + 1u;
      __syncwarp();                                                   // every lane has read the header image (clock) by now
      if (lane == 0) {
        unsigned long long* shw = reinterpret_cast<unsigned long long*>(X.hdr[parity]);
        const uint64_t H = digest_fold(shw[1], evl, evu, t_end);
        shw[1] = H;                                                   // (kept current for a further iteration)
        shw[0] = (unsigned long long)t_end;
        if constexpr (ADA) shw[15] += (unsigned long long)n_done | ((unsigned long long)ev_nrc << 32);
        if constexpr (MULTI) reinterpret_cast<uint32_t*>(UB_H64 + 19)[0] = n_done;   // Hdr::last_done (fenced runs: the router)
        const uint32_t pk = n > peak ? n : peak;
        shw[14] = (unsigned long long)swap_used | ((unsigned long long)pk << 32);
        if (same) atomicAdd(s.hist + (size_t)r * kTbtBins + tbt_bin(cost), same);
        __stcg(UB_H64 + 0, (unsigned long long)t_end);
        __stcg(UB_H64 + 1, (unsigned long long)H);
        shw[13] = (unsigned long long)n_new | (shw[13] & 0xFFFFFFFF00000000ull);
        __stcg(UB_H64 + 13, shw[13]);
        if (n > peak || swin_blocks || swout_blocks)
          __stcg(UB_H64 + 14, (unsigned long long)swap_used | ((unsigned long long)pk << 32));
        if (ndnew != nd) __stcg(reinterpret_cast<uint32_t*>(UB_H64 + 18), ndnew);
        atomicAdd(UB_H64 + 3, (unsigned long long)n);                    // request-steps
        atomicAdd(UB_H64 + 4, (unsigned long long)emit);
        if (pf) atomicAdd(UB_H64 + 5, (unsigned long long)pf);
        atomicAdd(UB_H64 + 6, (unsigned long long)dec);
        if (ev_lost) atomicAdd(UB_H64 + 7, (unsigned long long)ev_lost);
        atomicAdd(UB_H64 + 12, 1ull);                                    // iterations
        if (n_done | ev_nrc) atomicAdd(UB_H64 + 15, (unsigned long long)n_done | ((unsigned long long)ev_nrc << 32));
        if (ev_nsw | swin_cnt) atomicAdd(UB_H64 + 16, (unsigned long long)ev_nsw | ((unsigned long long)swin_cnt << 32));
      }
      n = n_new; wsize = n_new; nd = ndnew;
      if (n == 0 && (int64_t)sh[2] == kNever) {                       // finished its trace in this call
        if (lane == 0) atomicAdd(A.count + 5, 1u);
        it++;
        break;
      }
      if (MULTI) __syncwarp();                                        // window stores before the next iteration's loads
    }

    // ---------------- not handled here: queue the replica for the team kernels of this round
    if (slow && lane == 0) {
      reinterpret_cast<uint32_t*>(UB_H64 + 17)[1] = iters - it;                 // iterations it owes the team kernels
      push_list(A, s.all_stream ? 2u : (wsize <= A.thrS ? 0u : (wsize <= A.thrM ? 1u : 2u)), r);
    }
  }
  cp_wait<0>();
#undef UB_H64
#undef UB_GW
#undef UB_TR
#undef UB_DELTA
}

// ub_debug_keys_stream: the (class, key) this file's own scorer -- score(), the one the streaming kernel runs -- gives
// every request of one replica's window as it stands (kernel-level parity of a1, M3-M5); one warp, 32 records a time
__global__ void k_debug_keys_stream(const SimDev s, const uint32_t r, const uint32_t n, uint32_t* id, unsigned long long* okey) {
  const int lane = threadIdx.x & 31;
  const RepPar par = s.hdr[r].par;
  int64_t lutv = 0;
  if (par.policy == 2) lutv = __ldg(s.lut + par.lut_off + (size_t)s.hdr[r].level * 64u + lane);
  for (uint32_t base = 0; base < n; base += 32u) {
    const uint32_t p = base + (uint32_t)lane;
    Rec0 q0; Rec1 q1;
    q0.a = 0; q0.P = 1; q0.D = 1; q1.id = 0; q1.d = 0; q1.cached = 0; q1.flags = 0;
    if (p < n) { q0 = s.E0[(size_t)r * s.Q + p]; q1 = s.E1[(size_t)r * s.Q + p]; }
    uint64_t key; uint32_t bin;
    score(q0, q1, s.k, lutv, (par.policy == 0 || par.policy == 2) ? par.delta : 0ll, par.guard != 0, par.policy, key, bin);
    if (p < n) { id[p] = q1.id; okey[p] = key; }
  }
}
void launch_debug_keys_stream(const SimDev& s, uint32_t r, uint32_t n, uint32_t* id, unsigned long long* okey, cudaStream_t st) {
  k_debug_keys_stream<<<1, 32, 0, st>>>(s, r, n, id, okey);
}

// persistent grid: every warp takes replicas until none is left
template <bool ADA, bool MULTI, bool LIST, bool DRIFT, bool SPEC> static void launch_stream_t(const StepArgs& A0, cudaStream_t st) {
  StepArgs A = A0;
  static int ctas_per_sm = 0;
  if (!ctas_per_sm) {
    cudaFuncSetAttribute(k_stream<ADA, MULTI, LIST, DRIFT, SPEC>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, k_stream<ADA, MULTI, LIST, DRIFT, SPEC>, 32 * kSWarps, 0) != cudaSuccess ||
        ctas_per_sm < 1)
      ctas_per_sm = 4;
  }
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const uint32_t need = (A.rend - A.rbeg + kSWarps - 1) / kSWarps;
  uint32_t grid = (uint32_t)(sms * ctas_per_sm);
  if (grid > need) grid = need;
  // a warp takes 15/16 of an even share of the replicas by static striding (7/8 with several iterations per launch), the
  // rest by tickets (measured on config 5, the generic instance: 1/2 7.4e10, 3/4 8.15e10, 7/8 8.32e10, 15/16 8.29e10, all
  // static 7.97e10 request-steps/s; the BOOST + MemGuard instance: 13/16 8.27e10, 7/8 8.54e10, 15/16 .. 61/64 8.60e10,
  // the resident mode 1.03e11 at 7/8 and 1.005e11 at 15/16)
  const uint32_t nwarps = grid * kSWarps, share = ((A.rend - A.rbeg) / nwarps) * (MULTI ? 14u : 15u) / 16u;
  A.nstat = share > 2u ? share : 2u;
  A.dynbase = A.rbeg + A.nstat * nwarps;
  k_stream<ADA, MULTI, LIST, DRIFT, SPEC><<<grid, 32 * kSWarps, 0, st>>>(A);
}
template <bool SPEC> static void launch_main(const StepArgs& A, cudaStream_t st) {
  if (A.s.ada_ring) launch_stream_t<true, false, false, false, SPEC>(A, st);   // (gamma-Ada: one iteration per launch, no list: ub_api.cu)
  else if (A.iters > 1u) { if (A.live) launch_stream_t<false, true, true, false, SPEC>(A, st); else launch_stream_t<false, true, false, false, SPEC>(A, st); }
  else if (A.live) launch_stream_t<false, false, true, false, SPEC>(A, st);
  else launch_stream_t<false, false, false, false, SPEC>(A, st);
}
void launch_stream(const StepArgs& A, cudaStream_t st) {
  if (A.rend <= A.rbeg) return;
  if (A.drift) {                                                   // the drift group always comes as a list
    if (A.iters > 1u) launch_stream_t<false, true, true, true, false>(A, st); else launch_stream_t<false, false, true, true, false>(A, st);
  }
  else if (A.s.all_boost_guard) launch_main<true>(A, st);
  else launch_main<false>(A, st);
}

}  // namespace ub
