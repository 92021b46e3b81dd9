// ub_device.cuh -- device helpers shared by the step kernels (ub_stream.cu: streaming warp-per-replica path,
// ub_step.cu: general team-per-replica path).  Both kernels operate on the same HBM state (ub_internal.cuh),
// so a replica may be advanced by either one in any iteration.  Nothing here is shared with oracle/.
#pragma once
#include "ub_internal.cuh"

namespace ub {

// ceil(x / blk): a shift when the block size is a power of two (the usual 16), else a division
__device__ __forceinline__ uint32_t blocks_of(const SimDev& s, uint32_t x) {
  return s.blk_shift < 32u ? (x + s.blk - 1u) >> s.blk_shift : (x + s.blk - 1u) / s.blk;
}

// M12 (test plumbing): event hash = 32-bit mix of (id, type) times the odd number 2*payload+1; inside an
// iteration the low and high halves are summed separately modulo 2^32, so any reduction order (redux.sync,
// shared-memory atomics) gives the same result; one multiply-xorshift round folds the iteration into H.
enum { EV_ADMIT = 1, EV_EVICT_RECOMPUTE = 2, EV_EVICT_SWAP = 3, EV_SWAPIN = 4, EV_EMIT_FIRST = 5, EV_COMPLETE = 6 };
__device__ __forceinline__ void ev_add(uint32_t& lo, uint32_t& hi, uint32_t type, uint32_t id, uint32_t payload) {
  const uint32_t m = ((id + 1u) * 0x9E3779B1u) ^ (type * 0x85EBCA6Bu);
  const uint64_t h = (uint64_t)m * (uint64_t)(2u * payload + 1u);
  lo += (uint32_t)h;
  hi += (uint32_t)(h >> 32);
}
__device__ __forceinline__ uint64_t digest_fold(uint64_t H, uint32_t lo, uint32_t hi, int64_t t_end) {
  uint64_t x = (H ^ (((uint64_t)hi << 32) | (uint64_t)lo)) + (uint64_t)t_end * 0x9E3779B97F4A7C15ull;
  x ^= x >> 29;
  x *= 0xBF58476D1CE4E5B9ull;
  x ^= x >> 32;
  return x;
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

__device__ __forceinline__ uint32_t signal_of(const RepPar& par, uint32_t P, uint32_t D, uint32_t d) {
  if (par.signal_mode == 0) return P + d;                       // w~ = max(w, s_pre)
  if (par.signal_mode == 1) return (d == 0) ? P : d;            // SIGNAL
  return D - d;                                                 // remaining (tests: SRPT limit)
}
__device__ __forceinline__ uint32_t bin_of(const RepPar& par, uint32_t k, uint32_t sig) {
  return (par.quant_mode == 0) ? geo_bin(sig, k) : sig;         // QUANTIZE, Eq. 8
}

// a1 for every policy (M3-M5, M14): okey = class<<63 | (key + 2^62) of one request; the general form used by the team
// kernels and by ub_debug_keys (the streaming kernel has its own lean copy for FCFS / BOOST, ub_stream.cu score()).
// lut: the replica's boost table (already offset by its gamma-Ada level); tfirst / tlast: the replica's t_first / t_last
// rows; t: the replica clock (a request that emitted in the last iteration carries its t_last implicitly: == t).
__device__ __forceinline__ uint64_t okey_of(const SimDev& s, const RepPar& par, const int64_t* lut, const int64_t* tfirst,
                                            const int64_t* tlast, const int64_t t, const Rec0& q0, const Rec1& q1) {
  const uint32_t sig = signal_of(par, q0.P, q0.D, q1.d);
  const uint32_t bin = bin_of(par, s.k, sig);
  int64_t kv;
  if (par.policy == 0) kv = q0.a;                                                  // FCFS
  else if (par.policy == 1) kv = (int64_t)(q0.D - q1.d);                           // SRPT, perfect lengths
  else if (par.policy == 3) kv = (int64_t)sig;                                     // LAS
  else if (par.policy == 4) kv = (int64_t)q0.D;                                    // SJF, perfect lengths
  else if (par.policy == 5) kv = (int64_t)q0.P;                                    // SPF
  else if (par.policy == 6) {                                                      // DistBoost (M14), Eq. 3-4
    if (q1.d >= 1u) kv = __ldcg(tfirst + q1.id);
    else { const uint32_t pb = bin_of(par, s.k, q0.P); kv = q0.a - __ldg(lut + (pb < par.lut_nb ? pb : par.lut_nb - 1)); }
  }
  else if (par.policy == 7) {                                                      // Sarathi (M16)
    // decode queue round robin: by the time of the last token; prefill queue first come first served
    kv = q1.d >= 1u ? ((q1.flags & F_EMITPREV) ? t : __ldcg(tlast + q1.id)) : q0.a;
  }
  else kv = q0.a - __ldg(lut + (bin < par.lut_nb ? bin : par.lut_nb - 1));         // pi = a - b
  const bool res = (q1.flags & F_RESIDENT) != 0;
  if (res && (par.policy == 0 || par.policy == 2)) kv -= par.delta;                // Eq. 7 as a bias
  uint64_t klass = (par.guard && res && (q1.flags >> F_LOCK_SHIFT) == bin + 1u) ? 0ull : 1ull;   // MemGuard lock
  if (par.policy == 6 || par.policy == 7) klass = q1.d >= 1u ? 0ull : 1ull;        // decode batch first, Eq. 5-6 / PAPER.md:239
  return (klass << 63) | (uint64_t)(kv + kKeyBias);
}

__device__ __forceinline__ uint32_t warp_scan_incl(uint32_t v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += n;
  }
  return v;
}

__device__ __forceinline__ bool key_less(uint64_t ka, uint32_t ia, uint64_t kb, uint32_t ib) {
  return ka < kb || (ka == kb && ia < ib);
}

// ---------------------------------------------------------------------------------------------- work lists
// Per scheduler round: the streaming kernel visits every replica and queues the ones it does not handle itself into
// list[cls * R + i], count[cls]; cls 0 = S (1 warp), 1 = M (4 warps), 2 = L (8 warps), 3 = overflow (a window that
// outgrew its team during the round).  count[5] = replicas that have finished their trace (monotone).
struct StepArgs {
  SimDev s;
  uint32_t* list; uint32_t* count;
  uint32_t iters;
  uint32_t tick;                // which of the two ticket counters (count[4], count[6]) this launch draws from
  uint32_t nstat, dynbase;      // k_stream work distribution (set by launch_stream): static replicas per warp, first ticket
  uint32_t rbeg, rend;          // replicas [rbeg, rend) belong to this launch (a round may be split over two streams)
  uint32_t thrS, thrM;          // window size up to which a replica is queued for the S / M kernel
  const uint32_t* live;         // k_stream, list mode: the replicas to visit are live[rbeg .. rend) (else the indices themselves)
  uint32_t drift;               // this launch advances the drift group (SRPT / LAS replicas), see ub_stream.cu
  const int64_t* tlimit;        // time fence (rule M18, JSQ): replica r runs only iterations that start before tlimit[r]; null = none
};

__device__ __forceinline__ void push_list(const StepArgs& A, uint32_t slot, uint32_t r) {
  const uint32_t idx = atomicAdd(A.count + slot, 1u);
  A.list[(size_t)slot * A.s.R + idx] = r;
}

}  // namespace ub
