// ub_internal.cuh -- device-side data layout shared by the kernels and the C-ABI host code of libuniboost.so.
// (Nothing here is shared with oracle/.)
//
// HBM layout.  Per replica r the active window is a struct of two 16-byte record
// arrays kept in PRIORITY ORDER of the last executed iteration (so the next iteration finds it nearly sorted):
//   E0[r][Q] = { a: i64 arrival us, P: u32 prompt tokens, D: u32 hidden output tokens }   static per request
//   E1[r][Q] = { id: u32, d: u32 tokens emitted, cached: u32 KV tokens held, flags: u32 } dynamic
// plus one 256-byte header Hdr[r] -- 160 bytes of state (8-byte word i is addressed directly by the streaming kernel:
// keep the order), the replica's parameters and its dirty list, fetched together by one asynchronous copy --, the
// packed traces TR[trace][N] (same 16-byte record as E0), the
// per-request outputs t_first/t_last/n_evict/n_evict_unforced [R][N] and the TBT histogram [R][4352].
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace ub {

constexpr int      kTbtBins   = 4352;
constexpr uint32_t kMaxQueue  = 2048;
constexpr int64_t  kBoostMax  = (int64_t)1 << 60;
constexpr int64_t  kKeyBias   = (int64_t)1 << 62;
constexpr int64_t  kNever     = INT64_MAX;          // a_next when the trace is exhausted

// flags word of E1
constexpr uint32_t F_RESIDENT = 1u;        // KV on the device
constexpr uint32_t F_SWAPPED  = 2u;        // KV in the host swap pool
constexpr uint32_t F_EMITPREV = 4u;        // emitted a token in the previous executed iteration => t_last == clock
constexpr uint32_t F_DIRTY    = 8u;        // (class,key) may differ from the previous iteration's => listed in dlist
constexpr uint32_t F_ADMITNOW = 16u;       // admitted in the last executed iteration (read by the eviction pass only)
constexpr uint32_t F_KLASS1   = 32u;       // was in class 1 (not MemGuard-locked) in the last executed iteration
constexpr uint32_t F_PREEMPTED = 64u;      // evicted (swap or recompute) and not yet admitted again (rule M15: preemption time)
constexpr uint32_t F_PARKED  = F_SWAPPED | F_PREEMPTED;   // what a waiting request may carry besides F_KLASS1
constexpr int      F_LOCK_SHIFT = 7;       // bits 7..31: lockbin + 1 (0 = no lock)
constexpr uint32_t F_LOCK_MASK_LOW = (1u << F_LOCK_SHIFT) - 1u;   // the flag bits below the lock field
constexpr uint32_t kDirtyMax  = 32;        // entries of a replica's dirty list; Hdr::n_dirty > kDirtyMax = overflow

struct __align__(16) Rec0 { int64_t a; uint32_t P; uint32_t D; };
struct __align__(16) Rec1 { uint32_t id; uint32_t d; uint32_t cached; uint32_t flags; };

struct __align__(16) RepPar {   // per-replica parameters, read-only on the device (32 bytes: two cp.async pieces)
  int64_t  delta;               // hysteresis_us
  uint32_t trace_id;
  uint32_t lut_off;             // offset of this replica's boost table in lut[]
  uint32_t lut_nb;              // entries
  uint8_t  policy, guard, signal_mode, quant_mode;
  uint32_t pad[2];
};
struct __align__(16) Hdr {   // 256 bytes per replica: state (160), parameters (32), dirty list (64) -- one prefetch

  int64_t  t;                 // replica clock, us
  uint64_t H;                 // schedule digest (M12)
  int64_t  a_next;            // arrival of trace[next], kNever if exhausted
  int64_t  request_steps;
  int64_t  tokens_emitted, prefill_tokens, decode_seqs, tokens_lost;
  int64_t  sum_ttft, sum_ttlt, sum_tbt_num, sum_tbt_den;
  int64_t  iterations;
  uint32_t n_active, next, swap_used, peak_active;
  uint32_t n_completed, evict_recompute, evict_swap, swapins;
  uint32_t done, todo, n_dirty, level;  // todo: iterations of this round still to do (hand-over between kernels);
                                        // level: gamma-Ada grid level (0 for a static replica), selects the boost table
  uint32_t last_done;           // requests completed by the last executed iteration (read by the JSQ router, M18)
  uint32_t pad_state;
  RepPar   par;               // per-replica parameters (read-only after ub_set_replicas)
  uint16_t dl[kDirtyMax];     // window positions of the re-keyed ("dirty") requests
};
static_assert(sizeof(Hdr) == 256 && offsetof(Hdr, par) == 160, "Hdr: 160 bytes of state, then parameters and dirty list");

constexpr uint32_t kMaxSplit = 16;    // parts (streams) a scheduler round may be issued as, the drift group's included
constexpr uint32_t kWindowPad = 64;   // records allocated behind the last window (speculative chunk reads)

struct __align__(16) AdaState { int64_t gamma_u; unsigned long long n_updates; uint32_t level, seen, on, pad; };

struct SimDev {                 // kernel argument (by value)
  // configuration
  uint32_t R, NT, N, Q;
  uint32_t B, blk, M, c, T;
  uint32_t blk_shift;           // log2(blk) if blk is a power of two, else 32
  uint32_t preempt_mode, swap_ns, swap_pool, k;
  int64_t  c0, c_pf, c_dec;
  // state
  Rec0* E0; Rec1* E1; Hdr* hdr;
  const Rec0* TR;               // packed traces [NT][N]
  const uint32_t* n_req;        // [NT]
  const int64_t* lut;
  int64_t* t_first; int64_t* t_last;      // [R][N]
  int64_t* t_pre;                         // [R][N] preemption time (M15): minus the eviction times plus the re-admission times
  uint32_t* n_evict; uint32_t* n_evict_unf;
  uint32_t* hist;               // [R][kTbtBins]
  uint2*    evbuf;              // [R][evcap] scratch: per-request events of one iteration that wait for t_end
  uint32_t  evcap;              // min(M, Q)
  // gamma-Ada (M13); ada_ring == nullptr when off
  int64_t*  ada_ring;           // [R][ada_W] end-to-end latencies, slot = completion number mod ada_W
  struct AdaState* ada_state;   // [R]
  const int64_t* ada_grid;      // [ada_G] gamma_u thresholds
  uint32_t  ada_W, ada_G, ada_min, ada_shift;
  int64_t   ada_eps;
  uint32_t  all_stream;         // every replica is eligible for the streaming kernel: its rare hand-overs all go to the L team kernel
  uint32_t  all_boost_guard;    // every replica is BOOST with MemGuard, the paper's signal and quantiser (the method itself,
                                // PAPER.md:406-473), block size a power of two: k_stream's instance specialised for it runs
};

// kernels (ub_step.cu, ub_aux.cu)
void launch_step(const SimDev& s, uint32_t* list, uint32_t* count, uint32_t iters, uint32_t rbeg, uint32_t rend,
                 uint32_t tick, const uint32_t* live, bool drift, const int64_t* tlimit, cudaStream_t st);
void flush_slow(const SimDev& s, uint32_t* list, uint32_t* count, uint32_t rbeg, uint32_t rend, const int64_t* tlimit,
                cudaStream_t st);
struct JsqArgs {                // one global arrival stream per cluster of K replicas (rule M18)
  uint32_t K, C, NA; const int64_t* a; const int32_t* p; const int32_t* d; const uint32_t* n_arr;
  int64_t* tlimit; int32_t* assign; uint32_t* count; int* err;
};
void launch_jsq_dispatch(const SimDev& s, const JsqArgs& J, int64_t j, cudaStream_t st);
void launch_stream(const struct StepArgs& A, cudaStream_t st);    // ub_stream.cu
void launch_debug_keys_stream(const SimDev& s, uint32_t r, uint32_t n, uint32_t* id, unsigned long long* okey, cudaStream_t st);
void launch_gamma_ada(const SimDev& s, uint32_t rbeg, uint32_t rend, cudaStream_t st);   // ub_aux.cu
void launch_ada_init(const SimDev& s, cudaStream_t st);
int  step_configure(uint32_t Q);
void launch_pack_validate(const int64_t* a, const int32_t* p, const int32_t* d, const int32_t* hit, const uint32_t* n_req,
                          uint32_t NT, uint32_t N, uint32_t B, uint32_t blk, Rec0* out, int* err, cudaStream_t st);
void launch_reset(const SimDev& s, uint32_t* list, uint32_t* count, cudaStream_t st);
void launch_count_live(const uint32_t* count, uint32_t R, unsigned long long* live, cudaStream_t st);
void launch_compact_live(const SimDev& s, uint32_t rbeg, uint32_t rend, const uint32_t* in, bool drift_group, bool any_state,
                         uint32_t* out, uint32_t* cnt, cudaStream_t st);
void launch_flush_tlast(const SimDev& s, cudaStream_t st);
struct StatsDev {               // device-side result of the percentile reduction, one per replica
  int64_t ttft[3], ttlt[3], tbt[3];
};
void launch_stats(const SimDev& s, StatsDev* out, cudaStream_t st);
void launch_percentile_curve(const SimDev& s, uint32_t which, const uint32_t* permille, uint32_t n, int64_t* out,
                             cudaStream_t st);
// the same with the result staged in a static device array of kNoAllocCurveMax values (ub_aux.cu); *staged = its device
// address.  0, -1 (n_replicas x n beyond the array, or device number out of range) or -2 (symbol lookup failed)
constexpr size_t kNoAllocCurveMax = 65536;
int launch_percentile_curve_noalloc(const SimDev& s, int device, uint32_t which, const uint32_t* permille, uint32_t n,
                                    const int64_t** staged, cudaStream_t st);
void launch_class_percentiles(const SimDev& s, uint32_t which, uint32_t len_lo, uint32_t len_hi, const uint32_t* permille,
                              uint32_t n, int64_t* out, uint32_t* count, int64_t* sum, cudaStream_t st);
void launch_slo_count(const SimDev& s, uint32_t which, uint32_t n, const int64_t* thr, uint32_t* out, cudaStream_t st);

}  // namespace ub
