/*
 * uniboost.h -- C-ABI of libuniboost.so: the per-iteration scheduling step of a
 * continuous-batching LLM replica under the tail-aware scheduler of
 * arxiv 2606.18431 (UniBoost), batched over R independent replicas and run as
 * a trace-driven simulation on one B200 (sm_100a).
 *
 * Every step of the path runs in hand-written CUDA kernels; there is no CPU
 * fallback.  Operation definitions (rules M1..M12) follow
 *   Algorithm 1, PAPER.md:406-473   (rescore all active -> unified order ->
 *                                    admit under KV capacity -> evict -> execute -> stats)
 *   BOOST / QUANTIZE / SIGNAL,      PAPER.md:564-587, Eq. 2, Eq. 8
 *   unified priority + hysteresis,  PAPER.md:185-196 (Eq. 7)
 *   MemGuard minimum-run rule,
 *   problem statement,              PAPER.md:117-123 (requests a_i, s_pre, s_dec), PAPER.md:409 (B, M, c, k, gamma)
 * and the per-iteration cost model of BASELINE.json configs 1 and 3.
 *
 * Conventions
 *  - every call returns UB_OK (0) or a negative UB_E* code; nothing throws or aborts across the ABI;
 *  - "host" / "device" is stated per pointer; input arrays are caller-owned and copied (free after return);
 *    outputs go to caller-allocated buffers; the handle owns all its device memory;
 *  - the handle is not thread-safe; work is ordered on the borrowed CUDA stream; only the calls marked
 *    "synchronises" wait for the device;
 *  - all times are int64 microseconds; the only floating point is the host-side build of the boost table
 *    (fp64, M4) and the final us -> s conversion of the statistics.
 */
#ifndef UNIBOOST_H
#define UNIBOOST_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define UB_ABI_VERSION 1u
#define UB_MAX_QUEUE   2048u      /* largest queue_cap (active requests per replica) */
#define UB_TBT_BINS    4352u      /* log-linear TBT histogram, 7 sub-bits, gaps < 2^40 us (M11) */

enum { UB_OK = 0, UB_EINVAL = -1, UB_ENOMEM = -2, UB_ECUDA = -3, UB_ESTATE = -4,
       UB_EUNSORTED = -5, UB_EINFEASIBLE = -6, UB_ELIVELOCK = -7, UB_ETOOBIG = -8 };

/* policy (M5): key = a | D-d | a - b_gamma(w_hat) | sig */
enum { UB_FCFS = 0, UB_SRPT = 1, UB_BOOST = 2, UB_LAS = 3,
       UB_SJF = 4,    /* shortest job first: key = hidden output length D (perfect lengths) */
       UB_SPF = 5,    /* shortest prompt first: key = prompt length P */
       UB_DISTBOOST = 6,    /* Phase-1 strawman DistBoost: decode queue first, keyed by the time of
                               entering it (Eq. 4); prefill queue keyed by a - b_gamma(prompt) (Eq. 3); guard and
                               hysteresis are not applied */
       UB_SARATHI = 7 };    /* the Sarathi baseline ("chunk-prefill, decode-prioritized continuous batching,
                               with round-robin ordering in the decode and piggy-back prefills"; rule M16): decode queue
                               first, ordered by the time of the request's last token; prefill queue first come first
                               served; guard and hysteresis are not applied */
/* size signal (M3): P+d | SIGNAL of PAPER.md:575-587 | D-d (tests: SRPT limit) */
enum { UB_SIG_UNIFIED = 0, UB_SIG_PHASE = 1, UB_SIG_REMAINING = 2 };
/* quantiser (M3): Eq. 8 geometric bins | identity (vanilla boost, tests) */
enum { UB_Q_GEOMETRIC = 0, UB_Q_EXACT = 1 };
/* preemption (M8) */
enum { UB_PRE_RECOMPUTE = 0, UB_PRE_SWAP = 1, UB_PRE_AUTO = 2 };

typedef struct ub_sim ub_sim;     /* opaque */

/* Simulator-wide parameters ("Require: B, M, c, k"; cost model BASELINE.json). */
typedef struct {
  uint32_t struct_size;           /* sizeof(ub_config), checked */
  uint32_t abi_version;           /* UB_ABI_VERSION */
  uint32_t n_replicas;            /* R >= 1 */
  uint32_t n_traces;              /* distinct traces; replicas may share one */
  uint32_t max_requests;          /* N: row length of the trace arrays, < 2^29 */
  uint32_t queue_cap;             /* Q: max simultaneously active requests per replica, 1..UB_MAX_QUEUE */
  uint32_t kv_blocks;             /* B: KV capacity in blocks */
  uint32_t block_tokens;          /* blk: tokens per block (16) */
  uint32_t max_batch;             /* M: batch cap */
  uint32_t chunk_tokens;          /* c: prefill chunk, 1..65535 */
  uint32_t token_budget;          /* T: tokens per iteration, 1..65535 */
  uint32_t preempt_mode;          /* UB_PRE_* */
  uint32_t swap_ns_per_block;     /* swap time per block, ns (128 KiB / 25 GB/s = 5243) */
  uint32_t swap_pool_blocks;      /* host swap pool, blocks */
  uint32_t bin_tokens;            /* MemGuard k (Eq. 8) */
  uint32_t tok_us;                /* service us credited per token in the argument of b_gamma (reading G1) */
  int64_t  c0_us;                 /* iteration cost = c0 + c_prefill_tok * prefill tokens            (<= 2^40) */
  int64_t  c_prefill_tok_us;      /*                + c_decode_seq * decode sequences + swap time (M9); <= 2^20 */
  int64_t  c_decode_seq_us;       /* <= 2^30 */
  uint32_t iters_per_launch;      /* scheduler iterations one kernel launch advances; 0 or 1 = one iteration per
                                     launch with the state streamed HBM -> SM -> HBM every iteration */
  int32_t  device;                /* CUDA device ordinal */
  void*    stream;                /* cudaStream_t, borrowed; NULL = the legacy default stream */
} ub_config;

/* One per replica: policies / gamma points / trace seeds run side by side as the batch dimension. */
typedef struct {
  uint32_t trace_id;
  uint8_t  policy;                /* UB_FCFS .. UB_SARATHI */
  uint8_t  guard;                 /* MemGuard lock on/off */
  uint8_t  signal_mode;           /* UB_SIG_* */
  uint8_t  quant_mode;            /* UB_Q_* */
  int64_t  hysteresis_us;         /* delta_hyst of Eq. 7, 0 .. 2^60 */
  double   gamma;                 /* 1/s, > 0; +inf => boost 0 (== FCFS) */
} ub_replica;

/* Per-replica statistics (M11); identical field meaning to the oracle's. */
typedef struct {
  int64_t iterations, request_steps, n_completed;
  int64_t evict_recompute, evict_swap, swapins;
  int64_t tokens_lost, tokens_emitted, prefill_tokens, decode_seqs;
  int64_t t_end_us, peak_active, done, swap_used;
  int64_t ttft_us[3], ttlt_us[3], tbt_us[3];        /* P50, P90, P99: nearest rank */
  int64_t sum_ttft_us, sum_ttlt_us, sum_tbt_num_us, sum_tbt_den;
  double  ttft_s[3], ttlt_s[3], tbt_s[3];           /* the same in fp64 seconds */
  double  mean_ttft_s, mean_ttlt_s, mean_tbt_s, tokens_per_s;
} ub_replica_stats;

/* Create a simulator.  cfg: host.  Allocates all device state for R replicas. */
int  ub_create(const ub_config* cfg, ub_sim** out);
void ub_destroy(ub_sim*);

/* Load the request traces: [n_traces][max_requests] row-major, arrival-sorted per row,
 * n_req[n_traces] valid requests per row.  Pointers are host (ptrs_on_device = 0) or device (1); the data
 * is copied.  Validates on the device: UB_EUNSORTED if arrivals decrease, UB_EINFEASIBLE if some request has
 * P < 1, D < 1 or ceil((P+D)/blk) > B, UB_EINVAL if an arrival is outside [0, 2^61].  Synchronises. */
int  ub_load_trace(ub_sim*, const int64_t* arrival_us, const int32_t* prompt_tok, const int32_t* decode_tok,
                   const uint32_t* n_req, int ptrs_on_device);

/* Prefix / radix caching (A.5; rule M17 of DESIGN.md): as ub_load_trace plus hit_tok
 * [n_traces][max_requests] (host or device like the others), the prompt tokens of each request already in the prefix
 * cache, 0 <= h < P (else UB_EINVAL).  "Caching primarily reduces effective prefill work": the request prefills
 * s_pre - h tokens, and its size signal is w~ = max(w, s_pre - h) with w the tokens processed so far -- the device
 * record carries the effective prompt s_pre - h for both.  (The shared prefix's KV blocks belong to the cache and are
 * not charged to the request's footprint.)  Synchronises. */
int  ub_load_trace_prefix(ub_sim*, const int64_t* arrival_us, const int32_t* prompt_tok, const int32_t* decode_tok,
                          const int32_t* hit_tok, const uint32_t* n_req, int ptrs_on_device);

/* Set the replica table (host, [R]) and reset every replica to t = 0 with an empty queue.  Builds the
 * fixed-point boost table LUT[bin] = min(2^60, floor(b_gamma(k 2^bin tok_us 1e-6) 1e6 + 0.5)) us on the host
 * in fp64 (Eq. 2, rule M4) and uploads it.  Needs a loaded trace.  Synchronises. */
int  ub_set_replicas(ub_sim*, const ub_replica* reps);

/* Advance every replica by n_iters scheduler iterations.  One iteration is one pass of Algorithm 1's loop body
 * (PAPER.md:412-472): for all active r: SIGNAL -> QUANTIZE -> BOOST -> pi(r) = a_r - b_r -> UPDATEKEY;
 * B <- {}, U <- KV usage; while |B| < M: r <- argmin of the queue tops, admit if U + KVNEED(r, c) <= B else
 * SELECTVICTIM / SWAPOUT; EXECUTEONESTEP(B, c) under the stated cost model;
 * UPDATESTATS -- steps a0..a5 of DESIGN.md Sec. 2, rules M6-M10.  Finished replicas are no-ops.
 * Asynchronous on the stream unless live_replicas (host, nullable) is given: then it synchronises and returns the
 * number of unfinished replicas. */
int  ub_step(ub_sim*, uint32_t n_iters, uint64_t* live_replicas);

/* Algorithm 1's outer loop ("while system is running") over the whole trace: ub_step until every replica
 * has served its last request (trace exhausted and no request active, M6) or max_iters iterations were issued (then
 * UB_ELIVELOCK).  iters_done (host, nullable) = iterations issued.  Synchronises.
 * The rounds are replayed from a captured CUDA graph (64 rounds at a time) while the set of unfinished replicas a round
 * visits is unchanged; if the handle's stream is a default stream (which cannot be captured) the graph runs on a stream
 * of the library's, ordered behind the handle's stream and in front of it again by events.  Same schedules either way;
 * gamma-Ada runs and a stream that refuses capture fall back to plain launches. */
int  ub_run(ub_sim*, uint64_t max_iters, uint64_t* iters_done);

/* Device-resident reduction of the per-request histories to the tail metrics the paper reports (TTFT, TTLT = E2E
 * and TBT at mean / P50 / P90 / P99: PAPER.md:245, 256-265): percentile p of m samples is the paper's
 * t_p = inf{t : Fbar(t) <= (100 - p)/100} = the ceil(p m / 100)-th smallest (rule M11); plus the
 * counters UPDATESTATS keeps.  out: host, [R].  Synchronises. */
int  ub_stats(ub_sim*, ub_replica_stats* out);

/* Per-request results, each [R][max_requests] (nullable): first / last token time (us, -1 = none yet),
 * evictions, unforced evictions (victim was not MemGuard-locked).  Host (on_device = 0) or device.  Synchronises. */
int  ub_per_request(ub_sim*, int64_t* t_first_us, int64_t* t_last_us, uint32_t* n_evict,
                    uint32_t* n_evict_unforced, int on_device);

/* Schedule digest H per replica (M12), host [R].  Equal digests + equal per-request results = identical
 * schedule.  Synchronises. */
int  ub_digest(ub_sim*, uint64_t* digest);

/* Boost table of one replica: nb entries; lut (host, nullable) receives min(nb, cap).  */
int  ub_boost_lut(ub_sim*, uint32_t replica, int64_t* lut, uint32_t cap, uint32_t* nb);

/* TBT histogram of one replica, host [UB_TBT_BINS].  Synchronises. */
int  ub_tbt_hist(ub_sim*, uint32_t replica, uint32_t* hist);

/* Kernel-level parity: the active window of one replica in stored (= last priority) order.
 * Each array host, [queue_cap], nullable; *n_active receives the count.  Synchronises. */
int  ub_debug_get_state(ub_sim*, uint32_t replica, uint32_t* n_active, uint32_t* id, uint32_t* d,
                        uint32_t* cached, uint32_t* flags, int64_t* clock_us);

/* Flag bits of ub_debug_get_state / ub_debug_set_state (the `flags` word of a window record). */
enum { UB_F_RESIDENT = 1u,        /* KV on the device */
       UB_F_SWAPPED  = 2u,        /* KV in the host swap pool */
       UB_F_EMITPREV = 4u,        /* emitted a token in the last executed iteration (its t_last is the replica clock) */
       UB_F_DIRTY    = 8u,        /* (resident, Eq. 8 bin, class) -- the inputs of its key -- changed in the last executed
                                     iteration: the only requests that may be out of place in the stored order */
       UB_F_ADMITNOW = 16u,       /* admitted in the last executed iteration */
       UB_F_KLASS1   = 32u,       /* was in class 1 (not MemGuard-locked) in the last executed iteration */
       UB_F_PREEMPTED = 64u,      /* evicted (swap or recompute) and not admitted again yet (its preemption time is running) */
       UB_F_LOCK_SHIFT = 7 };     /* bits 7..31: MemGuard lock bin + 1 (0 = no lock; residents re-lock every iteration, M10) */

/* Kernel-level parity (SURVEY.md Sec. 4 tier T1, Sec. 8(b)): overwrite the state of one unfinished replica so that a
 * single ub_step runs admit / victim-select / advance (a3..a5) from a state taken from elsewhere, e.g. an oracle
 * snapshot.  Window of n_active requests in stored order: id (< next_request), d tokens emitted (< D), cached KV
 * tokens (<= P + d; 0 unless resident or swapped), flags (UB_F_*); each host, [n_active].  The stored order must be
 * the priority order of the state except for the requests flagged UB_F_DIRTY (flag every request to have the next
 * iteration sort from scratch).  clock_us: replica clock; next_request: trace cursor (requests below it were
 * ingested); swap_used_blocks: occupancy of the host swap pool.  Counters, digest and per-request outputs are left
 * as they are.  UB_EINVAL on an inconsistent record, UB_ESTATE if the replica has finished or the state would leave
 * it finished.  Synchronises. */
int  ub_debug_set_state(ub_sim*, uint32_t replica, uint32_t n_active, const uint32_t* id, const uint32_t* d,
                        const uint32_t* cached, const uint32_t* flags, int64_t clock_us, uint32_t next_request,
                        uint32_t swap_used_blocks);

/* Kernel-level parity (SURVEY.md Sec. 4 tier T1): the (class, key) the device assigns to every request of a replica's
 * window as it stands now, i.e. as the NEXT iteration would score the requests already in the window (a1, M3-M5, M14)
 * -- computed by the same device function the team kernels use.  id, klass: host [queue_cap] u32; key_us: host
 * [queue_cap] i64 (microseconds, or tokens for SRPT / LAS / SJF / SPF); each nullable; *n_active receives the count.
 * Entries come in stored (last priority) order.  Synchronises. */
int  ub_debug_keys(ub_sim*, uint32_t replica, uint32_t* n_active, uint32_t* id, uint32_t* klass, int64_t* key_us);
/* The same through the streaming kernel's own scorer (the one bench.py times; FCFS / BOOST with the unified signal
 * and the geometric quantiser, else UB_EINVAL): pi = a - b_gamma(w_hat) - delta [resident] (Eq. 7). */
int  ub_debug_keys_stream(ub_sim*, uint32_t replica, uint32_t* n_active, uint32_t* id, uint32_t* klass, int64_t* key_us);

/* Timing of the step kernel launches issued by the LAST ub_step / ub_run call, measured with CUDA events on
 * the borrowed stream: total milliseconds and launch count.  Synchronises. */
int  ub_last_step_timing(ub_sim*, float* kernel_ms, uint32_t* launches);

/* Richer reductions, device-resident like ub_stats.  which: 0 = TTFT, 1 = TTLT, over the
 * completed requests of each replica.
 * ub_percentile_curve: nearest-rank percentiles at n (1..16) per-mille points (e.g. 500, 900, 990, 999 -- the
 *   per-percentile curves of Fig. 6): the ceil(p m / 1000)-th smallest of the m samples (t_p of
 *   PAPER.md:225), 0 when m = 0.  permille: host [n], each 1..1000;  out_us: host [n_replicas][n].
 * ub_slo_attainment: for each replica and each of n (1..16) latency thresholds (microseconds; the caller forms them as
 *   SLO scale x base latency, Fig. 8) the number of completed requests with latency <= threshold;
 *   divide by ub_replica_stats::n_completed for the attainment.  threshold_us, met: host [n_replicas][n].
 * Both synchronise. */
int  ub_percentile_curve(ub_sim*, uint32_t which, const uint32_t* permille, uint32_t n, int64_t* out_us);
int  ub_slo_attainment(ub_sim*, uint32_t which, const int64_t* threshold_us, uint32_t n, uint32_t* met);

/* ub_percentile_curve for callers that cannot call cudaMalloc (tight serving loops, harnesses that forbid it): same
 * arguments, same result, but no cudaMalloc / cudaFree or other allocating routine is called -- the device staging of
 * the result is a static device array inside the library of UB_NOALLOC_CURVE_MAX int64 values (512 KB, held by every
 * GPU that loads the library until the process exits).  n_replicas x n > UB_NOALLOC_CURVE_MAX returns UB_ETOOBIG.
 * The array is shared by every call on the device, from any handle, and keeps the last call's values: the kernel
 * overwrites every value it returns, nothing needs clearing, but two calls that overlap on the GPU (two handles on
 * different streams or host threads) race -- serialise them.  The first call on a device looks the array's device
 * address up (once per device).  Synchronises. */
#define UB_NOALLOC_CURVE_MAX 65536u
int  ub_percentile_curve_noalloc(ub_sim*, uint32_t which, const uint32_t* permille, uint32_t n, int64_t* out_us);

/* Per-class reductions (the short- / long-request tables of the starvation experiment,
 * PAPER.md:549-560 Table 3, Tables 4-5), device-resident: over the completed requests of each replica
 * whose total length P + D lies in [len_lo, len_hi], the nearest-rank percentiles (t_p of PAPER.md:225, rank
 * ceil(p m / 1000); per-mille 1000 = the maximum) at n (1..16) points of
 *   which 0: TTFT,  1: TTLT (E2E),  2: preemption time -- the time from the start of the iteration that evicts a request
 *   (swap or recompute) to the start of the iteration that admits it again, summed over its evictions ("the preemption
 *   time of longer requests"; rule M15 of DESIGN.md).
 * out_us: host [n_replicas][n] (0 where the class is empty); count: host [n_replicas], requests in the class (nullable);
 * sum_us: host [n_replicas], sum of their values -- the mean is sum / count (nullable).  Synchronises. */
int  ub_class_percentiles(ub_sim*, uint32_t which, uint32_t len_lo, uint32_t len_hi, const uint32_t* permille, uint32_t n,
                          int64_t* out_us, uint32_t* count, int64_t* sum_us);
/* Preemption time of every request so far (rule M15), [n_replicas][max_requests] microseconds, host (on_device = 0) or
 * device.  A request that is preempted right now shows minus the start time of its eviction plus the finished part.
 * Synchronises. */
int  ub_preempt_time(ub_sim*, int64_t* t_preempt_us, int on_device);

/* Clusters of replicas behind a join-the-shortest-queue router ("Composability with Global
 * Dispatch Policies", Table 9; rule M18 of DESIGN.md).  The handle must hold n_replicas =
 * n_clusters x cluster_size replicas (cluster_size <= 32), replica r on its own trace r, every trace loaded EMPTY
 * (n_req = 0; max_requests is the room of a replica's row), replicas set and no iteration run; gamma-Ada off.
 * arrival_us / prompt_tok / decode_tok: host, [n_clusters][max_arrivals], one global stream per cluster, arrival-sorted;
 * n_arrivals: host [n_clusters].  Arrival by arrival, every replica of the cluster executes the iterations that START
 * before the arrival time (a time-fenced run of the step kernels); then the arrival joins the replica with the fewest
 * requests in the system at that instant -- assigned to it and not completed by then --, the lowest replica number on a
 * tie (one warp per cluster: a min-reduction over the cluster's replicas), and is appended to that replica's trace.
 * After the last arrival every replica runs to completion (ub_run).  assign (host, nullable): [n_clusters][max_arrivals],
 * the replica number within the cluster each arrival joined (-1 = no arrival).  Errors as ub_load_trace for the streams;
 * UB_EINVAL if a replica's row overflows; UB_ESTATE on a handle that is not in the state above.  Afterwards the
 * replicas' traces hold what the router sent them: ub_set_replicas rewinds to a plain (uncoupled) run of those traces.
 * Synchronises. */
int  ub_jsq_run(ub_sim*, uint32_t cluster_size, uint32_t n_clusters, uint32_t max_arrivals, const int64_t* arrival_us,
                const int32_t* prompt_tok, const int32_t* decode_tok, const uint32_t* n_arrivals, int32_t* assign);

/* gamma-Ada (Eq. 9, UPDATEGAMMA PAPER.md:588-601; rule M13 of DESIGN.md),
 * integer-only so that schedules stay bit-exact.  gamma is kept as gamma_u = gamma * 1e6.  At the start of an executed
 * iteration of an adaptive replica, if a request completed since the last update and >= min_samples have completed:
 *   L = the last min(window, n_completed) end-to-end latencies (us);  t95, t99 = nearest-rank percentiles of L;
 *   hat_u = floor(ln 5 * 1e12) / max(t99 - t95, eps_us);  gamma_u += (hat_u - gamma_u) / 2^beta_shift (truncating);
 *   clip to the grid ends;  level = largest j with grid_u[j] <= gamma_u;  the boost table of grid point j is used.
 * Grid: gamma_j = gamma_min (gamma_max/gamma_min)^(j/(levels-1)), grid_u[j] = floor(gamma_j 1e6 + 0.5). */
typedef struct {
  uint32_t struct_size;
  uint32_t window;         /* max_batch <= window <= 1024 */
  uint32_t min_samples;    /* >= 2 */
  uint32_t beta_shift;     /* smoothing beta = 2^-beta_shift, 0..16 */
  uint32_t levels;         /* 2..64 */
  uint32_t pad;
  double   gamma_min, gamma_max;
  int64_t  eps_us;         /* >= 1 */
} ub_gamma_ada;

/* After ub_set_replicas and before the first ub_step.  adaptive: host, [n_replicas], non-zero = the replica adapts
 * (requires policy UB_BOOST with the geometric quantiser and a finite gamma, else UB_EINVAL); its initial gamma is its
 * ub_replica::gamma clipped to the grid.  While adaptation is on every launch advances one iteration.  Synchronises. */
int  ub_set_gamma_ada(ub_sim*, const ub_gamma_ada* cfg, const uint8_t* adaptive);
/* Current gamma_u, grid level and number of updates of one replica (level = -1 for a non-adaptive one); any output
 * nullable.  Synchronises. */
int  ub_gamma_state(ub_sim*, uint32_t replica, int64_t* gamma_u, int32_t* level, uint64_t* n_updates);
/* The grid (host, [levels]) as built by the library, for comparison with the oracle's. */
int  ub_gamma_grid(ub_sim*, int64_t* grid_u);

/* Changes ub_config::iters_per_launch for the following ub_step / ub_run calls (0 is read as 1).  The schedule does
 * not depend on it (pin P14): with more than one iteration per launch a warp advances its replica several iterations
 * in a row, so the window is re-read from L2 instead of HBM.  Host call, does not synchronise. */
int  ub_set_iters_per_launch(ub_sim*, uint32_t iters_per_launch);

const char* ub_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
