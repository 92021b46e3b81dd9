/*
 * orc_uniboost.h -- CPU ORACLE for the UniBoost per-iteration scheduling step.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call
 * anything in oracle/.  The CUDA product path (paper_2606_18431_b200/) shares
 * no code, header, table or constant generator with this directory and never
 * calls it.
 *
 * What it is: a plain, slow, single-threaded simulator of one continuous-
 * batching LLM replica at a time under the paper's tail-aware scheduler
 * (arxiv 2606.18431, "Beyond Prediction: Tail-Aware Scheduling for LLM
 * Inference"), following Algorithm 1 and its helpers
 * BOOST / QUANTIZE / SIGNAL, Sec. 3.2 unified priority
 * and hysteresis (Eq. 7), Sec. 3.3 MemGuard (PAPER.md:198-215,
 * Eq. 8), on top of the per-iteration cost model that BASELINE.json states
 * (config 1 and config 3).  Where the paper is silent the readings are the
 * ones listed in DESIGN.md Sec. 3 (model rules M1..M18, readings G1..G28; M13 =
 * gamma-Ada, Eq. 9 / UPDATEGAMMA; M14 = DistBoost,
 * Eq. 3-6; baselines SJF / SPF as static keys).
 * The method is a policy (a heuristic driven by a priority rule), not a
 * faster route to a closed form, so the oracle is the algorithm written out
 * step by step in the paper's order: score every active request, sort,
 * walk the order admitting under the KV capacity, evict from the back,
 * execute one step with the cost model, update the statistics.
 *
 * Parity pins (tests/test_oracle_pins.py, -m "not gpu"):
 *   quantiser closed form + the paper's worked number,
 *   boost table vs 50-digit evaluation of Eq. 2,
 *   gamma -> inf == FCFS and gamma -> 0 == LAS,
 *   boost on remaining size with unbounded strength == SRPT (north_star),
 *   KV occupancy <= capacity, work conservation,
 *   G/G/1 FIFO Lindley recursion, brute force over all slot schedules on
 *   tiny traces, Eq. 6 arg-min subset, MemGuard logarithmic
 *   bound, Lemma A.1 boost bound,
 *   percentile definition vs numpy inverted_cdf, a hand-worked
 *   schedules (tests/golden/hand_traces.{md,json}); Smith's rule brute force
 *   (SJF / SPF); Lindley recursion and the Eq. 3-6 queue structure (DistBoost);
 *   tests/test_gamma_ada_pins.py: Eq. 9 on an exactly exponential tail, the
 *   log-spaced grid, no update == static gamma, the update rule re-derived every
 *   iteration; tests/test_reductions.py: numpy inverted_cdf at per-mille points
 *   and plain counts (percentile curve, SLO attainment);
 *   hand-worked goldens G, G2, H, I, J (PHASE signal, AUTO swap rule, swap-time rounding, one-token prefill tail);
 *   tests/test_class_reductions.py: preemption times (M15) read off the hand-derived schedules, the one-block
 *   closed form (t_last - t_first) - (D-1) c0, class filter + numpy inverted_cdf; tests/test_oracle_pins.py
 *   test_sarathi_*: Lindley recursion, round-robin structure, DistBoost at gamma = inf (M16);
 *   tests/test_prefix_cache.py: the signal max(w, s_pre - h) tracked per iteration, work balance (M17);
 *   tests/test_jsq.py: brute force over all assignments, post-hoc recount of the queue lengths, burst = round robin,
 *   one replica per cluster = plain trace (M18).
 * Parity UNPINNED: the paper's latency tables (Tables 2-10) -- they need real
 * GPUs, model weights and datasets that are not available.
 */
#ifndef ORC_UNIBOOST_H
#define ORC_UNIBOOST_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* policies (M5) */
enum { ORC_FCFS = 0, ORC_SRPT = 1, ORC_BOOST = 2, ORC_LAS = 3, ORC_SJF = 4, ORC_SPF = 5,
       ORC_DISTBOOST = 6,    /* Phase-1 strawman, PAPER.md:150-175 (rule M14) */
       ORC_SARATHI = 7 };    /* decode-prioritised, round-robin decode, FCFS chunked prefill piggy-backing (rule M16) */
/* size signal (M3) */
enum { ORC_SIG_UNIFIED = 0, ORC_SIG_PHASE = 1, ORC_SIG_REMAINING = 2 };
/* quantiser (M3) */
enum { ORC_Q_GEOMETRIC = 0, ORC_Q_EXACT = 1 };
/* preemption (M8) */
enum { ORC_PRE_RECOMPUTE = 0, ORC_PRE_SWAP = 1, ORC_PRE_AUTO = 2 };

typedef struct {
  int64_t n_replicas;     /* R */
  int64_t n_traces;       /* number of distinct traces */
  int64_t max_requests;   /* N: row length of the trace arrays */
  int64_t queue_cap;      /* Q: max simultaneously active requests */
  int64_t kv_blocks;      /* B */
  int64_t block_tokens;   /* blk */
  int64_t max_batch;      /* M */
  int64_t chunk_tokens;   /* c */
  int64_t token_budget;   /* T */
  int64_t c0_us, c_prefill_tok_us, c_decode_seq_us; /* iteration cost model */
  int64_t preempt_mode;
  int64_t swap_ns_per_block;
  int64_t swap_pool_blocks;
  int64_t bin_tokens;     /* MemGuard k */
  int64_t tok_us;         /* service microseconds credited per token in b_gamma's argument (G1) */
} orc_config;

typedef struct {
  int64_t trace_id;
  int64_t policy;
  int64_t guard;          /* MemGuard lock on/off */
  int64_t signal_mode;
  int64_t quant_mode;
  int64_t hysteresis_us;  /* delta_hyst, Eq. 7 */
  double  gamma;          /* 1/s; +inf => boost 0 */
} orc_replica;

typedef struct {
  int64_t iterations;       /* executed (non no-op) iterations */
  int64_t request_steps;    /* sum over iterations of the active count */
  int64_t n_completed;
  int64_t evict_recompute, evict_swap, swapins;
  int64_t tokens_lost;      /* KV tokens dropped by recompute evictions */
  int64_t tokens_emitted;
  int64_t prefill_tokens;   /* executed prefill tokens (incl. recomputation) */
  int64_t decode_seqs;      /* executed decode sequence-steps */
  int64_t t_end_us;         /* replica clock */
  int64_t peak_active;
  int64_t done;             /* 1 when trace exhausted and nothing active */
  int64_t swap_used;        /* blocks currently in the host swap pool */
  int64_t ttft_us[3], ttlt_us[3], tbt_us[3];     /* P50, P90, P99 (nearest rank, M11) */
  int64_t sum_ttft_us, sum_ttlt_us;              /* over completed requests */
  int64_t sum_tbt_num_us, sum_tbt_den;           /* sum(t_last-t_first), sum(D-1) */
  double  ttft_s[3], ttlt_s[3], tbt_s[3];        /* the same in fp64 seconds */
  double  mean_ttft_s, mean_ttlt_s, mean_tbt_s, tokens_per_s;
} orc_stats;

/* One entry of the per-step record (in priority order), for kernel-level checks. */
typedef struct {
  int64_t id, klass, key, bin;
  int64_t resident_before;  /* 0/1 */
  int64_t want;             /* tokens admitted this iteration, 0 = not admitted */
  int64_t evict;            /* 0 none, 1 recompute, 2 swap */
  int64_t cached_after, d_after, resident_after;
} orc_step_entry;

typedef struct {
  int64_t executed;         /* 0 if the step was a no-op (replica done) */
  int64_t n_active;         /* after ingestion */
  int64_t t_start_us, cost_us, t_end_us;
  int64_t claimed_blocks;   /* C after the admission walk */
  int64_t prefill_tokens, decode_seqs, swap_blocks;
  int64_t kv_resident_after;/* sum of ceil(cached/blk) over residents after the step */
} orc_step_info;

typedef struct orc_sim orc_sim;

int  orc_create(const orc_config* cfg, orc_sim** out);
void orc_destroy(orc_sim*);
/* arrays are [n_traces][max_requests] row-major, arrival-sorted; n_req[n_traces] */
int  orc_load_trace(orc_sim*, const int64_t* arrival_us, const int32_t* prompt_tok,
                    const int32_t* decode_tok, const uint32_t* n_req);
/* Rule M17 (prefix / radix caching): as orc_load_trace plus hit[n_traces][max_requests] cached prompt
 * tokens per request, 0 <= h < P: the request needs s_pre - h tokens of prefill and is signalled as w~ = max(w, s_pre - h). */
int  orc_load_trace_prefix(orc_sim*, const int64_t* arrival_us, const int32_t* prompt_tok, const int32_t* decode_tok,
                           const int32_t* hit_tok, const uint32_t* n_req);
int  orc_set_replicas(orc_sim*, const orc_replica* reps);
int  orc_step(orc_sim*, int64_t n_iters);                 /* every replica advances n_iters iterations */
int  orc_step_replica(orc_sim*, int64_t replica, orc_step_info* info,
                      orc_step_entry* entries /* [queue_cap] or NULL */);
int  orc_run(orc_sim*, int64_t max_iters, int64_t* iters_done);
int  orc_run_replica(orc_sim*, int64_t replica, int64_t max_iters, int64_t* iters_done);
int  orc_stats_get(orc_sim*, orc_stats* out /* [R] */);
int  orc_per_request(orc_sim*, int64_t* t_first_us, int64_t* t_last_us,
                     uint32_t* n_evict, uint32_t* n_evict_unforced /* each [R][N], nullable */);
int  orc_digest(orc_sim*, uint64_t* digest /* [R] */);
/* Richer reductions over the completed requests of each replica; which: 0 TTFT, 1 TTLT.
 * Percentile curve (Fig. 6): the ceil(p m / 1000)-th smallest of the m samples (t_p of PAPER.md:225).
 * SLO attainment (Fig. 8): number of samples <= threshold, per replica and threshold. */
int  orc_percentile_curve(orc_sim*, int64_t which, const int64_t* permille /* [n] */, int64_t n, int64_t* out_us /* [R][n] */);
int  orc_slo_attainment(orc_sim*, int64_t which, const int64_t* threshold_us /* [R][n] */, int64_t n, int64_t* met /* [R][n] */);
/* Rule M15 ("the preemption time of longer requests", Table 5): a request is
 * preempted from the start of the iteration that evicts it (swap or recompute) to the start of the iteration that
 * admits it again; its preemption time is the sum over its evictions.  out: [R][N] microseconds. */
int  orc_preempt_time(orc_sim*, int64_t* out);
/* Per-class reductions (Tables 3-5): over the completed requests of a replica whose total
 * length P + D lies in [len_lo, len_hi]: nearest-rank percentiles at n per-mille points of TTFT (which 0), TTLT (1) or
 * preemption time (2) -> out [R][n]; their number -> count [R] (nullable); their sum -> sum [R] (nullable). */
int  orc_class_percentiles(orc_sim*, int64_t which, int64_t len_lo, int64_t len_hi, const int64_t* permille, int64_t n,
                           int64_t* out, int64_t* count, int64_t* sum);
/* Rule M18: clusters of K replicas behind a join-the-shortest-queue router (Table 9).
 * The simulator must hold n_replicas = C K replicas, replica r on its own trace r, all traces empty, no iteration run.
 * arrival / prompt / decode: [C][NA] global streams (arrival-sorted per cluster), n_arr[C] their lengths.  Every arrival
 * goes to the replica of its cluster with the fewest requests in the system at its arrival time (lowest number on a
 * tie); then every replica runs to completion.  assign (nullable): [C][NA] replica number within the cluster. */
int  orc_jsq_run(orc_sim*, int64_t cluster_size, const int64_t* arrival_us, const int32_t* prompt_tok,
                 const int32_t* decode_tok, const uint32_t* n_arr, int64_t max_arrivals, int32_t* assign);
int  orc_boost_lut(orc_sim*, int64_t replica, int64_t* lut /* [cap] */, int64_t cap, int64_t* nb);
int  orc_tbt_hist(orc_sim*, int64_t replica, uint32_t* hist /* [4352] */);
/* stand-alone helpers exposed so the pins can hit them directly */
/* gamma-Ada (rule M13 of DESIGN.md; Eq. 9 and UPDATEGAMMA), integer-only:
 *   gamma is kept as gamma_u = gamma * 1e6 (1/s in micro units).  At the start of an executed iteration of an
 *   adaptive replica, if a request completed since the last update and at least min_samples have completed:
 *     L     = the last min(window, n_completed) E2E latencies (TTLT, us)
 *     t95, t99 = nearest-rank percentiles of L (t_p of PAPER.md:225)
 *     hat_u = floor(ln(5) * 1e12) / max(t99 - t95, eps_us)          (Eq. 9: -(ln 0.01 - ln 0.05)/(t99 - t95))
 *     gamma_u += (hat_u - gamma_u) / 2^beta_shift  (C division, truncating);  clip to [gamma_min_u, gamma_max_u]
 *     level = largest j with grid_u[j] <= gamma_u;  the boost table in use is the one of grid point j,
 *   grid: gamma_j = gamma_min * (gamma_max/gamma_min)^(j/(levels-1)), grid_u[j] = floor(gamma_j*1e6 + 0.5). */
typedef struct {
  int64_t window;        /* W: max_batch <= W <= 1024 */
  int64_t min_samples;   /* >= 2 */
  int64_t beta_shift;    /* beta = 2^-beta_shift, 0..16 */
  int64_t levels;        /* G: 2..64 */
  double  gamma_min, gamma_max;
  int64_t eps_us;        /* >= 1 */
} orc_gamma_ada;
/* after orc_set_replicas; adaptive[r] != 0 requires policy BOOST with the geometric quantiser */
int  orc_set_gamma_ada(orc_sim*, const orc_gamma_ada* cfg, const uint8_t* adaptive /* [R] */);
int  orc_gamma_state(orc_sim*, int64_t replica, int64_t* gamma_u, int64_t* level, int64_t* n_updates);
int  orc_gamma_grid(orc_sim*, int64_t* grid_u /* [levels] */);
int64_t orc_gamma_hat_u(int64_t t95_us, int64_t t99_us, int64_t eps_us);     /* Eq. 9 in fixed point */
int64_t orc_quant_bin(int64_t sig, int64_t k);                       /* Eq. 8 exponent */
int64_t orc_boost_us(double gamma, int64_t w_tokens, int64_t tok_us); /* Eq. 2 in fixed point */
int64_t orc_percentile_nearest_rank(const int64_t* sorted, int64_t m, int64_t p);
int64_t orc_tbt_bin(int64_t gap_us);
int64_t orc_tbt_edge(int64_t idx);
const char* orc_strerror(int);

#define ORC_OK 0
#define ORC_EINVAL (-1)
#define ORC_ENOMEM (-2)
#define ORC_ESTATE (-4)
#define ORC_EUNSORTED (-5)
#define ORC_EINFEASIBLE (-6)
#define ORC_ELIVELOCK (-7)

#ifdef __cplusplus
}
#endif
#endif
