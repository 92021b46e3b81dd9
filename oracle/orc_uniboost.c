/*
 * orc_uniboost.c -- CPU ORACLE (test infrastructure; see orc_uniboost.h).
 *
 * Plain single-threaded C, array-of-structs, one replica at a time, qsort for
 * the order, a literal sequential admission walk, back-to-front eviction.
 * No blocking, fusion or reordering beyond what Algorithm 1
 * and DESIGN.md Sec. 3 (M1..M12) state.  Shares nothing with the CUDA path.
 */
#include "orc_uniboost.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define TBT_BINS 4352
#define LUT_CAP_GEOM 64
#define BOOST_MAX ((int64_t)1 << 60)

typedef struct {
  int32_t d;          /* output tokens emitted so far (M1) */
  int32_t cached;     /* tokens whose KV is held (device if resident, host if swapped) */
  int32_t resident;
  int32_t swapped;
  int64_t lockbin;    /* MemGuard: bin at which the request was last (re)locked */
  int64_t t_first, t_last;
  uint32_t n_evict, n_evict_unforced;
  int32_t completed;
  int64_t preempt_since;  /* M15: start time of the iteration that evicted it, -1 while it is not preempted */
  int64_t t_preempt;      /* M15: total time spent preempted so far */
} orc_req;

typedef struct {
  orc_replica par;
  orc_req* req;        /* [n_req of its trace] */
  int32_t* active;     /* ids, ascending (= arrival order), length n_active */
  int64_t n_active;
  int64_t next;        /* trace cursor */
  int64_t t;           /* clock, us */
  int64_t swap_used;
  uint64_t H;          /* schedule digest (M12) */
  int64_t* lut; int64_t nb;
  uint32_t* hist;      /* pooled TBT gaps, log-linear (M11) */
  int64_t iterations, request_steps, n_completed, evict_recompute, evict_swap, swapins;
  int64_t tokens_lost, tokens_emitted, prefill_tokens, decode_seqs, peak_active;
  int64_t sum_ttft, sum_ttlt, sum_tbt_num, sum_tbt_den;
  /* gamma-Ada (M13) */
  int32_t ada;
  int64_t* ring;       /* [window] E2E latencies, slot = completion number mod window */
  int64_t* lut_levels; /* [levels][LUT_CAP_GEOM] */
  int64_t gamma_u, level, n_updates, seen;
} orc_rep;

struct orc_sim {
  orc_config cfg;
  int64_t* arrival; int32_t* prompt; int32_t* decode; uint32_t* n_req;
  int32_t* hit;        /* M17: prefix-cache hit tokens h_i per request (all 0 unless loaded with orc_load_trace_prefix) */
  int have_trace, have_reps;
  orc_rep* rep;
  orc_gamma_ada ada; int have_ada;
  int64_t* grid_u;     /* [levels] */
};

/* ---------- small closed-form helpers ---------- */

/* Eq. 8 / QUANTIZE: w_hat = k * 2^bin with
 * bin = floor(log2(max(sig,k)/k)); floor(log2(x)) == floor(log2(floor(x))) for x>=1. */
int64_t orc_quant_bin(int64_t sig, int64_t k) {
  int64_t q = (sig > k ? sig : k) / k;
  int64_t bin = 0;
  while (q > 1) { q >>= 1; bin++; }
  return bin;
}

/* Eq. 2 / BOOST in fixed point (M4):
 * x = w*tok_us*1e-6 s; b = (1/gamma) log(1/(1-exp(-gamma x))) = -log(-expm1(-gamma x))/gamma;
 * value = min(2^60, floor(b*1e6 + 0.5)) us.  x == 0 -> 2^60.  gamma == +inf -> 0. */
static int64_t boost_fixed(double gamma, double w_tokens, int64_t tok_us) {
  if (isinf(gamma) && gamma > 0) return 0;
  double x = w_tokens * (double)tok_us * 1e-6;
  if (!(x > 0.0)) return BOOST_MAX;
  double b = -log(-expm1(-gamma * x)) / gamma;
  double v = floor(b * 1e6 + 0.5);
  if (!(v > 0.0)) return 0;
  if (v >= (double)BOOST_MAX) return BOOST_MAX;
  return (int64_t)v;
}
int64_t orc_boost_us(double gamma, int64_t w_tokens, int64_t tok_us) {
  return boost_fixed(gamma, (double)w_tokens, tok_us);
}

/* t_p = inf{t : Fbar(t) <= (100-p)/100} == the ceil(p*m/100)-th smallest. */
int64_t orc_percentile_nearest_rank(const int64_t* sorted, int64_t m, int64_t p) {
  if (m <= 0) return 0;
  int64_t rank = (p * m + 99) / 100;
  if (rank < 1) rank = 1;
  if (rank > m) rank = m;
  return sorted[rank - 1];
}

/* M11: log-linear histogram with 7 sub-bits. */
int64_t orc_tbt_bin(int64_t g) {
  if (g < 0) g = 0;
  if (g >= ((int64_t)1 << 40)) g = ((int64_t)1 << 40) - 1;
  int64_t lg = 0; { int64_t q = g; while (q > 1) { q >>= 1; lg++; } }
  int64_t shift = lg - 7; if (shift < 0) shift = 0;
  return 128 * shift + (g >> shift);
}
int64_t orc_tbt_edge(int64_t idx) {
  int64_t s = idx / 128 - 1; if (s < 0) s = 0;
  return (idx - 128 * s) << s;
}

/* M12 (test plumbing, not part of the paper's method).  Event hash: a 32-bit mix of
 * (id, type) times the odd number 2*payload+1.  Inside an iteration the low and the high 32-bit halves of the
 * event hashes are summed separately, each modulo 2^32 (order-free), and the iteration is folded into H by one
 * multiply-xorshift round together with t_end. */
enum { EV_ADMIT = 1, EV_EVICT_RECOMPUTE = 2, EV_EVICT_SWAP = 3, EV_SWAPIN = 4, EV_EMIT_FIRST = 5, EV_COMPLETE = 6 };
typedef struct { uint32_t lo, hi; } ev_acc;
static void ev_add(ev_acc* e, uint32_t type, uint32_t id, uint32_t payload) {
  uint32_t m = ((id + 1u) * 0x9E3779B1u) ^ (type * 0x85EBCA6Bu);
  uint64_t h = (uint64_t)m * (uint64_t)(uint32_t)(2u * payload + 1u);
  e->lo += (uint32_t)h;
  e->hi += (uint32_t)(h >> 32);
}
static uint64_t digest_fold(uint64_t H, ev_acc e, int64_t t_end) {
  uint64_t x = (H ^ (((uint64_t)e.hi << 32) | (uint64_t)e.lo)) + (uint64_t)t_end * 0x9E3779B97F4A7C15ull;
  x ^= x >> 29;
  x *= 0xBF58476D1CE4E5B9ull;
  x ^= x >> 32;
  return x;
}

const char* orc_strerror(int e) {
  switch (e) {
    case ORC_OK: return "ok";
    case ORC_EINVAL: return "invalid argument";
    case ORC_ENOMEM: return "out of memory";
    case ORC_ESTATE: return "wrong call order";
    case ORC_EUNSORTED: return "arrivals not non-decreasing";
    case ORC_EINFEASIBLE: return "request does not fit the KV capacity or has P<1 or D<1";
    case ORC_ELIVELOCK: return "max_iters reached before all replicas finished";
    default: return "unknown";
  }
}

/* ---------- life cycle ---------- */

int orc_create(const orc_config* c, orc_sim** out) {
  if (!c || !out) return ORC_EINVAL;
  if (c->n_replicas < 1 || c->n_traces < 1 || c->max_requests < 1 || c->queue_cap < 1 ||
      c->kv_blocks < 1 || c->block_tokens < 1 || c->max_batch < 1 || c->chunk_tokens < 1 ||
      c->token_budget < 1 || c->c0_us < 0 || c->c_prefill_tok_us < 0 || c->c_decode_seq_us < 0 ||
      c->preempt_mode < 0 || c->preempt_mode > 2 || c->swap_ns_per_block < 0 || c->swap_pool_blocks < 0 ||
      c->bin_tokens < 1 || c->tok_us < 1)
    return ORC_EINVAL;
  orc_sim* s = (orc_sim*)calloc(1, sizeof(orc_sim));
  if (!s) return ORC_ENOMEM;
  s->cfg = *c;
  *out = s;
  return ORC_OK;
}

static void free_reps(orc_sim* s) {
  if (!s->rep) return;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    free(s->rep[r].req); free(s->rep[r].active); free(s->rep[r].hist);
    if (!s->rep[r].ada) free(s->rep[r].lut);          /* (an adaptive replica's lut points into lut_levels) */
    free(s->rep[r].ring); free(s->rep[r].lut_levels);
  }
  free(s->rep); s->rep = NULL; s->have_reps = 0;
  free(s->grid_u); s->grid_u = NULL; s->have_ada = 0;
}

void orc_destroy(orc_sim* s) {
  if (!s) return;
  free_reps(s);
  free(s->arrival); free(s->prompt); free(s->decode); free(s->n_req); free(s->hit);
  free(s);
}

int orc_load_trace(orc_sim* s, const int64_t* a, const int32_t* p, const int32_t* d, const uint32_t* n_req) {
  if (!s || !a || !p || !d || !n_req) return ORC_EINVAL;
  const orc_config* c = &s->cfg;
  int64_t NT = c->n_traces, N = c->max_requests;
  for (int64_t t = 0; t < NT; t++) {
    if ((int64_t)n_req[t] > N) return ORC_EINVAL;
    for (int64_t i = 0; i < (int64_t)n_req[t]; i++) {
      int64_t ai = a[t * N + i];
      if (ai < 0 || ai > ((int64_t)1 << 61)) return ORC_EINVAL;
      if (i > 0 && ai < a[t * N + i - 1]) return ORC_EUNSORTED;
      int64_t P = p[t * N + i], D = d[t * N + i];
      if (P < 1 || D < 1) return ORC_EINFEASIBLE;
      if ((P + D + c->block_tokens - 1) / c->block_tokens > c->kv_blocks) return ORC_EINFEASIBLE;
    }
  }
  free_reps(s);
  free(s->arrival); free(s->prompt); free(s->decode); free(s->n_req); free(s->hit);
  s->hit = (int32_t*)calloc((size_t)(NT * N > 0 ? NT * N : 1), sizeof(int32_t));
  s->arrival = (int64_t*)malloc(sizeof(int64_t) * NT * N);
  s->prompt = (int32_t*)malloc(sizeof(int32_t) * NT * N);
  s->decode = (int32_t*)malloc(sizeof(int32_t) * NT * N);
  s->n_req = (uint32_t*)malloc(sizeof(uint32_t) * NT);
  if (!s->arrival || !s->prompt || !s->decode || !s->n_req || !s->hit) return ORC_ENOMEM;
  memcpy(s->arrival, a, sizeof(int64_t) * NT * N);
  memcpy(s->prompt, p, sizeof(int32_t) * NT * N);
  memcpy(s->decode, d, sizeof(int32_t) * NT * N);
  memcpy(s->n_req, n_req, sizeof(uint32_t) * NT);
  s->have_trace = 1;
  return ORC_OK;
}

/* M17 prefix / radix caching (A.5): a request with h_i cached prompt tokens needs only s_pre - h_i
 * tokens of prefill ("caching primarily reduces effective prefill work") and its size signal becomes
 * w~ = max(w, s_pre - h_i), w = the tokens processed so far.  hit: [n_traces][max_requests], 0 <= h < P. */
int orc_load_trace_prefix(orc_sim* s, const int64_t* a, const int32_t* p, const int32_t* d, const int32_t* hit,
                          const uint32_t* n_req) {
  if (!hit) return ORC_EINVAL;
  int rc = orc_load_trace(s, a, p, d, n_req);
  if (rc) return rc;
  const int64_t NT = s->cfg.n_traces, N = s->cfg.max_requests;
  for (int64_t t = 0; t < NT; t++)
    for (int64_t i = 0; i < (int64_t)n_req[t]; i++)
      if (hit[t * N + i] < 0 || hit[t * N + i] >= p[t * N + i]) { s->have_trace = 0; return ORC_EINVAL; }
  memcpy(s->hit, hit, sizeof(int32_t) * (size_t)(NT * N));
  return ORC_OK;
}

int orc_set_replicas(orc_sim* s, const orc_replica* reps) {
  if (!s || !reps) return ORC_EINVAL;
  if (!s->have_trace) return ORC_ESTATE;
  const orc_config* c = &s->cfg;
  int64_t R = c->n_replicas, N = c->max_requests;
  for (int64_t r = 0; r < R; r++) {
    const orc_replica* q = &reps[r];
    if (q->trace_id < 0 || q->trace_id >= c->n_traces) return ORC_EINVAL;
    if (q->policy < 0 || q->policy > 7 || q->signal_mode < 0 || q->signal_mode > 2 ||
        q->quant_mode < 0 || q->quant_mode > 1 || q->hysteresis_us < 0 ||
        q->hysteresis_us > ((int64_t)1 << 60))
      return ORC_EINVAL;
    if ((q->policy == ORC_BOOST || q->policy == ORC_DISTBOOST) && !(q->gamma > 0.0)) return ORC_EINVAL; /* also rejects NaN */
  }
  free_reps(s);
  s->rep = (orc_rep*)calloc((size_t)R, sizeof(orc_rep));
  if (!s->rep) return ORC_ENOMEM;
  for (int64_t r = 0; r < R; r++) {
    orc_rep* x = &s->rep[r];
    x->par = reps[r];
    int64_t tr = x->par.trace_id, n = s->n_req[tr];
    x->req = (orc_req*)calloc((size_t)(N > 0 ? N : 1), sizeof(orc_req));   /* (row length: a JSQ router appends, M18) */
    x->active = (int32_t*)calloc((size_t)c->queue_cap, sizeof(int32_t));
    x->hist = (uint32_t*)calloc(TBT_BINS, sizeof(uint32_t));
    if (!x->req || !x->active || !x->hist) return ORC_ENOMEM;
    for (int64_t i = 0; i < N; i++) { x->req[i].t_first = -1; x->req[i].t_last = -1; x->req[i].lockbin = -1; x->req[i].preempt_since = -1; }
    /* boost table (M4): one entry per bin; EXACT quantiser => one entry per signal value */
    int64_t nb = LUT_CAP_GEOM;
    if (x->par.quant_mode == ORC_Q_EXACT) {
      int64_t mx = 0;
      for (int64_t i = 0; i < n; i++) {
        int64_t v = (int64_t)s->prompt[tr * N + i] + s->decode[tr * N + i];
        if (v > mx) mx = v;
      }
      nb = mx + 1;
    }
    x->nb = nb;
    x->lut = (int64_t*)calloc((size_t)nb, sizeof(int64_t));
    if (!x->lut) return ORC_ENOMEM;
    for (int64_t b = 0; b < nb; b++) {
      if (x->par.policy != ORC_BOOST && x->par.policy != ORC_DISTBOOST) { x->lut[b] = 0; continue; }
      /* w_hat = k * 2^b (Eq. 8), in fp64 so that absurd bins cannot overflow */
      double what = (x->par.quant_mode == ORC_Q_EXACT) ? (double)b : ldexp((double)c->bin_tokens, (int)b);
      x->lut[b] = boost_fixed(x->par.gamma, what, c->tok_us);
    }
  }
  s->have_reps = 1;
  return ORC_OK;
}


/* ---------- gamma-Ada (M13) ---------- */

#define LN5_E12 1609437912434LL   /* floor(ln(5) * 1e12) */

/* Eq. 9 with F(t95) = 0.05, F(t99) = 0.01: gamma_hat = ln 5 / (t99 - t95), times in seconds;
 * in micro units with times in microseconds: hat_u = ln5 * 1e12 / max(t99 - t95, eps). */
int64_t orc_gamma_hat_u(int64_t t95_us, int64_t t99_us, int64_t eps_us) {
  int64_t delta = t99_us - t95_us;
  if (delta < eps_us) delta = eps_us;
  return LN5_E12 / delta;
}

static int i64_cmp_(const void* a, const void* b) {
  int64_t x = *(const int64_t*)a, y = *(const int64_t*)b;
  return (x > y) - (x < y);
}

static int64_t level_of(const orc_sim* s, int64_t gamma_u) {
  int64_t j = 0;
  while (j + 1 < s->ada.levels && s->grid_u[j + 1] <= gamma_u) j++;
  return j;
}

/* UPDATEGAMMA, step by step */
static int update_gamma(orc_sim* s, orc_rep* x) {
  const orc_gamma_ada* g = &s->ada;
  if (x->n_completed == x->seen || x->n_completed < g->min_samples) return 0;
  int64_t m = x->n_completed < g->window ? x->n_completed : g->window;
  int64_t* L = (int64_t*)malloc(sizeof(int64_t) * (size_t)m);
  if (!L) return ORC_ENOMEM;
  memcpy(L, x->ring, sizeof(int64_t) * (size_t)m);      /* slots 0..m-1 hold the last m samples */
  qsort(L, (size_t)m, sizeof(int64_t), i64_cmp_);
  int64_t x95 = orc_percentile_nearest_rank(L, m, 95), x99 = orc_percentile_nearest_rank(L, m, 99);
  free(L);
  int64_t hat = orc_gamma_hat_u(x95, x99, g->eps_us);
  x->gamma_u += (hat - x->gamma_u) / ((int64_t)1 << g->beta_shift);          /* (1-beta) gamma + beta gamma_hat */
  if (x->gamma_u < s->grid_u[0]) x->gamma_u = s->grid_u[0];                   /* clip */
  if (x->gamma_u > s->grid_u[g->levels - 1]) x->gamma_u = s->grid_u[g->levels - 1];
  x->level = level_of(s, x->gamma_u);
  x->lut = x->lut_levels + x->level * LUT_CAP_GEOM;
  x->seen = x->n_completed;
  x->n_updates++;
  return 0;
}

int orc_set_gamma_ada(orc_sim* s, const orc_gamma_ada* g, const uint8_t* adaptive) {
  if (!s || !g || !adaptive) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  if (g->window < s->cfg.max_batch || g->window > 1024 || g->min_samples < 2 || g->beta_shift < 0 ||
      g->beta_shift > 16 || g->levels < 2 || g->levels > 64 || !(g->gamma_min > 0.0) ||
      !(g->gamma_max > g->gamma_min) || g->gamma_max > 1e6 || g->eps_us < 1)
    return ORC_EINVAL;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    const orc_rep* x = &s->rep[r];
    if (adaptive[r] && (x->par.policy != ORC_BOOST || x->par.quant_mode != ORC_Q_GEOMETRIC || isinf(x->par.gamma)))
      return ORC_EINVAL;
    if (x->iterations != 0 || x->ada) return ORC_ESTATE;
  }
  s->ada = *g; s->have_ada = 1;
  free(s->grid_u);
  s->grid_u = (int64_t*)calloc((size_t)g->levels, sizeof(int64_t));
  if (!s->grid_u) return ORC_ENOMEM;
  for (int64_t j = 0; j < g->levels; j++) {
    double gj = g->gamma_min * pow(g->gamma_max / g->gamma_min, (double)j / (double)(g->levels - 1));
    s->grid_u[j] = (int64_t)floor(gj * 1e6 + 0.5);
  }
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    orc_rep* x = &s->rep[r];
    if (!adaptive[r]) continue;
    x->ring = (int64_t*)calloc((size_t)g->window, sizeof(int64_t));
    x->lut_levels = (int64_t*)calloc((size_t)(g->levels * LUT_CAP_GEOM), sizeof(int64_t));
    if (!x->ring || !x->lut_levels) return ORC_ENOMEM;
    for (int64_t j = 0; j < g->levels; j++) {
      double gj = g->gamma_min * pow(g->gamma_max / g->gamma_min, (double)j / (double)(g->levels - 1));
      for (int64_t b = 0; b < LUT_CAP_GEOM; b++)
        x->lut_levels[j * LUT_CAP_GEOM + b] = boost_fixed(gj, ldexp((double)s->cfg.bin_tokens, (int)b), s->cfg.tok_us);
    }
    x->gamma_u = (int64_t)floor(x->par.gamma * 1e6 + 0.5);
    if (x->gamma_u < s->grid_u[0]) x->gamma_u = s->grid_u[0];
    if (x->gamma_u > s->grid_u[g->levels - 1]) x->gamma_u = s->grid_u[g->levels - 1];
    x->level = level_of(s, x->gamma_u);
    free(x->lut);
    x->lut = x->lut_levels + x->level * LUT_CAP_GEOM; x->nb = LUT_CAP_GEOM;
    x->ada = 1;
  }
  return ORC_OK;
}

int orc_gamma_state(orc_sim* s, int64_t r, int64_t* gamma_u, int64_t* level, int64_t* n_updates) {
  if (!s || !s->have_reps || r < 0 || r >= s->cfg.n_replicas) return ORC_EINVAL;
  const orc_rep* x = &s->rep[r];
  if (gamma_u) *gamma_u = x->ada ? x->gamma_u : 0;
  if (level) *level = x->ada ? x->level : -1;
  if (n_updates) *n_updates = x->n_updates;
  return ORC_OK;
}

int orc_gamma_grid(orc_sim* s, int64_t* grid_u) {
  if (!s || !grid_u || !s->have_ada) return ORC_EINVAL;
  memcpy(grid_u, s->grid_u, sizeof(int64_t) * (size_t)s->ada.levels);
  return ORC_OK;
}

/* ---------- one scheduler iteration of one replica ---------- */

typedef struct { int64_t klass, key, id, bin; int32_t resident_before; int64_t want; int32_t evict; } ent_t;

static int ent_cmp(const void* pa, const void* pb) {
  const ent_t* a = (const ent_t*)pa; const ent_t* b = (const ent_t*)pb;
  if (a->klass != b->klass) return a->klass < b->klass ? -1 : 1;
  if (a->key != b->key) return a->key < b->key ? -1 : 1;
  if (a->id != b->id) return a->id < b->id ? -1 : 1;
  return 0;
}

static int64_t ceil_div(int64_t x, int64_t y) { return (x + y - 1) / y; }

static int step_one(orc_sim* s, orc_rep* x, orc_step_info* info, orc_step_entry* out) {
  const orc_config* c = &s->cfg;
  const int64_t N = c->max_requests, tr = x->par.trace_id, nreq = s->n_req[tr];
  const int64_t* A = s->arrival + tr * N;
  const int32_t* Pp = s->prompt + tr * N;
  const int32_t* Hh = s->hit + tr * N;     /* M17: prefix-cache hits; P below is the effective prefill work s_pre - h */
  const int32_t* Dd = s->decode + tr * N;
  const int64_t blk = c->block_tokens, B = c->kv_blocks;
  if (info) memset(info, 0, sizeof(*info));

  /* M6 step start: idle jump, then ingest every arrival with a <= t */
  if (x->n_active == 0) {
    if (x->next >= nreq) return 0;            /* done: no-op */
    if (A[x->next] > x->t) x->t = A[x->next];
  }
  /* Algorithm 1 "gamma <- UPDATEGAMMA(S)" at the top of the loop */
  if (x->ada) { int rc = update_gamma(s, x); if (rc) return rc; }
  while (x->next < nreq && A[x->next] <= x->t && x->n_active < c->queue_cap)
    x->active[x->n_active++] = (int32_t)x->next++;
  const int64_t n = x->n_active;
  if (n > x->peak_active) x->peak_active = n;

  ent_t* e = (ent_t*)malloc(sizeof(ent_t) * (size_t)n);
  if (!e) return ORC_ENOMEM;

  /* Algorithm 1 lines 5-10: rescore every active request */
  for (int64_t j = 0; j < n; j++) {
    int64_t id = x->active[j];
    orc_req* q = &x->req[id];
    int64_t P = Pp[id] - Hh[id], D = Dd[id];
    /* M3 SIGNAL: UNIFIED w~ = max(w, s_pre) with w = tokens processed => P + d; with prefix-cache hits
       w~ = max(w, s_pre - h) => (s_pre - h) + d, P being the effective prefill work here (M17);
       PHASE: prompt tokens in prefill else attained decode tokens */
    int64_t sig;
    if (x->par.signal_mode == ORC_SIG_UNIFIED) sig = P + q->d;
    else if (x->par.signal_mode == ORC_SIG_PHASE) sig = (q->d == 0) ? P : q->d;
    else sig = D - q->d;
    /* M3 QUANTIZE (Eq. 8) */
    int64_t bin = (x->par.quant_mode == ORC_Q_GEOMETRIC) ? orc_quant_bin(sig, c->bin_tokens) : sig;
    /* M5 key: pi(r) = a_r - b_r; FCFS a; SRPT remaining tokens; LAS attained signal */
    int64_t key;
    if (x->par.policy == ORC_FCFS) key = A[id];
    else if (x->par.policy == ORC_SRPT) key = D - q->d;
    else if (x->par.policy == ORC_LAS) key = sig;
    /* baselines of PAPER.md:51, 239 as static keys: shortest job (output length, perfect) / shortest prompt first */
    else if (x->par.policy == ORC_SJF) key = D;
    else if (x->par.policy == ORC_SPF) key = P;
    else if (x->par.policy == ORC_DISTBOOST) {
      /* DistBoost (M14): decode queue Q_d = {prefill done} keyed by the time of entering it, Eq. 4; prefill queue
         keyed by a - b_gamma(s_pre), Eq. 3 */
      if (q->d >= 1) key = q->t_first;
      else {
        int64_t pb = (x->par.quant_mode == ORC_Q_GEOMETRIC) ? orc_quant_bin(P, c->bin_tokens) : P;
        key = A[id] - x->lut[pb < x->nb ? pb : x->nb - 1];
      }
    }
    else if (x->par.policy == ORC_SARATHI) {
      /* Sarathi (M16; "chunk-prefill, decode-prioritized continuous batching, with round-robin ordering in the decode
         and piggy-back prefills"): the decode queue goes round robin -- whoever emitted longest ago
         first --, the prefill queue is first come first served */
      key = (q->d >= 1) ? q->t_last : A[id];
    }
    else key = A[id] - x->lut[bin < x->nb ? bin : x->nb - 1];
    /* Eq. 7 hysteresis as a bias on requests that hold the device */
    if (q->resident && (x->par.policy == ORC_FCFS || x->par.policy == ORC_BOOST)) key -= x->par.hysteresis_us;
    /* MemGuard minimum-run lock: dispatched and still in the bin it was locked at */
    int64_t klass = (x->par.guard && q->resident && bin == q->lockbin) ? 0 : 1;
    /* DistBoost: the decode batch is selected first, prefill piggybacks on what is left (Eq. 5-6) */
    if (x->par.policy == ORC_DISTBOOST || x->par.policy == ORC_SARATHI) klass = (q->d >= 1) ? 0 : 1;
    e[j].klass = klass; e[j].key = key; e[j].id = id; e[j].bin = bin;
    e[j].resident_before = q->resident; e[j].want = 0; e[j].evict = 0;
  }

  /* unified ordering across phases: ascending (class, key, id) */
  qsort(e, (size_t)n, sizeof(ent_t), ent_cmp);

  /* M7 admission walk: B <- {}, U <- claims; while |B| < M ... */
  int64_t C = 0, tok = 0, cnt = 0, newblocked = 0;
  int64_t prefill_tokens = 0, decode_seqs = 0, swap_blocks = 0;
  ev_acc ev = {0u, 0u};
  for (int64_t j = 0; j < n; j++) {
    if (cnt == c->max_batch || tok == c->token_budget) break;
    orc_req* q = &x->req[e[j].id];
    int64_t P = Pp[e[j].id] - Hh[e[j].id];
    if (!q->resident && newblocked) continue;
    int64_t rem = P + q->d - q->cached;                 /* tokens still to process before the next emission */
    int64_t want = c->chunk_tokens;                     /* KVNEED(r, c): next prefill chunk or decode step */
    if (rem < want) want = rem;
    if (c->token_budget - tok < want) want = c->token_budget - tok;
    int64_t foot = ceil_div(q->cached + want, blk);
    if (C + foot > B) {                                  /* U + dU > B */
      if (q->resident) break;
      newblocked = 1; continue;
    }
    e[j].want = want; C += foot; tok += want; cnt++;
    if (q->preempt_since >= 0) {                         /* M15: back on the device -- the preemption ends where this iteration starts */
      q->t_preempt += x->t - q->preempt_since;
      q->preempt_since = -1;
    }
    if (q->d >= 1 && rem == 1) decode_seqs++; else prefill_tokens += want;   /* M9 */
    ev_add(&ev, EV_ADMIT, (uint32_t)e[j].id, (uint32_t)want);
    if (q->swapped) {                                    /* swap-in on admission (M9) */
      int64_t blocks = ceil_div(q->cached, blk);
      swap_blocks += blocks; x->swap_used -= blocks; x->swapins++;
      ev_add(&ev, EV_SWAPIN, (uint32_t)e[j].id, (uint32_t)blocks);
    }
  }

  /* M8 SELECTVICTIM / SWAPOUT: non-admitted residents must fit in B - C;
     evict the lowest-priority one (the last in the order) until they do */
  int64_t sumres = 0;
  for (int64_t j = 0; j < n; j++)
    if (e[j].want == 0 && x->req[e[j].id].resident) sumres += ceil_div(x->req[e[j].id].cached, blk);
  for (int64_t j = n - 1; j >= 0 && sumres > B - C; j--) {
    orc_req* q = &x->req[e[j].id];
    if (e[j].want != 0 || !q->resident) continue;
    int64_t res = ceil_div(q->cached, blk);
    int do_swap = 0;
    if (c->preempt_mode == ORC_PRE_SWAP) do_swap = (x->swap_used + res <= c->swap_pool_blocks);
    else if (c->preempt_mode == ORC_PRE_AUTO)
      do_swap = (x->swap_used + res <= c->swap_pool_blocks) &&
                (2 * res * c->swap_ns_per_block < 1000 * c->c_prefill_tok_us * (int64_t)q->cached);
    if (do_swap) {
      q->swapped = 1; x->swap_used += res; swap_blocks += res; x->evict_swap++;
      ev_add(&ev, EV_EVICT_SWAP, (uint32_t)e[j].id, (uint32_t)res);
      e[j].evict = 2;
    } else {
      x->tokens_lost += q->cached;
      ev_add(&ev, EV_EVICT_RECOMPUTE, (uint32_t)e[j].id, (uint32_t)q->cached);
      q->cached = 0; x->evict_recompute++;
      e[j].evict = 1;
    }
    q->resident = 0; q->lockbin = -1; q->n_evict++;
    q->preempt_since = x->t;                             /* M15: preempted from the start of this iteration on */
    if (e[j].klass == 1) q->n_evict_unforced++;
    sumres -= res;
  }

  /* M9 EXECUTEONESTEP replaced by the stated cost model (BASELINE.json configs 1 and 3) */
  int64_t cost = c->c0_us + c->c_prefill_tok_us * prefill_tokens + c->c_decode_seq_us * decode_seqs +
                 (swap_blocks * c->swap_ns_per_block + 500) / 1000;
  int64_t t_start = x->t, t_end = x->t + cost;
  x->t = t_end;

  /* M10 apply: update KV + token counters */
  for (int64_t j = 0; j < n; j++) {
    if (e[j].want == 0) continue;
    int64_t id = e[j].id;
    orc_req* q = &x->req[id];
    q->resident = 1; q->swapped = 0; q->cached += (int32_t)e[j].want;
    if (q->cached == Pp[id] - Hh[id] + q->d) {
      q->d++; x->tokens_emitted++;
      if (q->d == 1) { q->t_first = t_end; ev_add(&ev, EV_EMIT_FIRST, (uint32_t)id, 0); }
      else x->hist[orc_tbt_bin(t_end - q->t_last)]++;
      q->t_last = t_end;
      if (q->d == Dd[id]) {
        q->completed = 1; q->resident = 0; q->cached = 0;     /* KV freed at once */
        if (x->ada) x->ring[x->n_completed % s->ada.window] = q->t_last - A[id];   /* E2E latency sample (M13) */
        x->n_completed++;
        x->sum_ttft += q->t_first - A[id]; x->sum_ttlt += q->t_last - A[id];
        x->sum_tbt_num += q->t_last - q->t_first; x->sum_tbt_den += Dd[id] - 1;
        ev_add(&ev, EV_COMPLETE, (uint32_t)id, 0);
      }
    }
  }
  /* re-lock every resident at the bin its key was computed with this iteration (M10, G6) */
  int64_t kv_after = 0;
  for (int64_t j = 0; j < n; j++) {
    orc_req* q = &x->req[e[j].id];
    if (q->resident) { q->lockbin = e[j].bin; kv_after += ceil_div(q->cached, blk); }
  }
  /* remove completed requests, preserving id order */
  int64_t m = 0;
  for (int64_t j = 0; j < n; j++)
    if (!x->req[x->active[j]].completed) x->active[m++] = x->active[j];
  x->n_active = m;

  /* M12 digest */
  x->H = digest_fold(x->H, ev, t_end);
  x->iterations++; x->request_steps += n;
  x->prefill_tokens += prefill_tokens; x->decode_seqs += decode_seqs;

  if (info) {
    info->executed = 1; info->n_active = n; info->t_start_us = t_start; info->cost_us = cost;
    info->t_end_us = t_end; info->claimed_blocks = C; info->prefill_tokens = prefill_tokens;
    info->decode_seqs = decode_seqs; info->swap_blocks = swap_blocks; info->kv_resident_after = kv_after;
  }
  if (out) {
    for (int64_t j = 0; j < n; j++) {
      const orc_req* q = &x->req[e[j].id];
      out[j].id = e[j].id; out[j].klass = e[j].klass; out[j].key = e[j].key; out[j].bin = e[j].bin;
      out[j].resident_before = e[j].resident_before; out[j].want = e[j].want; out[j].evict = e[j].evict;
      out[j].cached_after = q->cached; out[j].d_after = q->d; out[j].resident_after = q->resident;
    }
  }
  free(e);
  return 1;
}

static int rep_done(const orc_sim* s, const orc_rep* x) {
  return x->n_active == 0 && x->next >= (int64_t)s->n_req[x->par.trace_id];
}

int orc_step(orc_sim* s, int64_t n_iters) {
  if (!s || n_iters < 0) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++)
    for (int64_t i = 0; i < n_iters; i++) {
      int rc = step_one(s, &s->rep[r], NULL, NULL);
      if (rc < 0) return rc;
      if (rc == 0) break;
    }
  return ORC_OK;
}

int orc_step_replica(orc_sim* s, int64_t r, orc_step_info* info, orc_step_entry* entries) {
  if (!s || r < 0 || r >= s->cfg.n_replicas) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  int rc = step_one(s, &s->rep[r], info, entries);
  return rc < 0 ? rc : ORC_OK;
}

int orc_run_replica(orc_sim* s, int64_t r, int64_t max_iters, int64_t* iters_done) {
  if (!s || r < 0 || r >= s->cfg.n_replicas || max_iters < 0) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  int64_t it = 0;
  while (it < max_iters) {
    int rc = step_one(s, &s->rep[r], NULL, NULL);
    if (rc < 0) return rc;
    if (rc == 0) break;
    it++;
  }
  if (iters_done) *iters_done = it;
  return rep_done(s, &s->rep[r]) ? ORC_OK : ORC_ELIVELOCK;
}

int orc_run(orc_sim* s, int64_t max_iters, int64_t* iters_done) {
  if (!s || max_iters < 0) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  int64_t mx = 0; int live = 0;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    int64_t it = 0;
    int rc = orc_run_replica(s, r, max_iters, &it);
    if (rc == ORC_ELIVELOCK) live = 1; else if (rc < 0) return rc;
    if (it > mx) mx = it;
  }
  if (iters_done) *iters_done = mx;
  return live ? ORC_ELIVELOCK : ORC_OK;
}

/* ---------- M18: a cluster of replicas behind a join-the-shortest-queue router (Table 9) ----------
 * "Cluster-level routers decide which instance a request is sent to; UniBoost decides how to schedule requests within
 * that instance."  Replicas c K .. c K + K - 1 form cluster c and start with empty traces; the cluster's arrivals come in
 * one global stream.  An arrival at time a goes to the replica with the fewest requests in the system at time a --
 * assigned to it and not completed by a (completion time t_last <= a counts as gone) --, the lowest replica number on
 * a tie.  A replica's state at time a is the result of every iteration that STARTS before a (an iteration that starts at
 * a would already ingest the arrival). */
static int64_t jsq_next_start(const orc_sim* s, const orc_rep* x) {
  if (x->n_active > 0) return x->t;
  const int64_t tr = x->par.trace_id;
  if (x->next >= (int64_t)s->n_req[tr]) return INT64_MAX;                  /* nothing to do */
  const int64_t a = s->arrival[tr * s->cfg.max_requests + x->next];
  return a > x->t ? a : x->t;                                              /* idle jump (M6) */
}

int orc_jsq_run(orc_sim* s, int64_t K, const int64_t* arrival, const int32_t* prompt, const int32_t* decode,
                const uint32_t* n_arr, int64_t NA, int32_t* assign) {
  if (!s || !arrival || !prompt || !decode || !n_arr || K < 1 || NA < 0) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  const orc_config* c = &s->cfg;
  const int64_t R = c->n_replicas, N = c->max_requests;
  if (R % K != 0 || c->n_traces != R) return ORC_EINVAL;
  const int64_t C = R / K;
  for (int64_t r = 0; r < R; r++)
    if (s->rep[r].par.trace_id != r || s->n_req[r] != 0 || s->rep[r].iterations != 0 || s->rep[r].ada) return ORC_ESTATE;
  for (int64_t cl = 0; cl < C; cl++) {
    if ((int64_t)n_arr[cl] > NA) return ORC_EINVAL;
    for (int64_t j = 0; j < (int64_t)n_arr[cl]; j++) {
      const int64_t a = arrival[cl * NA + j], P = prompt[cl * NA + j], D = decode[cl * NA + j];
      if (a < 0 || a > ((int64_t)1 << 61)) return ORC_EINVAL;
      if (j > 0 && a < arrival[cl * NA + j - 1]) return ORC_EUNSORTED;
      if (P < 1 || D < 1 || (P + D + c->block_tokens - 1) / c->block_tokens > c->kv_blocks) return ORC_EINFEASIBLE;
    }
  }
  for (int64_t cl = 0; cl < C; cl++) {
    for (int64_t j = 0; j < (int64_t)n_arr[cl]; j++) {
      const int64_t a = arrival[cl * NA + j];
      int64_t best = -1, best_n = 0;
      for (int64_t k = 0; k < K; k++) {
        orc_rep* x = &s->rep[cl * K + k];
        while (jsq_next_start(s, x) < a) { int rc = step_one(s, x, NULL, NULL); if (rc < 0) return rc; }
        int64_t in_system = 0;                                             /* assigned and not completed by time a */
        for (int64_t i = 0; i < (int64_t)s->n_req[cl * K + k]; i++)
          if (!(x->req[i].completed && x->req[i].t_last <= a)) in_system++;
        if (best < 0 || in_system < best_n) { best = k; best_n = in_system; }
      }
      const int64_t tr = cl * K + best;
      if ((int64_t)s->n_req[tr] >= N) return ORC_EINVAL;                   /* the replica's row is full */
      const int64_t at = tr * N + s->n_req[tr];
      s->arrival[at] = a; s->prompt[at] = prompt[cl * NA + j]; s->decode[at] = decode[cl * NA + j];
      s->n_req[tr]++;
      if (assign) assign[cl * NA + j] = (int32_t)best;
    }
  }
  return orc_run(s, INT64_MAX, NULL);                                      /* every replica serves what it got */
}

/* ---------- read-out ---------- */

static int i64_cmp(const void* a, const void* b) {
  int64_t x = *(const int64_t*)a, y = *(const int64_t*)b;
  return x < y ? -1 : (x > y ? 1 : 0);
}

int orc_stats_get(orc_sim* s, orc_stats* out) {
  if (!s || !out) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  const int64_t N = s->cfg.max_requests;
  static const int64_t PCT[3] = {50, 90, 99};
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    orc_rep* x = &s->rep[r];
    orc_stats* o = &out[r];
    memset(o, 0, sizeof(*o));
    int64_t tr = x->par.trace_id, nreq = s->n_req[tr];
    o->iterations = x->iterations; o->request_steps = x->request_steps; o->n_completed = x->n_completed;
    o->evict_recompute = x->evict_recompute; o->evict_swap = x->evict_swap; o->swapins = x->swapins;
    o->tokens_lost = x->tokens_lost; o->tokens_emitted = x->tokens_emitted;
    o->prefill_tokens = x->prefill_tokens; o->decode_seqs = x->decode_seqs;
    o->t_end_us = x->t; o->peak_active = x->peak_active; o->done = rep_done(s, x); o->swap_used = x->swap_used;
    o->sum_ttft_us = x->sum_ttft; o->sum_ttlt_us = x->sum_ttlt;
    o->sum_tbt_num_us = x->sum_tbt_num; o->sum_tbt_den = x->sum_tbt_den;
    /* M11: TTFT_i = t_first - a_i, TTLT_i = t_last - a_i over completed requests; nearest rank */
    int64_t m = 0;
    int64_t* f = (int64_t*)malloc(sizeof(int64_t) * (size_t)(nreq > 0 ? nreq : 1));
    int64_t* l = (int64_t*)malloc(sizeof(int64_t) * (size_t)(nreq > 0 ? nreq : 1));
    if (!f || !l) { free(f); free(l); return ORC_ENOMEM; }
    for (int64_t i = 0; i < nreq; i++)
      if (x->req[i].completed) {
        f[m] = x->req[i].t_first - s->arrival[tr * N + i];
        l[m] = x->req[i].t_last - s->arrival[tr * N + i];
        m++;
      }
    qsort(f, (size_t)m, sizeof(int64_t), i64_cmp);
    qsort(l, (size_t)m, sizeof(int64_t), i64_cmp);
    int64_t gaps = 0;
    for (int b = 0; b < TBT_BINS; b++) gaps += x->hist[b];
    for (int k = 0; k < 3; k++) {
      o->ttft_us[k] = orc_percentile_nearest_rank(f, m, PCT[k]);
      o->ttlt_us[k] = orc_percentile_nearest_rank(l, m, PCT[k]);
      int64_t v = 0;
      if (gaps > 0) {
        int64_t rank = (PCT[k] * gaps + 99) / 100, cum = 0;
        if (rank < 1) rank = 1;
        for (int b = 0; b < TBT_BINS; b++) { cum += x->hist[b]; if (cum >= rank) { v = orc_tbt_edge(b); break; } }
      }
      o->tbt_us[k] = v;
      o->ttft_s[k] = (double)o->ttft_us[k] * 1e-6;
      o->ttlt_s[k] = (double)o->ttlt_us[k] * 1e-6;
      o->tbt_s[k] = (double)o->tbt_us[k] * 1e-6;
    }
    free(f); free(l);
    o->mean_ttft_s = m ? ((double)x->sum_ttft / (double)m) * 1e-6 : 0.0;
    o->mean_ttlt_s = m ? ((double)x->sum_ttlt / (double)m) * 1e-6 : 0.0;
    o->mean_tbt_s = x->sum_tbt_den ? ((double)x->sum_tbt_num / (double)x->sum_tbt_den) * 1e-6 : 0.0;
    o->tokens_per_s = x->t > 0 ? (double)x->tokens_emitted / ((double)x->t * 1e-6) : 0.0;
  }
  return ORC_OK;
}

int orc_per_request(orc_sim* s, int64_t* tf, int64_t* tl, uint32_t* ne, uint32_t* neu) {
  if (!s) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  const int64_t N = s->cfg.max_requests;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    orc_rep* x = &s->rep[r];
    int64_t nreq = s->n_req[x->par.trace_id];
    for (int64_t i = 0; i < N; i++) {
      int in = i < nreq;
      if (tf) tf[r * N + i] = in ? x->req[i].t_first : -1;
      if (tl) tl[r * N + i] = in ? x->req[i].t_last : -1;
      if (ne) ne[r * N + i] = in ? x->req[i].n_evict : 0;
      if (neu) neu[r * N + i] = in ? x->req[i].n_evict_unforced : 0;
    }
  }
  return ORC_OK;
}

/* ---------- richer reductions (next row 3) ---------- */

/* latencies (which: 0 TTFT = t_first - a, 1 TTLT = t_last - a) of the completed requests of one replica */
static int64_t collect_latencies(const orc_sim* s, const orc_rep* x, int64_t which, int64_t* out) {
  const int64_t N = s->cfg.max_requests, tr = x->par.trace_id, nreq = s->n_req[tr];
  int64_t m = 0;
  for (int64_t i = 0; i < nreq; i++)
    if (x->req[i].completed)
      out[m++] = (which == 0 ? x->req[i].t_first : x->req[i].t_last) - s->arrival[tr * N + i];
  return m;
}

int orc_percentile_curve(orc_sim* s, int64_t which, const int64_t* permille, int64_t n, int64_t* out) {
  if (!s || !s->have_reps || !permille || !out || which < 0 || which > 1 || n < 1) return ORC_EINVAL;
  int64_t* v = (int64_t*)malloc(sizeof(int64_t) * (size_t)(s->cfg.max_requests > 0 ? s->cfg.max_requests : 1));
  if (!v) return ORC_ENOMEM;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    int64_t m = collect_latencies(s, &s->rep[r], which, v);
    qsort(v, (size_t)m, sizeof(int64_t), i64_cmp_);
    for (int64_t k = 0; k < n; k++) {
      if (permille[k] < 1 || permille[k] > 1000) { free(v); return ORC_EINVAL; }
      if (m == 0) { out[r * n + k] = 0; continue; }
      int64_t rank = (permille[k] * m + 999) / 1000;      /* ceil(p m / 1000), 1-based */
      if (rank < 1) rank = 1;
      if (rank > m) rank = m;
      out[r * n + k] = v[rank - 1];
    }
  }
  free(v);
  return ORC_OK;
}

/* M15 / per-class reductions (Tables 3-5): over the completed
 * requests of a replica whose total length P + D lies in [len_lo, len_hi], the nearest-rank percentiles (t_p of
 * PAPER.md:225, rank ceil(p m / 1000)) of TTFT (which 0), TTLT (1) or preemption time (2), their number and sum. */
int orc_preempt_time(orc_sim* s, int64_t* out) {
  if (!s || !s->have_reps || !out) return ORC_EINVAL;
  const int64_t N = s->cfg.max_requests;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    const orc_rep* x = &s->rep[r];
    const int64_t nreq = s->n_req[x->par.trace_id];
    for (int64_t i = 0; i < N; i++) out[r * N + i] = i < nreq ? x->req[i].t_preempt : 0;
  }
  return ORC_OK;
}

int orc_class_percentiles(orc_sim* s, int64_t which, int64_t len_lo, int64_t len_hi, const int64_t* permille, int64_t n,
                          int64_t* out, int64_t* count, int64_t* sum) {
  if (!s || !s->have_reps || !permille || !out || which < 0 || which > 2 || n < 1) return ORC_EINVAL;
  const int64_t N = s->cfg.max_requests;
  int64_t* v = (int64_t*)malloc(sizeof(int64_t) * (size_t)(N > 0 ? N : 1));
  if (!v) return ORC_ENOMEM;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    const orc_rep* x = &s->rep[r];
    const int64_t tr = x->par.trace_id, nreq = s->n_req[tr];
    int64_t m = 0, tot = 0;
    for (int64_t i = 0; i < nreq; i++) {
      const orc_req* q = &x->req[i];
      const int64_t len = (int64_t)s->prompt[tr * N + i] - (int64_t)s->hit[tr * N + i] + (int64_t)s->decode[tr * N + i];   /* (effective length, M17) */
      if (!q->completed || len < len_lo || len > len_hi) continue;
      const int64_t a = s->arrival[tr * N + i];
      v[m] = which == 0 ? q->t_first - a : (which == 1 ? q->t_last - a : q->t_preempt);
      tot += v[m];
      m++;
    }
    qsort(v, (size_t)m, sizeof(int64_t), i64_cmp_);
    for (int64_t k = 0; k < n; k++) {
      if (permille[k] < 1 || permille[k] > 1000) { free(v); return ORC_EINVAL; }
      if (m == 0) { out[r * n + k] = 0; continue; }
      int64_t rank = (permille[k] * m + 999) / 1000;
      if (rank < 1) rank = 1;
      if (rank > m) rank = m;
      out[r * n + k] = v[rank - 1];
    }
    if (count) count[r] = m;
    if (sum) sum[r] = tot;
  }
  free(v);
  return ORC_OK;
}

int orc_slo_attainment(orc_sim* s, int64_t which, const int64_t* thr, int64_t n, int64_t* met) {
  if (!s || !s->have_reps || !thr || !met || which < 0 || which > 1 || n < 1) return ORC_EINVAL;
  int64_t* v = (int64_t*)malloc(sizeof(int64_t) * (size_t)(s->cfg.max_requests > 0 ? s->cfg.max_requests : 1));
  if (!v) return ORC_ENOMEM;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) {
    int64_t m = collect_latencies(s, &s->rep[r], which, v);
    for (int64_t k = 0; k < n; k++) {
      int64_t c = 0;
      for (int64_t i = 0; i < m; i++) if (v[i] <= thr[r * n + k]) c++;
      met[r * n + k] = c;
    }
  }
  free(v);
  return ORC_OK;
}

int orc_digest(orc_sim* s, uint64_t* dg) {
  if (!s || !dg) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  for (int64_t r = 0; r < s->cfg.n_replicas; r++) dg[r] = s->rep[r].H;
  return ORC_OK;
}

int orc_boost_lut(orc_sim* s, int64_t r, int64_t* lut, int64_t cap, int64_t* nb) {
  if (!s || r < 0 || r >= s->cfg.n_replicas || !nb) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  *nb = s->rep[r].nb;
  if (lut) for (int64_t b = 0; b < s->rep[r].nb && b < cap; b++) lut[b] = s->rep[r].lut[b];
  return ORC_OK;
}

int orc_tbt_hist(orc_sim* s, int64_t r, uint32_t* hist) {
  if (!s || r < 0 || r >= s->cfg.n_replicas || !hist) return ORC_EINVAL;
  if (!s->have_reps) return ORC_ESTATE;
  memcpy(hist, s->rep[r].hist, sizeof(uint32_t) * TBT_BINS);
  return ORC_OK;
}
