/* spd_oracle.c — CPU oracle for the SPD step.  TEST INFRASTRUCTURE ONLY; see spd_oracle.h.
 *
 * Written from /root/reference/PAPER.md (cited as PAPER.md:<line>) and the readings C-1 / C-2.x of
 * SURVEY.md §8(c) (also listed in DESIGN.md).  Plain loops, fp32 tensors, fp64 accumulation,
 * OpenMP only over independent output rows.  No blocking/fusion except ora_prefill(block>1), which
 * only interchanges the (token, row) loops.
 */
#include "spd_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ scalars and bf16 ---------- */

static inline float bf16_to_f32(uint16_t b) {
  uint32_t u = (uint32_t)b << 16;
  float f;
  memcpy(&f, &u, 4);
  return f;
}

/* fp32 -> bf16, round to nearest even (C-2.17: the only rounding below fp32 on the path). */
uint16_t ora_op_f32_to_bf16(float x) {
  uint32_t u;
  memcpy(&u, &x, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40); /* NaN stays NaN */
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

/* C-2.19: the forced-acceptance draw is a pure integer function of (seed, step counter). */
uint64_t ora_op_splitmix64(uint64_t x) {
  uint64_t z = x + 0x9e3779b97f4a7c15ull;
  z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
  z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
  return z ^ (z >> 31);
}

int32_t ora_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* Dot product of a bf16 weight row with an fp32 vector, accumulated in fp64.  Sixteen interleaved
 * partial sums (element i goes to partial i mod 16) are added in index order at the end, so the
 * value does not depend on how the compiler vectorises the loop. */
static inline double dot_row(const uint16_t *w, const float *x, int k) {
  double acc[16];
  for (int j = 0; j < 16; ++j) acc[j] = 0.0;
  int i = 0;
  for (; i + 16 <= k; i += 16)
    for (int j = 0; j < 16; ++j) acc[j] += (double)bf16_to_f32(w[i + j]) * (double)x[i + j];
  for (int j = 0; i < k; ++i, ++j) acc[j] += (double)bf16_to_f32(w[i]) * (double)x[i];
  double s = 0.0;
  for (int j = 0; j < 16; ++j) s += acc[j];
  return s;
}

/* ------------------------------------------------------------------ single operations --------- */

/* RMSNorm(x, g) = x * (mean(x^2) + eps)^(-1/2) * g   (C-1; eps from BASELINE.json). */
void ora_op_rmsnorm(const float *x, const uint16_t *gain, int32_t d, float eps, float *out) {
  double ss = 0.0;
  for (int i = 0; i < d; ++i) ss += (double)x[i] * (double)x[i];
  double r = 1.0 / sqrt(ss / (double)d + (double)eps);
  for (int i = 0; i < d; ++i) out[i] = (float)((double)x[i] * r * (double)bf16_to_f32(gain[i]));
}

/* out = W x, W bf16 [rows, k] row-major. */
void ora_op_gemv(const uint16_t *w, int32_t rows, int32_t k, const float *x, float *out) {
  /* rows are independent, so threading never changes a value; products below 2^20 multiply-adds (every product of
   * the small test models) stay on the calling thread: no worker wake-ups or spinning between tiny regions */
#pragma omp parallel for schedule(static) if ((size_t)rows * (size_t)k >= 1048576)
  for (int r = 0; r < rows; ++r) out[r] = (float)dot_row(w + (size_t)r * k, x, k);
}

/* Same product for a block of vectors: Y[t][r] = W[r] . X[t].  Rows outside, tokens inside, so a
 * weight row is read once per block; each (t, r) value is the same dot_row call as in ora_op_gemv. */
static void gemv_block(const uint16_t *w, int rows, int k, const float *x, int ldx, float *y, int ldy,
                       int nt) {
#pragma omp parallel for schedule(static) if ((size_t)rows * (size_t)k * (size_t)nt >= 1048576)
  for (int r = 0; r < rows; ++r)
    for (int t = 0; t < nt; ++t) y[(size_t)t * ldy + r] = (float)dot_row(w + (size_t)r * k, x + (size_t)t * ldx, k);
}

/* RoPE, rotate-half pairing (C-2.14): pair (i, i+hd/2), theta_i = base^(-2i/hd), angle = pos*theta_i,
 * cos/sin evaluated in double and rounded to fp32. */
void ora_op_rope(float *vec, int32_t n_heads, int32_t head_dim, int32_t pos, float base) {
  int half = head_dim / 2;
  for (int i = 0; i < half; ++i) {
    double theta = pow((double)base, -2.0 * (double)i / (double)head_dim);
    double ang = (double)pos * theta;
    float c = (float)cos(ang), s = (float)sin(ang);
    for (int h = 0; h < n_heads; ++h) {
      float *v = vec + (size_t)h * head_dim;
      double a = v[i], b = v[i + half];
      v[i] = (float)(a * (double)c - b * (double)s);
      v[i + half] = (float)(b * (double)c + a * (double)s);
    }
  }
}

/* GQA decode attention for one token (C-1): for q-head hq, kv-head kvh = hq / (Hq/Hkv),
 * s_t = q_hq . K[t][kvh] / sqrt(hd) for t = 0..t_len-1, w = softmax(s), o_hq = sum_t w_t V[t][kvh].
 * kc, vc: bf16 [t_len, Hkv*hd] (row t = position t). */
void ora_op_attention(const float *q, const uint16_t *kc, const uint16_t *vc, int32_t t_len,
                      int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, float *out) {
  int group = n_q_heads / n_kv_heads;
  size_t row = (size_t)n_kv_heads * head_dim;
#pragma omp parallel for schedule(static) if ((size_t)n_q_heads * (size_t)t_len * (size_t)head_dim >= 1048576)
  for (int hq = 0; hq < n_q_heads; ++hq) {
    int kvh = hq / group;
    const float *qh = q + (size_t)hq * head_dim;
    float *s = (float *)malloc(sizeof(float) * (size_t)t_len);
    float m = -INFINITY;
    for (int t = 0; t < t_len; ++t) {
      double dot = dot_row(kc + (size_t)t * row + (size_t)kvh * head_dim, qh, head_dim);
      s[t] = (float)(dot / sqrt((double)head_dim));
      if (s[t] > m) m = s[t];
    }
    double *w = (double *)malloc(sizeof(double) * (size_t)t_len);
    double denom = 0.0;
    for (int t = 0; t < t_len; ++t) { w[t] = exp((double)s[t] - (double)m); denom += w[t]; }
    /* o_e = sum_t w_t V[t][e] / denom: every element's sum runs over t in ascending order; the t loop is the outer
     * one only so that a V row is read contiguously (same operations per element, same order, same result) */
    double *acc = (double *)calloc((size_t)head_dim, sizeof(double));
    for (int t = 0; t < t_len; ++t) {
      const uint16_t *vr = vc + (size_t)t * row + (size_t)kvh * head_dim;
      for (int e = 0; e < head_dim; ++e) acc[e] += w[t] * (double)bf16_to_f32(vr[e]);
    }
    for (int e = 0; e < head_dim; ++e) out[(size_t)hq * head_dim + e] = (float)(acc[e] / denom);
    free(acc);
    free(w);
    free(s);
  }
}

/* a = silu(gate) * up, silu(z) = z / (1 + exp(-z))  (C-1). */
void ora_op_silu_mul(const float *gate, const float *up, int32_t n, float *out) {
  for (int i = 0; i < n; ++i) {
    double z = gate[i];
    out[i] = (float)(z / (1.0 + exp(-z)) * (double)up[i]);
  }
}

/* Greedy argmax: maximum value, lowest index among exact ties (C-2.8). */
int32_t ora_op_argmax(const float *x, int32_t n) {
  int best = 0;
  for (int i = 1; i < n; ++i)
    if (x[i] > x[best]) best = i;
  return best;
}

static void top2_margin(const float *x, int n, float *gap, float *maxabs) {
  float a = -INFINITY, b = -INFINITY, mx = 0.f;
  for (int i = 0; i < n; ++i) {
    float v = x[i];
    if (v > a) { b = a; a = v; } else if (v > b) b = v;
    if (fabsf(v) > mx) mx = fabsf(v);
  }
  *gap = a - b;
  *maxabs = mx;
}

/* ------------------------------------------------------------------ context ------------------- */

struct ora_ctx {
  ora_config cfg;
  ora_weights w;
  uint16_t *kc, *vc; /* [L][max_seq][Hkv*hd] bf16 */
  int32_t *len;      /* [L] valid KV rows (C-2.11) */
  float *hfin;       /* [max_seq][d] final (pre-norm) hidden state of committed positions (C-2.4) */
  int32_t c;         /* committed length */
  int32_t a;         /* in-flight tokens, oldest first */
  int32_t *r_pos, *r_tok, *r_k;
  float *r_h;        /* [n][d] */
  int64_t steps;     /* K */
  int32_t emitted;   /* N */
  int32_t prompt_len, prefilled;
  const int32_t *truth;
  int32_t n_truth;
  int32_t forced_on;
  uint64_t forced_thresh, forced_seed;
  /* last-step records */
  float *exit_logits, *pdm_logits, *pdm_u, *pdm_feat;
  float gap[2], maxabs[2];
  int32_t ties[2];   /* tie hints adopted: [0] verify, [1] PDM */
  float *ar_trace;
  int32_t reverse_forward;
  /* NEXT-2 sampling verification */
  int32_t sampling_on, top_k;
  float temperature;
  uint64_t samp_seed;
  ora_dist *r_q;     /* [n] the draft distribution each in-flight token was drawn from */
  ora_sample_record rec;
  /* NEXT-1 the paper's PDM */
  int32_t pdm_on, pdm_m, pdm_anchor[ORA_PDM_MAX_ANCHORS];
  ora_pdm_weights pw;
  float *anch;       /* [max_seq][m][d]  H_pos^{b_i}: the residual stream entering layer b_i */
  uint16_t *pkc, *pvc; /* [L_s][max_seq][Hkv*hd] bf16: the PDM's own KV cache */
  int32_t pdm_final; /* F: positions whose PDM cache rows are final (depth n) */
  float *pdm_x;      /* [rows][d] features / residual streams of the rows of the last PDM run */
  float *pdm_g;      /* [rows][d] the features g as built (kept for the pins) */
  float *pdm_lg;     /* [V_s] */
  float *pdm_h;      /* [d] */
  int32_t pdm_rows, pdm_first, pdm_cap, *pdm_depth;
  /* scratch */
  float *x, *q, *kk, *vv, *att, *o, *g, *u, *act, *dn, *z;
};

static size_t kv_row(const ora_config *c) { return (size_t)c->n_kv_heads * c->head_dim; }

/* ------------------------------------------------------------------ NEXT-2: sampling ops ------ */

/* S-6: 24-bit uniform in [0, 1), exactly representable in fp32 and fp64. */
double ora_op_uniform(uint64_t seed, int64_t K, int32_t j) {
  uint64_t r = ora_op_splitmix64(seed + 3ull * (uint64_t)K + (uint64_t)j) >> 40;
  return (double)r * (1.0 / 16777216.0);
}

/* S-2: top-k filter + temperature softmax ("top-k=50 and top-p=1.0", T = 1). */
void ora_op_topk_softmax(const float *logits, int32_t vocab, int32_t top_k, float temperature,
                         const int32_t *support, ora_dist *out) {
  int k = top_k < vocab ? top_k : vocab;
  if (k > ORA_MAX_TOPK) k = ORA_MAX_TOPK;
  int ids[ORA_MAX_TOPK];
  if (support) {
    for (int i = 0; i < k; ++i) ids[i] = support[i];
  } else {
    /* k passes; pass r takes the best entry not taken yet: larger value first, lower index on ties */
    for (int r = 0; r < k; ++r) {
      int best = -1;
      for (int i = 0; i < vocab; ++i) {
        int taken = 0;
        for (int t = 0; t < r; ++t) taken |= ids[t] == i;
        if (taken) continue;
        if (best < 0 || logits[i] > logits[best]) best = i;
      }
      ids[r] = best;
    }
  }
  /* ascending token id */
  for (int i = 1; i < k; ++i) {
    int v = ids[i], j = i - 1;
    while (j >= 0 && ids[j] > v) { ids[j + 1] = ids[j]; --j; }
    ids[j + 1] = v;
  }
  double m = -INFINITY, e[ORA_MAX_TOPK], Z = 0.0;
  for (int i = 0; i < k; ++i)
    if ((double)logits[ids[i]] > m) m = (double)logits[ids[i]];
  for (int i = 0; i < k; ++i) {
    e[i] = exp(((double)logits[ids[i]] - m) / (double)temperature);
    Z += e[i];
  }
  memset(out, 0, sizeof *out);
  out->k = k;
  for (int i = 0; i < k; ++i) { out->id[i] = ids[i]; out->p[i] = (float)(e[i] / Z); }
}

/* S-3: inverse CDF over weights w[0..k) in list order: the smallest i with u * W < w_0 + .. + w_i.
 * lo/hi (may be NULL) receive that entry's interval [C_{i-1}, C_i) / W for every entry. */
static int pick_index(const double *w, int k, double u, double *lo, double *hi) {
  double W = 0.0;
  for (int i = 0; i < k; ++i) W += w[i];
  double c = 0.0;
  int chosen = -1, last = -1;
  for (int i = 0; i < k; ++i) {
    if (lo) lo[i] = c / W;
    c += w[i];
    if (hi) hi[i] = c / W;
    if (w[i] > 0.0) last = i;
    if (chosen < 0 && u * W < c) chosen = i;
  }
  return chosen >= 0 ? chosen : last;
}

static double dist_prob(const ora_dist *D, int token) {
  for (int i = 0; i < D->k; ++i)
    if (D->id[i] == token) return (double)D->p[i];
  return 0.0;
}

int32_t ora_op_sample_cdf(const ora_dist *D, double u) {
  double w[ORA_MAX_TOPK];
  for (int i = 0; i < D->k; ++i) w[i] = (double)D->p[i];
  return D->id[pick_index(w, D->k, u, NULL, NULL)];
}

/* PAPER.md:129 "standard rejection sampling": accept x ~ Q with probability min(1, P(x)/Q(x)). */
int32_t ora_op_accept(const ora_dist *P, const ora_dist *Q, int32_t token, double u) {
  return u * dist_prob(Q, token) < dist_prob(P, token);
}

static void residual_weights(const ora_dist *P, const ora_dist *Q, double *w) {
  double W = 0.0;
  for (int i = 0; i < P->k; ++i) {
    double r = (double)P->p[i] - dist_prob(Q, P->id[i]);
    w[i] = r > 0.0 ? r : 0.0;
    W += w[i];
  }
  if (!(W > 0.0))
    for (int i = 0; i < P->k; ++i) w[i] = (double)P->p[i];
}

/* the replacement of a rejected token; standard rejection sampling draws it from
 * norm(max(0, P - Q)) so that the emitted token is distributed as P. */
int32_t ora_op_sample_residual(const ora_dist *P, const ora_dist *Q, double u) {
  double w[ORA_MAX_TOPK];
  residual_weights(P, Q, w);
  return P->id[pick_index(w, P->k, u, NULL, NULL)];
}

int ora_set_sampling(ora_ctx *o, float temperature, int32_t top_k, uint64_t seed) {
  if (top_k < 1) { o->sampling_on = 0; return 0; }
  if (top_k > ORA_MAX_TOPK || !(temperature > 0.f) || o->forced_on || o->pdm_on) return -1;   /* P-9: the paper's PDM is greedy only */
  o->sampling_on = 1; o->top_k = top_k; o->temperature = temperature; o->samp_seed = seed;
  /* tokens already in flight were not drawn from a filtered distribution: whoever put them there acted as a
   * deterministic drafter, Q = one-hot on the token (accepted with probability P(x)) */
  for (int i = 0; i < o->a; ++i) {
    memset(&o->r_q[i], 0, sizeof(ora_dist));
    o->r_q[i].k = 1; o->r_q[i].id[0] = o->r_tok[i]; o->r_q[i].p[0] = 1.f;
  }
  return 0;
}

void ora_get_sample_record(const ora_ctx *o, ora_sample_record *out) { *out = o->rec; }

/* Test hook: is `ids` (k distinct entries) a top-k set of `logits` up to `band`? */
static int support_hint_valid(const float *logits, int vocab, const int32_t *ids, int k, float band) {
  float mn = INFINITY, mx = -INFINITY;
  for (int i = 0; i < k; ++i) {
    if (ids[i] < 0 || ids[i] >= vocab) return 0;
    for (int j = 0; j < i; ++j)
      if (ids[j] == ids[i]) return 0;
    if (logits[ids[i]] < mn) mn = logits[ids[i]];
  }
  for (int i = 0; i < vocab; ++i) {
    int in = 0;
    for (int j = 0; j < k; ++j) in |= ids[j] == i;
    if (!in && logits[i] > mx) mx = logits[i];
  }
  return mn >= mx - band;
}

/* Filtered distribution of a head's logits; a valid differing support hint is adopted (counted). */
static void head_dist(ora_ctx *o, const float *logits, const int32_t *hint_ids, int hint_k, float band,
                      ora_dist *out) {
  int V = o->cfg.vocab;
  ora_op_topk_softmax(logits, V, o->top_k, o->temperature, NULL, out);
  if (hint_ids && hint_k == out->k) {
    int same = 1;
    for (int i = 0; i < hint_k; ++i) {
      int found = 0;
      for (int j = 0; j < out->k; ++j) found |= out->id[j] == hint_ids[i];
      same &= found;
    }
    if (!same && support_hint_valid(logits, V, hint_ids, hint_k, band)) {
      ora_op_topk_softmax(logits, V, o->top_k, o->temperature, hint_ids, out);
      o->rec.ties_support += 1;
    }
  }
}

/* Own inverse-CDF draw over weights w on support ids; a differing hint token is adopted iff u lies within
 * eps (in units of normalised mass) of the hint's interval. */
static int draw_with_hint(const int32_t *ids, const double *w, int k, double u, int hint, double eps,
                          int32_t *ties) {
  double lo[ORA_MAX_TOPK], hi[ORA_MAX_TOPK];
  int own = pick_index(w, k, u, lo, hi);
  if (hint >= 0 && hint != ids[own])
    for (int i = 0; i < k; ++i)
      if (ids[i] == hint && u >= lo[i] - eps && u < hi[i] + eps) { *ties += 1; return hint; }
  return ids[own];
}


ora_ctx *ora_create(const ora_config *cfg, const ora_weights *w) {
  if (!cfg || !w) return NULL;
  if (cfg->n_stages < 1 || cfg->n_layers % cfg->n_stages != 0) return NULL;      /* C-2.7 */
  if (cfg->n_kv_heads < 1 || cfg->n_q_heads % cfg->n_kv_heads != 0 || cfg->head_dim % 2 != 0) return NULL;
  ora_ctx *o = (ora_ctx *)calloc(1, sizeof(ora_ctx));
  o->cfg = *cfg;
  o->w = *w;
  int d = cfg->d_model, n = cfg->n_stages, L = cfg->n_layers, F = cfg->d_ffn, V = cfg->vocab;
  size_t row = kv_row(cfg);
  o->kc = (uint16_t *)calloc((size_t)L * cfg->max_seq * row, 2);
  o->vc = (uint16_t *)calloc((size_t)L * cfg->max_seq * row, 2);
  o->len = (int32_t *)calloc(L, 4);
  o->hfin = (float *)calloc((size_t)cfg->max_seq * d, 4);
  o->r_pos = (int32_t *)calloc(n, 4);
  o->r_tok = (int32_t *)calloc(n, 4);
  o->r_k = (int32_t *)calloc(n, 4);
  o->r_h = (float *)calloc((size_t)n * d, 4);
  o->r_q = (ora_dist *)calloc(n, sizeof(ora_dist));
  o->exit_logits = (float *)calloc(V, 4);
  o->pdm_logits = (float *)calloc(V, 4);
  o->pdm_u = (float *)calloc(d, 4);
  o->pdm_feat = (float *)calloc((size_t)n * d, 4);
  int qd = cfg->n_q_heads * cfg->head_dim;
  o->x = (float *)calloc(d, 4);
  o->q = (float *)calloc(qd, 4);
  o->kk = (float *)calloc(row, 4);
  o->vv = (float *)calloc(row, 4);
  o->att = (float *)calloc(qd, 4);
  o->o = (float *)calloc(d, 4);
  o->g = (float *)calloc(F, 4);
  o->u = (float *)calloc(F, 4);
  o->act = (float *)calloc(F, 4);
  o->dn = (float *)calloc(d, 4);
  o->z = (float *)calloc(d, 4);
  return o;
}

void ora_destroy(ora_ctx *o) {
  if (!o) return;
  free(o->kc); free(o->vc); free(o->len); free(o->hfin); free(o->r_pos); free(o->r_tok); free(o->r_k);
  free(o->r_h); free(o->exit_logits); free(o->pdm_logits); free(o->pdm_u); free(o->pdm_feat);
  free(o->x); free(o->q); free(o->kk); free(o->vv); free(o->att); free(o->o); free(o->g); free(o->u);
  free(o->act); free(o->dn); free(o->z); free(o->r_q);
  free(o->anch); free(o->pkc); free(o->pvc); free(o->pdm_x); free(o->pdm_g); free(o->pdm_lg); free(o->pdm_h); free(o->pdm_depth);
  free(o);
}

static void embed_row(const ora_ctx *o, int tok, float *h) {
  const uint16_t *e = o->w.embed + (size_t)tok * o->cfg.d_model;
  for (int i = 0; i < o->cfg.d_model; ++i) h[i] = bf16_to_f32(e[i]);
}

/* A stack of decoder layers with its KV cache: the target's L layers, or the PDM's L_s layers (same structure, C-2.13 /
 * reading P-3).  len == NULL: rows may be rewritten (the PDM refreshes its trailing rows every cycle). */
typedef struct {
  const uint16_t *const *attn_norm, *const *wq, *const *wk, *const *wv, *const *wo, *const *mlp_norm, *const *w_gate,
      *const *w_up, *const *w_down;
  uint16_t *kc, *vc;
  int32_t *len;
  int32_t capture;   /* 1: the target stack — capture the anchors H^b of the paper's PDM on the way (Eq. 4) */
} layer_set;

static layer_set target_set(ora_ctx *o) {
  layer_set S = {o->w.attn_norm, o->w.wq, o->w.wk, o->w.wv, o->w.wo, o->w.mlp_norm, o->w.w_gate, o->w.w_up, o->w.w_down,
                 o->kc, o->vc, o->len, 1};
  return S;
}

static layer_set pdm_set(ora_ctx *o) {
  layer_set S = {o->pw.attn_norm, o->pw.wq, o->pw.wk, o->pw.wv, o->pw.wo, o->pw.mlp_norm, o->pw.w_gate, o->pw.w_up,
                 o->pw.w_down, o->pkc, o->pvc, NULL, 0};
  return S;
}

/* PAPER.md:91 "H_t^l denote the hidden state of token x_t after layer l (l = 0 is the embedding)": the residual stream
 * ENTERING layer l.  Stored for the anchors l in B when the paper's PDM is attached. */
static void capture_anchor(ora_ctx *o, int l, const float *h, int pos) {
  if (!o->pdm_on) return;
  for (int i = 0; i < o->pdm_m; ++i)
    if (o->pdm_anchor[i] == l)
      memcpy(o->anch + ((size_t)pos * o->pdm_m + i) * o->cfg.d_model, h, sizeof(float) * (size_t)o->cfg.d_model);
}

/* The per-token attention sub-step of Layer: RoPE(q,k,pos); require len[l]==pos; append bf16(k),
 * bf16(v) as row pos; attend over rows 0..pos (causal incl. self).  Returns -1 if the causality
 * precondition of north_star ("every earlier-position token already deeper") is violated. */
static int attend_token(ora_ctx *o, const layer_set *S, int l, int pos, float *q, float *kk, const float *vv, float *att) {
  const ora_config *c = &o->cfg;
  size_t row = kv_row(c);
  ora_op_rope(q, c->n_q_heads, c->head_dim, pos, c->rope_base);
  ora_op_rope(kk, c->n_kv_heads, c->head_dim, pos, c->rope_base);
  if (pos >= c->max_seq || (S->len && S->len[l] != pos)) return -1;
  uint16_t *kd = S->kc + ((size_t)l * c->max_seq + pos) * row;
  uint16_t *vd = S->vc + ((size_t)l * c->max_seq + pos) * row;
  for (size_t i = 0; i < row; ++i) { kd[i] = ora_op_f32_to_bf16(kk[i]); vd[i] = ora_op_f32_to_bf16(vv[i]); }
  if (S->len) S->len[l] = pos + 1;
  ora_op_attention(q, S->kc + (size_t)l * c->max_seq * row, S->vc + (size_t)l * c->max_seq * row, pos + 1,
                   c->n_q_heads, c->n_kv_heads, c->head_dim, att);
  return 0;
}

/* Layer(l, h, pos) of C-1: pre-norm attention block then pre-norm SwiGLU block, residual stream h. */
static int layer_forward_set(ora_ctx *o, const layer_set *S, int l, float *h, int pos) {
  const ora_config *c = &o->cfg;
  int d = c->d_model, qd = c->n_q_heads * c->head_dim, kd = c->n_kv_heads * c->head_dim, F = c->d_ffn;
  if (S->capture) capture_anchor(o, l, h, pos);
  ora_op_rmsnorm(h, S->attn_norm[l], d, c->rms_eps, o->x);
  ora_op_gemv(S->wq[l], qd, d, o->x, o->q);
  ora_op_gemv(S->wk[l], kd, d, o->x, o->kk);
  ora_op_gemv(S->wv[l], kd, d, o->x, o->vv);
  if (attend_token(o, S, l, pos, o->q, o->kk, o->vv, o->att)) return -1;
  ora_op_gemv(S->wo[l], d, qd, o->att, o->o);
  for (int i = 0; i < d; ++i) h[i] += o->o[i];
  ora_op_rmsnorm(h, S->mlp_norm[l], d, c->rms_eps, o->x);
  ora_op_gemv(S->w_gate[l], F, d, o->x, o->g);
  ora_op_gemv(S->w_up[l], F, d, o->x, o->u);
  ora_op_silu_mul(o->g, o->u, F, o->act);
  ora_op_gemv(S->w_down[l], d, F, o->act, o->dn);
  for (int i = 0; i < d; ++i) h[i] += o->dn[i];
  return 0;
}

static int layer_forward(ora_ctx *o, int l, float *h, int pos) {
  layer_set S = target_set(o);
  return layer_forward_set(o, &S, l, h, pos);
}

/* logits = E . RMSNorm(h, gain); returns argmax and records the margin. */
static int head_argmax(ora_ctx *o, const float *h, const uint16_t *gain, float *logits, int which) {
  const ora_config *c = &o->cfg;
  ora_op_rmsnorm(h, gain, c->d_model, c->rms_eps, o->z);
  ora_op_gemv(o->w.embed, c->vocab, c->d_model, o->z, logits);
  top2_margin(logits, c->vocab, &o->gap[which], &o->maxabs[which]);
  return ora_op_argmax(logits, c->vocab);
}

static void ring_set_single(ora_ctx *o, int pos, int tok) {
  o->a = 1;
  o->r_pos[0] = pos; o->r_tok[0] = tok; o->r_k[0] = 0;
  embed_row(o, tok, o->r_h);
}

/* Blocked variant of "for every prompt token: Layer(l, h, pos)" for one layer and tokens t0..t1-1. */
static int layer_forward_block(ora_ctx *o, int l, float *H, int t0, int t1) {
  const ora_config *c = &o->cfg;
  int d = c->d_model, qd = c->n_q_heads * c->head_dim, kd = c->n_kv_heads * c->head_dim, F = c->d_ffn;
  int nt = t1 - t0;
  float *X = (float *)malloc(sizeof(float) * (size_t)nt * (F > qd ? F : qd));
  float *Q = (float *)malloc(sizeof(float) * (size_t)nt * qd);
  float *Kb = (float *)malloc(sizeof(float) * (size_t)nt * kd);
  float *Vb = (float *)malloc(sizeof(float) * (size_t)nt * kd);
  float *A = (float *)malloc(sizeof(float) * (size_t)nt * qd);
  float *O = (float *)malloc(sizeof(float) * (size_t)nt * d);
  float *G = (float *)malloc(sizeof(float) * (size_t)nt * F);
  float *U = (float *)malloc(sizeof(float) * (size_t)nt * F);
  int rc = 0;
  layer_set S = target_set(o);
  for (int t = 0; t < nt; ++t) capture_anchor(o, l, H + (size_t)(t0 + t) * d, t0 + t);
  for (int t = 0; t < nt; ++t) ora_op_rmsnorm(H + (size_t)(t0 + t) * d, o->w.attn_norm[l], d, c->rms_eps, X + (size_t)t * d);
  gemv_block(o->w.wq[l], qd, d, X, d, Q, qd, nt);
  gemv_block(o->w.wk[l], kd, d, X, d, Kb, kd, nt);
  gemv_block(o->w.wv[l], kd, d, X, d, Vb, kd, nt);
  for (int t = 0; t < nt && !rc; ++t)
    rc = attend_token(o, &S, l, t0 + t, Q + (size_t)t * qd, Kb + (size_t)t * kd, Vb + (size_t)t * kd, A + (size_t)t * qd);
  if (!rc) {
    gemv_block(o->w.wo[l], d, qd, A, qd, O, d, nt);
    for (int t = 0; t < nt; ++t)
      for (int i = 0; i < d; ++i) H[(size_t)(t0 + t) * d + i] += O[(size_t)t * d + i];
    for (int t = 0; t < nt; ++t) ora_op_rmsnorm(H + (size_t)(t0 + t) * d, o->w.mlp_norm[l], d, c->rms_eps, X + (size_t)t * d);
    gemv_block(o->w.w_gate[l], F, d, X, d, G, F, nt);
    gemv_block(o->w.w_up[l], F, d, X, d, U, F, nt);
    for (int t = 0; t < nt; ++t) ora_op_silu_mul(G + (size_t)t * F, U + (size_t)t * F, F, X + (size_t)t * F);
    gemv_block(o->w.w_down[l], d, F, X, F, O, d, nt);
    for (int t = 0; t < nt; ++t)
      for (int i = 0; i < d; ++i) H[(size_t)(t0 + t) * d + i] += O[(size_t)t * d + i];
  }
  free(X); free(Q); free(Kb); free(Vb); free(A); free(O); free(G); free(U);
  return rc;
}

/* Prefill (C-1): for pos in order: h = E[tok]; for l: h = Layer(l, h, pos); Hfin[pos] = h.
 * y_P = argmax(E . RMSNorm(Hfin[P-1], g_final)).  State: c = P, len[l] = P, ring = {(P, y_P, k=0, E[y_P])},
 * emitted = [y_P], K = 0.  ("the prefill prefix ... fully processed"; prefill is outside
 * the paper's timed region.) */
int ora_prefill(ora_ctx *o, const int32_t *tokens, int32_t P, int32_t block, int32_t *first_token) {
  const ora_config *c = &o->cfg;
  int d = c->d_model, L = c->n_layers;
  if (P < 1 || P >= c->max_seq) return -1;
  for (int i = 0; i < P; ++i)
    if (tokens[i] < 0 || tokens[i] >= c->vocab) return -1;
  for (int l = 0; l < L; ++l) o->len[l] = 0;
  o->pdm_final = 0;   /* the first cycle's PDM run builds the prompt's full-depth rows */
  if (block <= 1) {
    for (int pos = 0; pos < P; ++pos) {
      float *h = o->hfin + (size_t)pos * d;
      embed_row(o, tokens[pos], h);
      for (int l = 0; l < L; ++l)
        if (layer_forward(o, l, h, pos)) return -2;
    }
  } else {
    for (int pos = 0; pos < P; ++pos) embed_row(o, tokens[pos], o->hfin + (size_t)pos * d);
    for (int l = 0; l < L; ++l)
      for (int t0 = 0; t0 < P; t0 += block) {
        int t1 = t0 + block < P ? t0 + block : P;
        if (layer_forward_block(o, l, o->hfin, t0, t1)) return -2;
      }
  }
  int y = head_argmax(o, o->hfin + (size_t)(P - 1) * d, o->w.final_norm, o->exit_logits, 0);
  if (o->sampling_on) { /* the first token is drawn from P as well ("x ~ P"), u(seed, 0, 2) */
    memset(&o->rec, 0, sizeof o->rec);
    head_dist(o, o->exit_logits, NULL, 0, 0.f, &o->rec.target);
    o->rec.u_resid = ora_op_uniform(o->samp_seed, 0, 2);
    y = ora_op_sample_cdf(&o->rec.target, o->rec.u_resid);
  }
  o->c = P;
  o->prompt_len = P;
  o->steps = 0;
  o->emitted = 1;
  o->prefilled = 1;
  ring_set_single(o, P, y);
  if (first_token) *first_token = y;
  return 0;
}

int ora_set_forced(ora_ctx *o, const int32_t *truth, int32_t n_truth, float p, uint64_t seed) {
  if (p < 0.f) { o->forced_on = 0; return 0; }
  if (p > 1.f || (!truth && n_truth > 0) || o->sampling_on) return -1;
  o->truth = truth; o->n_truth = n_truth; o->forced_on = 1; o->forced_seed = seed;
  o->forced_thresh = (uint64_t)floor((double)p * 9007199254740992.0); /* floor(p * 2^53) */
  return 0;
}

/* ------------------------------------------------------------------ NEXT-1: the paper's PDM ---- */

static int apply_hint(const float *logits, int own, int hint, int vocab, float band, int32_t *ties);

/* Reading P-1: B = [0, L/4, L/2, 3L/4, L-1] (integer division), duplicates removed — for L = 32 the paper's
 * [0, 8, 16, 24, 31] (the last anchor is taken literally as L-1, C-2.6). */
static int anchor_set(int L, int32_t *b) {
  int cand[5] = {0, L / 4, L / 2, (3 * L) / 4, L - 1}, m = 0;
  for (int i = 0; i < 5; ++i)
    if (m == 0 || cand[i] > b[m - 1]) b[m++] = cand[i];
  return m;
}

int32_t ora_pdm_anchors(const ora_ctx *o, int32_t *anchors) {
  int32_t b[ORA_PDM_MAX_ANCHORS];
  int m = anchor_set(o->cfg.n_layers, b);
  if (anchors) memcpy(anchors, b, sizeof(int32_t) * (size_t)m);
  return m;
}

/* Eq. 3: l_max(k) = min(L, k L/n); f(k) = max{ i | b_i <= l_max(k) }. */
int32_t ora_pdm_f(const ora_ctx *o, int32_t k) {
  int32_t b[ORA_PDM_MAX_ANCHORS];
  int m = anchor_set(o->cfg.n_layers, b), L = o->cfg.n_layers, n = o->cfg.n_stages;
  int lmax = k * (L / n) < L ? k * (L / n) : L, f = 0;
  for (int i = 0; i < m; ++i)
    if (b[i] <= lmax) f = i;
  return f;
}

int ora_pdm_attach(ora_ctx *o, const ora_pdm_weights *pw) {
  const ora_config *c = &o->cfg;
  if (!pw || pw->n_layers < 1 || pw->vocab < 1 || pw->vocab > c->vocab || o->sampling_on || o->prefilled) return -1;
  if (!pw->fc || !pw->attn_norm || !pw->wq || !pw->wk || !pw->wv || !pw->wo || !pw->mlp_norm || !pw->w_gate || !pw->w_up ||
      !pw->w_down || !pw->final_norm || !pw->head || !pw->vocab_map)
    return -1;
  for (int i = 0; i < pw->vocab; ++i)
    if (pw->vocab_map[i] < 0 || pw->vocab_map[i] >= c->vocab || (i > 0 && pw->vocab_map[i] <= pw->vocab_map[i - 1])) return -1;
  o->pw = *pw;
  o->pdm_m = anchor_set(c->n_layers, o->pdm_anchor);
  size_t row = kv_row(c);
  o->anch = (float *)calloc((size_t)c->max_seq * o->pdm_m * c->d_model, 4);
  o->pkc = (uint16_t *)calloc((size_t)pw->n_layers * c->max_seq * row, 2);
  o->pvc = (uint16_t *)calloc((size_t)pw->n_layers * c->max_seq * row, 2);
  o->pdm_lg = (float *)calloc((size_t)pw->vocab, 4);
  o->pdm_h = (float *)calloc((size_t)c->d_model, 4);
  o->pdm_cap = 0;
  o->pdm_final = 0;
  o->pdm_on = 1;
  return 0;
}

/* The draft of one cycle (see spd_oracle.h).  Returns the drafted TARGET token id. */
static int pdm_paper_draft(ora_ctx *o, int32_t draft_hint, float band) {
  const ora_config *c = &o->cfg;
  int d = c->d_model, n = c->n_stages, m = o->pdm_m;
  int a = o->a, p_new = o->r_pos[a - 1];
  int first = o->pdm_final, rows = p_new - first + 1;
  if (rows > o->pdm_cap) {
    free(o->pdm_x); free(o->pdm_g); free(o->pdm_depth);
    o->pdm_cap = rows + 64;
    o->pdm_x = (float *)calloc((size_t)o->pdm_cap * d, 4);
    o->pdm_g = (float *)calloc((size_t)o->pdm_cap * d, 4);
    o->pdm_depth = (int32_t *)calloc((size_t)o->pdm_cap, 4);
  }
  o->pdm_rows = rows; o->pdm_first = first;
  float *cat = (float *)malloc(sizeof(float) * (size_t)m * d);
  /* features (Eq. 4): committed positions q < c take the full-depth rule k = n (Eq. 2 / Eq. 5); an in-flight token
   * takes its depth BEFORE this cycle's forward (pre-step); the newest contributes only g^0 */
  for (int r = 0; r < rows; ++r) {
    int q = first + r, k;
    if (q < o->c) k = n;
    else k = o->r_k[q - o->c];
    o->pdm_depth[r] = k;
    int f = ora_pdm_f(o, k);
    for (int i = 0; i <= f; ++i) {
      float *dst = cat + (size_t)i * d;
      /* an in-flight token's deepest eligible state H^{k L/n} is the residual stream it currently holds (the input of
       * its next stage; k = 0: the embedding row) — the capture below layer_forward stores it only when that stage runs */
      if (q >= o->c && o->pdm_anchor[i] == k * (c->n_layers / n)) memcpy(dst, o->r_h + (size_t)(q - o->c) * d, sizeof(float) * d);
      else memcpy(dst, o->anch + ((size_t)q * m + i) * d, sizeof(float) * d);
    }
    ora_op_gemv(o->pw.fc[f], d, (f + 1) * d, cat, o->pdm_x + (size_t)r * d);
  }
  free(cat);
  memcpy(o->pdm_g, o->pdm_x, sizeof(float) * (size_t)rows * d);
  /* the PDM decoder over those rows, layer by layer, rows in position order (causal); every row rewrites its K/V row
   * of the PDM cache (the trailing features are refreshed on every advance) */
  layer_set S = pdm_set(o);
  for (int l = 0; l < o->pw.n_layers; ++l)
    for (int r = 0; r < rows; ++r)
      if (layer_forward_set(o, &S, l, o->pdm_x + (size_t)r * d, first + r)) return -1;
  o->pdm_final = o->c;   /* rows below c were built at depth n: final */
  /* independent head on the last position (Eq. 1), reduced vocabulary */
  memcpy(o->pdm_h, o->pdm_x + (size_t)(rows - 1) * d, sizeof(float) * d);
  ora_op_rmsnorm(o->pdm_h, o->pw.final_norm, d, c->rms_eps, o->z);
  ora_op_gemv(o->pw.head, o->pw.vocab, d, o->z, o->pdm_lg);
  top2_margin(o->pdm_lg, o->pw.vocab, &o->gap[1], &o->maxabs[1]);
  int idx = ora_op_argmax(o->pdm_lg, o->pw.vocab);
  int hint_idx = -1;
  if (draft_hint >= 0)
    for (int i = 0; i < o->pw.vocab; ++i)
      if (o->pw.vocab_map[i] == draft_hint) hint_idx = i;
  idx = apply_hint(o->pdm_lg, idx, hint_idx, o->pw.vocab, band, &o->ties[1]);
  return o->pw.vocab_map[idx];
}

void ora_pdm_get_anchor(const ora_ctx *o, int32_t pos, int32_t i, float *out) {
  memcpy(out, o->anch + ((size_t)pos * o->pdm_m + i) * o->cfg.d_model, 4 * (size_t)o->cfg.d_model);
}

void ora_pdm_get_last(const ora_ctx *o, int32_t what, float *out) {
  if (what == 0) memcpy(out, o->pdm_lg, 4 * (size_t)o->pw.vocab);
  else if (what == 1) memcpy(out, o->pdm_h, 4 * (size_t)o->cfg.d_model);
  else if (what == 2) memcpy(out, o->pdm_g, 4 * (size_t)o->pdm_rows * o->cfg.d_model);
}

void ora_pdm_last_rows(const ora_ctx *o, int32_t *first_pos, int32_t *rows, int32_t *depths) {
  if (first_pos) *first_pos = o->pdm_first;
  if (rows) *rows = o->pdm_rows;
  if (depths) memcpy(depths, o->pdm_depth, 4 * (size_t)o->pdm_rows);
}

void ora_pdm_get_kv(const ora_ctx *o, int32_t layer, int32_t which, int32_t rows, uint16_t *out, int32_t *final_len) {
  size_t row = kv_row(&o->cfg);
  const uint16_t *src = (which ? o->pvc : o->pkc) + (size_t)layer * o->cfg.max_seq * row;
  memcpy(out, src, 2 * row * (size_t)rows);
  if (final_len) *final_len = o->pdm_final;
}

/* One SPD cycle — "Step" of C-1, in the paper's order: (1) read the ring, (2) PDM on PRE-step
 * features, (3) every in-flight token runs its own stage's layer slice
 * (PAPER.md:67-69), (4) the oldest token exits, its logits judge its successor,
 * accept -> the draft enters stage 1; reject -> truncate KV, flush, reseed,
 * (5) no exit (warm-up): the draft simply enters. */
int ora_step(ora_ctx *o, int32_t draft_override, ora_step_result *out) {
  return ora_step_follow(o, draft_override, -1, -1, 0.f, out);
}

/* A tie hint (test hook): `hint` is the token the CUDA path chose.  If it
 * is not the oracle's argmax but its oracle logit lies within `band` (ABSOLUTE, in logit units: the test
 * passes a small multiple of the logit difference it measured between the two implementations) of the
 * oracle's maximum, both are valid choices at that measured difference: the oracle continues with the hint
 * and counts a tie.  band <= 0, an out-of-range hint, or a hint further below the maximum: the oracle
 * keeps its own argmax (and the caller reports the mismatch). */
static int apply_hint(const float *logits, int own, int hint, int vocab, float band, int32_t *ties) {
  if (hint < 0 || hint >= vocab || hint == own || !(band > 0.f)) return own;
  if (logits[own] - logits[hint] <= band) { *ties += 1; return hint; }
  return own;
}

static int step_impl(ora_ctx *o, int32_t draft_override, int32_t draft_hint, int32_t verify_hint, float band,
                     const ora_sample_hints *sh, ora_step_result *out);

/* The same cycle with tie hints for the PDM argmax and the verify argmax (either may be -1). */
int ora_step_follow(ora_ctx *o, int32_t draft_override, int32_t draft_hint, int32_t verify_hint, float band,
                    ora_step_result *out) {
  return step_impl(o, draft_override, draft_hint, verify_hint, band, NULL, out);
}

/* Sampling mode with the CUDA path's decisions as hints (NULL: none). */
int ora_step_sample_follow(ora_ctx *o, int32_t draft_override, const ora_sample_hints *hints, ora_step_result *out) {
  if (!o->sampling_on) return -1;
  return step_impl(o, draft_override, -1, -1, 0.f, hints, out);
}

static int step_impl(ora_ctx *o, int32_t draft_override, int32_t draft_hint, int32_t verify_hint, float band,
                     const ora_sample_hints *sh, ora_step_result *out) {
  const ora_config *c = &o->cfg;
  int d = c->d_model, n = c->n_stages, L = c->n_layers, per = L / n;
  if (!o->prefilled) return -1;
  /* 1 */
  int a = o->a;
  int p_new = o->r_pos[a - 1];
  if (p_new + 1 >= c->max_seq) return -3; /* capacity: the draft would need row p_new+1 next step */
  o->steps += 1;
  ora_step_result r;
  memset(&r, 0, sizeof r);
  r.step_index = (int32_t)o->steps;
  r.fill = a;
  r.emitted_token = -1;

  /* 2: slot j <-> position p_new - j <-> depth j (C-2.2).  In-flight token: its state before this
   * step's forward (C-2.5; depth 0 = the bare embedding row).  Committed token: Hfin (Eq. 5, C-2.4).
   * Negative position: zero vector. */
  for (int j = 0; j < n; ++j) {
    float *f = o->pdm_feat + (size_t)j * d;
    int q = p_new - j;
    if (j < a) memcpy(f, o->r_h + (size_t)(a - 1 - j) * d, sizeof(float) * d);
    else if (q >= 0) memcpy(f, o->hfin + (size_t)q * d, sizeof(float) * d);
    else memset(f, 0, sizeof(float) * d);
  }
  int draft;
  if (o->pdm_on) {   /* NEXT-1: the paper's PDM replaces the simplified one (same pre-step schedule) */
    draft = pdm_paper_draft(o, draft_hint, band);
    if (draft < 0) return -2;
  } else {
    ora_op_gemv(o->w.pdm_proj, d, n * d, o->pdm_feat, o->pdm_u);
    draft = head_argmax(o, o->pdm_u, o->w.pdm_norm, o->pdm_logits, 1);
    draft = apply_hint(o->pdm_logits, draft, draft_hint, c->vocab, band, &o->ties[1]);
  }
  ora_dist Qd; /* the distribution the entering draft is drawn from (sampling mode) */
  memset(&Qd, 0, sizeof Qd);
  if (o->sampling_on) { /* x^ ~ Q_t = filtered PDM distribution (S-2, S-3; j = 0) */
    double w[ORA_MAX_TOPK];
    head_dist(o, o->pdm_logits, sh && sh->draft_k ? sh->draft_ids : NULL, sh ? sh->draft_k : 0,
              sh ? sh->logit_band : 0.f, &Qd);
    o->rec.draft = Qd;
    memset(&o->rec.target, 0, sizeof o->rec.target);
    o->rec.u_draft = ora_op_uniform(o->samp_seed, o->steps, 0);
    o->rec.u_accept = o->rec.u_resid = -1.0;
    o->rec.succ_token = -1; o->rec.succ_q = o->rec.succ_p = 0.f;
    for (int i = 0; i < Qd.k; ++i) w[i] = (double)Qd.p[i];
    draft = draw_with_hint(Qd.id, w, Qd.k, o->rec.u_draft, sh ? sh->draft_token : -1,
                           sh ? (double)sh->prob_eps : 0.0, &o->rec.ties_draft);
    if (draft_override >= 0) { /* a deterministic drafter: Q = one-hot on the override */
      memset(&Qd, 0, sizeof Qd);
      Qd.k = 1; Qd.id[0] = draft_override; Qd.p[0] = 1.f;
    }
  }
  if (o->forced_on) {
    uint64_t draw = ora_op_splitmix64(o->forced_seed + (uint64_t)o->steps) >> 11;
    int ti = p_new + 1 - o->prompt_len;
    if (draw < o->forced_thresh && ti >= 0 && ti < o->n_truth) { draft = o->truth[ti]; r.draft_forced = 1; }
  }
  if (draft_override >= 0) draft = draft_override;
  r.draft_token = draft;

  /* 3: the in-flight tokens touch disjoint layer slices, so their order is irrelevant. */
  for (int ii = 0; ii < a; ++ii) {
    int i = o->reverse_forward ? a - 1 - ii : ii;
    int k = o->r_k[i];
    for (int l = k * per; l < (k + 1) * per; ++l)
      if (layer_forward(o, l, o->r_h + (size_t)i * d, o->r_pos[i])) return -2;
    o->r_k[i] = k + 1;
  }

  /* 4 */
  if (o->r_k[0] == n) {
    int e_pos = o->r_pos[0];
    memcpy(o->hfin + (size_t)e_pos * d, o->r_h, sizeof(float) * d);
    o->c = e_pos + 1;
    int y = head_argmax(o, o->r_h, o->w.final_norm, o->exit_logits, 0);
    y = apply_hint(o->exit_logits, y, verify_hint, c->vocab, band, &o->ties[0]);
    o->emitted += 1;
    r.exited = 1;
    /* pop the oldest */
    for (int i = 1; i < a; ++i) {
      o->r_pos[i - 1] = o->r_pos[i]; o->r_tok[i - 1] = o->r_tok[i]; o->r_k[i - 1] = o->r_k[i];
      o->r_q[i - 1] = o->r_q[i];
      memcpy(o->r_h + (size_t)(i - 1) * d, o->r_h + (size_t)i * d, sizeof(float) * d);
    }
    a -= 1;
    int succ = a > 0 ? o->r_tok[0] : draft; /* n = 1: the successor is the draft itself (C-2.12) */
    int ok = succ == y;                     /* greedy: exact argmax match */
    if (o->sampling_on) {                   /* sampling: standard rejection sampling */
      const ora_dist *Qs = a > 0 ? &o->r_q[0] : &Qd;
      ora_dist *Pt = &o->rec.target;
      head_dist(o, o->exit_logits, sh && sh->verify_k ? sh->verify_ids : NULL, sh ? sh->verify_k : 0,
                sh ? sh->logit_band : 0.f, Pt);
      double eps = sh ? (double)sh->prob_eps : 0.0;
      double qx = dist_prob(Qs, succ), px = dist_prob(Pt, succ);
      o->rec.succ_token = succ; o->rec.succ_q = (float)qx; o->rec.succ_p = (float)px;
      o->rec.u_accept = ora_op_uniform(o->samp_seed, o->steps, 1);
      ok = ora_op_accept(Pt, Qs, succ, o->rec.u_accept);
      if (sh && sh->accepted >= 0 && sh->accepted != ok && fabs(o->rec.u_accept * qx - px) <= eps * qx) {
        ok = sh->accepted;
        o->rec.ties_accept += 1;
      }
      if (ok) {
        y = succ;
      } else {
        double w[ORA_MAX_TOPK], W = 0.0;
        residual_weights(Pt, Qs, w);
        for (int i = 0; i < Pt->k; ++i) W += w[i];
        o->rec.u_resid = ora_op_uniform(o->samp_seed, o->steps, 2);
        y = draw_with_hint(Pt->id, w, Pt->k, o->rec.u_resid, sh ? sh->emitted_token : -1, eps / W,
                           &o->rec.ties_resid);
      }
    }
    r.emitted_token = y;
    if (ok) {
      r.accepted = 1;
      o->r_pos[a] = p_new + 1; o->r_tok[a] = draft; o->r_k[a] = 0;
      o->r_q[a] = Qd;
      embed_row(o, draft, o->r_h + (size_t)a * d);
      o->a = a + 1;
    } else {
      r.accepted = 0;
      r.discarded = a;
      for (int l = 0; l < L; ++l)
        if (o->len[l] > o->c) o->len[l] = o->c;
      ring_set_single(o, o->c, y); /* the draft is dropped (C-2.10) */
    }
  } else {
    /* 5 */
    o->r_pos[a] = p_new + 1; o->r_tok[a] = draft; o->r_k[a] = 0;
    o->r_q[a] = Qd;
    embed_row(o, draft, o->r_h + (size_t)a * d);
    o->a = a + 1;
  }
  r.committed_len = o->c;
  if (out) *out = r;
  return 0;
}

int ora_rollback(ora_ctx *o, int32_t new_len, int32_t reseed_token) {
  if (!o->prefilled) return -1;
  if (new_len < 0 || new_len > o->c || reseed_token < 0 || reseed_token >= o->cfg.vocab) return -1;
  o->c = new_len;
  if (o->pdm_final > new_len) o->pdm_final = new_len;
  o->emitted = new_len - o->prompt_len + 1; /* tokens emitted up to and including the reseed token */
  if (o->emitted < 1) o->emitted = 1;       /* a rollback into the prompt: the reseed token is the first emitted one */
  for (int l = 0; l < o->cfg.n_layers; ++l)
    if (o->len[l] > new_len) o->len[l] = new_len;
  ring_set_single(o, new_len, reseed_token);
  return 0;
}

/* O-AR: plain greedy decode, one token through all L layers (the single-GPU autoregressive
 * baseline of PAPER.md:145).  The pending token is ring entry 0 left by ora_prefill. */
int ora_ar_step(ora_ctx *o, int32_t *next_token) {
  const ora_config *c = &o->cfg;
  int d = c->d_model;
  if (!o->prefilled || o->a != 1 || o->r_k[0] != 0) return -1;
  int pos = o->r_pos[0];
  if (pos + 1 >= c->max_seq) return -3;
  float *h = o->r_h;
  if (o->ar_trace) memcpy(o->ar_trace, h, sizeof(float) * d);
  for (int l = 0; l < c->n_layers; ++l) {
    if (layer_forward(o, l, h, pos)) return -2;
    if (o->ar_trace) memcpy(o->ar_trace + (size_t)(l + 1) * d, h, sizeof(float) * d);
  }
  memcpy(o->hfin + (size_t)pos * d, h, sizeof(float) * d);
  o->c = pos + 1;
  int y = head_argmax(o, h, o->w.final_norm, o->exit_logits, 0);
  o->steps += 1;
  o->emitted += 1;
  ring_set_single(o, pos + 1, y);
  if (next_token) *next_token = y;
  return 0;
}

void ora_ar_set_trace(ora_ctx *o, float *trace) { o->ar_trace = trace; }
void ora_set_forward_order(ora_ctx *o, int32_t reverse) { o->reverse_forward = reverse; }

/* ------------------------------------------------------------------ readers ------------------- */

int32_t ora_committed_len(const ora_ctx *o) { return o->c; }
int32_t ora_fill(const ora_ctx *o) { return o->a; }
int64_t ora_steps(const ora_ctx *o) { return o->steps; }
int32_t ora_emitted(const ora_ctx *o) { return o->emitted; }
void ora_get_kv_len(const ora_ctx *o, int32_t *len) { memcpy(len, o->len, 4 * (size_t)o->cfg.n_layers); }

void ora_get_kv(const ora_ctx *o, int32_t layer, int32_t which, int32_t rows, uint16_t *out) {
  size_t row = kv_row(&o->cfg);
  const uint16_t *src = (which ? o->vc : o->kc) + (size_t)layer * o->cfg.max_seq * row;
  memcpy(out, src, 2 * row * (size_t)rows);
}

int ora_get_ring(const ora_ctx *o, int32_t i, int32_t *pos, int32_t *tok, int32_t *k, float *hidden) {
  if (i < 0 || i >= o->a) return -1;
  if (pos) *pos = o->r_pos[i];
  if (tok) *tok = o->r_tok[i];
  if (k) *k = o->r_k[i];
  if (hidden) memcpy(hidden, o->r_h + (size_t)i * o->cfg.d_model, 4 * (size_t)o->cfg.d_model);
  return 0;
}

void ora_get_hfin(const ora_ctx *o, int32_t pos, float *out) {
  memcpy(out, o->hfin + (size_t)pos * o->cfg.d_model, 4 * (size_t)o->cfg.d_model);
}

void ora_get_last(const ora_ctx *o, int32_t what, float *out) {
  const ora_config *c = &o->cfg;
  if (what == 0) memcpy(out, o->exit_logits, 4 * (size_t)c->vocab);
  else if (what == 1) memcpy(out, o->pdm_logits, 4 * (size_t)c->vocab);
  else if (what == 2) memcpy(out, o->pdm_u, 4 * (size_t)c->d_model);
  else if (what == 3) memcpy(out, o->pdm_feat, 4 * (size_t)c->d_model * c->n_stages);
}

void ora_get_ties(const ora_ctx *o, int32_t *verify_ties, int32_t *pdm_ties) {
  *verify_ties = o->ties[0];
  *pdm_ties = o->ties[1];
}

void ora_get_margin(const ora_ctx *o, int32_t which, float *gap, float *maxabs) {
  *gap = o->gap[which & 1];
  *maxabs = o->maxabs[which & 1];
}

/* ------------------------------------------------------------------ timing-only helpers ------- */

void ora_load_kv(ora_ctx *o, int32_t layer, const uint16_t *k, const uint16_t *v, int32_t rows) {
  size_t row = kv_row(&o->cfg);
  memcpy(o->kc + (size_t)layer * o->cfg.max_seq * row, k, 2 * row * (size_t)rows);
  memcpy(o->vc + (size_t)layer * o->cfg.max_seq * row, v, 2 * row * (size_t)rows);
}

int ora_assume_prefilled(ora_ctx *o, int32_t committed_len, int32_t first_token) {
  if (committed_len < 1 || committed_len >= o->cfg.max_seq) return -1;
  for (int l = 0; l < o->cfg.n_layers; ++l) o->len[l] = committed_len;
  o->c = committed_len;
  o->prompt_len = committed_len;
  o->steps = 0;
  o->emitted = 1;
  o->prefilled = 1;
  ring_set_single(o, committed_len, first_token);
  return 0;
}
