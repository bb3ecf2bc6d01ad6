/* spd_oracle.h — CPU oracle for one Speculative Pipeline Decoding (SPD) step.
 *
 * TEST INFRASTRUCTURE ONLY.  This is the plain, slow, obviously-correct implementation the CUDA
 * path is checked against.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` legs may call it.  It shares no code, header, table or helper with the CUDA
 * library (include/spd.h, paper_2605_30852_b200/csrc/); the two only ever see the same input bytes.
 *
 * What it computes (citations are /root/reference/PAPER.md lines; "C-x.y" are the readings listed in
 * SURVEY.md §8(c) and DESIGN.md):
 *   O-AR   plain greedy token-by-token decode of the dense decoder with a KV cache — the sequence
 *          every greedy SPD run must reproduce (PAPER.md:125 "lossless", :129 "exact argmax match").
 *   O-SPD  the SPD cycle, step by step: n-stage token pipeline, pre-step Pipeline
 *          Draft Module on the depth staircase (PAPER.md:77-85 Eq.1-2, :102-107 Eq.5, :115),
 *          streaming greedy verification and rollback; with
 *          ora_set_sampling, verification by standard rejection sampling —
 *          pinned by tests/test_oracle_sampling.py (library softmax, the lossless identity measured in u,
 *          top_k = 1 == greedy, the exact autoregressive sampling law on a micro decoder).
 *
 * Numeric contract (C-2.17): every tensor is fp32 except K/V cache rows, which are rounded to bf16
 * (round-to-nearest-even) when appended; weights are bf16 widened exactly.  Every reduction (dot
 * product, sum of squares, softmax denominator, weighted V sum) is accumulated in fp64 and rounded
 * to fp32 once, so the oracle's fp32 tensors are the correctly-rounded values of the contract.
 *
 * Parity pins: see tests/test_oracle_*.py.  The simplified PDM (linear n*d->d + RMSNorm + tied
 * head, BASELINE.json) has no counterpart in the paper: draft-token parity vs the paper is
 * UNPINNED ("parity unpinned"); it is pinned only as a pure function of its n slot vectors.
 * The paper's own PDM (ora_pdm_attach, NEXT-1) is pinned by tests/test_oracle_pdm.py: a float64 whole-prefix
 * numpy model of the PDM decoder over the feature sequence (no cache), the anchors against O-AR's per-layer
 * trace, f(k) against Eq. 3 by brute force, the staircase layouts of Eq. 2 / Eq. 5, lossless-ness unchanged.
 */
#ifndef SPD_ORACLE_H
#define SPD_ORACLE_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t d_model, n_layers, n_stages, n_q_heads, n_kv_heads, head_dim, d_ffn, vocab, max_seq;
  float rms_eps, rope_base;
} ora_config;

/* All pointers are HOST pointers to bf16 bit patterns, row-major [out, in]; borrowed. */
typedef struct {
  const uint16_t *embed;                 /* [V, d]  tied: embedding = LM head = PDM head (C-2.3) */
  const uint16_t *const *attn_norm;      /* [L] -> [d]            */
  const uint16_t *const *wq;             /* [L] -> [Hq*hd, d]     */
  const uint16_t *const *wk;             /* [L] -> [Hkv*hd, d]    */
  const uint16_t *const *wv;             /* [L] -> [Hkv*hd, d]    */
  const uint16_t *const *wo;             /* [L] -> [d, Hq*hd]     */
  const uint16_t *const *mlp_norm;       /* [L] -> [d]            */
  const uint16_t *const *w_gate;         /* [L] -> [F, d]         */
  const uint16_t *const *w_up;           /* [L] -> [F, d]         */
  const uint16_t *const *w_down;         /* [L] -> [d, F]         */
  const uint16_t *final_norm;            /* [d]                   */
  const uint16_t *pdm_proj;              /* [d, n*d]; column block j multiplies the depth-j slot  */
  const uint16_t *pdm_norm;              /* [d]                   */
} ora_weights;

typedef struct {
  int32_t step_index, fill, exited, accepted, emitted_token, draft_token, draft_forced, discarded,
      committed_len;
} ora_step_result;

typedef struct ora_ctx ora_ctx;

ora_ctx *ora_create(const ora_config *cfg, const ora_weights *w);
void ora_destroy(ora_ctx *);

/* Prefill: token-by-token through all L layers.  block<=1: the plain path;
 * block>1: prompt tokens are processed `block` at a time per layer so weight rows are reused —
 * per-token arithmetic and its order are unchanged (tested bitwise against block=1). */
int ora_prefill(ora_ctx *, const int32_t *tokens, int32_t n_tokens, int32_t block, int32_t *first_token);

/* O-SPD: one cycle.  draft_override >= 0 replaces the PDM's token for this step (adversarial-draft
 * tests); -1 keeps the PDM / forced-acceptance token. */
int ora_step(ora_ctx *, int32_t draft_override, ora_step_result *out);
/* The same cycle with tie hints (test hook): draft_hint / verify_hint are
 * the tokens the CUDA path chose (-1: none).  A hint that is not the oracle's argmax but whose oracle
 * logit is within `band` of the oracle's maximum is adopted and counted by ora_get_ties; any other hint is
 * ignored.  `band` is ABSOLUTE (logit units): the caller passes a small multiple of the logit difference it
 * MEASURED between the two implementations, so a hint is adopted only where that difference can flip the
 * argmax; band <= 0 never adopts.  Pinned by tests/test_oracle_model.py::test_tie_hint_*. */
int ora_step_follow(ora_ctx *, int32_t draft_override, int32_t draft_hint, int32_t verify_hint, float band,
                    ora_step_result *out);
void ora_get_ties(const ora_ctx *, int32_t *verify_ties, int32_t *pdm_ties);
/* External truncate + flush + reseed with c := new_len. */
int ora_rollback(ora_ctx *, int32_t new_len, int32_t reseed_token);
/* Forced acceptance (C-2.19): force <=> (splitmix64(seed + K) >> 11) < floor(p * 2^53); p<0 disables.
 * truth[i] is the token at absolute position prompt_len + i. */
int ora_set_forced(ora_ctx *, const int32_t *truth, int32_t n_truth, float p, uint64_t seed);

/* O-AR: after ora_prefill, run the pending token (position c) through all L layers, commit it, and
 * return the next greedy token.  Never mixed with ora_step on the same ctx. */
int ora_ar_step(ora_ctx *, int32_t *next_token);
/* Optional trace for the in-flight-state pin: when set (non-NULL), ora_ar_step writes the residual
 * stream of the token it runs after every layer: trace[(layer+1)*d .. ] and trace[0..d) = embedding. */
void ora_ar_set_trace(ora_ctx *, float *trace /* [(L+1)*d] */);

/* Test hook for the independence pin: run step 3's in-flight tokens newest-first instead of
 * oldest-first (they touch disjoint layer slices, so the state must come out bitwise identical). */
void ora_set_forward_order(ora_ctx *, int32_t reverse);

/* State readers. */
int32_t ora_committed_len(const ora_ctx *);
int32_t ora_fill(const ora_ctx *);
int64_t ora_steps(const ora_ctx *);
int32_t ora_emitted(const ora_ctx *);
void ora_get_kv_len(const ora_ctx *, int32_t *len /* [L] */);
/* K or V rows of one layer as bf16 bits, [rows, Hkv*hd]. */
void ora_get_kv(const ora_ctx *, int32_t layer, int32_t which /*0=K,1=V*/, int32_t rows, uint16_t *out);
/* ring entry i (0 = oldest): pos, tok, depth k; hidden [d] (may be NULL). */
int ora_get_ring(const ora_ctx *, int32_t i, int32_t *pos, int32_t *tok, int32_t *k, float *hidden);
void ora_get_hfin(const ora_ctx *, int32_t pos, float *out /* [d] */);
/* Last computed: what 0 = exit (verify) logits [V], 1 = PDM logits [V], 2 = PDM pre-norm u [d],
 * 3 = PDM slot features [n*d] (slot j = depth j). */
void ora_get_last(const ora_ctx *, int32_t what, float *out);
/* top1-top2 gap and max|logit| of the last verify (which=0) / PDM (which=1) argmax (C-4). */
void ora_get_margin(const ora_ctx *, int32_t which, float *gap, float *maxabs);

/* ---- NEXT-1: the paper's Pipeline Draft Module (readings P-1..P-9 of DESIGN.md section 14) ----
 * PAPER.md:71 "an L_s-layer Transformer decoder f_theta with an independent LM head W_lm"; :77-85 Eq. 1-2 the
 * depth-conditioned feature sequence G_t and the depth staircase; :91-100 Eq. 3-4 multi-depth feature aggregation
 * (anchors B with b_0 = 0, l_max(k) = min(L, k L/n), f(k) = max{i | b_i <= l_max(k)},
 * g_t^k = FC_f(k)(Concat(H_t^b0 .. H_t^bf(k)))); :102-107 Eq. 5 warm-up layout; :115 pre-step features; :139 reduced
 * vocabulary head; :299 App. A.1 PDM KV cache ("caching appends only the trailing (n+1) refreshed features each step").
 *
 * One cycle's draft (replaces the simplified PDM when attached):
 *   rows q = F .. p_new, F = positions whose cached PDM rows are already final (depth n), p_new = newest position;
 *   depth k(q) = n for committed q < c, else the in-flight token's completed stages BEFORE this cycle's forward;
 *   g_q = FC_f(k(q)) . Concat(H_q^b0 .. H_q^bf) (H^b = the target's residual stream entering layer b; H^0 = E[tok]);
 *   the L_s PDM layers (the target's layer structure, C-2.13, own weights) run over those rows in position order, each
 *   row rewriting its K/V row of the PDM cache and attending rows 0 .. q; then F := c;
 *   x^ = vocab_map[argmax(W_lm . RMSNorm(h_last; g_pdm))].
 * Tensors fp32, reductions fp64, K/V rows bf16 — the same numeric contract as the target (C-2.17). */
#define ORA_PDM_MAX_ANCHORS 8
typedef struct {
  int32_t n_layers;                    /* L_s >= 1 */
  int32_t vocab;                       /* V_s <= V: rows of the independent head */
  const uint16_t *const *fc;           /* [m] -> [d, (i+1) d]: FC_i multiplies Concat(H^b0 .. H^bi) */
  const uint16_t *const *attn_norm, *const *wq, *const *wk, *const *wv, *const *wo, *const *mlp_norm, *const *w_gate,
      *const *w_up, *const *w_down;    /* [L_s] each, shapes as the target's */
  const uint16_t *final_norm;          /* [d] */
  const uint16_t *head;                /* [V_s, d] */
  const int32_t *vocab_map;            /* [V_s] draft index -> target token id, strictly ascending */
} ora_pdm_weights;
/* Attaches the paper's PDM (before ora_prefill).  -1: bad arguments or sampling is on (greedy only, reading P-9). */
int ora_pdm_attach(ora_ctx *, const ora_pdm_weights *);
/* The anchor set B of the ctx's L (reading P-1: [0, L/4, L/2, 3L/4, L-1], duplicates removed); returns m. */
int32_t ora_pdm_anchors(const ora_ctx *, int32_t *anchors /* [ORA_PDM_MAX_ANCHORS] */);
/* f(k) of Eq. 3 for the ctx's (L, n). */
int32_t ora_pdm_f(const ora_ctx *, int32_t k);
/* H_pos^{b_i} as captured by the target's forward (fp32 [d]). */
void ora_pdm_get_anchor(const ora_ctx *, int32_t pos, int32_t i, float *out);
/* Last PDM run: what 0 = logits [V_s], 1 = final hidden h_last [d] (pre-norm), 2 = features g of its rows [rows, d]. */
void ora_pdm_get_last(const ora_ctx *, int32_t what, float *out);
/* Rows of the last PDM run: first position, row count, per-row depth k (may be NULL). */
void ora_pdm_last_rows(const ora_ctx *, int32_t *first_pos, int32_t *rows, int32_t *depths);
/* K or V rows of one PDM layer as bf16 bits, [rows, Hkv*hd]; *final_len = F. */
void ora_pdm_get_kv(const ora_ctx *, int32_t layer, int32_t which, int32_t rows, uint16_t *out, int32_t *final_len);

/* ---- NEXT-2: sampling verification (readings S-1..S-10 of DESIGN.md §11) ----------
 * PAPER.md:129 "under sampling we apply standard rejection sampling"; PAPER.md:131 on a reject the
 * pipeline is reseeded "from x ~ P(x | x_1:t-n+1)"; "Sampling runs (T=1) use top-k=50 and
 * top-p=1.0".  Standard rejection sampling of speculative decoding: a token x drafted from Q is accepted
 * with probability min(1, P(x)/Q(x)); on a reject the replacement is drawn from norm(max(0, P - Q)), so
 * the emitted token is distributed exactly as P (pinned by enumeration in tests/test_oracle_sampling.py).
 *
 * S-2  filtered distribution of a logit vector l: support S = the top_k entries in the order (value
 *      descending, index ascending); p_i = exp((l_i - max l)/T) / Z on S (Z summed in fp64 in ascending
 *      token id, p rounded to fp32), 0 elsewhere.  Distributions list their support in ASCENDING TOKEN ID.
 * S-3  every draw is inverse-CDF over the support in ascending token id: the smallest i with
 *      u * W < w_0 + .. + w_i (fp64), W the total weight.
 * S-6  uniforms: u(seed, K, j) = (splitmix64(seed + 3 K + j) >> 40) * 2^-24, j = 0 draft, 1 accept,
 *      2 residual / first token; K = the cycle counter after its increment (0 at the prefill's final head). */
#define ORA_MAX_TOPK 64
typedef struct {
  int32_t k;
  int32_t id[ORA_MAX_TOPK]; /* ascending */
  float p[ORA_MAX_TOPK];
} ora_dist;

/* S-2.  support == NULL: the top_k set is selected here; otherwise `support` lists top_k distinct ids that
 * are used as the support as given (test hook: the CUDA path's set, validated by the caller). */
void ora_op_topk_softmax(const float *logits, int32_t vocab, int32_t top_k, float temperature,
                         const int32_t *support, ora_dist *out);
/* S-6 */
double ora_op_uniform(uint64_t seed, int64_t K, int32_t j);
/* S-3 on the distribution's own probabilities; returns the token id. */
int32_t ora_op_sample_cdf(const ora_dist *dist, double u);
/* Accept test of token x drafted from Q under target P: 1 iff u * Q(x) < P(x) (fp64 on the fp32
 * probabilities; a token outside a support has probability 0). */
int32_t ora_op_accept(const ora_dist *P, const ora_dist *Q, int32_t token, double u);
/* Residual draw: weights w_i = max(0, P(i) - Q(i)) over P's support (all zero -> w = P), S-3 with u. */
int32_t ora_op_sample_residual(const ora_dist *P, const ora_dist *Q, double u);

/* Enables sampling for the ctx (top_k < 1 disables = greedy).  1 <= top_k <= ORA_MAX_TOPK, T > 0.
 * Called before ora_prefill the first token is drawn from P as well (u(seed, 0, 2)); forced acceptance
 * and sampling are mutually exclusive (-1).  In sampling mode a cycle drafts x ~ Q_t (S-3, j = 0) and
 * keeps Q_t with the in-flight token; at the exit the successor is judged by ora_op_accept (j = 1) and
 * on a reject replaced by ora_op_sample_residual (j = 2); emitted_token = the accepted successor or the
 * replacement.  draft_override >= 0 acts as a deterministic drafter (Q = one-hot on the override). */
int ora_set_sampling(ora_ctx *, float temperature, int32_t top_k, uint64_t seed);

/* Test hook: what the CUDA path decided in this cycle.  A hint that differs
 * from the oracle's own decision is adopted only when the difference is implied by the logit difference
 * the test measured: a support is adopted iff min over it >= max over the rest - logit_band; a token /
 * accept bit iff the uniform lies within prob_eps (probability mass) of the oracle's decision boundary. */
typedef struct {
  int32_t draft_k, draft_ids[ORA_MAX_TOPK];   /* draft_k = 0: no support hint */
  int32_t verify_k, verify_ids[ORA_MAX_TOPK];
  int32_t draft_token, accepted, emitted_token; /* -1: no hint */
  float logit_band, prob_eps;
} ora_sample_hints;
typedef struct {
  ora_dist draft;   /* Q_t of the last cycle */
  ora_dist target;  /* P of the last exit (or of the prefill's final head) */
  double u_draft, u_accept, u_resid;
  int32_t succ_token;
  float succ_q, succ_p;
  int32_t ties_support, ties_draft, ties_accept, ties_resid; /* hints adopted so far */
} ora_sample_record;
int ora_step_sample_follow(ora_ctx *, int32_t draft_override, const ora_sample_hints *hints, ora_step_result *out);
void ora_get_sample_record(const ora_ctx *, ora_sample_record *out);

/* Timing-only helpers (bench cpu_baseline): load KV rows / declare a committed length without a
 * prefill.  Never used by a parity test. */
void ora_load_kv(ora_ctx *, int32_t layer, const uint16_t *k, const uint16_t *v, int32_t rows);
int ora_assume_prefilled(ora_ctx *, int32_t committed_len, int32_t first_token);

/* Single operations, exported for per-kernel parity. */
void ora_op_rmsnorm(const float *x, const uint16_t *gain, int32_t d, float eps, float *out);
void ora_op_gemv(const uint16_t *w, int32_t rows, int32_t k, const float *x, float *out);
void ora_op_rope(float *vec, int32_t n_heads, int32_t head_dim, int32_t pos, float base);
void ora_op_attention(const float *q, const uint16_t *kc, const uint16_t *vc, int32_t t_len,
                      int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, float *out);
void ora_op_silu_mul(const float *gate, const float *up, int32_t n, float *out);
int32_t ora_op_argmax(const float *x, int32_t n);
uint16_t ora_op_f32_to_bf16(float x);
uint64_t ora_op_splitmix64(uint64_t x);
int32_t ora_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
