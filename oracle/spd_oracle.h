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
 *          streaming greedy verification and rollback.
 *
 * Numeric contract (C-2.17): every tensor is fp32 except K/V cache rows, which are rounded to bf16
 * (round-to-nearest-even) when appended; weights are bf16 widened exactly.  Every reduction (dot
 * product, sum of squares, softmax denominator, weighted V sum) is accumulated in fp64 and rounded
 * to fp32 once, so the oracle's fp32 tensors are the correctly-rounded values of the contract.
 *
 * Parity pins: see tests/test_oracle_*.py.  The simplified PDM (linear n*d->d + RMSNorm + tied
 * head, BASELINE.json) has no counterpart in the paper: draft-token parity vs the paper is
 * UNPINNED ("parity unpinned"); it is pinned only as a pure function of its n slot vectors.
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
 * logit is within band * max|logit| of the oracle's maximum is adopted (both are valid at the stated
 * logit tolerance) and counted by ora_get_ties; any other hint is ignored. */
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
