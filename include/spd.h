/* spd.h — C ABI of the B200-native Speculative Pipeline Decoding (SPD) step library.
 *
 * One SPD pipeline step of a batch-1 sequence on one GPU (sm_100a).  Every step of the path runs in
 * this library's CUDA kernels; callers hand in plain pointers and sizes.  Citations "PAPER.md:<line>"
 * are lines of /root/reference/PAPER.md (arxiv/paper_2605_30852); "C-2.x" are the readings listed in
 * DESIGN.md ("Readings of the paper").
 *
 * The operation (PAPER.md:67-69 §3.1, :115 §3.3, :125-131 §3.4):
 *   The target decoder's L layers are split into n contiguous stages; up to n tokens of ONE sequence
 *   are in flight, the token that has completed k stages runs stage k this cycle.  A cycle
 *     1. drafts the next token with the Pipeline Draft Module (PDM) from PRE-step hidden states of
 *        the n most recent positions (slot j = position p_new - j at depth j; committed positions give
 *        their final hidden state, Eq. 5),
 *     2. runs every in-flight token through its stage's L/n layers (RMSNorm, QKV GEMV, RoPE, KV append,
 *        GQA attention over that layer's cache, O GEMV, RMSNorm, SwiGLU GEMVs),
 *     3. if the oldest token finished stage n: commits it, y = argmax(E . RMSNorm(h)) judges its
 *        in-flight successor; equal -> the draft enters stage 0; different -> every layer's KV length
 *        is truncated to the committed length, the pipeline is flushed and reseeded with y.
 *   Greedy by default: the emitted tokens equal plain greedy decoding ("lossless").
 *   spd_set_sampling switches step 3 to sampling verification ("under sampling we apply
 *   standard rejection sampling"): the emitted tokens are then distributed as sampling from the target.
 *
 * Numeric contract (C-2.17): weights bf16, every activation fp32 with fp32 accumulation, K/V cache
 * rows rounded to bf16 (round-to-nearest-even) when appended.  argmax = max value, lowest index (C-2.8).
 *
 * Memory and ownership: the library never allocates device memory.  The caller allocates three
 * device buffers of the sizes spd_query_sizes reports (any 256-byte aligned allocation, e.g.
 * torch.empty) plus two CUDA streams, and keeps them and all weight tensors alive until spd_destroy.
 * The ctx owns only host metadata, CUDA events/graphs and one small pinned host buffer.
 * Threading: one ctx is used from one host thread at a time.
 * Errors: every call returns spd_status; out-parameters are written only on SPD_OK; no exception or
 * foreign object crosses the ABI.  After SPD_ECUDA the ctx is unusable except for spd_last_error and
 * spd_destroy.  There is NO CPU fallback: without a CUDA device spd_create returns SPD_ECUDA.
 */
#ifndef SPD_H
#define SPD_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spd_ctx spd_ctx; /* opaque */

typedef enum {
  SPD_OK = 0,
  SPD_EINVAL = 1,    /* bad argument or unsupported configuration; state unchanged              */
  SPD_ESTATE = 2,    /* call out of order (e.g. spd_step before spd_prefill); state unchanged   */
  SPD_ECAPACITY = 3, /* the step would need a KV row >= max_seq; state unchanged                */
  SPD_ECUDA = 4,     /* a CUDA call failed or a device-side check fired; see spd_last_error     */
  SPD_ENOMEM = 5     /* a caller buffer is missing or too small                                 */
} spd_status;

/* Decoder shape (BASELINE.json configs; C-2.13: pre-norm, no biases, no QK-norm, GQA, SwiGLU, RoPE
 * rotate-half on all head dims, scale 1/sqrt(head_dim)).  Requirements (else SPD_EINVAL):
 * n_layers % n_stages == 0 (C-2.7), n_q_heads % n_kv_heads == 0, head_dim in {64, 128},
 * d_model, d_ffn, n_q_heads*head_dim multiples of 8, 1 <= n_stages <= 32, vocab >= 2, max_seq >= 2. */
typedef struct {
  int32_t d_model, n_layers, n_stages, n_q_heads, n_kv_heads, head_dim, d_ffn, vocab, max_seq;
  float rms_eps, rope_base;
  int32_t device; /* CUDA device ordinal */
} spd_config;

/* Weights: DEVICE pointers to bf16 bit patterns, row-major [out, in].  The nine per-layer members
 * are HOST arrays of n_layers DEVICE pointers (the arrays themselves are only read during
 * spd_create).  All tensors are borrowed until spd_destroy. */
typedef struct {
  const uint16_t *embed;            /* [vocab, d]  tied: input embedding = LM head = PDM head (C-2.3) */
  const uint16_t *const *attn_norm; /* [L] -> [d]                */
  const uint16_t *const *wq;        /* [L] -> [n_q_heads*hd, d]  */
  const uint16_t *const *wk;        /* [L] -> [n_kv_heads*hd, d] */
  const uint16_t *const *wv;        /* [L] -> [n_kv_heads*hd, d] */
  const uint16_t *const *wo;        /* [L] -> [d, n_q_heads*hd]  */
  const uint16_t *const *mlp_norm;  /* [L] -> [d]                */
  const uint16_t *const *w_gate;    /* [L] -> [d_ffn, d]         */
  const uint16_t *const *w_up;      /* [L] -> [d_ffn, d]         */
  const uint16_t *const *w_down;    /* [L] -> [d, d_ffn]         */
  const uint16_t *final_norm;       /* [d]                       */
  const uint16_t *pdm_proj;         /* [d, n*d]; column block j multiplies the depth-j slot (C-2.2) */
  const uint16_t *pdm_norm;         /* [d]                       */
} spd_weights;

typedef struct {
  size_t repack_bytes; /* streaming layout of the layer weights, written once by spd_create */
  size_t kv_bytes;     /* K/V cache, bf16, [layer][K|V][kv_head][max_seq][head_dim]          */
  size_t work_bytes;   /* step state, activations, hidden-state history, result ring         */
} spd_sizes;

typedef struct {
  void *repack, *kv, *work;        /* DEVICE, >= the sizes above, 256-byte aligned            */
  void *stream_main, *stream_pdm;  /* cudaStream_t handles (e.g. torch.cuda.Stream.cuda_stream) */
  size_t repack_bytes, kv_bytes, work_bytes; /* what the caller allocated: spd_create returns SPD_ENOMEM if any is
                                      smaller than spd_query_sizes reports (an undersized buffer never reaches a kernel) */
} spd_buffers;

/* What one cycle did.  step_index = K after the step (K counts cycles since prefill);
 * fill = tokens in flight when the step began; exited/accepted are 0/1; emitted_token is the verified
 * token y of an exit step (-1 otherwise); draft_token is what the PDM (or the forced rule) proposed;
 * discarded = in-flight tokens dropped by a reject (n-1 in saturation); committed_len = c after it. */
typedef struct {
  int32_t step_index, fill, exited, accepted, emitted_token, draft_token, draft_forced, discarded,
      committed_len;
} spd_step_result;

/* Engine options (spd_set_option). */
enum {
  SPD_OPT_ENGINE = 0,      /* 0 = one kernel per operation (reference engine), 1 = persistent fused step kernel, one stage
                              chain per CTA (spd_mega.cu), 2 = persistent fused step kernel with multiplexed stage chains
                              (spd_mega2.cu; default when available, else 1, else 0)                                  */
  SPD_OPT_DEBUG_LOGITS = 1,/* 1 = also write full verify/PDM logit vectors (for parity tests)    */
  SPD_OPT_PHASE_PROFILE = 2,/* 1 = the fused kernel records per-phase clock stamps (SPD_DBG_PHASE_PROFILE) */
  SPD_OPT_CHAINS = 4,      /* engine 2 only: stage chains a CTA serves in turn, 1..4 (default 2; 3 for n_stages > 8; results
                              do not depend on it)                                                                  */
  SPD_OPT_PREFILL = 3      /* 1 = batched tensor-core prefill (tcgen05 GEMMs over chunks of the prompt; default when the
                              configuration supports it: d_model, n_q_heads*head_dim, d_ffn multiples of 64),
                              0 = the prompt runs through the decode kernel, one token entering per cycle          */
};

/* spd_debug_read selectors.  `index` meaning in brackets. */
enum {
  SPD_DBG_SLOT_HIDDEN = 0, /* [depth k] fp32[d]: hidden state of the in-flight token at depth k     */
  SPD_DBG_EXIT_LOGITS = 1, /* fp32[vocab] of the last verify (needs SPD_OPT_DEBUG_LOGITS)           */
  SPD_DBG_PDM_LOGITS = 2,  /* fp32[vocab] of the last PDM   (needs SPD_OPT_DEBUG_LOGITS)           */
  SPD_DBG_PDM_PRENORM = 3, /* fp32[d]: u = W_p . concat(slots) of the last PDM                     */
  SPD_DBG_PDM_FEAT = 4,    /* fp32[n*d]: the slot vectors the last PDM read (slot j = depth j)     */
  SPD_DBG_KV_K = 5,        /* [layer] bf16 [rows, n_kv_heads*hd], rows = bytes / row size          */
  SPD_DBG_KV_V = 6,        /* [layer] same for V                                                   */
  SPD_DBG_KV_LEN = 7,      /* int32[L]: valid KV rows per layer (C-2.11)                           */
  SPD_DBG_RING = 8,        /* int32[2 + 3n]: fill a, committed c, then per depth k: occupied, pos, tok */
  SPD_DBG_HFIN = 9,        /* [position] fp32[d]: final hidden state of a committed position        */
  SPD_DBG_SAMPLE = 11,     /* spd_sample_record of the last cycle (needs spd_set_sampling)                */
  SPD_DBG_Q = 12,          /* [stage k] fp32[n_q_heads*hd]: q (after RoPE) of the token that ran stage k in the
                              last cycle, at that stage's LAST layer (k+1)*L/n - 1 (per-kernel attention parity)  */
  SPD_DBG_ATT = 13,        /* [stage k] fp32[n_q_heads*hd]: that layer's attention output (input of the O GEMV)   */
  SPD_DBG_CYCLE_TIMES = 14,/* uint64[1024][2]: %globaltimer (ns) at which the controller of the cycle with step_index K
                              began [(K-1) % 1024][0] (kernel entry of the fused engine) and finished [..][1]; the
                              difference of consecutive finish stamps of back-to-back cycles is the step latency   */
  SPD_DBG_PDM2_LOGITS = 15,/* fp32[V_s]: logits of the paper PDM's last draft (reduced vocabulary)                   */
  SPD_DBG_PDM2_HIDDEN = 16,/* fp32[d]: its last row's hidden state before the final norm                            */
  SPD_DBG_PDM2_RUN = 17,   /* int32[3]: first position, row count of the last draft, F (final rows)                 */
  SPD_DBG_PDM2_FEAT = 18,  /* [rows] fp32[rows, d]: the features g of those rows (Eq. 4)                             */
  SPD_DBG_PDM2_K = 19,     /* [PDM layer] bf16 [rows, n_kv_heads*hd] of the PDM's cache, rows = bytes / row size    */
  SPD_DBG_PDM2_V = 20,
  SPD_DBG_ANCHOR = 21,     /* [position * 8 + i] fp32[d]: H^{b_i} of that position                                  */
  SPD_DBG_PHASE_PROFILE = 10 /* uint64[160][168][6]: per (CTA, phase) clock stamps of the last fused cycle:
                              0 inputs ready, 1 activations staged, 2 tiles consumed, 3/4 producer issued the
                              phase's first/last tile (SM clock); 5 = %globaltimer at stamp 0; phase 167 holds
                              (clock, %globaltimer) after the schedule [0,1] and at kernel entry [2,3]; CTA 0 also
                              at the end of the controller [4,5] (needs SPD_OPT_PHASE_PROFILE)               */
};

/* Buffer sizes for a configuration.  SPD_EINVAL if the configuration is unsupported. */
int spd_query_sizes(const spd_config *cfg, spd_sizes *out);

/* Creates a context: validates, repacks the layer weights into `bufs->repack` (streaming layout of
 * the fused step kernel), zeroes the state.  Blocks until done. */
int spd_create(const spd_config *cfg, const spd_weights *w, const spd_buffers *bufs, spd_ctx **out);
int spd_destroy(spd_ctx *ctx);

/* Prefill (outside the paper's timed region): runs the prompt (HOST int32 ids,
 * 1 <= n_tokens < max_seq - 1) through all layers.  Default (SPD_OPT_PREFILL = 1): layer by layer over chunks of
 * 1024 prompt tokens — GEMMs with M = tokens on the tcgen05 tensor cores (fp32 activations as three bf16 parts, exact,
 * against the exact bf16 weights, fp32 accumulation in TMEM), causal GQA attention over the cache, the same RMSNorm /
 * RoPE / bf16 KV append / SwiGLU arithmetic as the step.  SPD_OPT_PREFILL = 0: the prompt runs through the step's
 * own kernel, n tokens pipelined over the n stages (one full weight sweep per token).  Either way, afterwards:
 * committed length = n_tokens, every layer holds n_tokens KV rows, the final hidden state of every prompt position is
 * kept (Eq. 5 warm-up features), *first_token = argmax of the last position's logits is the single in-flight
 * token, K = 0.  May be called again to start a new sequence. */
int spd_prefill(spd_ctx *ctx, const int32_t *tokens, int32_t n_tokens, int32_t *first_token);

/* One SPD cycle including verification and, on reject, the internal rollback.  Returns after the
 * result is on the host (one small D2H copy + stream sync). */
int spd_step(spd_ctx *ctx, spd_step_result *out);
/* n_steps cycles enqueued back to back (the state lives on the device), one sync at the end;
 * results[0..n_steps) in order.  SPD_ECAPACITY (nothing run) unless all n_steps are guaranteed to fit. */
int spd_step_many(spd_ctx *ctx, int32_t n_steps, spd_step_result *results);

/* External truncate + flush + reseed (PAPER.md:131 with c := new_len): every layer's KV length becomes
 * min(len, new_len), in-flight tokens are dropped, reseed_token becomes the single in-flight token at
 * position new_len.  0 <= new_len <= committed length, 0 <= reseed_token < vocab, else SPD_EINVAL.
 * O(L) integers; no KV data moves. */
int spd_rollback(spd_ctx *ctx, int32_t new_len, int32_t reseed_token);

/* Bench mode (north_star: controlled acceptance from random-init weights; C-2.19): at cycle K the
 * PDM's token is replaced by truth[p_new + 1 - prompt_len] iff
 * (splitmix64(seed + K) >> 11) < floor(p * 2^53) and that entry exists.  truth: HOST int32[n_truth],
 * copied.  p < 0 disables; p > 1 or n_truth > max_seq -> SPD_EINVAL. */
int spd_set_forced(spd_ctx *ctx, const int32_t *truth, int32_t n_truth, float p, uint64_t seed);

/* Sampling verification.  PAPER.md:129: "under sampling we apply standard rejection
 * sampling"; on a reject the pipeline is reseeded "from x ~ P(x | x_1:t-n+1)"; PAPER.md:141:
 * "Sampling runs (T=1) use top-k=50 and top-p=1.0".  With sampling on (1 <= top_k <= SPD_MAX_TOPK,
 * temperature > 0):
 *   - a logit vector l is filtered to its top_k entries (value descending, index ascending) with
 *     p = softmax(l / temperature) over them (sum in fp64, p in fp32); supports are listed in ascending token id;
 *   - the PDM's token is DRAWN from its filtered distribution Q_t, which stays with the in-flight token;
 *   - at the exit the successor x (drafted from Q) is accepted iff u * Q(x) < P(x), P the filtered exit
 *     distribution; a rejected x is replaced by a draw from norm(max(0, P - Q)) and the pipeline is flushed and
 *     reseeded with it (KV truncation as in the greedy path); emitted_token = x or the replacement;
 *   - spd_prefill draws first_token from P;
 *   - every draw is the inverse CDF in ascending token id in fp64 with the uniform
 *     u(seed, K, j) = (splitmix64(seed + 3 K + j) >> 40) * 2^-24, j = 0 draft, 1 accept, 2 replacement / first
 *     token, K = step_index of the cycle (0 in spd_prefill).
 * The emitted tokens are distributed exactly as autoregressive sampling from the filtered target (not
 * token-identical to any other run).  top_k < 1 switches back to greedy.  top_k = 1 is the greedy path.
 * Switched on in the middle of a sequence, the tokens already in flight count as deterministic drafts
 * (Q = one-hot: accepted with probability P(x)).
 * SPD_EINVAL: top_k > SPD_MAX_TOPK or temperature <= 0.  SPD_ESTATE: forced acceptance is on (and
 * spd_set_forced while sampling is on).  Logits must be finite.  May be called before or after spd_prefill. */
#define SPD_MAX_TOPK 64
typedef struct {
  int32_t k;
  int32_t id[SPD_MAX_TOPK]; /* ascending token id */
  float p[SPD_MAX_TOPK];
} spd_sample_dist;
/* What the sampler of the last cycle saw and decided (spd_debug_read(SPD_DBG_SAMPLE), parity tests). */
typedef struct {
  spd_sample_dist draft;   /* Q_t of this cycle's PDM (k = 0: the PDM did not run)                      */
  spd_sample_dist target;  /* P of this cycle's exit or of spd_prefill's final head (k = 0: no exit)    */
  float u_draft, u_accept, u_resid; /* -1: not drawn                                                    */
  int32_t succ_token;      /* the judged token (-1: none), its stored draft probability, its target probability */
  float succ_q, succ_p;
  int32_t exact_rounds;    /* selections of this cycle that took the exact k-round path (0..2)          */
  int32_t prefiltered;     /* selections served by the head pass's threshold list, no scan (0..2)       */
} spd_sample_record;
int spd_set_sampling(spd_ctx *ctx, float temperature, int32_t top_k, uint64_t seed);

/* ---- The paper's Pipeline Draft Module ----------------------------------------------------
 * PAPER.md:71 "an L_s-layer Transformer decoder f_theta with an independent LM head"; :91-100 Eq. 3-4 (anchors
 * B = [0, L/4, L/2, 3L/4, L-1] — [0, 8, 16, 24, 31] for L = 32 —, l_max(k) = min(L, k L/n), f(k) = max{i | b_i <= l_max(k)},
 * g_t^k = FC_f(k)(Concat(H_t^b0 .. H_t^bf(k))), H^b = the target's residual stream entering layer b); :102-107 Eq. 5;
 * :115 pre-step features; :139 reduced-vocabulary head; :299 the PDM's KV cache, whose trailing n + 1 rows are rewritten
 * every cycle.  Once attached it REPLACES the simplified PDM of spd_weights (pdm_proj / pdm_norm are then unused): every
 * cycle, before the stage forward, the rows F .. p_new (F = positions whose rows are final, p_new = newest position)
 * run through FC_f(k) and the L_s PDM layers (the target's layer structure C-2.13 with its own weights and its own
 * cache), the last row goes through RMSNorm(final_norm) and the head, and draft = vocab_map[argmax].  spd_prefill
 * also builds the prompt's full-depth rows; spd_rollback rewinds F.  Greedy verification only (spd_set_sampling then
 * returns SPD_ESTATE, reading P-9).  Weights: DEVICE pointers to bf16 bit patterns, row-major [out, in]; the per-layer
 * members and `fc` are HOST arrays of DEVICE pointers (read during spd_pdm_attach only); vocab_map is a DEVICE int32
 * array, strictly ascending target token ids.  Buffers: DEVICE, sizes from spd_pdm_query_sizes, 256-byte aligned,
 * caller-owned until spd_destroy.  Attach before spd_prefill (SPD_ESTATE afterwards); SPD_EINVAL on bad arguments. */
typedef struct spd_pdm_weights {
  int32_t n_layers;                 /* L_s >= 1 */
  int32_t vocab;                    /* V_s <= vocab */
  const uint16_t *const *fc;        /* [m] -> [d, (i+1) d], m = anchors (5 unless L < 8) */
  const uint16_t *const *attn_norm, *const *wq, *const *wk, *const *wv, *const *wo, *const *mlp_norm, *const *w_gate,
      *const *w_up, *const *w_down; /* [L_s] each, shapes as spd_weights */
  const uint16_t *final_norm;       /* [d] */
  const uint16_t *head;             /* [V_s, d] */
  const int32_t *vocab_map;         /* DEVICE int32[V_s] */
} spd_pdm_weights;
typedef struct {
  size_t kv_bytes;   /* the PDM's cache: bf16 [L_s][K|V][kv_head][max_seq][head_dim] */
  size_t work_bytes; /* row scratch, anchors H^b of every position [max_seq][m][d] fp32 */
} spd_pdm_sizes;
int spd_pdm_query_sizes(const spd_config *cfg, int32_t pdm_layers, int32_t pdm_vocab, spd_pdm_sizes *out);
int spd_pdm_attach(spd_ctx *ctx, const spd_pdm_weights *w, void *pdm_kv, void *pdm_work);

int spd_set_option(spd_ctx *ctx, int32_t option, int32_t value);
/* The option's current value (SPD_OPT_ENGINE: the engine that runs the next cycle; SPD_OPT_CHAINS: 0 when engine 2 is not
 * available for this configuration).  Returns SPD_OK / SPD_EINVAL. */
int spd_get_option(spd_ctx *ctx, int32_t option, int32_t *value);

/* Copies internal state to HOST memory (parity tests).  bytes must match the selector's size
 * (KV selectors: a multiple of the row size, at most max_seq rows). */
int spd_debug_read(spd_ctx *ctx, int32_t what, int32_t index, void *host_out, size_t bytes);

/* Counters since the last spd_prefill: cycles K, emitted tokens N (alpha = N/K), and the
 * number of this library's kernel launches since spd_create. */
int spd_get_counters(spd_ctx *ctx, int64_t *steps, int64_t *emitted, int64_t *kernel_launches);

/* Last error text of the ctx (never NULL; static string if ctx is NULL). */
const char *spd_last_error(const spd_ctx *ctx);

/* ---- single operations, for per-kernel parity tests (DEVICE pointers, launched on `stream`,
 *      asynchronous; the kernels are the reference engine's).  Return SPD_OK / SPD_EINVAL / SPD_ECUDA. */
/* out[i] = x[i] * rsqrt(mean(x^2) + eps) * gain[i] */
int spd_op_rmsnorm(const float *x, const uint16_t *gain, int32_t d, float eps, float *out, void *stream);
/* out = W x, W bf16 [rows, k] row-major, k % 8 == 0 */
int spd_op_gemv(const uint16_t *w, int32_t rows, int32_t k, const float *x, float *out, void *stream);
/* RoPE (C-2.14) in place on vec = n_heads heads of head_dim at position pos */
int spd_op_rope(float *vec, int32_t n_heads, int32_t head_dim, int32_t pos, float base, void *stream);
/* GQA decode attention of one token over t_len rows.  kc, vc: bf16 [n_kv_heads][t_stride][head_dim]
 * (the cache's head-major layout); scratch: fp32, >= spd_op_attention_scratch(...) bytes. */
int spd_op_attention(const float *q, const uint16_t *kc, const uint16_t *vc, int32_t t_len, int32_t t_stride,
                     int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, float *out, float *scratch,
                     void *stream);
size_t spd_op_attention_scratch(int32_t t_len, int32_t n_q_heads, int32_t head_dim);
/* spd_op_attention for callers that cannot allocate device memory (CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same operation (the stage forward's attention; fixed 128-row splits merged in
 * split order), same arguments minus `scratch` — the split partials live in a file-scope device array of
 * spd_op_attention_static_max_bytes() = 2 MiB inside the library (held by every GPU that loads the library until the
 * process exits).  q, kc, vc, out: DEVICE, caller-owned, layouts as spd_op_attention.  Allocates nothing (no cudaMalloc /
 * cudaFree / allocating library call).  Returns SPD_OK; SPD_EINVAL (bad argument); SPD_ECAPACITY when
 * ceil(t_len / 128) * n_q_heads * (head_dim + 2) * 4 bytes exceed the array (use spd_op_attention with a caller buffer);
 * SPD_ECUDA.  All calls on a device SHARE the array, which keeps the last call's contents (nothing needs to start at zero:
 * every slot is written before it is read); calls that overlap on the GPU (different streams without a dependency) race
 * on it — calls on one stream are ordered.  Asynchronous on `stream` like the other spd_op_* calls. */
int spd_op_attention_static(const float *q, const uint16_t *kc, const uint16_t *vc, int32_t t_len, int32_t t_stride,
                            int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, float *out, void *stream);
size_t spd_op_attention_static_max_bytes(void);
/* The prefill GEMM as one operation: y[M, N] = x[M, K] . W[N, K]^T, x fp32 (split exactly into three bf16 parts), W bf16 row-major,
 * y fp32, on the tcgen05 tensor cores.  K % 64 == 0, N % 4 == 0.  scratch: DEVICE, >= spd_op_gemm_scratch(M, K) bytes. */
int spd_op_gemm(const float *x, const uint16_t *w, int32_t m, int32_t n, int32_t k, float *y, void *scratch, void *stream);
size_t spd_op_gemm_scratch(int32_t m, int32_t k);
/* out[i] = silu(gate[i]) * up[i] */
int spd_op_silu_mul(const float *gate, const float *up, int32_t n, float *out, void *stream);
/* argmax with lowest-index ties of x[0..n); result int32 on the device */
int spd_op_argmax(const float *x, int32_t n, int32_t *out_index, void *stream);
/* The filtered distribution of spd_set_sampling: top_k + temperature softmax of x[0..n) into *out (DEVICE
 * spd_sample_dist).  use_candidates != 0: threshold scan seeded by 128 chunk maxima (the step's path);
 * 0: no candidates (the exact k-round selection when n > 2048).  scratch: DEVICE, >= spd_op_topk_scratch() bytes. */
int spd_op_topk_softmax(const float *x, int32_t n, int32_t top_k, float temperature, int32_t use_candidates,
                        spd_sample_dist *out, void *scratch, void *stream);
size_t spd_op_topk_scratch(void);

#ifdef __cplusplus
}
#endif
#endif
