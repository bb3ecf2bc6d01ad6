// spd_api.cu — the C ABI of include/spd.h: context, buffer map, prefill / step / rollback drivers.
// Host code only launches kernels and moves the small result structs; every step of the SPD path
// itself runs on the device.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../include/spd.h"
#include "spd_engine.h"
#include "spd_kernels.cuh"

using namespace spd;

struct spd_ctx {
  spd_config cfg;
  DevPtrs P;
  spd_buffers bufs;
  spd_sizes sizes;
  cudaStream_t sm, sp;
  cudaEvent_t ev_fork, ev_join;
  cudaGraphExec_t graph[3];
  int graph_tried[3];
  int engine;
  int has_mega, has_mega2;
  MegaPlan mega;
  Mega2Plan mega2;
  PdmPlan *pdm;            // the paper's PDM, if attached (spd_pdm_attach)
  int prefill_mode;        // 1: batched tensor-core prefill (spd_prefill.cu), 0: the decode kernel's prefill mode
  PrefillPlan *pf;
  StepResult *h_results;   // pinned
  StepState *h_state;      // pinned mirror
  int prefilled, dead;
  int forced_on, sampling_on;   // host mirrors (the two modes exclude each other)
  long long launches;
  long long launches_per_step[3];
  char err[512];
};

static const char *kNullCtxErr = "spd: null context";

static int fail(spd_ctx *c, int code, const char *fmt, const char *a = "") {
  if (c) snprintf(c->err, sizeof c->err, fmt, a);
  return code;
}

#define CU(call)                                                                              \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      ctx->dead = 1;                                                                          \
      snprintf(ctx->err, sizeof ctx->err, "CUDA error %s at %s:%d", cudaGetErrorString(e_), __FILE__, __LINE__); \
      return SPD_ECUDA;                                                                       \
    }                                                                                         \
  } while (0)

// ------------------------------------------------------------------ configuration -------------
static int validate(const spd_config *c) {
  if (!c) return 0;
  if (c->n_stages < 1 || c->n_stages > kMaxStages || c->n_layers < 1 || c->n_layers % c->n_stages) return 0;
  if (c->n_kv_heads < 1 || c->n_q_heads < 1 || c->n_q_heads % c->n_kv_heads) return 0;
  if (c->n_q_heads / c->n_kv_heads > 8) return 0;
  if (c->head_dim != 64 && c->head_dim != 128) return 0;
  if (c->d_model < 8 || c->d_model % 8 || c->d_ffn < 8 || c->d_ffn % 8) return 0;
  if (c->vocab < 2 || c->max_seq < 2) return 0;
  if (!(c->rms_eps >= 0.f) || !(c->rope_base > 0.f)) return 0;
  return 1;
}

static Dims make_dims(const spd_config *c) {
  Dims D;
  D.d = c->d_model; D.L = c->n_layers; D.n = c->n_stages; D.Hq = c->n_q_heads; D.Hkv = c->n_kv_heads;
  D.hd = c->head_dim; D.F = c->d_ffn; D.V = c->vocab; D.max_seq = c->max_seq; D.per = c->n_layers / c->n_stages;
  D.eps = c->rms_eps;
  return D;
}

// One pass over the work buffer: with base == nullptr it only measures.
struct Carver {
  char *base;
  size_t off;
  template <typename T> T *take(size_t count) {
    off = (off + 255) & ~(size_t)255;
    T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
    off += count * sizeof(T);
    return p;
  }
};

static size_t carve_work(const spd_config *c, void *base, DevPtrs *P, const uint16_t ***tables) {
  Dims D = make_dims(c);
  Carver cv{(char *)base, 0};
  int nsplit = (D.max_seq + kAttnSplit - 1) / kAttnSplit;
  size_t qd = (size_t)D.Hq * D.hd, kd = (size_t)D.Hkv * D.hd, n = D.n;
  DevPtrs Q;
  memset(&Q, 0, sizeof Q);
  Q.dim = D;
  Q.nsplit_max = nsplit;
  Q.st = cv.take<StepState>(1);
  Q.len = cv.take<int32_t>(D.L);
  Q.h = cv.take<float>(n * D.d);
  Q.x = cv.take<float>(n * D.d);
  Q.act = cv.take<float>(n * D.F);
  Q.q = cv.take<float>(n * qd);
  Q.kvtmp = cv.take<float>(n * 2 * kd);
  Q.att = cv.take<float>(n * qd);
  Q.part_o = cv.take<float>(n * D.Hq * nsplit * D.hd);
  Q.part_ml = cv.take<float2>(n * D.Hq * nsplit);
  Q.att_cnt = cv.take<int32_t>(n * D.Hq);
  Q.feat = cv.take<float>(n * D.d);
  Q.pdm_part = cv.take<float>(n * D.d);
  Q.pdm_u = cv.take<float>(D.d);
  Q.xv = cv.take<float>(D.d);
  Q.xp = cv.take<float>(D.d);
  Q.logits_v = cv.take<float>(D.V);
  Q.logits_p = cv.take<float>(D.V);
  Q.cand_val = cv.take<float>(2 * kMaxCand);
  Q.cand_idx = cv.take<int32_t>(2 * kMaxCand);
  Q.rope = cv.take<float2>(n * (D.hd / 2));
  Q.inv_freq = cv.take<double>(D.hd / 2);
  Q.hfin = cv.take<float>((size_t)D.max_seq * D.d);
  Q.truth = cv.take<int32_t>(D.max_seq);
  Q.pf_tokens = cv.take<int32_t>(D.max_seq);
  Q.results = cv.take<StepResult>(kResultRing);
  Q.cycle_ts = cv.take<unsigned long long>(2 * (size_t)kResultRing);
  Q.bar = cv.take<unsigned int>(kBarWords);
  Q.claim = cv.take<unsigned int>((size_t)kClaimPhases * kMaxStages);
  Q.prof = cv.take<unsigned long long>((size_t)kProfCtas * kProfPhases * kProfStamps);
  Q.samp = cv.take<SampleState>(1);
  Q.samp_val = cv.take<float>(kSampCap);
  Q.samp_idx = cv.take<int32_t>(kSampCap);
  Q.pre_val = cv.take<float>(2 * kSampCap);
  Q.pre_idx = cv.take<int32_t>(2 * kSampCap);
  if (prefill_supported(D)) {
    size_t mc = (size_t)prefill_chunk_tokens(D);
    size_t ymax = qd + 2 * kd > 2 * (size_t)D.F ? qd + 2 * kd : 2 * (size_t)D.F;
    if ((size_t)D.d > ymax) ymax = D.d;
    size_t xmax = (size_t)D.d > qd ? D.d : qd;
    if ((size_t)D.F > xmax) xmax = D.F;
    if (5 * (size_t)D.d > xmax) xmax = 5 * (size_t)D.d;   // the paper PDM's prefill: K = m d concatenated anchors (m <= 5)
    Q.pf_chunk = (int32_t)mc;
    Q.pf_H = cv.take<float>(mc * D.d);
    Q.pf_Q = cv.take<float>(mc * qd);
    Q.pf_Y = cv.take<float>(mc * ymax);
    Q.pf_plane = mc * xmax;
    Q.pf_x3 = cv.take<uint16_t>(3 * mc * xmax);
  }
  const uint16_t **tabs[9];
  for (int i = 0; i < 9; ++i) tabs[i] = cv.take<const uint16_t *>(D.L);
  Q.attn_norm = tabs[0]; Q.wq = tabs[1]; Q.wk = tabs[2]; Q.wv = tabs[3]; Q.wo = tabs[4];
  Q.mlp_norm = tabs[5]; Q.w_gate = tabs[6]; Q.w_up = tabs[7]; Q.w_down = tabs[8];
  if (P) *P = Q;
  if (tables) for (int i = 0; i < 9; ++i) tables[i] = tabs[i];
  return (cv.off + 255) & ~(size_t)255;
}

static size_t kv_bytes_of(const spd_config *c) {
  return (size_t)c->n_layers * 2 * c->n_kv_heads * c->max_seq * c->head_dim * sizeof(uint16_t);
}

extern "C" int spd_query_sizes(const spd_config *cfg, spd_sizes *out) {
  if (!validate(cfg) || !out) return SPD_EINVAL;
  spd_sizes s;
  s.work_bytes = carve_work(cfg, nullptr, nullptr, nullptr);
  s.kv_bytes = kv_bytes_of(cfg);
  s.repack_bytes = mega_repack_bytes(make_dims(cfg));
  *out = s;
  return SPD_OK;
}

// ------------------------------------------------------------------ small state kernels --------
namespace spd {
__global__ void k_state_init(DevPtrs P, int mode, int pf_n) {
  StepState *st = P.st;
  if (threadIdx.x == 0) {
    long long K = 0, N = 0;
    int forced_on = st->forced_on, n_truth = st->n_truth;
    unsigned long long th = st->forced_thresh, sd = st->forced_seed;
    memset(st, 0, sizeof(StepState));
    st->forced_on = forced_on; st->n_truth = n_truth; st->forced_thresh = th; st->forced_seed = sd;
    st->mode = mode; st->K = K; st->N = N; st->pf_n = pf_n; st->prompt_len = pf_n;
    for (int k = 0; k < kMaxStages; ++k) st->hbuf[k] = k;
  }
  for (int l = threadIdx.x; l < P.dim.L; l += blockDim.x) P.len[l] = 0;
}
__global__ void k_set_mode(DevPtrs P, int mode) { P.st->mode = mode; }
// After the batched prefill: every layer holds n rows, the committed length is n, nothing is in flight.
__global__ void k_prefill_done(DevPtrs P, int n) {
  if (threadIdx.x == 0) { P.st->c = n; P.st->pf_next = n; }
  for (int l = threadIdx.x; l < P.dim.L; l += blockDim.x) P.len[l] = n;
}
__global__ void k_set_forced(DevPtrs P, int on, int n_truth, unsigned long long thresh, unsigned long long seed) {
  P.st->forced_on = on; P.st->n_truth = n_truth; P.st->forced_thresh = thresh; P.st->forced_seed = seed;
}
__global__ void k_set_sampling(DevPtrs P, int on, int top_k, float temperature, unsigned long long seed) {
  P.samp->on = on; P.samp->top_k = top_k; P.samp->temperature = temperature; P.samp->seed = seed;
  for (int b = 0; b < kMaxStages; ++b) P.samp->q[b].k = 0;   // nothing in flight carries a draft distribution yet
  P.samp->pre_cnt[0] = P.samp->pre_cnt[1] = 0;
  P.samp->tau_guess[0] = P.samp->tau_guess[1] = INFINITY;
}
// External truncate + flush + reseed (PAPER.md:131 with c := new_len).
__global__ void k_rollback(DevPtrs P, int new_len, int tok) {
  StepState *st = P.st;
  for (int l = threadIdx.x; l < P.dim.L; l += blockDim.x) if (P.len[l] > new_len) P.len[l] = new_len;
  int buf = st->hbuf[0];
  __syncthreads();
  if (threadIdx.x == 0) {
    st->c = new_len;
    const long long nn = (long long)new_len - st->prompt_len + 1;   // tokens emitted up to and including the reseed token
    st->N = nn > 1 ? nn : 1;                           // a rollback into the prompt: the reseed token is the first emitted one
    for (int k = 1; k < P.dim.n; ++k) st->occ[k] = 0;
    st->occ[0] = 1; st->pos[0] = new_len; st->tok[0] = tok;
  }
  const uint16_t *e = P.embed + (size_t)tok * P.dim.d;
  for (int i = threadIdx.x; i < P.dim.d; i += blockDim.x) P.h[(size_t)buf * P.dim.d + i] = bf16_to_f32(e[i]);
}
}  // namespace spd

// ------------------------------------------------------------------ create / destroy -----------
// Everything a half-built context may own (events, pinned buffers, plans): one exit for every failure of spd_create.
static void create_cleanup(spd_ctx *ctx) {
  if (!ctx) return;
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
  if (ctx->h_results) cudaFreeHost(ctx->h_results);
  if (ctx->h_state) cudaFreeHost(ctx->h_state);
  free(ctx->pf);
  free(ctx);
  cudaGetLastError();
}

extern "C" int spd_create(const spd_config *cfg, const spd_weights *w, const spd_buffers *bufs, spd_ctx **out) {
  if (!out) return SPD_EINVAL;
  if (!validate(cfg) || !w || !bufs) return SPD_EINVAL;
  if (!w->embed || !w->final_norm || !w->pdm_proj || !w->pdm_norm || !w->attn_norm || !w->wq || !w->wk || !w->wv ||
      !w->wo || !w->mlp_norm || !w->w_gate || !w->w_up || !w->w_down)
    return SPD_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || cfg->device < 0 || cfg->device >= ndev) return SPD_ECUDA;
  spd_sizes need;
  spd_query_sizes(cfg, &need);
  if (!bufs->kv || !bufs->work || (need.repack_bytes && !bufs->repack)) return SPD_ENOMEM;
  if (bufs->kv_bytes < need.kv_bytes || bufs->work_bytes < need.work_bytes || bufs->repack_bytes < need.repack_bytes)
    return SPD_ENOMEM;
  spd_ctx *ctx = (spd_ctx *)calloc(1, sizeof(spd_ctx));
  if (!ctx) return SPD_ENOMEM;
  ctx->cfg = *cfg; ctx->bufs = *bufs; ctx->sizes = need;
  ctx->sm = (cudaStream_t)bufs->stream_main; ctx->sp = (cudaStream_t)bufs->stream_pdm;
#define CUC(call)                                                                                         \
  do {                                                                                                    \
    cudaError_t e_ = (call);                                                                              \
    if (e_ != cudaSuccess) { fprintf(stderr, "spd_create: %s\n", cudaGetErrorString(e_)); create_cleanup(ctx); return SPD_ECUDA; } \
  } while (0)
  CUC(cudaSetDevice(cfg->device));
  const uint16_t **tables[9];
  carve_work(cfg, bufs->work, &ctx->P, tables);
  DevPtrs &P = ctx->P;
  P.kv = (uint16_t *)bufs->kv;
  P.embed = w->embed; P.final_norm = w->final_norm; P.pdm_proj = w->pdm_proj; P.pdm_norm = w->pdm_norm;
  CUC(cudaMemsetAsync(bufs->work, 0, need.work_bytes, ctx->sm));
  const uint16_t *const *src[9] = {w->attn_norm, w->wq, w->wk, w->wv, w->wo, w->mlp_norm, w->w_gate, w->w_up, w->w_down};
  for (int i = 0; i < 9; ++i) {
    for (int l = 0; l < cfg->n_layers; ++l)
      if (!src[i][l]) { create_cleanup(ctx); return SPD_EINVAL; }
    CUC(cudaMemcpyAsync((void *)tables[i], src[i], sizeof(void *) * cfg->n_layers, cudaMemcpyHostToDevice, ctx->sm));
  }
  int half = cfg->head_dim / 2;
  double inv[64];
  for (int i = 0; i < half; ++i) inv[i] = pow((double)cfg->rope_base, -2.0 * (double)i / (double)cfg->head_dim);
  CUC(cudaMemcpyAsync(P.inv_freq, inv, sizeof(double) * half, cudaMemcpyHostToDevice, ctx->sm));
  k_state_init<<<1, 256, 0, ctx->sm>>>(P, MODE_IDLE, 0);
  CUC(cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming));
  CUC(cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming));
  CUC(cudaMallocHost(&ctx->h_results, sizeof(StepResult) * kResultRing));
  CUC(cudaMallocHost(&ctx->h_state, sizeof(StepState)));
  // fused engine: plan + weight repack into the caller's buffer
  ctx->has_mega = 0;
  ctx->engine = 0;
  int mrc = mega_create(P, src, bufs->repack, need.repack_bytes, ctx->sm, &ctx->mega);
  if (mrc == 0) { ctx->has_mega = 1; ctx->engine = 1; }
  // the multiplexed-chain schedule of the same building blocks (spd_mega2.cu); shares the repacked weights
  ctx->has_mega2 = 0;
  if (ctx->has_mega && mega2_create(P, ctx->mega, &ctx->mega2) == 0) { ctx->has_mega2 = 1; ctx->engine = SPD_DEFAULT_FUSED_ENGINE == 2 ? 2 : 1; }
  ctx->pf = (PrefillPlan *)calloc(1, sizeof(PrefillPlan));
  ctx->prefill_mode = (ctx->pf && prefill_create(P, src, ctx->pf) == 0) ? 1 : 0;
  CUC(cudaStreamSynchronize(ctx->sm));
  CUC(cudaGetLastError());
#undef CUC
  snprintf(ctx->err, sizeof ctx->err, "ok");
  *out = ctx;
  return SPD_OK;
}

extern "C" int spd_destroy(spd_ctx *ctx) {
  if (!ctx) return SPD_EINVAL;
  cudaStreamSynchronize(ctx->sm);
  cudaStreamSynchronize(ctx->sp);
  for (int e = 0; e < 3; ++e) if (ctx->graph[e]) cudaGraphExecDestroy(ctx->graph[e]);
  cudaEventDestroy(ctx->ev_fork);
  cudaEventDestroy(ctx->ev_join);
  cudaFreeHost(ctx->h_results);
  cudaFreeHost(ctx->h_state);
  free(ctx->pf);
  pdm_destroy(ctx->pdm);
  free(ctx);
  return SPD_OK;
}

extern "C" const char *spd_last_error(const spd_ctx *ctx) { return ctx ? ctx->err : kNullCtxErr; }

// ------------------------------------------------------------------ running cycles -------------
static int enqueue_raw(spd_ctx *ctx, long long *cnt) {
  // NEXT-1: the paper's PDM drafts from the pre-step state, in front of the cycle's kernels
  if (ctx->pdm && pdm_enqueue_draft(ctx->P, ctx->pdm, ctx->sm, cnt)) return -1;
  if (ctx->engine == 2) return mega2_enqueue_step(ctx->P, ctx->mega, ctx->mega2, ctx->sm, cnt);
  if (ctx->engine == 1) return mega_enqueue_step(ctx->P, ctx->mega, ctx->sm, cnt);
  return ref_enqueue_step(ctx->P, ctx->sm, ctx->sp, ctx->ev_fork, ctx->ev_join, cnt);
}

// One cycle on the main stream: a replay of the captured CUDA graph of the engine (captured once), or
// the plain launches if capture is not possible.
static int enqueue_cycle(spd_ctx *ctx) {
  int e = ctx->engine;
  if (!ctx->graph[e] && !ctx->graph_tried[e]) {
    ctx->graph_tried[e] = 1;
    cudaGraph_t g = nullptr;
    long long cnt = 0;
    if (cudaStreamBeginCapture(ctx->sm, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      int rc = enqueue_raw(ctx, &cnt);
      cudaError_t ce = cudaStreamEndCapture(ctx->sm, &g);
      if (rc == 0 && ce == cudaSuccess && g && cudaGraphInstantiate(&ctx->graph[e], g, 0) == cudaSuccess)
        ctx->launches_per_step[e] = cnt;
      else
        ctx->graph[e] = nullptr;
      if (g) cudaGraphDestroy(g);
    }
    cudaGetLastError();
  }
  if (ctx->graph[e]) {
    CU(cudaGraphLaunch(ctx->graph[e], ctx->sm));
    ctx->launches += ctx->launches_per_step[e];
    return SPD_OK;
  }
  if (enqueue_raw(ctx, &ctx->launches)) { ctx->dead = 1; return fail(ctx, SPD_ECUDA, "kernel launch failed%s"); }
  return SPD_OK;
}

static int sync_state(spd_ctx *ctx) {
  CU(cudaMemcpyAsync(ctx->h_state, ctx->P.st, sizeof(StepState), cudaMemcpyDeviceToHost, ctx->sm));
  CU(cudaStreamSynchronize(ctx->sm));
  if (ctx->h_state->err) { ctx->dead = 1; return fail(ctx, SPD_ECUDA, "device-side check failed (KV length != position or capacity)%s"); }
  return SPD_OK;
}

extern "C" int spd_prefill(spd_ctx *ctx, const int32_t *tokens, int32_t n_tokens, int32_t *first_token) {
  if (!ctx) return SPD_EINVAL;
  if (ctx->dead) return SPD_ECUDA;
  if (!tokens || n_tokens < 1 || n_tokens >= ctx->cfg.max_seq - 1) return fail(ctx, SPD_EINVAL, "spd_prefill: bad n_tokens%s");
  for (int i = 0; i < n_tokens; ++i)
    if (tokens[i] < 0 || tokens[i] >= ctx->cfg.vocab) return fail(ctx, SPD_EINVAL, "spd_prefill: token id out of range%s");
  CU(cudaSetDevice(ctx->cfg.device));
  ctx->prefilled = 0;
  CU(cudaMemcpyAsync(ctx->P.pf_tokens, tokens, sizeof(int32_t) * n_tokens, cudaMemcpyHostToDevice, ctx->sm));
  if (ctx->prefill_mode == 1) {
    // batched prefill: per-layer tcgen05 GEMMs + causal attention over chunks of the prompt (spd_prefill.cu); the
    // state is then what the pipelined prefill leaves before its final cycle: c = len[l] = P, nothing in flight
    k_state_init<<<1, 256, 0, ctx->sm>>>(ctx->P, MODE_PREFILL_FINAL, n_tokens);
    ++ctx->launches;
    if (prefill_run(ctx->P, *ctx->pf, n_tokens, ctx->sm, &ctx->launches)) {
      ctx->dead = 1;
      return fail(ctx, SPD_ECUDA, "batched prefill launch failed%s");
    }
    k_prefill_done<<<1, 256, 0, ctx->sm>>>(ctx->P, n_tokens);
    ++ctx->launches;
  } else {
    k_state_init<<<1, 256, 0, ctx->sm>>>(ctx->P, MODE_PREFILL, n_tokens);
    ++ctx->launches;
    // cycle 0 only enters token 0; cycles 1..P-1 forward and enter; n more drain the pipeline
    int total = n_tokens + ctx->cfg.n_stages;
    for (int i = 0; i < total; ++i) {
      int rc = enqueue_cycle(ctx);
      if (rc) return rc;
    }
    k_set_mode<<<1, 1, 0, ctx->sm>>>(ctx->P, MODE_PREFILL_FINAL);
    ++ctx->launches;
  }
  if (ctx->pdm && pdm_prefill(ctx->P, ctx->pdm, n_tokens, ctx->prefill_mode, ctx->sm, &ctx->launches)) {
    ctx->dead = 1;
    return fail(ctx, SPD_ECUDA, "PDM prefill launch failed%s");
  }
  int rc = enqueue_cycle(ctx);
  if (rc) return rc;
  CU(cudaMemcpyAsync(ctx->h_results, ctx->P.results, sizeof(StepResult), cudaMemcpyDeviceToHost, ctx->sm));
  rc = sync_state(ctx);
  if (rc) return rc;
  if (ctx->h_state->c != n_tokens || ctx->h_state->mode != MODE_SPD) { ctx->dead = 1; return fail(ctx, SPD_ECUDA, "prefill left an inconsistent state%s"); }
  ctx->prefilled = 1;
  if (first_token) *first_token = ctx->h_results[0].emitted_token;
  return SPD_OK;
}

extern "C" int spd_step_many(spd_ctx *ctx, int32_t n_steps, spd_step_result *results) {
  if (!ctx) return SPD_EINVAL;
  if (ctx->dead) return SPD_ECUDA;
  if (!ctx->prefilled) return fail(ctx, SPD_ESTATE, "spd_step before spd_prefill%s");
  if (n_steps < 1 || n_steps > kResultRing || !results) return fail(ctx, SPD_EINVAL, "spd_step_many: bad n_steps%s");
  int p_new = ctx->h_state->pos[0];
  if ((long long)p_new + n_steps >= ctx->cfg.max_seq) return fail(ctx, SPD_ECAPACITY, "KV capacity (max_seq) reached%s");
  CU(cudaSetDevice(ctx->cfg.device));
  long long K0 = ctx->h_state->K;
  for (int i = 0; i < n_steps; ++i) {
    int rc = enqueue_cycle(ctx);
    if (rc) return rc;
  }
  int first = (int)(K0 % kResultRing);
  int run1 = n_steps < kResultRing - first ? n_steps : kResultRing - first;
  CU(cudaMemcpyAsync(ctx->h_results, ctx->P.results + first, sizeof(StepResult) * run1, cudaMemcpyDeviceToHost, ctx->sm));
  if (run1 < n_steps)
    CU(cudaMemcpyAsync(ctx->h_results + run1, ctx->P.results, sizeof(StepResult) * (n_steps - run1), cudaMemcpyDeviceToHost, ctx->sm));
  int rc = sync_state(ctx);
  if (rc) return rc;
  static_assert(sizeof(StepResult) == sizeof(spd_step_result), "result layout");
  static_assert(sizeof(SampleRecord) == sizeof(spd_sample_record) && kMaxTopK == SPD_MAX_TOPK, "sample record layout");
  memcpy(results, ctx->h_results, sizeof(StepResult) * n_steps);
  return SPD_OK;
}

extern "C" int spd_step(spd_ctx *ctx, spd_step_result *out) {
  spd_step_result r;
  int rc = spd_step_many(ctx, 1, &r);
  if (rc == SPD_OK && out) *out = r;
  return rc;
}

extern "C" int spd_rollback(spd_ctx *ctx, int32_t new_len, int32_t reseed_token) {
  if (!ctx) return SPD_EINVAL;
  if (ctx->dead) return SPD_ECUDA;
  if (!ctx->prefilled) return fail(ctx, SPD_ESTATE, "spd_rollback before spd_prefill%s");
  if (new_len < 0 || new_len > ctx->h_state->c || reseed_token < 0 || reseed_token >= ctx->cfg.vocab)
    return fail(ctx, SPD_EINVAL, "spd_rollback: bad new_len or token%s");
  if (new_len + 1 >= ctx->cfg.max_seq) return fail(ctx, SPD_ECAPACITY, "KV capacity (max_seq) reached%s");
  CU(cudaSetDevice(ctx->cfg.device));
  k_rollback<<<1, 256, 0, ctx->sm>>>(ctx->P, new_len, reseed_token);
  ++ctx->launches;
  if (ctx->pdm) { pdm_rollback(ctx->pdm, new_len, ctx->sm); ++ctx->launches; }
  return sync_state(ctx);
}

extern "C" int spd_set_forced(spd_ctx *ctx, const int32_t *truth, int32_t n_truth, float p, uint64_t seed) {
  if (!ctx) return SPD_EINVAL;
  if (ctx->dead) return SPD_ECUDA;
  CU(cudaSetDevice(ctx->cfg.device));
  if (p >= 0.f && ctx->sampling_on) return fail(ctx, SPD_ESTATE, "spd_set_forced: sampling verification is on%s");
  if (p < 0.f) {
    k_set_forced<<<1, 1, 0, ctx->sm>>>(ctx->P, 0, 0, 0ull, 0ull);
    ctx->forced_on = 0;
  } else {
    if (p > 1.f || n_truth < 0 || n_truth > ctx->cfg.max_seq || (n_truth > 0 && !truth))
      return fail(ctx, SPD_EINVAL, "spd_set_forced: bad arguments%s");
    ctx->forced_on = 1;
    if (n_truth) CU(cudaMemcpyAsync(ctx->P.truth, truth, sizeof(int32_t) * n_truth, cudaMemcpyHostToDevice, ctx->sm));
    unsigned long long thresh = (unsigned long long)floor((double)p * 9007199254740992.0);
    k_set_forced<<<1, 1, 0, ctx->sm>>>(ctx->P, 1, n_truth, thresh, (unsigned long long)seed);
  }
  ++ctx->launches;
  CU(cudaStreamSynchronize(ctx->sm));
  return SPD_OK;
}

static void drop_graphs(spd_ctx *ctx) {   // a kernel parameter changed: captured graphs must be rebuilt
  cudaStreamSynchronize(ctx->sm);
  for (int e = 0; e < 3; ++e) {
    if (ctx->graph[e]) cudaGraphExecDestroy(ctx->graph[e]);
    ctx->graph[e] = nullptr; ctx->graph_tried[e] = 0;
  }
}

extern "C" int spd_set_sampling(spd_ctx *ctx, float temperature, int32_t top_k, uint64_t seed) {
  if (!ctx) return SPD_EINVAL;
  if (ctx->dead) return SPD_ECUDA;
  const int on = top_k >= 1;
  if (on && (top_k > kMaxTopK || !(temperature > 0.f))) return fail(ctx, SPD_EINVAL, "spd_set_sampling: bad arguments%s");
  if (on && ctx->forced_on) return fail(ctx, SPD_ESTATE, "spd_set_sampling: forced acceptance is on%s");
  if (on && ctx->pdm) return fail(ctx, SPD_ESTATE, "spd_set_sampling: the paper's PDM is attached (greedy verification only)%s");
  CU(cudaSetDevice(ctx->cfg.device));
  if (ctx->P.sampling != on) { ctx->P.sampling = on; drop_graphs(ctx); }
  ctx->sampling_on = on;
  k_set_sampling<<<1, 1, 0, ctx->sm>>>(ctx->P, on, on ? top_k : 0, on ? temperature : 1.f, (unsigned long long)seed);
  ++ctx->launches;
  CU(cudaStreamSynchronize(ctx->sm));
  return SPD_OK;
}

extern "C" int spd_set_option(spd_ctx *ctx, int32_t option, int32_t value) {
  if (!ctx) return SPD_EINVAL;
  if (option == SPD_OPT_ENGINE) {
    if (value == 0 || (value == 1 && ctx->has_mega) || (value == 2 && ctx->has_mega2)) { ctx->engine = value; return SPD_OK; }
    return fail(ctx, SPD_EINVAL, "engine not available%s");
  }
  if (option == SPD_OPT_CHAINS) {
    if (!ctx->has_mega2 || value < 1 || value > kMega2MaxChains) return fail(ctx, SPD_EINVAL, "chains: 1..4, engine 2 only%s");
    if (ctx->mega2.chains != value) { ctx->mega2.chains = value; drop_graphs(ctx); }
    return SPD_OK;
  }
  if (option == SPD_OPT_PREFILL) {
    if (value == 0 || (value == 1 && ctx->pf && ctx->pf->available)) { ctx->prefill_mode = value; return SPD_OK; }
    return fail(ctx, SPD_EINVAL, "batched prefill not available for this configuration%s");
  }
  if (option == SPD_OPT_DEBUG_LOGITS || option == SPD_OPT_PHASE_PROFILE) {
    int v = value ? 1 : 0;
    int32_t *field = option == SPD_OPT_DEBUG_LOGITS ? &ctx->P.debug_logits : &ctx->P.prof_on;
    if (v != *field) {
      *field = v;
      drop_graphs(ctx);
    }
    return SPD_OK;
  }
  return fail(ctx, SPD_EINVAL, "unknown option%s");
}

extern "C" int spd_get_option(spd_ctx *ctx, int32_t option, int32_t *value) {
  if (!ctx || !value) return SPD_EINVAL;
  switch (option) {
    case SPD_OPT_ENGINE: *value = ctx->engine; return SPD_OK;
    case SPD_OPT_DEBUG_LOGITS: *value = ctx->P.debug_logits; return SPD_OK;
    case SPD_OPT_PHASE_PROFILE: *value = ctx->P.prof_on; return SPD_OK;
    case SPD_OPT_PREFILL: *value = ctx->prefill_mode; return SPD_OK;
    case SPD_OPT_CHAINS: *value = ctx->has_mega2 ? ctx->mega2.chains : 0; return SPD_OK;
    default: return fail(ctx, SPD_EINVAL, "unknown option%s");
  }
}

extern "C" int spd_get_counters(spd_ctx *ctx, int64_t *steps, int64_t *emitted, int64_t *kernel_launches) {
  if (!ctx) return SPD_EINVAL;
  if (steps) *steps = ctx->prefilled ? ctx->h_state->K : 0;
  if (emitted) *emitted = ctx->prefilled ? ctx->h_state->N : 0;
  if (kernel_launches) *kernel_launches = ctx->launches;
  return SPD_OK;
}

extern "C" int spd_debug_read(spd_ctx *ctx, int32_t what, int32_t index, void *host_out, size_t bytes) {
  if (!ctx || !host_out) return SPD_EINVAL;
  if (ctx->dead) return SPD_ECUDA;
  const Dims &D = ctx->P.dim;
  const DevPtrs &P = ctx->P;
  CU(cudaSetDevice(ctx->cfg.device));
  int rc = sync_state(ctx);
  if (rc) return rc;
  const StepState *st = ctx->h_state;
  const void *src = nullptr;
  size_t want = 0;
  switch (what) {
    case SPD_DBG_SLOT_HIDDEN:
      if (index < 0 || index >= D.n) return fail(ctx, SPD_EINVAL, "debug_read: depth out of range%s");
      src = P.h + (size_t)st->hbuf[index] * D.d; want = sizeof(float) * D.d; break;
    case SPD_DBG_EXIT_LOGITS:
    case SPD_DBG_PDM_LOGITS:
      if (!P.debug_logits && !P.sampling && ctx->engine >= 1) return fail(ctx, SPD_ESTATE, "debug_read: enable SPD_OPT_DEBUG_LOGITS first%s");
      src = what == SPD_DBG_EXIT_LOGITS ? P.logits_v : P.logits_p; want = sizeof(float) * D.V; break;
    case SPD_DBG_PDM_PRENORM: src = P.pdm_u; want = sizeof(float) * D.d; break;
    case SPD_DBG_PDM_FEAT: src = P.feat; want = sizeof(float) * D.d * D.n; break;
    case SPD_DBG_KV_LEN: src = P.len; want = sizeof(int32_t) * D.L; break;
    case SPD_DBG_HFIN:
      if (index < 0 || index >= D.max_seq) return fail(ctx, SPD_EINVAL, "debug_read: position out of range%s");
      src = P.hfin + (size_t)index * D.d; want = sizeof(float) * D.d; break;
    case SPD_DBG_Q:
    case SPD_DBG_ATT:
      if (index < 0 || index >= D.n) return fail(ctx, SPD_EINVAL, "debug_read: stage out of range%s");
      src = (what == SPD_DBG_Q ? P.q : P.att) + (size_t)index * D.Hq * D.hd; want = sizeof(float) * D.Hq * D.hd; break;
    case SPD_DBG_SAMPLE:
      if (!P.sampling) return fail(ctx, SPD_ESTATE, "debug_read: sampling verification is off%s");
      src = &P.samp->rec; want = sizeof(SampleRecord); break;
    case SPD_DBG_PDM2_LOGITS: case SPD_DBG_PDM2_HIDDEN: case SPD_DBG_PDM2_RUN: case SPD_DBG_PDM2_FEAT:
    case SPD_DBG_PDM2_K: case SPD_DBG_PDM2_V:
      if (!ctx->pdm) return fail(ctx, SPD_ESTATE, "debug_read: the paper's PDM is not attached%s");
      if (pdm_debug_read(P, ctx->pdm, what - SPD_DBG_PDM2_LOGITS, index, host_out, bytes))
        return fail(ctx, SPD_EINVAL, "debug_read: bad PDM selector arguments%s");
      return SPD_OK;
    case SPD_DBG_ANCHOR:
      if (!ctx->pdm || index < 0 || index / 8 >= D.max_seq || index % 8 >= P.pdm_m) return fail(ctx, SPD_EINVAL, "debug_read: bad anchor index%s");
      src = P.anch + ((size_t)(index / 8) * P.pdm_m + index % 8) * D.d; want = sizeof(float) * D.d; break;
    case SPD_DBG_CYCLE_TIMES:
      src = P.cycle_ts; want = sizeof(unsigned long long) * 2 * kResultRing; break;
    case SPD_DBG_PHASE_PROFILE:
      src = P.prof; want = sizeof(unsigned long long) * kProfCtas * kProfPhases * kProfStamps; break;
    case SPD_DBG_RING: {
      want = sizeof(int32_t) * (2 + 3 * D.n);
      if (bytes != want) return fail(ctx, SPD_EINVAL, "debug_read: size mismatch%s");
      int32_t *o = (int32_t *)host_out;
      int fill = 0;
      for (int k = 0; k < D.n; ++k) fill += st->occ[k];
      o[0] = fill; o[1] = st->c;
      for (int k = 0; k < D.n; ++k) { o[2 + 3 * k] = st->occ[k]; o[3 + 3 * k] = st->pos[k]; o[4 + 3 * k] = st->tok[k]; }
      return SPD_OK;
    }
    case SPD_DBG_KV_K:
    case SPD_DBG_KV_V: {
      size_t rowb = (size_t)D.Hkv * D.hd * sizeof(uint16_t);
      if (index < 0 || index >= D.L || bytes % rowb || bytes / rowb > (size_t)D.max_seq)
        return fail(ctx, SPD_EINVAL, "debug_read: bad layer or size%s");
      size_t rows = bytes / rowb;
      if (!rows) return SPD_OK;
      for (int hh = 0; hh < D.Hkv; ++hh)   // head-major cache -> position-major rows
        CU(cudaMemcpy2D((char *)host_out + (size_t)hh * D.hd * 2, rowb,
                        P.kv + kv_offset(D, index, what == SPD_DBG_KV_V, hh), (size_t)D.hd * 2, (size_t)D.hd * 2, rows,
                        cudaMemcpyDeviceToHost));
      return SPD_OK;
    }
    default: return fail(ctx, SPD_EINVAL, "debug_read: unknown selector%s");
  }
  if (bytes != want) return fail(ctx, SPD_EINVAL, "debug_read: size mismatch%s");
  CU(cudaMemcpy(host_out, src, want, cudaMemcpyDeviceToHost));
  return SPD_OK;
}

// ------------------------------------------------------------------ the prefill GEMM as one operation ----------
extern "C" size_t spd_op_gemm_scratch(int32_t m, int32_t k) { return (size_t)3 * (m > 0 ? m : 0) * (k > 0 ? k : 0) * sizeof(uint16_t); }
extern "C" int spd_op_gemm(const float *x, const uint16_t *w, int32_t m, int32_t n, int32_t k, float *y, void *scratch,
                           void *stream) {
  if (!x || !w || !y || !scratch || m < 1 || n < 1 || k < 64 || k % 64 || n % 4) return SPD_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return SPD_ECUDA;
  return prefill_op_gemm(x, w, m, n, k, y, scratch, (cudaStream_t)stream) == 0 ? SPD_OK : SPD_ECUDA;
}

// ------------------------------------------------------------------ the paper's PDM (NEXT-1) -------------------
extern "C" int spd_pdm_query_sizes(const spd_config *cfg, int32_t pdm_layers, int32_t pdm_vocab, spd_pdm_sizes *out) {
  if (!validate(cfg) || !out || pdm_layers < 1 || pdm_layers > kPrefillMaxLayers || pdm_vocab < 1 || pdm_vocab > cfg->vocab)
    return SPD_EINVAL;
  Dims D = make_dims(cfg);
  out->kv_bytes = pdm_kv_bytes(D, pdm_layers);
  out->work_bytes = pdm_work_bytes(D, pdm_layers, pdm_vocab);
  return SPD_OK;
}

extern "C" int spd_pdm_attach(spd_ctx *ctx, const spd_pdm_weights *w, void *pdm_kv, void *pdm_work) {
  if (!ctx) return SPD_EINVAL;
  if (ctx->dead) return SPD_ECUDA;
  if (ctx->prefilled || ctx->pdm) return fail(ctx, SPD_ESTATE, "spd_pdm_attach: attach once, before spd_prefill%s");
  if (ctx->sampling_on) return fail(ctx, SPD_ESTATE, "spd_pdm_attach: sampling verification is on%s");
  if (!w || !pdm_kv || !pdm_work || !w->fc || !w->attn_norm || !w->wq || !w->wk || !w->wv || !w->wo || !w->mlp_norm ||
      !w->w_gate || !w->w_up || !w->w_down || !w->final_norm || !w->head || !w->vocab_map)
    return fail(ctx, SPD_EINVAL, "spd_pdm_attach: missing argument%s");
  CU(cudaSetDevice(ctx->cfg.device));
  ctx->pdm = pdm_create(&ctx->P, w, pdm_kv, pdm_work, ctx->sm);
  if (!ctx->pdm) return fail(ctx, SPD_EINVAL, "spd_pdm_attach: bad PDM configuration%s");
  drop_graphs(ctx);   // the kernels' parameters changed
  return SPD_OK;
}
