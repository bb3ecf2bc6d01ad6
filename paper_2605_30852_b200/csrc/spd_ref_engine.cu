// spd_ref_engine.cu — the reference engine: one plain CUDA kernel per operation of the SPD cycle,
// stage-batched over gridDim.y, PDM on the second stream.  It is the simple, easy-to-check GPU path
// (and the kernels behind the spd_op_* entry points); the fused persistent engine (spd_mega.cu) is the
// fast one.  The two engines use different reduction orders, so each is compared with the CPU oracle,
// not bitwise with the other.
#include "../../include/spd.h"
#include "spd_engine.h"
#include "spd_kernels.cuh"

namespace spd {

// ------------------------------------------------------------------ controller kernels ---------
__global__ void k_begin(DevPtrs P) {
  if (threadIdx.x == 0) controller_begin(P);
  __syncthreads();
  rope_table_fill(P, threadIdx.x, blockDim.x);
}

// PDM slot vectors (pre-step): slot j = token at depth j, else Hfin[p_new - j], else 0.
__global__ void k_pdm_gather(DevPtrs P) {
  const StepState *st = P.st;
  if (!st->run_pdm) return;
  int j = blockIdx.y, d = P.dim.d;
  int q = st->p_new - j;
  const float *src = nullptr;
  if (st->occ[j]) src = P.h + (size_t)st->hbuf[j] * d;
  else if (q >= 0) src = P.hfin + (size_t)q * d;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < d; i += gridDim.x * blockDim.x)
    P.feat[(size_t)j * d + i] = src ? src[i] : 0.f;
}

__global__ void k_end(DevPtrs P, int ncand) {
  __shared__ SampSmem sm;
  controller_end(P, ncand, &sm);
}

// ------------------------------------------------------------------ per-op kernels -------------
// which: 0 attn_norm, 1 mlp_norm (per stage); 2 verify head input; 3 PDM head input
__global__ void k_rmsnorm(DevPtrs P, int which, int pass) {
  __shared__ float red[33];
  const StepState *st = P.st;
  const Dims &D = P.dim;
  if (which <= 1) {
    int k = blockIdx.x;
    if (!st->occ[k]) return;
    int layer = k * D.per + pass;
    const uint16_t *g = which == 0 ? P.attn_norm[layer] : P.mlp_norm[layer];
    const int ai = which == 0 ? anchor_index(P, layer) : -1;
    if (ai >= 0 && st->pos[k] < D.max_seq)   // NEXT-1: H^layer of the paper PDM's anchor set
      for (int i = threadIdx.x; i < D.d; i += blockDim.x)
        P.anch[((size_t)st->pos[k] * P.pdm_m + ai) * D.d + i] = P.h[(size_t)st->hbuf[k] * D.d + i];
    block_rmsnorm(P.h + (size_t)st->hbuf[k] * D.d, g, D.d, D.eps, P.x + (size_t)k * D.d, red);
  } else if (which == 2) {
    if (!st->run_verify) return;
    const float *src = st->mode == MODE_PREFILL_FINAL ? P.hfin + (size_t)(st->c - 1) * D.d
                                                      : P.h + (size_t)st->hbuf[D.n - 1] * D.d;
    block_rmsnorm(src, P.final_norm, D.d, D.eps, P.xv, red);
  } else {
    if (!st->run_pdm) return;
    block_rmsnorm(P.pdm_u, P.pdm_norm, D.d, D.eps, P.xp, red);
  }
}

enum GemvMode { G_QKV = 0, G_O = 1, G_GATEUP = 2, G_DOWN = 3, G_PDM = 4, G_HEAD = 5 };

// Stage-batched GEMV: gridDim.y = stage (depth k), one warp per output row, 8 rows per CTA.
template <int MODE>
__global__ void __launch_bounds__(256) k_gemv(DevPtrs P, int pass) {
  const StepState *st = P.st;
  const Dims &D = P.dim;
  int k = blockIdx.y;
  int row = blockIdx.x * 8 + (threadIdx.x >> 5);
  int lane = threadIdx.x & 31;
  if (MODE <= G_DOWN) {
    if (!st->occ[k]) return;
    int layer = k * D.per + pass;
    float *h = P.h + (size_t)st->hbuf[k] * D.d;
    const float *x = P.x + (size_t)k * D.d;
    int qd = D.Hq * D.hd, kd = D.Hkv * D.hd;
    if (MODE == G_QKV) {
      if (row >= qd + 2 * kd) return;
      const uint16_t *w;
      float *out;
      if (row < qd) { w = P.wq[layer] + (size_t)row * D.d; out = P.q + (size_t)k * qd + row; }
      else if (row < qd + kd) { w = P.wk[layer] + (size_t)(row - qd) * D.d; out = P.kvtmp + (size_t)k * 2 * kd + (row - qd); }
      else { w = P.wv[layer] + (size_t)(row - qd - kd) * D.d; out = P.kvtmp + (size_t)k * 2 * kd + (row - qd); }
      float v = warp_dot_row(w, x, D.d);
      if (lane == 0) *out = v;
    } else if (MODE == G_O) {
      if (row >= D.d) return;
      float v = warp_dot_row(P.wo[layer] + (size_t)row * qd, P.att + (size_t)k * qd, qd);
      if (lane == 0) h[row] += v;
    } else if (MODE == G_GATEUP) {
      if (row >= D.F) return;
      float g = warp_dot_row(P.w_gate[layer] + (size_t)row * D.d, x, D.d);
      float u = warp_dot_row(P.w_up[layer] + (size_t)row * D.d, x, D.d);
      if (lane == 0) P.act[(size_t)k * D.F + row] = silu_mul(g, u);
    } else {  // G_DOWN
      if (row >= D.d) return;
      float v = warp_dot_row(P.w_down[layer] + (size_t)row * D.F, P.act + (size_t)k * D.F, D.F);
      if (lane == 0) h[row] += v;
    }
  } else if (MODE == G_PDM) {
    if (!st->run_pdm || row >= D.d) return;
    float v = warp_dot_row(P.pdm_proj + (size_t)row * D.n * D.d, P.feat, D.n * D.d);
    if (lane == 0) P.pdm_u[row] = v;
  } else {  // G_HEAD: the tied matrix E once, against both head inputs (verify, PDM)
    if (row >= D.V) return;
    const uint16_t *w = P.embed + (size_t)row * D.d;
    if (st->run_verify) { float v = warp_dot_row(w, P.xv, D.d); if (lane == 0) P.logits_v[row] = v; }
    if (st->run_pdm) { float v = warp_dot_row(w, P.xp, D.d); if (lane == 0) P.logits_p[row] = v; }
  }
}

// RoPE on q and k, bf16 rounding of k and v, KV append at row pos (requires len[layer] == pos).
__global__ void k_rope_append(DevPtrs P, int pass) {
  StepState *st = P.st;
  const Dims &D = P.dim;
  int k = blockIdx.x;
  if (!st->occ[k]) return;
  int layer = k * D.per + pass, pos = st->pos[k];
  if (P.len[layer] != pos || pos >= D.max_seq) {   // causality / capacity precondition
    if (threadIdx.x == 0) st->err = 1;
    return;
  }
  int half = D.hd / 2, qd = D.Hq * D.hd, kd = D.Hkv * D.hd;
  float *q = P.q + (size_t)k * qd;
  const float *kk = P.kvtmp + (size_t)k * 2 * kd, *vv = kk + kd;
  const float2 *tab = P.rope + (size_t)k * half;
  for (int i = threadIdx.x; i < D.Hq * half; i += blockDim.x) {
    int hh = i / half, j = i - hh * half;
    float2 cs = tab[j];
    float a = q[hh * D.hd + j], b = q[hh * D.hd + j + half];
    q[hh * D.hd + j] = a * cs.x - b * cs.y;
    q[hh * D.hd + j + half] = b * cs.x + a * cs.y;
  }
  for (int i = threadIdx.x; i < D.Hkv * half; i += blockDim.x) {
    int hh = i / half, j = i - hh * half;
    float2 cs = tab[j];
    float a = kk[hh * D.hd + j], b = kk[hh * D.hd + j + half];
    uint16_t *dst = P.kv + kv_offset(D, layer, 0, hh) + (size_t)pos * D.hd;
    dst[j] = f32_to_bf16(a * cs.x - b * cs.y);
    dst[j + half] = f32_to_bf16(b * cs.x + a * cs.y);
  }
  for (int i = threadIdx.x; i < kd; i += blockDim.x) {
    int hh = i / D.hd, j = i - hh * D.hd;
    P.kv[kv_offset(D, layer, 1, hh) + (size_t)pos * D.hd + j] = f32_to_bf16(vv[i]);
  }
  if (threadIdx.x == 0) P.len[layer] = pos + 1;
}

// grid (split, kv head, stage); block = group warps (one per q head of the group)
template <int HD>
__global__ void k_attn_partial(DevPtrs P, int pass) {
  const StepState *st = P.st;
  const Dims &D = P.dim;
  int k = blockIdx.z;
  if (!st->occ[k]) return;
  int T = st->pos[k] + 1;
  int split = blockIdx.x, t0 = split * kAttnSplit;
  if (t0 >= T) return;
  int t1 = min(T, t0 + kAttnSplit);
  int layer = k * D.per + pass, kvh = blockIdx.y, group = D.Hq / D.Hkv;
  int hq = kvh * group + (threadIdx.x >> 5);
  const uint16_t *kc = P.kv + kv_offset(D, layer, 0, kvh), *vc = P.kv + kv_offset(D, layer, 1, kvh);
  size_t slot = ((size_t)k * D.Hq + hq) * P.nsplit_max + split;
  attn_partial_warp<HD>(P.q + ((size_t)k * D.Hq + hq) * HD, kc, vc, t0, t1, P.part_o + slot * HD, P.part_ml + slot);
}

// grid (q head, stage); block = hd threads
__global__ void k_attn_merge(DevPtrs P) {
  const StepState *st = P.st;
  const Dims &D = P.dim;
  int k = blockIdx.y, hq = blockIdx.x;
  if (!st->occ[k]) return;
  int nsplit = (st->pos[k] + kAttnSplit) / kAttnSplit;
  size_t slot = ((size_t)k * D.Hq + hq) * P.nsplit_max;
  P.att[((size_t)k * D.Hq + hq) * D.hd + threadIdx.x] =
      attn_merge_elem(P.part_o + slot * D.hd, P.part_ml + slot, nsplit, D.hd, threadIdx.x);
}

// Per-CTA argmax candidates of the logit vectors (grid (ncand, 2)); reduced by k_end.
__global__ void k_argmax_cand(DevPtrs P) {
  __shared__ float sv[32];
  __shared__ int si[32];
  const StepState *st = P.st;
  int which = blockIdx.y;
  if ((which == 0 && !st->run_verify) || (which == 1 && !st->run_pdm)) return;
  const float *x = which == 0 ? P.logits_v : P.logits_p;
  int V = P.dim.V;
  int chunk = (V + gridDim.x - 1) / gridDim.x;
  int lo = blockIdx.x * chunk, hi = min(V, lo + chunk);
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  for (int i = lo + threadIdx.x; i < hi; i += blockDim.x) {
    float v = x[i];
    if (cand_better(v, i, bv, bi)) { bv = v; bi = i; }
  }
  for (int o = 16; o > 0; o >>= 1) {
    float ov = __shfl_xor_sync(0xffffffffu, bv, o);
    int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (cand_better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
  }
  if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = bv; si[threadIdx.x >> 5] = bi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w)
      if (cand_better(sv[w], si[w], bv, bi)) { bv = sv[w]; bi = si[w]; }
    P.cand_val[which * kMaxCand + blockIdx.x] = bv;
    P.cand_idx[which * kMaxCand + blockIdx.x] = lo < hi ? bi : -1;
  }
}

// ------------------------------------------------------------------ one cycle, enqueued --------
static inline unsigned cdiv(unsigned a, unsigned b) { return (a + b - 1) / b; }

int ref_enqueue_step(const DevPtrs &P, cudaStream_t sm, cudaStream_t sp, cudaEvent_t ev_fork, cudaEvent_t ev_join,
                     long long *launches) {
  const Dims &D = P.dim;
  int n = D.n, qd = D.Hq * D.hd, kd = D.Hkv * D.hd, group = D.Hq / D.Hkv;
  long long cnt = 0;
  k_begin<<<1, 256, 0, sm>>>(P); ++cnt;
  k_pdm_gather<<<dim3(cdiv(D.d, 256), n), 256, 0, sm>>>(P); ++cnt;
  // PDM branch on the second stream: it only needs the pre-step slot vectors gathered above
  cudaEventRecord(ev_fork, sm);
  cudaStreamWaitEvent(sp, ev_fork, 0);
  k_gemv<G_PDM><<<dim3(cdiv(D.d, 8), 1), 256, 0, sp>>>(P, 0); ++cnt;
  k_rmsnorm<<<1, 256, 0, sp>>>(P, 3, 0); ++cnt;
  cudaEventRecord(ev_join, sp);
  for (int pass = 0; pass < D.per; ++pass) {
    k_rmsnorm<<<n, 256, 0, sm>>>(P, 0, pass); ++cnt;
    k_gemv<G_QKV><<<dim3(cdiv(qd + 2 * kd, 8), n), 256, 0, sm>>>(P, pass); ++cnt;
    k_rope_append<<<n, 256, 0, sm>>>(P, pass); ++cnt;
    dim3 ga(P.nsplit_max, D.Hkv, n);
    if (D.hd == 128) k_attn_partial<128><<<ga, group * 32, 0, sm>>>(P, pass);
    else k_attn_partial<64><<<ga, group * 32, 0, sm>>>(P, pass);
    ++cnt;
    k_attn_merge<<<dim3(D.Hq, n), D.hd, 0, sm>>>(P); ++cnt;
    k_gemv<G_O><<<dim3(cdiv(D.d, 8), n), 256, 0, sm>>>(P, pass); ++cnt;
    k_rmsnorm<<<n, 256, 0, sm>>>(P, 1, pass); ++cnt;
    k_gemv<G_GATEUP><<<dim3(cdiv(D.F, 8), n), 256, 0, sm>>>(P, pass); ++cnt;
    k_gemv<G_DOWN><<<dim3(cdiv(D.d, 8), n), 256, 0, sm>>>(P, pass); ++cnt;
  }
  k_rmsnorm<<<1, 256, 0, sm>>>(P, 2, 0); ++cnt;
  cudaStreamWaitEvent(sm, ev_join, 0);
  k_gemv<G_HEAD><<<dim3(cdiv(D.V, 8), 1), 256, 0, sm>>>(P, 0); ++cnt;
  const int ncand = 128;
  k_argmax_cand<<<dim3(ncand, 2), 256, 0, sm>>>(P); ++cnt;
  k_end<<<1, 256, 0, sm>>>(P, ncand); ++cnt;
  if (launches) *launches += cnt;
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

// ------------------------------------------------------------------ spd_op_* kernels ------------
__global__ void k_op_rmsnorm(const float *x, const uint16_t *g, int d, float eps, float *out) {
  __shared__ float red[33];
  block_rmsnorm(x, g, d, eps, out, red);
}
__global__ void k_op_gemv(const uint16_t *w, int rows, int k, const float *x, float *out) {
  int row = blockIdx.x * 8 + (threadIdx.x >> 5);
  if (row >= rows) return;
  float v = warp_dot_row(w + (size_t)row * k, x, k);
  if ((threadIdx.x & 31) == 0) out[row] = v;
}
__global__ void k_op_rope(float *vec, int n_heads, int hd, int pos, double base) {
  int half = hd / 2;
  for (int i = threadIdx.x; i < n_heads * half; i += blockDim.x) {
    int hh = i / half, j = i - hh * half;
    double inv = pow(base, -2.0 * (double)j / (double)hd);
    double s, c;
    sincos((double)pos * inv, &s, &c);
    float cf = (float)c, sf = (float)s;
    float a = vec[hh * hd + j], b = vec[hh * hd + j + half];
    vec[hh * hd + j] = a * cf - b * sf;
    vec[hh * hd + j + half] = b * cf + a * sf;
  }
}
template <int HD>
__global__ void k_op_attn_partial(const float *q, const uint16_t *kc, const uint16_t *vc, int T, int t_stride, int Hq,
                                  int Hkv, int nsplit, float *part_o, float2 *part_ml) {
  int split = blockIdx.x, kvh = blockIdx.y, group = Hq / Hkv;
  int t0 = split * kAttnSplit, t1 = min(T, t0 + kAttnSplit);
  if (t0 >= T) return;
  int hq = kvh * group + (threadIdx.x >> 5);
  size_t slot = (size_t)hq * nsplit + split;
  attn_partial_warp<HD>(q + (size_t)hq * HD, kc + (size_t)kvh * t_stride * HD, vc + (size_t)kvh * t_stride * HD, t0, t1,
                        part_o + slot * HD, part_ml + slot);
}
__global__ void k_op_attn_merge(const float *part_o, const float2 *part_ml, int nsplit, int hd, float *out) {
  int hq = blockIdx.x;
  size_t slot = (size_t)hq * nsplit;
  out[(size_t)hq * hd + threadIdx.x] = attn_merge_elem(part_o + slot * hd, part_ml + slot, nsplit, hd, threadIdx.x);
}
__global__ void k_op_silu_mul(const float *g, const float *u, int n, float *out) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = silu_mul(g[i], u[i]);
}
__global__ void k_op_argmax(const float *x, int n, int *out) {
  __shared__ float sv[32];
  __shared__ int si[32];
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  for (int i = threadIdx.x; i < n; i += blockDim.x)
    if (cand_better(x[i], i, bv, bi)) { bv = x[i]; bi = i; }
  for (int o = 16; o > 0; o >>= 1) {
    float ov = __shfl_xor_sync(0xffffffffu, bv, o);
    int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (cand_better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
  }
  if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = bv; si[threadIdx.x >> 5] = bi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w)
      if (cand_better(sv[w], si[w], bv, bi)) { bv = sv[w]; bi = si[w]; }
    *out = bi;
  }
}

// Chunk maxima of x (grid = ncand CTAs): the argmax candidates that seed topk_dist's threshold.
__global__ void k_op_cand(const float *x, int n, float *cand_val, int32_t *cand_idx) {
  __shared__ float sv[32];
  __shared__ int si[32];
  int chunk = (n + gridDim.x - 1) / gridDim.x;
  int lo = blockIdx.x * chunk, hi = min(n, lo + chunk);
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  for (int i = lo + threadIdx.x; i < hi; i += blockDim.x)
    if (cand_better(x[i], i, bv, bi)) { bv = x[i]; bi = i; }
  for (int o = 16; o > 0; o >>= 1) {
    float ov = __shfl_xor_sync(0xffffffffu, bv, o);
    int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (cand_better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
  }
  if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = bv; si[threadIdx.x >> 5] = bi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w)
      if (cand_better(sv[w], si[w], bv, bi)) { bv = sv[w]; bi = si[w]; }
    cand_val[blockIdx.x] = bv;
    cand_idx[blockIdx.x] = lo < hi ? bi : -1;
  }
}
__global__ void __launch_bounds__(256) k_op_topk(const float *x, int n, int top_k, float temperature, int ncand,
                                                 const float *cand_val, const int32_t *cand_idx, float *surv_val,
                                                 int32_t *surv_idx, SampleDist *out) {
  __shared__ TopkSmem ts;
  topk_dist(x, n, cand_val, cand_idx, ncand, top_k, temperature, surv_val, surv_idx, out, nullptr, &ts);
}
}  // namespace spd

using namespace spd;

static int op_done() { return cudaGetLastError() == cudaSuccess ? 0 : 4; }

extern "C" int spd_op_rmsnorm(const float *x, const uint16_t *gain, int32_t d, float eps, float *out, void *stream) {
  if (!x || !gain || !out || d < 1) return 1;
  k_op_rmsnorm<<<1, 256, 0, (cudaStream_t)stream>>>(x, gain, d, eps, out);
  return op_done();
}
extern "C" int spd_op_gemv(const uint16_t *w, int32_t rows, int32_t k, const float *x, float *out, void *stream) {
  if (!w || !x || !out || rows < 1 || k < 8 || k % 8) return 1;
  k_op_gemv<<<cdiv(rows, 8), 256, 0, (cudaStream_t)stream>>>(w, rows, k, x, out);
  return op_done();
}
extern "C" int spd_op_rope(float *vec, int32_t n_heads, int32_t head_dim, int32_t pos, float base, void *stream) {
  if (!vec || n_heads < 1 || head_dim < 2 || head_dim % 2 || pos < 0) return 1;
  k_op_rope<<<1, 256, 0, (cudaStream_t)stream>>>(vec, n_heads, head_dim, pos, (double)base);
  return op_done();
}
extern "C" size_t spd_op_attention_scratch(int32_t t_len, int32_t n_q_heads, int32_t head_dim) {
  size_t nsplit = (size_t)(t_len + kAttnSplit - 1) / kAttnSplit;
  return nsplit * n_q_heads * ((size_t)head_dim + 2) * sizeof(float);
}
extern "C" int spd_op_attention(const float *q, const uint16_t *kc, const uint16_t *vc, int32_t t_len, int32_t t_stride,
                                int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, float *out, float *scratch,
                                void *stream) {
  if (!q || !kc || !vc || !out || !scratch || t_len < 1 || t_stride < t_len || n_kv_heads < 1 ||
      n_q_heads % n_kv_heads || n_q_heads / n_kv_heads > 32 || (head_dim != 64 && head_dim != 128))
    return 1;
  int nsplit = (t_len + kAttnSplit - 1) / kAttnSplit, group = n_q_heads / n_kv_heads;
  float *part_o = scratch;
  float2 *part_ml = reinterpret_cast<float2 *>(scratch + (size_t)nsplit * n_q_heads * head_dim);
  cudaStream_t s = (cudaStream_t)stream;
  if (head_dim == 128)
    k_op_attn_partial<128><<<dim3(nsplit, n_kv_heads), group * 32, 0, s>>>(q, kc, vc, t_len, t_stride, n_q_heads,
                                                                            n_kv_heads, nsplit, part_o, part_ml);
  else
    k_op_attn_partial<64><<<dim3(nsplit, n_kv_heads), group * 32, 0, s>>>(q, kc, vc, t_len, t_stride, n_q_heads,
                                                                           n_kv_heads, nsplit, part_o, part_ml);
  k_op_attn_merge<<<n_q_heads, head_dim, 0, s>>>(part_o, part_ml, nsplit, head_dim, out);
  return op_done();
}
extern "C" int spd_op_silu_mul(const float *gate, const float *up, int32_t n, float *out, void *stream) {
  if (!gate || !up || !out || n < 1) return 1;
  k_op_silu_mul<<<cdiv(n, 256), 256, 0, (cudaStream_t)stream>>>(gate, up, n, out);
  return op_done();
}
extern "C" int spd_op_argmax(const float *x, int32_t n, int32_t *out_index, void *stream) {
  if (!x || !out_index || n < 1) return 1;
  k_op_argmax<<<1, 1024, 0, (cudaStream_t)stream>>>(x, n, out_index);
  return op_done();
}

static const int kOpCand = 128;
extern "C" size_t spd_op_topk_scratch(void) { return (size_t)kOpCand * 8 + (size_t)kSampCap * 8; }
extern "C" int spd_op_topk_softmax(const float *x, int32_t n, int32_t top_k, float temperature, int32_t use_candidates,
                                   spd_sample_dist *out, void *scratch, void *stream) {
  static_assert(sizeof(spd_sample_dist) == sizeof(SampleDist), "dist layout");
  if (!x || !out || !scratch || n < 1 || top_k < 1 || top_k > kMaxTopK || !(temperature > 0.f)) return 1;
  float *cand_val = (float *)scratch;
  int32_t *cand_idx = (int32_t *)(cand_val + kOpCand);
  float *surv_val = (float *)(cand_idx + kOpCand);
  int32_t *surv_idx = (int32_t *)(surv_val + kSampCap);
  cudaStream_t s = (cudaStream_t)stream;
  if (use_candidates) k_op_cand<<<kOpCand, 256, 0, s>>>(x, n, cand_val, cand_idx);
  k_op_topk<<<1, 256, 0, s>>>(x, n, top_k, temperature, use_candidates ? kOpCand : 0, cand_val, cand_idx, surv_val,
                              surv_idx, reinterpret_cast<SampleDist *>(out));
  return op_done();
}
