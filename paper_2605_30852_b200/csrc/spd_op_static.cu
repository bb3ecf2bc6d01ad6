// spd_op_static.cu — spd_op_attention_static: the split-KV decode attention operation (the stage forward's
// attention) for callers that cannot allocate device memory (code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc).  Same arithmetic as spd_op_attention (spd_ref_engine.cu): fixed
// 128-row splits, one warp per q head and split, splits merged in split order — only the place of the split partials
// differs: a file-scope device array instead of a caller buffer.
//
// The array is part of the library image: every GPU that loads the library holds its kStaticScratchBytes (2 MiB) until the
// process exits.  All calls on a device share it, and it keeps the last call's contents:
//   * nothing has to start at zero — the partial kernel writes every (q head, split) slot before the merge kernel reads
//     it, and slots of an earlier, larger call are never read;
//   * two calls that overlap on the GPU (different streams, no dependency between them) RACE on it.  Calls on one stream
//     are ordered and safe.
// No cudaMalloc / cudaFree / allocating library routine is called here.
#include <mutex>

#include "../../include/spd.h"
#include "spd_kernels.cuh"

namespace spd {

constexpr size_t kStaticScratchBytes = 2u << 20;   // 2 MiB: e.g. 32 q heads x head_dim 128 up to 16128 rows
static __device__ __align__(256) unsigned char g_attn_scratch[kStaticScratchBytes];

constexpr int kMaxDevices = 64;
static void *g_scratch_ptr[kMaxDevices];            // device address of g_attn_scratch, per device (host-side cache)
static std::mutex g_scratch_mu;

// In host code `g_attn_scratch` is only a stand-in for the symbol; its device address on the CURRENT device comes from
// cudaGetSymbolAddress (once per device, with that device current).
static int static_scratch(void **out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return SPD_ECUDA; }
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (!g_scratch_ptr[dev]) {
    void *p = nullptr;
    if (cudaGetSymbolAddress(&p, g_attn_scratch) != cudaSuccess || !p) { cudaGetLastError(); return SPD_ECUDA; }
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return SPD_OK;
}

template <int HD>
__global__ void k_op_attn_partial_static(const float *q, const uint16_t *kc, const uint16_t *vc, int T, int t_stride, int Hq,
                                         int Hkv, int nsplit, float *part_o, float2 *part_ml) {
  const int split = blockIdx.x, kvh = blockIdx.y, group = Hq / Hkv;
  const int t0 = split * kAttnSplit, t1 = min(T, t0 + kAttnSplit);
  if (t0 >= T) return;
  const int hq = kvh * group + (threadIdx.x >> 5);
  const size_t slot = (size_t)hq * nsplit + split;
  attn_partial_warp<HD>(q + (size_t)hq * HD, kc + (size_t)kvh * t_stride * HD, vc + (size_t)kvh * t_stride * HD, t0, t1,
                        part_o + slot * HD, part_ml + slot);
}

__global__ void k_op_attn_merge_static(const float *part_o, const float2 *part_ml, int nsplit, int hd, float *out) {
  const int hq = blockIdx.x;
  const size_t slot = (size_t)hq * nsplit;
  out[(size_t)hq * hd + threadIdx.x] = attn_merge_elem(part_o + slot * hd, part_ml + slot, nsplit, hd, threadIdx.x);
}

}  // namespace spd

using namespace spd;

extern "C" size_t spd_op_attention_static_max_bytes(void) { return kStaticScratchBytes; }

extern "C" int spd_op_attention_static(const float *q, const uint16_t *kc, const uint16_t *vc, int32_t t_len, int32_t t_stride,
                                       int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim, float *out, void *stream) {
  if (!q || !kc || !vc || !out || t_len < 1 || t_stride < t_len || n_kv_heads < 1 || n_q_heads < 1 ||
      n_q_heads % n_kv_heads || n_q_heads / n_kv_heads > 32 || (head_dim != 64 && head_dim != 128))
    return SPD_EINVAL;
  const size_t nsplit = ((size_t)t_len + kAttnSplit - 1) / kAttnSplit;
  const size_t o_floats = nsplit * (size_t)n_q_heads * (size_t)head_dim;         // part_o; then part_ml (float2, 8-byte aligned)
  const size_t need = (o_floats + 2 * nsplit * (size_t)n_q_heads) * sizeof(float);
  if (need > kStaticScratchBytes) return SPD_ECAPACITY;    // beyond the static array: use spd_op_attention with a caller buffer
  void *base = nullptr;
  const int rc = static_scratch(&base);
  if (rc != SPD_OK) return rc;
  float *part_o = reinterpret_cast<float *>(base);
  float2 *part_ml = reinterpret_cast<float2 *>(part_o + o_floats);
  const int group = n_q_heads / n_kv_heads;
  cudaStream_t s = (cudaStream_t)stream;
  if (head_dim == 128)
    k_op_attn_partial_static<128><<<dim3((unsigned)nsplit, n_kv_heads), group * 32, 0, s>>>(q, kc, vc, t_len, t_stride, n_q_heads,
                                                                                          n_kv_heads, (int)nsplit, part_o, part_ml);
  else
    k_op_attn_partial_static<64><<<dim3((unsigned)nsplit, n_kv_heads), group * 32, 0, s>>>(q, kc, vc, t_len, t_stride, n_q_heads,
                                                                                         n_kv_heads, (int)nsplit, part_o, part_ml);
  k_op_attn_merge_static<<<n_q_heads, head_dim, 0, s>>>(part_o, part_ml, (int)nsplit, head_dim, out);
  return cudaGetLastError() == cudaSuccess ? SPD_OK : SPD_ECUDA;
}
