// spd_mega_dev.cuh — device-side building blocks shared by the two fused persistent engines (spd_mega.cu: one stage
// chain per CTA; spd_mega2.cu: two or three chains per CTA with a background stager): tile geometry, PTX wrappers (mbarrier,
// TMA bulk copies, ldmatrix / mma.sync), the consumer side of a GEMV phase (gemv_stream), of the LM-head pass
// (head_stream), attention items (scalar and tensor-core), the split merge and the fused unit epilogues.
// (CUDA path only; nothing here is used by, or taken from, oracle/.)
#pragma once
#include <cuda.h>
#include <stdio.h>
#include <string.h>

#include "spd_engine.h"
#include "spd_kernels.cuh"

namespace spd {

constexpr int kTileRows = 16;
constexpr int kTileCols = 512;
constexpr int kTileBytes = kTileRows * kTileCols * 2;   // 16 KB
constexpr int kStages = 11;                              // ring depth
constexpr int kXFloats = 12288;                          // activation vector capacity (48 KB)
constexpr int kConsumerThreads = 256;
constexpr int kThreads = kConsumerThreads + 32;
constexpr int kEndMark = -1;                             // slot tag: no more work in this phase
constexpr int kAttnScratchFloats = 2 * 8 * kAttnSplit + 8 * 8 * 128;   // scores, probabilities, per-warp partial outputs (G <= 8, hd <= 128)
constexpr int kQPairStride = 68;                         // u32 (bf16 pairs) per q head in the staged hi / lo arrays: 64 + 4 (bank spread)
constexpr int kAttnDoneMax = 32;                         // items whose completion counts are published together
static_assert(kAttnScratchFloats + kAttnDoneMax * 9 + 1 <= kXFloats, "attention scratch must fit the activation buffer");

enum PhaseType { PH_PDM = 0, PH_QKV = 1, PH_ATTN = 2, PH_O = 3, PH_GATEUP = 4, PH_DOWN = 5, PH_HEAD = 6 };

struct MegaLayout {
  const uint8_t *repack;
  unsigned long long layer_bytes, off_o, off_gu, off_dn, off_dnb, off_pdm, off_head, pdm_job_bytes;
  int u_qkv, u_o, u_gu, u_dn, u_pdm, u_head;   // 16-row units per job
  int nc_d, nc_qd, nc_f;                        // 512-column chunks for K = d, Hq*hd, F
  int attn_mma;                                 // full 128-row attention items go through the tensor cores
  // W_down is stored as two K parts: columns [0, nc_fa * 512) of every unit at off_dn, the other nc_f - nc_fa chunks at
  // off_dnb.  The one-chain engine streams a unit's tiles from both places in column order (same products, same order);
  // the two-chain engine runs the parts as two phases so that an activation buffer is 24 KB.
  int nc_fa;
  int chains;                                   // spd_mega2.cu: stage chains a CTA serves at most (SPD_OPT_CHAINS)
};

// Per-cycle schedule, computed identically by every CTA from the device state.
struct Sched {
  int mode, n_act, run_pdm, run_verify, p_new, c;
  int act[kMaxStages];                          // active stages (depth k), ascending
  int pos[kMaxStages], hbuf[kMaxStages], occ[kMaxStages];
  int my_stage;                                 // this CTA's stage in the layer phases (-1: none)
  int my_idx;                                   // index inside the stage's CTA group
  int my_gsize;                                 // CTAs in this CTA's stage group
  int exit_gsize;                               // CTAs in the group of stage n - 1 (0: that stage is empty)
  int pdm_slot, pdm_idx;                        // this CTA's slot (column block of W_p) in the PDM phase
  int attn_ns;                                  // 128-row splits of this CTA's stage in this cycle
  int attn_total;                               // attention items (kv head, split) of this CTA's stage in one pass
  int attn_nonfinal;                            // ... of which do not contain the row appended in this pass
};

struct PhaseDesc {                              // what one phase means for this CTA
  int type, job, U, nc;                         // job < 0: nothing to stream
  const uint8_t *base;                          // unit 0 of the job
  const uint8_t *base2;                         // W_down only: unit 0 of the second K part (tiles nc1 .. nc - 1 of a unit)
  int nc1;                                      // tiles of a unit that come from `base` (= nc except for W_down)
  unsigned int *ctr;                            // claim counter
};

struct AttnItem { int stage, kvh, split, nsplit, t0, rows; };

// ------------------------------------------------------------------ PTX helpers ----------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_n(uint64_t *bar, uint32_t n) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(n) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ void tma_load_1d(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
      ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy) : "memory");
}
// One 64 x 64 bf16 box (8 KB, 128-byte swizzled) of the K/V tensor map -> shared memory.
__device__ __forceinline__ void tma_load_box(void *dst_smem, const CUtensorMap *tmap, int c0, int c1, int c2, uint64_t *bar,
                                             uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;"
      ::"r"(smem_u32(dst_smem)), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)), "l"(policy) : "memory");
}
__device__ __forceinline__ void ldmatrix_x4(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
// D (16 x 8, fp32) += A (16 x 16, bf16, row) * B (16 x 8, bf16, col)
__device__ __forceinline__ void mma_bf16_16816(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                               uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// fp32 pair -> (bf16 hi pair, bf16 lo pair) with x = hi + lo to 16 mantissa bits: products with exact bf16 operands
// accumulated in fp32 keep ~fp32 accuracy.  Low half of a register = first element.
__device__ __forceinline__ void split_bf16x2(float x0, float x1, uint32_t &hi, uint32_t &lo) {
  const uint16_t h0 = f32_to_bf16(x0), h1 = f32_to_bf16(x1);
  const uint16_t l0 = f32_to_bf16(x0 - bf16_to_f32(h0)), l1 = f32_to_bf16(x1 - bf16_to_f32(h1));
  hi = (uint32_t)h0 | ((uint32_t)h1 << 16);
  lo = (uint32_t)l0 | ((uint32_t)l1 << 16);
}
// Orders generic-proxy accesses (st.global of the KV append) against async-proxy accesses (TMA reads).
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ void prof_stamp(const DevPtrs &P, int cta, int phase, int stamp) {
  if (P.prof_on && cta < kProfCtas && phase < kProfPhases)
    P.prof[((size_t)cta * kProfPhases + phase) * kProfStamps + stamp] = (unsigned long long)clock64();
}
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ void red_release_add_u32(unsigned int *p, unsigned int v) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_add_u64(unsigned long long *p, unsigned long long v) {
  asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int *p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ int phase_type(int p, int np) {
  if (p == 0) return PH_PDM;
  if (p == np - 1) return PH_HEAD;
  return PH_QKV + (p - 1) % 5;
}

// Pure function of (Sched, layout, phase) — the producer and the consumers both call it and must agree.
__device__ __forceinline__ PhaseDesc phase_desc(int p, int np, const Sched &S, const MegaLayout &ML, const Dims &D,
                                                unsigned int *claim) {
  PhaseDesc w;
  w.type = phase_type(p, np);
  w.job = -1; w.U = 0; w.nc = 0; w.nc1 = 0; w.base = nullptr; w.base2 = nullptr; w.ctr = claim + (size_t)p * kMaxStages;
  if (w.type == PH_PDM) {
    if (!S.run_pdm) return w;
    w.job = S.pdm_slot; w.U = ML.u_pdm; w.nc = ML.nc_d;
    w.base = ML.repack + ML.off_pdm + (unsigned long long)w.job * ML.pdm_job_bytes;
  } else if (w.type == PH_HEAD) {
    if (!S.run_pdm && !S.run_verify) return w;
    w.job = 0; w.U = ML.u_head; w.nc = ML.nc_d;
    w.base = ML.repack + ML.off_head;
  } else if (w.type == PH_ATTN) {
    if (S.my_stage >= 0) { w.job = S.my_stage; w.U = S.attn_total; }
  } else {
    if (S.my_stage < 0) return w;
    int pass = (p - 1) / 5;
    int layer = S.my_stage * D.per + pass;
    w.job = S.my_stage;
    const uint8_t *lb = ML.repack + (unsigned long long)layer * ML.layer_bytes;
    if (w.type == PH_QKV) { w.U = ML.u_qkv; w.nc = ML.nc_d; w.base = lb; }
    else if (w.type == PH_O) { w.U = ML.u_o; w.nc = ML.nc_qd; w.base = lb + ML.off_o; }
    else if (w.type == PH_GATEUP) { w.U = ML.u_gu; w.nc = ML.nc_d; w.base = lb + ML.off_gu; }
    else { w.U = ML.u_dn; w.nc = ML.nc_f; w.base = lb + ML.off_dn; w.base2 = lb + ML.off_dnb; w.nc1 = ML.nc_fa; }
  }
  if (w.base2 == nullptr) w.nc1 = w.nc;
  if (w.job >= 0) w.ctr += w.job;
  return w;
}

// Attention item of this CTA's stage -> (kv head, split).  Items [0, attn_nonfinal) are the splits that do
// not contain the row appended in this pass (kv head major) — their K/V rows are old and can be fetched
// before the QKV phase has finished; items [attn_nonfinal, attn_total) are the last split of every kv head.
__device__ __forceinline__ void attn_decode(int stage, int nsplit, int nonfinal, int pos, int item, AttnItem &it) {
  it.stage = stage; it.nsplit = nsplit;
  if (item < nonfinal) {
    it.kvh = item / (it.nsplit - 1);
    it.split = item - it.kvh * (it.nsplit - 1);
  } else {
    it.kvh = item - nonfinal;
    it.split = it.nsplit - 1;
  }
  it.t0 = it.split * kAttnSplit;
  it.rows = min(pos + 1 - it.t0, kAttnSplit);
}
__device__ __forceinline__ void attn_decode(const Sched &S, const Dims &D, int item, AttnItem &it) {
  attn_decode(S.my_stage, S.attn_ns, S.attn_nonfinal, S.pos[S.my_stage], item, it);
}

// ------------------------------------------------------------------ consumer pieces ------------
// 8 fp32 FMAs of one 16-byte weight chunk against two float4 of x.
__device__ __forceinline__ float fma8(uint4 w, float4 xa, float4 xb, float acc) {
  acc = fmaf(bf16_lo(w.x), xa.x, acc); acc = fmaf(bf16_hi(w.x), xa.y, acc);
  acc = fmaf(bf16_lo(w.y), xa.z, acc); acc = fmaf(bf16_hi(w.y), xa.w, acc);
  acc = fmaf(bf16_lo(w.z), xb.x, acc); acc = fmaf(bf16_hi(w.z), xb.y, acc);
  acc = fmaf(bf16_lo(w.w), xb.z, acc); acc = fmaf(bf16_hi(w.w), xb.w, acc);
  return acc;
}

// Sum over the 256 consumer threads with a fixed tree: warp xor-tree, then the 8 warp partials in order.
__device__ __forceinline__ float consumer_sum(float v, float *red) {
  v = warp_sum(v);
  consumer_sync();                      // protect `red` against a previous use
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  consumer_sync();
  float t = 0.f;
#pragma unroll
  for (int w = 0; w < 8; ++w) t += red[w];
  return t;
}

// Copies K fp32 values (K % 4 == 0) written by other CTAs (ld.global.cg, 128-bit) into shared memory;
// returns this thread's sum of squares.  Thread t owns float4 t, t + 256, ...
__device__ __forceinline__ float stage_copy(const float *src, float *dst, int K) {
  const float4 *s4 = reinterpret_cast<const float4 *>(src);
  float4 *d4 = reinterpret_cast<float4 *>(dst);
  const int n4 = K >> 2;
  float ss = 0.f;
#pragma unroll 4
  for (int i = threadIdx.x; i < n4; i += kConsumerThreads) {
    float4 v = __ldcg(s4 + i);
    d4[i] = v;
    ss = fmaf(v.x, v.x, ss); ss = fmaf(v.y, v.y, ss); ss = fmaf(v.z, v.z, ss); ss = fmaf(v.w, v.w, ss);
  }
  return ss;
}

// xs[i] *= r * gain[i] for the float4s this thread wrote in stage_copy.
__device__ __forceinline__ void stage_scale(float *xs, const uint16_t *gain, int K, float r) {
  float4 *d4 = reinterpret_cast<float4 *>(xs);
  const uint2 *g2 = reinterpret_cast<const uint2 *>(gain);
  const int n4 = K >> 2;
  for (int i = threadIdx.x; i < n4; i += kConsumerThreads) {
    float4 v = d4[i];
    uint2 g = __ldg(g2 + i);
    v.x = v.x * r * bf16_lo(g.x); v.y = v.y * r * bf16_hi(g.x);
    v.z = v.z * r * bf16_lo(g.y); v.w = v.w * r * bf16_hi(g.y);
    d4[i] = v;
  }
}

// Transposed butterfly reduction.  Every lane holds N partial sums v[0..N); the lanes that differ in the
// bits below 2*OFF hold partials of the same N quantities.  Each level halves the values a lane keeps
// (lane bit set: the upper half) and adds the partner's partials of the kept half; when one value is
// left the remaining levels are plain xor-sums.  Afterwards v[0..max(N/W,1)) are complete sums of the
// quantities base * max(N/W,1) + i, where `base` collects the lane bits of the halving levels (first
// level = most significant).  N - 1 shuffles instead of N * log2(W).
template <int N, int OFF>
struct XReduce {
  static __device__ __forceinline__ void run(float *v, int lane, int &base) {
    if constexpr (OFF >= 1) {
      if constexpr (N > 1) {
        constexpr int H = N / 2;
        const bool up = (lane & OFF) != 0;
#pragma unroll
        for (int i = 0; i < H; ++i) {
          float send = up ? v[i] : v[i + H];
          float keep = up ? v[i + H] : v[i];
          v[i] = keep + __shfl_xor_sync(0xffffffffu, send, OFF);
        }
        base = base * 2 + (up ? 1 : 0);
        XReduce<H, OFF / 2>::run(v, lane, base);
      } else {
        v[0] += __shfl_xor_sync(0xffffffffu, v[0], OFF);
        XReduce<1, OFF / 2>::run(v, lane, base);
      }
    }
  }
};

// One attention item: the G q heads of kv head `kvh` of the token at stage `stage`, over K/V rows
// [t0, t0 + rows) that the producer placed in ring slots seq0.. (K: nk slots, then V: nk slots).
// Writes the unnormalised partial output and (max, sum) of every head; the caller merges.
// scratch (the activation buffer, free during attention): sc[G][128] scores, ps[128][G] probabilities,
// red[8][G][HD] per-warp partial outputs.
template <int HD, int G>
__device__ __forceinline__ void attn_item(const DevPtrs &P, const AttnItem &it, const uint8_t *ring, uint32_t seq0, int nk,
                                          float *scratch, uint64_t *empty, const float *qsm = nullptr, int qslot = -1) {
  constexpr int CH = HD / 8;            // 16-byte chunks (= lanes) per K row
  constexpr int RPI = 32 / CH;          // rows covered by one warp-wide LDS.128
  constexpr int NI = 16 / RPI;          // iterations for a warp's 16 rows
  constexpr int NV = NI * G;            // partial scores per lane
  constexpr int NF = NV >= CH ? NV / CH : 1;
  constexpr int RPS = kTileBytes / (HD * 2);   // rows per ring slot
  constexpr int EPL = HD / 32;          // head-dim elements per lane in P.V
  const Dims &D = P.dim;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  float *sc = scratch, *ps = scratch + G * kAttnSplit, *red = scratch + 2 * G * kAttnSplit;
  const int hq0 = it.kvh * G;
  const int rows = it.rows;

  // ---- scores: lane (rsel, c) owns chunk c of rows 16*warp + i*RPI + rsel ----
  {
    const int c = lane % CH, rsel = lane / CH;
    float qv[G][8];
#pragma unroll
    for (int h = 0; h < G; ++h) {
      // q of the G heads: from the ring slot the producer filled (qsm, engine 2) or from global memory (written by other CTAs)
      const float4 *q4 = reinterpret_cast<const float4 *>((qsm ? qsm + (size_t)h * HD : P.q + ((size_t)it.stage * D.Hq + hq0 + h) * HD) + c * 8);
      float4 a, b;
      if (qsm) { a = q4[0]; b = q4[1]; } else { a = __ldcg(q4); b = __ldcg(q4 + 1); }
      qv[h][0] = a.x; qv[h][1] = a.y; qv[h][2] = a.z; qv[h][3] = a.w;
      qv[h][4] = b.x; qv[h][5] = b.y; qv[h][6] = b.z; qv[h][7] = b.w;
    }
    float v[NV];
#pragma unroll
    for (int i = 0; i < NI; ++i) {
      const int row = 16 * warp + i * RPI + rsel;
      uint4 kw = make_uint4(0u, 0u, 0u, 0u);
      if (row < rows) {
        const uint8_t *tile = ring + (size_t)((seq0 + row / RPS) % kStages) * kTileBytes;
        kw = *reinterpret_cast<const uint4 *>(tile + (size_t)(row % RPS) * (HD * 2) + c * 16);
      }
      const float k0 = bf16_lo(kw.x), k1 = bf16_hi(kw.x), k2 = bf16_lo(kw.y), k3 = bf16_hi(kw.y);
      const float k4 = bf16_lo(kw.z), k5 = bf16_hi(kw.z), k6 = bf16_lo(kw.w), k7 = bf16_hi(kw.w);
#pragma unroll
      for (int h = 0; h < G; ++h) {
        float a = k0 * qv[h][0];
        a = fmaf(k1, qv[h][1], a); a = fmaf(k2, qv[h][2], a); a = fmaf(k3, qv[h][3], a);
        a = fmaf(k4, qv[h][4], a); a = fmaf(k5, qv[h][5], a); a = fmaf(k6, qv[h][6], a); a = fmaf(k7, qv[h][7], a);
        v[i * G + h] = a;
      }
    }
    int base = 0;
    XReduce<NV, CH / 2>::run(v, lane, base);
    const float scale = 1.0f / sqrtf((float)HD);
#pragma unroll
    for (int i = 0; i < NF; ++i) {
      const int idx = base * NF + i, itn = idx / G, h = idx % G;
      sc[h * kAttnSplit + 16 * warp + itn * RPI + rsel] = v[i] * scale;
    }
  }
  consumer_sync();
  if (lane == 0) {
    for (int j = 0; j < nk; ++j) mbar_arrive(&empty[(seq0 + j) % kStages]);   // K slots are free
    if (qslot >= 0) mbar_arrive(&empty[qslot]);                               // ... and the q slot
  }
  // ---- softmax of the split, one warp per head: m = max, p = exp(s - m), l = sum p ----
  if (warp < G) {
    float s[kAttnSplit / 32], m = -INFINITY;
#pragma unroll
    for (int j = 0; j < kAttnSplit / 32; ++j) {
      int r = lane + 32 * j;
      s[j] = r < rows ? sc[warp * kAttnSplit + r] : -INFINITY;
      m = fmaxf(m, s[j]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    float l = 0.f;
#pragma unroll
    for (int j = 0; j < kAttnSplit / 32; ++j) {
      int r = lane + 32 * j;
      float p = r < rows ? expf(s[j] - m) : 0.f;
      ps[r * G + warp] = p;
      l += p;
    }
    l = warp_sum(l);
    if (lane == 0) {
      size_t slot = ((size_t)it.stage * D.Hq + hq0 + warp) * P.nsplit_max + it.split;
      P.part_ml[slot] = make_float2(m, l);
    }
  }
  consumer_sync();
  // ---- P.V: warp w sums its 16 rows for all G heads; lane owns EPL consecutive head-dim elements ----
  {
    float acc[G][EPL];
#pragma unroll
    for (int h = 0; h < G; ++h)
#pragma unroll
      for (int e = 0; e < EPL; ++e) acc[h][e] = 0.f;
#pragma unroll 4
    for (int i = 0; i < 16; ++i) {
      const int row = 16 * warp + i;
      if (row < rows) {
        const uint8_t *tile = ring + (size_t)((seq0 + nk + row / RPS) % kStages) * kTileBytes;
        const uint8_t *vr = tile + (size_t)(row % RPS) * (HD * 2) + lane * (EPL * 2);
        float vv[EPL];
        if constexpr (EPL == 4) {
          uint2 w = *reinterpret_cast<const uint2 *>(vr);
          vv[0] = bf16_lo(w.x); vv[1] = bf16_hi(w.x); vv[2] = bf16_lo(w.y); vv[3] = bf16_hi(w.y);
        } else {
          uint32_t w = *reinterpret_cast<const uint32_t *>(vr);
          vv[0] = bf16_lo(w); vv[1] = bf16_hi(w);
        }
        float pr[G];
        if constexpr (G == 4) {
          float4 t = *reinterpret_cast<const float4 *>(ps + row * G);
          pr[0] = t.x; pr[1] = t.y; pr[2] = t.z; pr[3] = t.w;
        } else if constexpr (G == 8) {
          float4 t = *reinterpret_cast<const float4 *>(ps + row * G), u = *reinterpret_cast<const float4 *>(ps + row * G + 4);
          pr[0] = t.x; pr[1] = t.y; pr[2] = t.z; pr[3] = t.w; pr[4] = u.x; pr[5] = u.y; pr[6] = u.z; pr[7] = u.w;
        } else {
#pragma unroll
          for (int h = 0; h < G; ++h) pr[h] = ps[row * G + h];
        }
#pragma unroll
        for (int h = 0; h < G; ++h)
#pragma unroll
          for (int e = 0; e < EPL; ++e) acc[h][e] = fmaf(pr[h], vv[e], acc[h][e]);
      }
    }
    __syncwarp();
    if (lane == 0) for (int j = 0; j < nk; ++j) mbar_arrive(&empty[(seq0 + nk + j) % kStages]);   // V slots are free
#pragma unroll
    for (int h = 0; h < G; ++h)
#pragma unroll
      for (int e = 0; e < EPL; ++e) red[((size_t)warp * G + h) * HD + lane * EPL + e] = acc[h][e];
  }
  consumer_sync();
  // ---- cross-warp sum in warp order (fixed), unnormalised partial output of the split ----
  for (int o = tid; o < G * HD; o += kConsumerThreads) {
    const int h = o / HD, e = o - h * HD;
    float t = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) t += red[((size_t)w * G + h) * HD + e];
    size_t slot = ((size_t)it.stage * D.Hq + hq0 + h) * P.nsplit_max + it.split;
    P.part_o[slot * HD + e] = t;
  }
}

// Tensor-core version of attn_item for a FULL split (128 rows) at head_dim 128.  The scalar path spends ~1000 issue
// slots per warp and item (4 q heads x 128 dims x 128 rows of fp32 FMAs on unpacked bf16) and makes the attention
// phase issue-bound; here scores (Q K^T) and P.V run as mma.sync m16n8k16 with the G q heads in rows 0..G-1 of the
// 16-row A operand.  q and the probabilities are fp32 (C-2.17), so each is split into bf16 hi + lo parts (hi in rows
// 0..G-1, lo in rows 8..8+G-1 of the same A operand, the two result rows are added): K and V are exact bf16,
// products are exact and accumulate in fp32, which keeps ~2^-17 relative accuracy per element.  K/V arrive as 128-byte-swizzled 64 x 64 boxes (tma_load_box): chunk c of row r sits at
// r * 128 + ((c ^ (r & 7)) << 4), so every ldmatrix phase touches 8 distinct 16-byte bank groups.  Warp w owns rows
// 16 w .. 16 w + 15 of the split (fixed) and runs scores -> softmax over its 16 rows -> P.V entirely in registers (the
// score fragment of thread (g, t) is the P.V A fragment); the 8 warps' (max, sum, output) are merged in warp order
// after one CTA barrier, the splits in split order: results do not depend on who ran the item.
template <int G>
__device__ __forceinline__ void attn_item_mma(const DevPtrs &P, const AttnItem &it, const uint8_t *ring, uint32_t seq0,
                                              float *scratch, uint64_t *empty, const uint32_t *qs, const float *qsm = nullptr,
                                              int qslot = -1) {
  constexpr int HD = 128, nk = 2;
  const Dims &D = P.dim;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, t = lane & 3;          // mma fragment coordinates
  const int mi = lane >> 3, mr = lane & 7;        // ldmatrix: this lane addresses row mr of matrix mi
  float2 *wml = reinterpret_cast<float2 *>(scratch);   // [8 warps][G] (max, sum) of a warp's 16 rows
  float *red = scratch + 2 * G * kAttnSplit;           // [8 warps][G][HD] unnormalised outputs (same place as attn_item)
  const int hq0 = it.kvh * G;
  const int rb = warp >> 2, r0 = (warp & 3) * 16; // this warp's rows: slot rb, local rows r0 .. r0 + 15
  float p0, p1, p2, p3;                           // probabilities of head g at rows 2t, 2t+1, 8+2t, 9+2t

  // ---- scores S[head][row] = q . K[row]: A = Q (head g in row g < G, other rows zero), B = K^T ----
  {
    uint32_t qh[8][2], ql[8][2];                  // per k-step: a0 (dims 16 ks + 2t, +1), a2 (dims 16 ks + 8 + 2t, +1)
#pragma unroll
    for (int ks = 0; ks < 8; ++ks) { qh[ks][0] = qh[ks][1] = ql[ks][0] = ql[ks][1] = 0u; }
    if (g < G) {
      if (qs) {                                   // staged once per phase: hi pairs, then lo pairs, kQPairStride per head
        const uint32_t *h = qs + (size_t)(hq0 + g) * kQPairStride, *l = h + (size_t)D.Hq * kQPairStride;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
          qh[ks][0] = h[8 * ks + t]; qh[ks][1] = h[8 * ks + 4 + t];
          ql[ks][0] = l[8 * ks + t]; ql[ks][1] = l[8 * ks + 4 + t];
        }
      } else if (qsm) {                           // fp32 q of the G heads in a ring slot (engine 2: brought by the producer)
        const float *q = qsm + (size_t)g * HD;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
          const float2 x = *reinterpret_cast<const float2 *>(q + 16 * ks + 2 * t);
          const float2 y = *reinterpret_cast<const float2 *>(q + 16 * ks + 8 + 2 * t);
          split_bf16x2(x.x, x.y, qh[ks][0], ql[ks][0]);
          split_bf16x2(y.x, y.y, qh[ks][1], ql[ks][1]);
        }
      } else {
        const float *q = P.q + ((size_t)it.stage * D.Hq + hq0 + g) * HD;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
          const float2 x = __ldcg(reinterpret_cast<const float2 *>(q + 16 * ks + 2 * t));
          const float2 y = __ldcg(reinterpret_cast<const float2 *>(q + 16 * ks + 8 + 2 * t));
          split_bf16x2(x.x, x.y, qh[ks][0], ql[ks][0]);
          split_bf16x2(y.x, y.y, qh[ks][1], ql[ks][1]);
        }
      }
    }
    float sa[2][4];
#pragma unroll
    for (int i = 0; i < 2; ++i) { sa[i][0] = sa[i][1] = sa[i][2] = sa[i][3] = 0.f; }
    const uint32_t kbase = smem_u32(ring + (size_t)((seq0 + rb) % kStages) * kTileBytes);
    const int krow = r0 + (mi >> 1) * 8 + mr;     // matrices 0, 1: rows 0..7 (dims lo, hi); 2, 3: rows 8..15
#pragma unroll
    for (int ks = 0; ks < 8; ++ks) {
      const int cc = 2 * ks + (mi & 1);           // 16-byte chunk of the 256-byte row
      uint32_t b[4];
      ldmatrix_x4(b, kbase + (cc >> 3) * (kTileBytes / 2) + krow * 128 + (((cc & 7) ^ (krow & 7)) << 4));
      mma_bf16_16816(sa[0], qh[ks][0], ql[ks][0], qh[ks][1], ql[ks][1], b[0], b[1]);   // rows g: hi part, rows g + 8: lo part
      mma_bf16_16816(sa[1], qh[ks][0], ql[ks][0], qh[ks][1], ql[ks][1], b[2], b[3]);
    }
    // ---- softmax of this warp's 16 rows, in registers (flash-attention style): thread (g, t) holds the scores of
    //      head g for rows 2t, 2t+1, 8+2t, 9+2t, which is exactly the A fragment P.V needs ----
    const float scale = 1.0f / sqrtf((float)HD);
    const float s0 = (sa[0][0] + sa[0][2]) * scale, s1 = (sa[0][1] + sa[0][3]) * scale;
    const float s2 = (sa[1][0] + sa[1][2]) * scale, s3 = (sa[1][1] + sa[1][3]) * scale;
    float m = fmaxf(fmaxf(s0, s1), fmaxf(s2, s3));
    m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 1));
    m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 2));
    p0 = expf(s0 - m); p1 = expf(s1 - m); p2 = expf(s2 - m); p3 = expf(s3 - m);
    float l = (p0 + p1) + (p2 + p3);
    l += __shfl_xor_sync(0xffffffffu, l, 1);
    l += __shfl_xor_sync(0xffffffffu, l, 2);
    if (g < G && t == 0) wml[warp * G + g] = make_float2(m, l);
  }
  __syncwarp();
  if (lane == 0) {
    for (int j = 0; j < nk; ++j) mbar_arrive(&empty[(seq0 + j) % kStages]);   // this warp is done with K
    if (qslot >= 0) mbar_arrive(&empty[qslot]);                               // ... and with q
  }
  // ---- P.V: O[head][dim] = sum over this warp's 16 rows: A = P (k = rows), B = V via ldmatrix.trans ----
  {
    uint32_t ph[2] = {0u, 0u}, pl[2] = {0u, 0u};  // a0: rows 2t, 2t+1; a2: rows 2t+8, 2t+9 (of the warp's 16)
    if (g < G) {
      split_bf16x2(p0, p1, ph[0], pl[0]);
      split_bf16x2(p2, p3, ph[1], pl[1]);
    }
    float oa[16][4];
#pragma unroll
    for (int j = 0; j < 16; ++j) { oa[j][0] = oa[j][1] = oa[j][2] = oa[j][3] = 0.f; }
    const uint32_t vbase = smem_u32(ring + (size_t)((seq0 + nk + rb) % kStages) * kTileBytes);
    const int vrow = r0 + (mi & 1) * 8 + mr;      // matrices 0, 1: rows 0..7, 8..15 of dims tile 2 jj; 2, 3: of tile 2 jj + 1
#pragma unroll
    for (int jj = 0; jj < 8; ++jj) {
      const int cc = 2 * jj + (mi >> 1);
      uint32_t b[4];
      ldmatrix_x4_trans(b, vbase + (cc >> 3) * (kTileBytes / 2) + vrow * 128 + (((cc & 7) ^ (vrow & 7)) << 4));
      mma_bf16_16816(oa[2 * jj], ph[0], pl[0], ph[1], pl[1], b[0], b[1]);              // rows g: hi part, rows g + 8: lo part
      mma_bf16_16816(oa[2 * jj + 1], ph[0], pl[0], ph[1], pl[1], b[2], b[3]);
    }
    __syncwarp();
    if (lane == 0) for (int j = 0; j < nk; ++j) mbar_arrive(&empty[(seq0 + nk + j) % kStages]);   // ... and with V
    if (g < G) {
#pragma unroll
      for (int j = 0; j < 16; ++j)
        *reinterpret_cast<float2 *>(red + ((size_t)warp * G + g) * HD + 8 * j + 2 * t) =
            make_float2(oa[j][0] + oa[j][2], oa[j][1] + oa[j][3]);
    }
  }
  consumer_sync();
  // ---- the 8 warps' (max, sum, unnormalised output) of every head, merged in warp order (fixed):
  //      M = max m_w, o = sum_w o_w e^(m_w - M), l = sum_w l_w e^(m_w - M) -> the split's partial ----
  for (int o = tid; o < G * HD; o += kConsumerThreads) {
    const int h = o / HD, e = o - h * HD;
    float M = -INFINITY;
#pragma unroll
    for (int w = 0; w < 8; ++w) M = fmaxf(M, wml[w * G + h].x);
    float acc = 0.f, L = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
      const float2 ml = wml[w * G + h];
      const float f = expf(ml.x - M);
      acc = fmaf(red[((size_t)w * G + h) * HD + e], f, acc);
      L = fmaf(ml.y, f, L);
    }
    const size_t slot = ((size_t)it.stage * D.Hq + hq0 + h) * P.nsplit_max + it.split;
    P.part_o[slot * HD + e] = acc;
    if (e == 0) P.part_ml[slot] = make_float2(M, L);
  }
  consumer_sync();                                // red / wml are rewritten by the next item
}

// Merge of the splits of one q head by one warp, in split order (fixed): out = sum_j o_j e^(m_j-M) / sum_j l_j e^(m_j-M).
// Lane owns EPL consecutive elements; the loads of different splits are independent and batched.
template <int HD>
__device__ __forceinline__ void attn_merge_warp(const DevPtrs &P, int stage, int hq, int nsplit, int lane) {
  constexpr int EPL = HD / 32;
  const Dims &D = P.dim;
  const size_t slot = ((size_t)stage * D.Hq + hq) * P.nsplit_max;
  const float2 *ml = P.part_ml + slot;
  float M = -INFINITY;
  for (int j = lane; j < nsplit; j += 32) M = fmaxf(M, __ldcg(&ml[j].x));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
  float L = 0.f, acc[EPL];
#pragma unroll
  for (int e = 0; e < EPL; ++e) acc[e] = 0.f;
  const float *po = P.part_o + slot * HD + lane * EPL;
#pragma unroll 8
  for (int j = 0; j < nsplit; ++j) {
    float2 mlj = __ldcg(&ml[j]);
    float v[EPL];
    if constexpr (EPL == 4) {
      float4 t = __ldcg(reinterpret_cast<const float4 *>(po + (size_t)j * HD));
      v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
    } else {
      float2 t = __ldcg(reinterpret_cast<const float2 *>(po + (size_t)j * HD));
      v[0] = t.x; v[1] = t.y;
    }
    float wj = expf(mlj.x - M);
    L = fmaf(mlj.y, wj, L);
#pragma unroll
    for (int e = 0; e < EPL; ++e) acc[e] = fmaf(v[e], wj, acc[e]);
  }
  float *out = P.att + ((size_t)stage * D.Hq + hq) * HD + lane * EPL;
#pragma unroll
  for (int e = 0; e < EPL; ++e) out[e] = acc[e] / L;
}

// Fused epilogue of one 16-row unit (lane 0 of every warp; rows r0, r0 + 1 of the repacked matrix).
template <class SchedT>
__device__ __forceinline__ void unit_epilogue(const DevPtrs &P, const SchedT &S, int t, int k, int pass, int r0, float y0,
                                              float y1, const float2 *rope_s) {
  const Dims &D = P.dim;
  if (t == PH_QKV) {
    const int qd = D.Hq * D.hd, kd = D.Hkv * D.hd, half = D.hd / 2, pos = S.pos[k];
    const int layer = k * D.per + pass;
    if (r0 < qd) {                           // q pair (i, i + hd/2) of head hh: RoPE (C-2.14)
      int hh = r0 / D.hd, i = (r0 - hh * D.hd) >> 1;
      float2 cs = rope_s[i];
      float *q = P.q + (size_t)k * qd + hh * D.hd;
      q[i] = y0 * cs.x - y1 * cs.y;
      q[i + half] = y1 * cs.x + y0 * cs.y;
    } else if (r0 < qd + kd) {               // k pair: RoPE, bf16 (RNE), append at row pos
      int rr = r0 - qd, hh = rr / D.hd, i = (rr - hh * D.hd) >> 1;
      float2 cs = rope_s[i];
      if (pos < D.max_seq) {
        uint16_t *dst = P.kv + kv_offset(D, layer, 0, hh) + (size_t)pos * D.hd;
        dst[i] = f32_to_bf16(y0 * cs.x - y1 * cs.y);
        dst[i + half] = f32_to_bf16(y1 * cs.x + y0 * cs.y);
      }
    } else if (r0 < qd + 2 * kd) {           // two consecutive v elements: bf16, append
      int rr = r0 - qd - kd, hh = rr / D.hd, i = rr - hh * D.hd;
      if (pos < D.max_seq) {
        uint16_t *dst = P.kv + kv_offset(D, layer, 1, hh) + (size_t)pos * D.hd;
        *reinterpret_cast<uint32_t *>(dst + i) = (uint32_t)f32_to_bf16(y0) | ((uint32_t)f32_to_bf16(y1) << 16);
      }
    }
  } else if (t == PH_O || t == PH_DOWN) {    // residual add
    float *h = P.h + (size_t)S.hbuf[k] * D.d;
    if (r0 + 1 < D.d) {
      float2 v = __ldcg(reinterpret_cast<const float2 *>(h + r0));
      *reinterpret_cast<float2 *>(h + r0) = make_float2(v.x + y0, v.y + y1);
    } else if (r0 < D.d) {
      h[r0] = __ldcg(h + r0) + y0;
    }
  } else if (t == PH_GATEUP) {               // rows (gate_i, up_i): SwiGLU
    int i = r0 >> 1;
    if (i < D.F) P.act[(size_t)k * D.F + i] = silu_mul(y0, y1);
  } else if (t == PH_PDM) {
    if (r0 < D.d) P.pdm_part[(size_t)k * D.d + r0] = y0;
    if (r0 + 1 < D.d) P.pdm_part[(size_t)k * D.d + r0 + 1] = y1;
  }                                          // PH_HEAD: head_stream() has its own epilogue
}

template <int HD>
__device__ __forceinline__ void attn_item_g(const DevPtrs &P, const AttnItem &it, const uint8_t *ring, uint32_t seq0, int nk,
                                            float *scratch, uint64_t *empty, int G, const float *qsm = nullptr, int qslot = -1) {
  if (G == 4) attn_item<HD, 4>(P, it, ring, seq0, nk, scratch, empty, qsm, qslot);
  else if (G == 2) attn_item<HD, 2>(P, it, ring, seq0, nk, scratch, empty, qsm, qslot);
  else if (G == 8) attn_item<HD, 8>(P, it, ring, seq0, nk, scratch, empty, qsm, qslot);
  else attn_item<HD, 1>(P, it, ring, seq0, nk, scratch, empty, qsm, qslot);
}

// Slot protocol of the tile-per-warp-pair mapping.  Only the owner pair of a tile reads its data, but EVERY
// consumer warp still waits on every slot's full barrier in ring order and arrives on its empty barrier (the
// non-owners right away, without touching the tile).  A slot is therefore recycled only after all 8 warps have
// passed it, exactly as when all warps read every tile: a parity wait can never observe a slot two phases late.
// One GEMV phase (M = 1) over the units the producer claimed for this CTA.  A tile (16 rows x 512 columns) is
// consumed by ONE warp pair: pair p = warp >> 1 owns the chunks c = p, p + 4, ... of every unit and its two
// warps take rows 0..7 / 8..15 of the tile, so a tile's slice of x is read from shared memory by 2 warps
// instead of 8 (the old row-per-warp mapping moved 48 KB of shared-memory traffic per 16 KB tile and capped an
// SM at ~60 GB/s; this one moves 36 KB).  Per unit a lane accumulates 8 rows over its columns, a transposed
// butterfly leaves the warp's partial of row q = lane >> 2 of its half in 4 lanes, the partials go through
// shared memory (double-buffered, one named barrier per unit) and warp (unit count mod 8) adds the 4 pair
// partials of every row in pair order and runs the fused epilogue on row pairs (even lanes 0..14).
template <class SchedT>
__device__ __forceinline__ void gemv_stream(const DevPtrs &P, const SchedT &S, int t, int k, int pass, int nc,
                                            const uint8_t *ring, uint64_t *full, uint64_t *empty, const int *meta,
                                            const float *xs, float *part, uint32_t &seq, const float2 *rope_s) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int pair = warp >> 1, half = warp & 1;
  const float4 *xv4 = reinterpret_cast<const float4 *>(xs);
  int ucount = 0;
  while (true) {
    const uint32_t s0 = seq;
    mbar_wait(&full[s0 % kStages], (s0 / kStages) & 1);
    const int u = meta[s0 % kStages];
    if (u == kEndMark) {
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s0 % kStages]);
      ++seq;
      break;
    }
    float acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = 0.f;
    for (int c = 0; c < nc; ++c) {
      const uint32_t sq = s0 + c, slot = sq % kStages;
      if (c > 0) mbar_wait(&full[slot], (sq / kStages) & 1);
      if ((c & 3) == pair) {
        const uint4 *wt = reinterpret_cast<const uint4 *>(ring + (size_t)slot * kTileBytes) + half * (8 * 64);
        const float4 *x4 = xv4 + c * (kTileCols / 4);
        const float4 x00 = x4[lane], x01 = x4[32 + lane], x10 = x4[64 + lane], x11 = x4[96 + lane];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          const uint4 w0 = wt[r * 64 + lane], w1 = wt[r * 64 + 32 + lane];
          acc[r] = fma8(w0, x00, x01, acc[r]);
          acc[r] = fma8(w1, x10, x11, acc[r]);
        }
        __syncwarp();
      }
      if (lane == 0) mbar_arrive(&empty[slot]);
    }
    seq += nc;
    int q = 0;
    XReduce<8, 16>::run(acc, lane, q);                   // q == lane >> 2: row q of this warp's half
    if ((lane & 3) == 0) part[(ucount & 1) * 64 + warp * 8 + q] = acc[0];
    consumer_sync();
    if (warp == (ucount & 7)) {
      const int r16 = lane & 15;
      const float *pp = part + (ucount & 1) * 64 + (r16 >> 3) * 8 + (r16 & 7);
      float y = 0.f;
#pragma unroll
      for (int pr = 0; pr < 4; ++pr) y += pp[pr * 16];   // warps 2 pr + (r16 >> 3), pr ascending
      const float y1 = __shfl_down_sync(0xffffffffu, y, 1);
      if (lane < 16 && (lane & 1) == 0) unit_epilogue(P, S, t, k, pass, u * kTileRows + r16, y, y1, rope_s);
    }
    ++ucount;
  }
}

// LM-head pass (M = 2: the verify and the PDM vector against the tied matrix E, read once).  With both vectors
// in shared memory the pass is bound by shared-memory bandwidth (16 KB of TMA writes + 16 KB of weight reads +
// 32 KB of x reads per tile), not by HBM.  Here K is split across the consumer warps by whole tiles: the warp
// pair p = warp >> 1 owns the chunks c = p, p + 4, ... of every unit (its two warps take rows 0..7 and 8..15 of
// the tile), so the pair's 512-column slices of both vectors live in REGISTERS and a tile costs only its own
// 16 KB of reads.  Per unit a lane accumulates 8 rows x 2 vectors over its columns, a transposed butterfly
// leaves the warp's partial of quantity q (vector q >> 3, row q & 7 of the warp's half) in lanes 2q, 2q + 1, the
// warp partials go through shared memory (double-buffered, one named barrier per unit) and are added in warp
// order by warp (unit count mod 8), whose lanes keep a running (value, index) maximum.  Fixed mapping and
// order: a logit never depends on which CTA claimed the unit.
template <int NXS>
__device__ __forceinline__ void head_stream(const DevPtrs &P, int nc, bool do_v, bool do_p, const uint8_t *ring,
                                            uint64_t *full, uint64_t *empty, const int *meta, float *xs, uint32_t &seq,
                                            float *cbest_v, int *cbest_i) {
  const Dims &D = P.dim;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int pair = warp >> 1, half = warp & 1;
  float4 xv[NXS][4], xp[NXS][4];
#pragma unroll
  for (int s = 0; s < NXS; ++s) {
    const int c = pair + 4 * s;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      xv[s][i] = make_float4(0.f, 0.f, 0.f, 0.f);
      xp[s][i] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (c < nc) {
        if (do_v) xv[s][i] = reinterpret_cast<const float4 *>(xs)[c * (kTileCols / 4) + 32 * i + lane];
        if (do_p) xp[s][i] = reinterpret_cast<const float4 *>(xs + kXFloats / 2)[c * (kTileCols / 4) + 32 * i + lane];
      }
    }
  }
  consumer_sync();                       // both vectors are in registers: xs is free for the warp partials
  float *part = xs;                      // [2][8 warps][16 quantities]
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  int ucount = 0;
  // sampling: every logit >= the guessed k-th value is listed while it is in a register (topk_dist, step 0)
  const float tguess = P.sampling ? __ldcg(&P.samp->tau_guess[lane >> 4]) : INFINITY;
  while (true) {
    const uint32_t s0 = seq;
    mbar_wait(&full[s0 % kStages], (s0 / kStages) & 1);
    const int u = meta[s0 % kStages];
    if (u == kEndMark) {
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s0 % kStages]);
      ++seq;
      break;
    }
    float acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = 0.f;
    if (pair != 0 && lane == 0) mbar_arrive(&empty[s0 % kStages]);   // first slot: the other warps right away
    // The unit's first slot is passed by all 8 warps (it carries the unit tag); every other tile is waited on and
    // released by its owner pair alone, so a tile is recycled as soon as its two readers are done.  An owner's
    // slot last held a tile of the previous unit (or this unit's first tile, nc <= 12): consumed before the
    // per-unit barrier this warp has passed, so the parity wait always targets the slot's next phase.
#pragma unroll
    for (int s = 0; s < NXS; ++s) {
      const int c = pair + 4 * s;
      if (c < nc) {
        const uint32_t sq = s0 + c, slot = sq % kStages;
        if (c > 0) mbar_wait(&full[slot], (sq / kStages) & 1);
        const uint4 *wt = reinterpret_cast<const uint4 *>(ring + (size_t)slot * kTileBytes) + half * (8 * 64);
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          const uint4 w0 = wt[r * 64 + lane], w1 = wt[r * 64 + 32 + lane];
          if (do_v) { acc[r] = fma8(w0, xv[s][0], xv[s][1], acc[r]); acc[r] = fma8(w1, xv[s][2], xv[s][3], acc[r]); }
          if (do_p) { acc[8 + r] = fma8(w0, xp[s][0], xp[s][1], acc[8 + r]); acc[8 + r] = fma8(w1, xp[s][2], xp[s][3], acc[8 + r]); }
        }
        __syncwarp();
        if (c > 0 && lane == 0) mbar_arrive_n(&empty[slot], 4);
      }
      if (s == 0 && pair == 0 && lane == 0) mbar_arrive(&empty[s0 % kStages]);   // first slot: pair 0 after reading it
    }
    seq += nc;
    int q = 0;
    XReduce<16, 16>::run(acc, lane, q);                  // q == lane >> 1: quantity (vector q >> 3, row q & 7)
    if ((lane & 1) == 0) part[(ucount & 1) * 128 + warp * 16 + q] = acc[0];
    consumer_sync();
    if (warp == (ucount & 7)) {
      const int vec = lane >> 4, r16 = lane & 15;        // this lane's logit: row r16 of the unit, vector vec
      const float *pp = part + (ucount & 1) * 128 + (r16 >> 3) * 16 + vec * 8 + (r16 & 7);
      float y = 0.f;
#pragma unroll
      for (int pr = 0; pr < 4; ++pr) y += pp[pr * 32];   // warps 2 pr + (r16 >> 3), pr ascending
      const int row = u * kTileRows + r16;
      if ((vec ? do_p : do_v) && row < D.V) {
        if (cand_better(y, row, bv, bi)) { bv = y; bi = row; }
        if (P.debug_logits | P.sampling) (vec ? P.logits_p : P.logits_v)[row] = y;
        if (y >= tguess) {
          const int pos = atomicAdd(&P.samp->pre_cnt[vec], 1);
          if (pos < kSampCap) { P.pre_val[vec * kSampCap + pos] = y; P.pre_idx[vec * kSampCap + pos] = row; }
        }
      }
    }
    ++ucount;
  }
  // lanes 0..15 hold verify candidates, lanes 16..31 PDM candidates: reduce inside each half
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (cand_better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
  }
  if ((lane & 15) == 0) { cbest_v[(lane >> 4) * 8 + warp] = bv; cbest_i[(lane >> 4) * 8 + warp] = bi; }
}

}  // namespace spd
