// spd_mega.cu — the fused persistent engine: ONE cooperative kernel per SPD cycle.
//
// Shape of the problem: a cycle streams every layer's weights once (12.3 GB at
// the 9B-class config) through (L/n)*5 + 2 dependent phases; every product is an M=1 GEMV, so the
// bound is HBM bandwidth and the enemy is the idle time at each phase boundary.  Design:
//   * grid = one CTA per SM, resident for the whole cycle; 8 consumer warps + 1 producer warp.
//   * weights are repacked once (spd_create) into 16 KB tiles — 16 rows x 512 columns; a "unit" is the
//     nc tiles of 16 output rows, contiguous in memory.
//   * the stages (the n in-flight tokens) own disjoint CTA groups (CTA c -> active stage c mod a), so a
//     CTA keeps one activation vector per phase; inside a group the units of a phase are CLAIMED
//     dynamically from a per-(phase, stage) counter, so SMs with less bandwidth simply take fewer units
//     and every CTA reaches the phase barrier at about the same time.
//   * the producer lane streams the claimed units with 1-D TMA bulk copies (cp.async.bulk + mbarrier
//     complete_tx) into an 11-deep shared-memory ring, tagging each slot with its unit index and closing
//     each phase with an END slot.  Unit claims do not depend on activations, so the producer runs
//     AHEAD of the activation dependency, across phase boundaries: while the consumers wait at a grid
//     barrier the next phase's tiles are already landing.
//   * consumers: a tile is read by ONE warp pair (pair = chunk index mod 4; its two warps take rows 0..7 /
//     8..15) with 128-bit conflict-free LDS of the weights and of the fp32 activation vector (staged in smem
//     once per phase with 128-bit L2 loads), fp32 FMA, a transposed butterfly per warp, the 8 warp partials
//     of a 16-row unit meet in shared memory under one named barrier, and one warp runs the fused epilogue
//     (RoPE + bf16 KV append, residual add, SiLU*mul, PDM partials).  The LM head (two vectors against the
//     tied matrix) keeps both vectors in registers.  Every warp still passes every slot's barriers in ring
//     order (gemv_stream) or the unit's first slot (head_stream), which keeps slot recycling race-free.
//   * attention: items (stage, kv head, 128-row split) are claimed dynamically by all CTAs; the
//     producer brings the K and V rows of an item through the same ring (TMA), the 8 consumer warps
//     compute the G q heads of the kv group together (scores with a transposed butterfly reduction,
//     softmax per head, P.V with a fixed cross-warp reduction); the last split of a head merges.
//   * phases are separated by arrive/poll barriers per stage group (red.release / ld.acquire at gpu scope on
//     per-cycle counters); cross-CTA activations are read with ld.global.cg.
// Every row's dot product is computed with a fixed warp/lane/column mapping and a fixed order of partial sums,
// attention splits are fixed 128-row blocks merged in split order, so a token's result never depends
// on n, slot, fill, history or on which CTA happened to claim the work (batch invariance).
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
  unsigned long long layer_bytes, off_o, off_gu, off_dn, off_pdm, off_head, pdm_job_bytes;
  int u_qkv, u_o, u_gu, u_dn, u_pdm, u_head;   // 16-row units per job
  int nc_d, nc_qd, nc_f;                        // 512-column chunks for K = d, Hq*hd, F
  int attn_mma;                                 // full 128-row attention items go through the tensor cores
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
  w.job = -1; w.U = 0; w.nc = 0; w.base = nullptr; w.ctr = claim + (size_t)p * kMaxStages;
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
    else { w.U = ML.u_dn; w.nc = ML.nc_f; w.base = lb + ML.off_dn; }
  }
  if (w.job >= 0) w.ctr += w.job;
  return w;
}

// Attention item of this CTA's stage -> (kv head, split).  Items [0, attn_nonfinal) are the splits that do
// not contain the row appended in this pass (kv head major) — their K/V rows are old and can be fetched
// before the QKV phase has finished; items [attn_nonfinal, attn_total) are the last split of every kv head.
__device__ __forceinline__ void attn_decode(const Sched &S, const Dims &D, int item, AttnItem &it) {
  it.stage = S.my_stage; it.nsplit = S.attn_ns;
  if (item < S.attn_nonfinal) {
    it.kvh = item / (it.nsplit - 1);
    it.split = item - it.kvh * (it.nsplit - 1);
  } else {
    it.kvh = item - S.attn_nonfinal;
    it.split = it.nsplit - 1;
  }
  it.t0 = it.split * kAttnSplit;
  int T = S.pos[it.stage] + 1;
  it.rows = min(T - it.t0, kAttnSplit);
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
                                          float *scratch, uint64_t *empty) {
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
      const float4 *q4 = reinterpret_cast<const float4 *>(P.q + ((size_t)it.stage * D.Hq + hq0 + h) * HD + c * 8);
      float4 a = __ldcg(q4), b = __ldcg(q4 + 1);
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
  if (lane == 0) for (int j = 0; j < nk; ++j) mbar_arrive(&empty[(seq0 + j) % kStages]);   // K slots are free
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
                                              float *scratch, uint64_t *empty, const uint32_t *qs) {
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
  if (lane == 0) for (int j = 0; j < nk; ++j) mbar_arrive(&empty[(seq0 + j) % kStages]);   // this warp is done with K
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
__device__ __forceinline__ void unit_epilogue(const DevPtrs &P, const Sched &S, int t, int k, int pass, int r0, float y0,
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
                                            float *scratch, uint64_t *empty, int G) {
  if (G == 4) attn_item<HD, 4>(P, it, ring, seq0, nk, scratch, empty);
  else if (G == 2) attn_item<HD, 2>(P, it, ring, seq0, nk, scratch, empty);
  else if (G == 8) attn_item<HD, 8>(P, it, ring, seq0, nk, scratch, empty);
  else attn_item<HD, 1>(P, it, ring, seq0, nk, scratch, empty);
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
__device__ __forceinline__ void gemv_stream(const DevPtrs &P, const Sched &S, int t, int k, int pass, int nc,
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

// The fused kernel ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads, 1) k_spd_cycle(DevPtrs P, MegaLayout ML, const __grid_constant__ CUtensorMap kv_tmap) {
  extern __shared__ __align__(1024) uint8_t smem[];   // ring slots must be 1024-byte aligned (128-byte swizzle)
  uint8_t *ring = smem;                                                  // kStages * 16 KB
  float *xs = reinterpret_cast<float *>(smem + kStages * kTileBytes);    // kXFloats
  uint64_t *full = reinterpret_cast<uint64_t *>(xs + kXFloats);          // [kStages]
  uint64_t *empty = full + kStages;                                      // [kStages]
  float2 *rope_s = reinterpret_cast<float2 *>(empty + kStages);          // [64]
  float *red = reinterpret_cast<float *>(rope_s + 64);                   // [16]
  float *cbest_v = red + 16;                                             // [2][8]
  int *cbest_i = reinterpret_cast<int *>(cbest_v + 16);                  // [2][8]
  int *meta = cbest_i + 16;                                              // [kStages] slot tags (+ padding to 16)
  float *gpart = reinterpret_cast<float *>(meta + 16);                     // [2][8][8] warp partials of a unit
  Sched *Sp = reinterpret_cast<Sched *>(gpart + 128);

  const Dims &D = P.dim;
  const int cta = blockIdx.x, ncta = gridDim.x;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int np = 2 + 5 * D.per;
  // Synchronisation words (each on its own 128-byte line): bar_count = CTAs that finished the cycle (monotonic over
  // launches), bar_launch = cycles completed; per cycle (zeroed by CTA 0 at the end): gbar[k] = phase arrivals of the
  // CTA group of stage k, pdm_staged = CTAs that have read their PDM slot vector, pdm_done = CTAs past the PDM phase.
  unsigned long long *bar_count = reinterpret_cast<unsigned long long *>(P.bar);
  unsigned long long *bar_launch = reinterpret_cast<unsigned long long *>(P.bar + 32);
  unsigned int *gbar = P.bar + kBarGroup0;
  unsigned int *pdm_staged = gbar + 32 * kMaxStages, *pdm_done = pdm_staged + 32;

  if (P.prof_on && tid == 0 && cta < kProfCtas) {
    unsigned long long *pr = P.prof + ((size_t)cta * kProfPhases + (kProfPhases - 1)) * kProfStamps;
    pr[2] = (unsigned long long)clock64(); pr[3] = globaltimer_ns();
  }
  // ---- schedule (every CTA computes the same thing from the state the previous cycle left) ----
  if (tid == 0) {
    const StepState *st = P.st;
    Sched &S = *Sp;
    S.mode = st->mode; S.c = st->c;
    int a = 0;
    for (int k = 0; k < D.n; ++k) {
      S.occ[k] = st->occ[k]; S.pos[k] = st->pos[k]; S.hbuf[k] = st->hbuf[k];
      if (st->occ[k]) S.act[a++] = k;
    }
    S.n_act = a;
    S.p_new = st->occ[0] ? st->pos[0] : -1;
    S.run_pdm = st->mode == MODE_SPD && !P.paper_pdm;
    S.run_verify = (st->mode == MODE_SPD && st->occ[D.n - 1]) || st->mode == MODE_PREFILL_FINAL;
    // CTA c serves active stage c mod a (every group gets the same mix of SMs); PDM slot c mod n
    S.my_stage = a > 0 ? S.act[cta % a] : -1;
    S.my_idx = a > 0 ? cta / a : 0;
    S.my_gsize = a > 0 ? ncta / a + (cta % a < ncta % a ? 1 : 0) : 0;
    S.exit_gsize = (a > 0 && st->occ[D.n - 1]) ? ncta / a + (a - 1 < ncta % a ? 1 : 0) : 0;   // stage n-1 = act[a-1]
    S.attn_ns = a > 0 ? (S.pos[S.my_stage] + kAttnSplit) / kAttnSplit : 0;                      // ceil((pos + 1) / split)
    S.attn_total = D.Hkv * S.attn_ns;
    S.attn_nonfinal = D.Hkv * (S.attn_ns - 1);
    S.pdm_slot = cta % D.n;
    S.pdm_idx = cta / D.n;
    for (int s = 0; s < kStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const Sched &S = *Sp;
  const unsigned long long launch = ld_acquire_u64(bar_launch);
  if (cta == 0 && tid == 0) controller_begin(P);   // writes only fields no other CTA reads in this kernel
  if (P.prof_on && tid == 0 && cta < kProfCtas) {
    unsigned long long *pr = P.prof + ((size_t)cta * kProfPhases + (kProfPhases - 1)) * kProfStamps;
    pr[0] = (unsigned long long)clock64(); pr[1] = globaltimer_ns();
  }
  if (S.my_stage >= 0 && tid < D.hd / 2) {         // RoPE table of this CTA's stage (C-2.14)
    double s_, c_;
    sincos((double)S.pos[S.my_stage] * P.inv_freq[tid], &s_, &c_);
    rope_s[tid] = make_float2((float)c_, (float)s_);
  }
  __syncthreads();
  const int RPS = kTileBytes / (D.hd * 2);         // K/V rows per ring slot

  if (warp == 8) {
    // =========================== producer: claim and stream every phase's work, running ahead =====
    if (lane == 0) {
      uint64_t pol_w, pol_kv;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_w));
      asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol_kv));
      uint32_t seq = 0;
      for (int p = 0; p < np; ++p) {
        PhaseDesc w = phase_desc(p, np, S, ML, D, P.claim);
        if (w.job >= 0) {
          unsigned int next = atomicAdd(w.ctr, 1u);
          if (w.type == PH_ATTN) {
            const int pass = (p - 1) / 5;
            bool first = true, kv_ready = false;
            while (next < (unsigned int)w.U) {
              AttnItem it;
              attn_decode(S, D, (int)next, it);
              const int item = (int)next;
              next = atomicAdd(w.ctr, 1u);
              if (item >= S.attn_nonfinal && !kv_ready) {
                // the last split holds the row appended by the group's CTAs in this pass's QKV phase: wait for it
                const unsigned int target = (unsigned int)(p - 1) * (unsigned int)S.my_gsize;
                while (ld_acquire_u32(gbar + 32 * S.my_stage) < target) {}
                fence_proxy_async();
                kv_ready = true;
              }
              const int layer = it.stage * D.per + pass;
              const int nk = (it.rows + RPS - 1) / RPS;
              const bool boxed = ML.attn_mma && it.rows == kAttnSplit;   // full split: swizzled boxes for the MMA path
              for (int kvsel = 0; kvsel < 2; ++kvsel) {
                const uint16_t *src = P.kv + kv_offset(D, layer, kvsel, it.kvh) + (size_t)it.t0 * D.hd;
                const int plane = (layer * 2 + kvsel) * D.Hkv + it.kvh;
                for (int j = 0; j < nk; ++j, ++seq) {
                  uint32_t slot = seq % kStages, itn = seq / kStages;
                  int r = min(RPS, it.rows - j * RPS);
                  uint32_t bytes = (uint32_t)r * D.hd * 2;
                  mbar_wait(&empty[slot], (itn & 1) ^ 1);
                  meta[slot] = item;
                  mbar_expect_tx(&full[slot], bytes);
                  uint8_t *dst = ring + (size_t)slot * kTileBytes;
                  if (boxed) {           // 64 rows: head-dim halves [0, 64) and [64, 128) as two 8 KB boxes
                    tma_load_box(dst, &kv_tmap, 0, it.t0 + j * RPS, plane, &full[slot], pol_kv);
                    tma_load_box(dst + kTileBytes / 2, &kv_tmap, 64, it.t0 + j * RPS, plane, &full[slot], pol_kv);
                  } else {
                    tma_load_1d(dst, src + (size_t)j * RPS * D.hd, bytes, &full[slot], pol_kv);
                  }
                  if (first) { prof_stamp(P, cta, p, 3); first = false; }
                }
              }
            }
          } else {
            bool first = true;
            while (next < (unsigned int)w.U) {
              const int u = (int)next;
              next = atomicAdd(w.ctr, 1u);         // claim ahead: its latency hides behind this unit's tiles
              const uint8_t *src = w.base + (unsigned long long)u * w.nc * kTileBytes;
              for (int i = 0; i < w.nc; ++i, ++seq, src += kTileBytes) {
                uint32_t slot = seq % kStages, itn = seq / kStages;
                mbar_wait(&empty[slot], (itn & 1) ^ 1);
                meta[slot] = u;
                mbar_expect_tx(&full[slot], kTileBytes);
                tma_load_1d(ring + (size_t)slot * kTileBytes, src, kTileBytes, &full[slot], pol_w);
                if (first) { prof_stamp(P, cta, p, 3); first = false; }
              }
            }
          }
          prof_stamp(P, cta, p, 4);
        }
        // END slot: closes the phase for the consumers
        uint32_t slot = seq % kStages, itn = seq / kStages;
        mbar_wait(&empty[slot], (itn & 1) ^ 1);
        meta[slot] = kEndMark;
        mbar_arrive(&full[slot]);
        ++seq;
      }
    }
  } else {
    // =========================== consumers ======================================================
    uint32_t seq = 0;
    const int G = D.Hq / D.Hkv;
    for (int p = 0; p < np; ++p) {
      const int pass = (p - 1) / 5;
      // ---- wait for the producers of this phase's inputs.  The n stages are independent chains, so a layer
      //      phase waits only for its own stage's CTA group (the groups drift apart and one group's attention or
      //      barrier wait is covered by the other groups' weight streams); the first O phase, the first to
      //      overwrite a residual stream, also waits until every CTA has read its pre-step PDM slot vector;
      //      the LM head waits for the exit stage's group and for the PDM partial products -----------------
      if (tid == 0) {
        if (p == np - 1) {
          if (S.run_verify && S.exit_gsize > 0) {
            const unsigned int target = (unsigned int)(np - 2) * (unsigned int)S.exit_gsize;
            while (ld_acquire_u32(gbar + 32 * (D.n - 1)) < target) {}
          }
          if (S.run_pdm) while (ld_acquire_u32(pdm_done) < (unsigned int)ncta) {}
        } else if (p >= 2 && S.my_stage >= 0) {
          const unsigned int target = (unsigned int)(p - 1) * (unsigned int)S.my_gsize;
          while (ld_acquire_u32(gbar + 32 * S.my_stage) < target) {}
          if (p == 3 && S.run_pdm) while (ld_acquire_u32(pdm_staged) < (unsigned int)ncta) {}
        }
      }
      consumer_sync();   // also: every warp is done with the previous phase's xs
      if (tid == 0) {
        prof_stamp(P, cta, p, 0);
        if (P.prof_on && cta < kProfCtas && p < kProfPhases) P.prof[((size_t)cta * kProfPhases + p) * kProfStamps + 5] = globaltimer_ns();
      }
      PhaseDesc w = phase_desc(p, np, S, ML, D, P.claim);
      const int t = w.type;
      const int k = w.job;                    // stage (layer phases) / slot (PDM)
      if (t == PH_ATTN) {
        if (tid == 0) prof_stamp(P, cta, p, 1);
        // ---- split-KV decode attention: items claimed by the producer arrive through the ring; the
        //      split-completion counts of the items this CTA processed are published together at the end
        //      of the phase (one fence), and whoever completes a q head merges its splits ------------------
        int *done_list = reinterpret_cast<int *>(xs + kAttnScratchFloats);   // [kAttnDoneMax] item ids
        int *merge_cnt = done_list + kAttnDoneMax;                           // [1]
        int *merge_list = merge_cnt + 1;                                     // [kAttnDoneMax * 8] (item slot, head)
        int n_done = 0;
        bool more = true;
        // q of this CTA's stage, split into bf16 hi / lo pairs, staged once per phase for the tensor-core items
        // (behind the score / probability / partial-output scratch, if it fits in front of the done lists)
        const uint32_t *qs = nullptr;
        if (ML.attn_mma && S.my_stage >= 0 && S.attn_ns > 1 &&
            10 * G * kAttnSplit + 2 * D.Hq * kQPairStride <= kAttnScratchFloats) {
          uint32_t *qw = reinterpret_cast<uint32_t *>(xs) + 10 * G * kAttnSplit;
          const float2 *q2 = reinterpret_cast<const float2 *>(P.q + (size_t)S.my_stage * D.Hq * D.hd);
          for (int i = tid; i < D.Hq * 64; i += kConsumerThreads) {
            const float2 v = __ldcg(q2 + i);
            uint32_t hi, lo;
            split_bf16x2(v.x, v.y, hi, lo);
            const int o = (i >> 6) * kQPairStride + (i & 63);
            qw[o] = hi;
            qw[D.Hq * kQPairStride + o] = lo;
          }
          qs = qw;
          consumer_sync();
        }
        while (more) {
          uint32_t slot = seq % kStages, itn = seq / kStages;
          mbar_wait(&full[slot], itn & 1);
          const int item = meta[slot];
          if (item == kEndMark) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[slot]);
            ++seq;
            more = false;
          } else {
            AttnItem it;
            attn_decode(S, D, item, it);
            const int nk = (it.rows + RPS - 1) / RPS;
            for (int j = 1; j < 2 * nk; ++j) mbar_wait(&full[(seq + j) % kStages], ((seq + j) / kStages) & 1);
            if (ML.attn_mma && it.rows == kAttnSplit) {
              if (G == 4) attn_item_mma<4>(P, it, ring, seq, xs, empty, qs);
              else if (G == 8) attn_item_mma<8>(P, it, ring, seq, xs, empty, qs);
              else if (G == 2) attn_item_mma<2>(P, it, ring, seq, xs, empty, qs);
              else attn_item_mma<1>(P, it, ring, seq, xs, empty, qs);
            } else if (D.hd == 128) attn_item_g<128>(P, it, ring, seq, nk, xs, empty, G);
            else attn_item_g<64>(P, it, ring, seq, nk, xs, empty, G);
            seq += 2 * nk;
            if (tid == 0) done_list[n_done] = item;
            ++n_done;
          }
          if (n_done == kAttnDoneMax || (!more && n_done > 0)) {
            if (tid == 0) *merge_cnt = 0;
            __threadfence();                       // this CTA's partial outputs, before their completion counts
            consumer_sync();
            for (int e = tid; e < n_done * G; e += kConsumerThreads) {
              AttnItem it;
              attn_decode(S, D, done_list[e / G], it);
              const int hq = it.kvh * G + e % G;
              if (atomicAdd(&P.att_cnt[it.stage * D.Hq + hq], 1) == it.nsplit - 1) merge_list[atomicAdd(merge_cnt, 1)] = e;
            }
            consumer_sync();
            const int nm = *merge_cnt;
            if (nm > 0) {
              __threadfence();
              for (int m = warp; m < nm; m += 8) {   // the last split of a q head to finish merges them (fixed split order)
                const int e = merge_list[m];
                AttnItem it;
                attn_decode(S, D, done_list[e / G], it);
                const int hq = it.kvh * G + e % G;
                if (D.hd == 128) attn_merge_warp<128>(P, it.stage, hq, it.nsplit, lane);
                else attn_merge_warp<64>(P, it.stage, hq, it.nsplit, lane);
                if (lane == 0) P.att_cnt[it.stage * D.Hq + hq] = 0;
              }
            }
            consumer_sync();                         // done_list / merge_list are reused
            n_done = 0;
          }
        }
      } else {
        // ---- stage the activation vector(s) of this phase in shared memory ----------------------
        if (k >= 0) {
          int K = 0;
          if (t == PH_QKV || t == PH_GATEUP) {
            int layer = k * D.per + pass;
            const float *h = P.h + (size_t)S.hbuf[k] * D.d;
            const uint16_t *g = t == PH_QKV ? P.attn_norm[layer] : P.mlp_norm[layer];
            float ss = consumer_sum(stage_copy(h, xs, D.d), red);
            if (t == PH_QKV && S.my_idx == 0) {   // NEXT-1: H^layer of the paper PDM's anchor set (the raw residual stream)
              const int ai = anchor_index(P, layer);
              if (ai >= 0 && S.pos[k] < D.max_seq) {
                float4 *dst = reinterpret_cast<float4 *>(P.anch + ((size_t)S.pos[k] * P.pdm_m + ai) * D.d);
                const float4 *src = reinterpret_cast<const float4 *>(xs);
                for (int i = tid; i < (D.d >> 2); i += kConsumerThreads) dst[i] = src[i];   // this thread's own float4s
              }
            }
            stage_scale(xs, g, D.d, 1.0f / sqrtf(ss / (float)D.d + D.eps));
            K = D.d;
          } else if (t == PH_O) {
            K = D.Hq * D.hd;
            stage_copy(P.att + (size_t)k * K, xs, K);
          } else if (t == PH_DOWN) {
            K = D.F;
            stage_copy(P.act + (size_t)k * K, xs, K);
          } else if (t == PH_PDM) {
            // slot j = k: pre-step state of the token at depth j, else Hfin[p_new - j], else zero (Eq. 5)
            K = D.d;
            int q = S.p_new - k;
            const float *src = S.occ[k] ? P.h + (size_t)S.hbuf[k] * D.d : (q >= 0 ? P.hfin + (size_t)q * D.d : nullptr);
            if (src) stage_copy(src, xs, K);
            else for (int i = tid; i < K; i += kConsumerThreads) xs[i] = 0.f;
            consumer_sync();
            if (tid == 0) { __threadfence(); atomicAdd(pdm_staged, 1u); }   // the pre-step state has been read
            if (S.pdm_idx == 0)               // kept for the parity tests (SPD_DBG_PDM_FEAT)
              for (int i = tid; i < K; i += kConsumerThreads) P.feat[(size_t)k * D.d + i] = xs[i];
          } else {  // PH_HEAD: verify input at xs[0..d), PDM input at xs[kXFloats/2 ..)
            K = D.d;
            if (S.run_verify) {
              const float *h = S.mode == MODE_PREFILL_FINAL ? P.hfin + (size_t)(S.c - 1) * D.d
                                                            : P.h + (size_t)S.hbuf[D.n - 1] * D.d;
              float ss = consumer_sum(stage_copy(h, xs, D.d), red);
              stage_scale(xs, P.final_norm, D.d, 1.0f / sqrtf(ss / (float)D.d + D.eps));
            }
            if (S.run_pdm) {
              float *xp = xs + kXFloats / 2;
              float4 *xp4w = reinterpret_cast<float4 *>(xp);
              float ss = 0.f;
              for (int i = tid; i < (D.d >> 2); i += kConsumerThreads) {   // u = sum_j W_p[:, block j] f_j, j ascending
                float4 u = make_float4(0.f, 0.f, 0.f, 0.f);
                for (int j = 0; j < D.n; ++j) {
                  float4 v = __ldcg(reinterpret_cast<const float4 *>(P.pdm_part + (size_t)j * D.d) + i);
                  u.x += v.x; u.y += v.y; u.z += v.z; u.w += v.w;
                }
                xp4w[i] = u;
                if (cta == 0) reinterpret_cast<float4 *>(P.pdm_u)[i] = u;    // kept for the parity tests (SPD_DBG_PDM_PRENORM)
                ss = fmaf(u.x, u.x, ss); ss = fmaf(u.y, u.y, ss); ss = fmaf(u.z, u.z, ss); ss = fmaf(u.w, u.w, ss);
              }
              ss = consumer_sum(ss, red);
              stage_scale(xp, P.pdm_norm, D.d, 1.0f / sqrtf(ss / (float)D.d + D.eps));
            }
          }
          int kpad = w.nc * kTileCols;
          for (int i = K + tid; i < kpad; i += kConsumerThreads) xs[i] = 0.f;
          if (t == PH_HEAD) for (int i = K + tid; i < kpad; i += kConsumerThreads) xs[kXFloats / 2 + i] = 0.f;
        }
        if (t == PH_QKV && S.my_stage >= 0 && S.my_idx == 0 && tid == 0) {
          // causality / capacity precondition of the KV append, and the new length (one CTA per stage)
          int layer = S.my_stage * D.per + pass, pos = S.pos[S.my_stage];
          if (P.len[layer] != pos || pos >= D.max_seq) P.st->err = 1;
          else P.len[layer] = pos + 1;
        }
        consumer_sync();
        if (tid == 0) prof_stamp(P, cta, p, 1);
        // ---- stream the claimed units ------------------------------------------------------------
        if (k < 0) {                               // nothing to stream: one END slot, read by every warp
          const uint32_t slot = seq % kStages;
          mbar_wait(&full[slot], (seq / kStages) & 1);
          __syncwarp();
          if (lane == 0) mbar_arrive(&empty[slot]);
          ++seq;
        } else if (t == PH_HEAD) {
          const bool do_v = S.run_verify, do_p = S.run_pdm;
          if (w.nc <= 4) head_stream<1>(P, w.nc, do_v, do_p, ring, full, empty, meta, xs, seq, cbest_v, cbest_i);
          else if (w.nc <= 8) head_stream<2>(P, w.nc, do_v, do_p, ring, full, empty, meta, xs, seq, cbest_v, cbest_i);
          else head_stream<3>(P, w.nc, do_v, do_p, ring, full, empty, meta, xs, seq, cbest_v, cbest_i);
        } else {
          gemv_stream(P, S, t, k, pass, w.nc, ring, full, empty, meta, xs, gpart, seq, rope_s);
        }
        if (t == PH_HEAD) {   // CTA-level candidates -> global
          consumer_sync();
          if (tid < 2) {
            float bv = -INFINITY;
            int bi = 0x7fffffff;
            for (int ww = 0; ww < 8; ++ww)
              if (cand_better(cbest_v[tid * 8 + ww], cbest_i[tid * 8 + ww], bv, bi)) { bv = cbest_v[tid * 8 + ww]; bi = cbest_i[tid * 8 + ww]; }
            P.cand_val[tid * kMaxCand + cta] = bv;
            P.cand_idx[tid * kMaxCand + cta] = bi == 0x7fffffff ? -1 : bi;
          }
        }
        if (t == PH_QKV) fence_proxy_async();   // the appended K/V rows are read by TMA (async proxy) next
      }
      // ---- publish this phase's outputs: arrive at the counter that the dependent phase waits on ----
      if (tid == 0) prof_stamp(P, cta, p, 2);
      if (p == np - 1 || (p == 0 && S.run_pdm) || (p > 0 && S.my_stage >= 0)) {
        // one release at gpu scope by thread 0 after the CTA barrier publishes every consumer's writes of this
        // phase (release is cumulative over what the barrier ordered before it); the waiters acquire
        consumer_sync();
        if (tid == 0) {
          if (p == np - 1) red_release_add_u64(bar_count, 1ull);
          else if (p == 0) red_release_add_u32(pdm_done, 1u);
          else red_release_add_u32(gbar + 32 * S.my_stage, 1u);
        }
      }
    }
  }
  // ---- last: CTA 0 waits for every CTA's head candidates, then runs the controller ---------------
  __syncthreads();
  if (cta == 0) {
    if (tid == 0) {
      unsigned long long target = (launch + 1) * (unsigned long long)ncta;
      while (ld_acquire_u64(bar_count) < target) {}
      __threadfence();
    }
    __syncthreads();
    controller_end(P, ncta, reinterpret_cast<SampSmem *>(ring), true);   // the tile ring is idle: every tile of the cycle was consumed
    for (int i = tid; i < np * kMaxStages; i += kThreads) P.claim[i] = 0u;   // every producer is done claiming
    if (tid < kMaxStages + 2) gbar[32 * tid] = 0u;                           // ... and every CTA with its group counters
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      atomicAdd(bar_launch, 1ull);
      if (P.prof_on) {
        unsigned long long *pr = P.prof + ((size_t)(kProfPhases - 1)) * kProfStamps;
        pr[4] = (unsigned long long)clock64(); pr[5] = globaltimer_ns();
      }
    }
  }
}

// ------------------------------------------------------------------ weight repack --------------
// dst tile layout: [unit u][chunk c][row r (16)][column group g (2)][lane l (32)][j (8)] bf16, where the
// logical column of (g, l, j) inside the chunk is g*256 + (j < 4 ? 4l + j : 128 + 4l + j - 4): a lane's
// 16-byte weight chunk multiplies the two float4 x[4l..4l+3] and x[128+4l..128+4l+3] of the group, both
// read as conflict-free LDS.128.  Row maps: QKV -> RoPE pairs (i, i+hd/2) adjacent, q heads, k heads,
// then v rows; GATEUP -> (gate_i, up_i) adjacent; others identity.  Padding rows/columns are zero.
enum RowMap { RM_PLAIN = 0, RM_QKV = 1, RM_GATEUP = 2 };

__global__ void k_repack(uint16_t *dst, int units, int nc, int rowmap, const uint16_t *s0, const uint16_t *s1,
                         const uint16_t *s2, int rows0, int rows1, int rows2, int K, int src_ld, int src_col0, int hd) {
  size_t total = (size_t)units * nc * kTileRows * 64;      // 16-byte chunks
  for (size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x; id < total; id += (size_t)gridDim.x * blockDim.x) {
    int l = id & 31, g = (id >> 5) & 1, r = (id >> 6) & 15;
    size_t tile = id >> 10;
    int c = tile % nc, u = tile / nc;
    int rho = u * kTileRows + r;
    const uint16_t *src = nullptr;
    int row = -1;
    if (rowmap == RM_PLAIN) {
      if (rho < rows0) { src = s0; row = rho; }
    } else if (rowmap == RM_GATEUP) {
      int i = rho >> 1;
      if (i < rows0) { src = (rho & 1) ? s1 : s0; row = i; }
    } else {
      int half = hd / 2;
      if (rho < rows0 + rows1) {                           // q or k heads: pairs adjacent
        int base = rho < rows0 ? 0 : rows0;
        int rr = rho - base, hh = rr / hd, e = rr - hh * hd;
        row = hh * hd + (e >> 1) + ((e & 1) ? half : 0);
        src = rho < rows0 ? s0 : s1;
      } else if (rho < rows0 + rows1 + rows2) { src = s2; row = rho - rows0 - rows1; }
    }
    uint16_t out[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      int col = c * kTileCols + g * 256 + (j < 4 ? 4 * l + j : 128 + 4 * l + j - 4);
      out[j] = (src && col < K) ? src[(size_t)row * src_ld + src_col0 + col] : (uint16_t)0;
    }
    reinterpret_cast<uint4 *>(dst)[id] = *reinterpret_cast<uint4 *>(out);
  }
}

// ------------------------------------------------------------------ host side ------------------
static inline int cdiv_i(int a, int b) { return (a + b - 1) / b; }

static void make_layout(const Dims &D, MegaLayout *ML, size_t *total) {
  int qd = D.Hq * D.hd, kd = D.Hkv * D.hd;
  ML->nc_d = cdiv_i(D.d, kTileCols); ML->nc_qd = cdiv_i(qd, kTileCols); ML->nc_f = cdiv_i(D.F, kTileCols);
  ML->u_qkv = cdiv_i(qd + 2 * kd, kTileRows); ML->u_o = cdiv_i(D.d, kTileRows); ML->u_gu = cdiv_i(2 * D.F, kTileRows);
  ML->u_dn = cdiv_i(D.d, kTileRows); ML->u_pdm = cdiv_i(D.d, kTileRows); ML->u_head = cdiv_i(D.V, kTileRows);
  unsigned long long b_qkv = (unsigned long long)ML->u_qkv * ML->nc_d * kTileBytes;
  unsigned long long b_o = (unsigned long long)ML->u_o * ML->nc_qd * kTileBytes;
  unsigned long long b_gu = (unsigned long long)ML->u_gu * ML->nc_d * kTileBytes;
  unsigned long long b_dn = (unsigned long long)ML->u_dn * ML->nc_f * kTileBytes;
  ML->off_o = b_qkv; ML->off_gu = b_qkv + b_o; ML->off_dn = b_qkv + b_o + b_gu;
  ML->layer_bytes = b_qkv + b_o + b_gu + b_dn;
  ML->pdm_job_bytes = (unsigned long long)ML->u_pdm * ML->nc_d * kTileBytes;
  ML->off_pdm = ML->layer_bytes * D.L;
  ML->off_head = ML->off_pdm + ML->pdm_job_bytes * D.n;
  *total = ML->off_head + (unsigned long long)ML->u_head * ML->nc_d * kTileBytes;
}

static bool mega_supported(const Dims &D) {
  int qd = D.Hq * D.hd;
  int G = D.Hq / D.Hkv;
  // 2 + 5 * (L / n) phases must fit the claim-counter / profile tables (P.claim is [kProfPhases][kMaxStages])
  return D.d <= kXFloats / 2 && qd <= kXFloats && D.F <= kXFloats && (G == 1 || G == 2 || G == 4 || G == 8) &&
         (qd + 2 * D.Hkv * D.hd) % 2 == 0 && D.hd % 2 == 0 && 2 + 5 * D.per <= kProfPhases;
}

size_t mega_repack_bytes(const Dims &D) {
  if (!mega_supported(D)) return 256;
  MegaLayout ML;
  size_t total;
  make_layout(D, &ML, &total);
  return total;
}

int mega_create(const DevPtrs &P, const uint16_t *const *const *src, void *repack, size_t repack_bytes,
                cudaStream_t stream, MegaPlan *plan) {
  const Dims &D = P.dim;
  plan->available = 0;
  if (!mega_supported(D) || !repack) return -1;
  MegaLayout ML;
  size_t total;
  make_layout(D, &ML, &total);
  if (repack_bytes < total) return -1;
  int dev = 0, sms = 0, coop = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  int smem = kStages * kTileBytes + kXFloats * 4 + 2 * kStages * 8 + 64 * 8 + 16 * 4 + 32 * 4 + 16 * 4 + 128 * 4 + (int)sizeof(Sched);
  if (!coop || sms < D.n || sms > kMaxCand) return -1;   // one argmax candidate slot per CTA
  if (cudaFuncSetAttribute(k_spd_cycle, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  int occ = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_spd_cycle, kThreads, smem) != cudaSuccess || occ < 1) {
    cudaGetLastError();
    return -1;
  }
  // K/V cache as a rank-3 bf16 tensor {hd, max_seq, L * 2 * Hkv}; boxes of 64 head-dim elements (128 bytes) x 64
  // rows land 128-byte-swizzled, so ldmatrix on a landed tile is bank-conflict-free.  The encoder is a driver
  // entry point fetched at run time (the library does not link libcuda).
  plan->has_kv_tmap = 0;
  ML.attn_mma = 0;
  if (D.hd == 128 && (D.Hq / D.Hkv) <= 8) {
    typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                 const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess && fn &&
        qres == cudaDriverEntryPointSuccess) {
      CUtensorMap tm;
      cuuint64_t gdim[3] = {(cuuint64_t)D.hd, (cuuint64_t)D.max_seq, (cuuint64_t)D.L * 2 * D.Hkv};
      cuuint64_t gstr[2] = {(cuuint64_t)D.hd * 2, (cuuint64_t)D.max_seq * D.hd * 2};
      cuuint32_t box[3] = {64, 64, 1}, estr[3] = {1, 1, 1};
      CUresult r = ((EncodeFn)fn)(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, (void *)P.kv, gdim, gstr, box, estr,
                                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (r == CUDA_SUCCESS) {
        static_assert(sizeof(CUtensorMap) == sizeof(plan->kv_tmap), "tensor map storage");
        memcpy(plan->kv_tmap, &tm, sizeof tm);
        plan->has_kv_tmap = 1;
        ML.attn_mma = 1;
      }
    } else {
      cudaGetLastError();
    }
  }
  ML.repack = (const uint8_t *)repack;
  uint8_t *base = (uint8_t *)repack;
  int qd = D.Hq * D.hd, kd = D.Hkv * D.hd;
  const int RB = 1184, RT = 256;
  for (int l = 0; l < D.L; ++l) {
    uint8_t *lb = base + (size_t)l * ML.layer_bytes;
    // spd_weights order: 0 attn_norm 1 wq 2 wk 3 wv 4 wo 5 mlp_norm 6 w_gate 7 w_up 8 w_down
    k_repack<<<RB, RT, 0, stream>>>((uint16_t *)lb, ML.u_qkv, ML.nc_d, RM_QKV, src[1][l], src[2][l], src[3][l], qd, kd, kd,
                                    D.d, D.d, 0, D.hd);
    k_repack<<<RB, RT, 0, stream>>>((uint16_t *)(lb + ML.off_o), ML.u_o, ML.nc_qd, RM_PLAIN, src[4][l], nullptr, nullptr,
                                    D.d, 0, 0, qd, qd, 0, D.hd);
    k_repack<<<RB, RT, 0, stream>>>((uint16_t *)(lb + ML.off_gu), ML.u_gu, ML.nc_d, RM_GATEUP, src[6][l], src[7][l],
                                    nullptr, D.F, D.F, 0, D.d, D.d, 0, D.hd);
    k_repack<<<RB, RT, 0, stream>>>((uint16_t *)(lb + ML.off_dn), ML.u_dn, ML.nc_f, RM_PLAIN, src[8][l], nullptr, nullptr,
                                    D.d, 0, 0, D.F, D.F, 0, D.hd);
  }
  for (int j = 0; j < D.n; ++j)   // W_p column block j: [d, d] at columns j*d
    k_repack<<<RB, RT, 0, stream>>>((uint16_t *)(base + ML.off_pdm + (size_t)j * ML.pdm_job_bytes), ML.u_pdm, ML.nc_d,
                                    RM_PLAIN, P.pdm_proj, nullptr, nullptr, D.d, 0, 0, D.d, D.n * D.d, j * D.d, D.hd);
  k_repack<<<RB, RT, 0, stream>>>((uint16_t *)(base + ML.off_head), ML.u_head, ML.nc_d, RM_PLAIN, P.embed, nullptr, nullptr,
                                  D.V, 0, 0, D.d, D.d, 0, D.hd);
  if (cudaGetLastError() != cudaSuccess) return -1;
  plan->repack = (const uint16_t *)repack;
  plan->n_cta = sms;
  plan->smem_bytes = smem;
  plan->available = 1;
  static_assert(sizeof(MegaLayout) <= sizeof(plan->layout), "layout storage");
  memcpy(plan->layout, &ML, sizeof ML);
  return 0;
}

int mega_enqueue_step(const DevPtrs &P, const MegaPlan &plan, cudaStream_t sm, long long *launches) {
  if (!plan.available) return -1;
  MegaLayout ML;
  memcpy(&ML, plan.layout, sizeof ML);
  DevPtrs Pc = P;
  CUtensorMap tm;
  memcpy(&tm, plan.kv_tmap, sizeof tm);
  void *args[] = {(void *)&Pc, (void *)&ML, (void *)&tm};
  cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_spd_cycle, dim3(plan.n_cta), dim3(kThreads), args,
                                              (size_t)plan.smem_bytes, sm);
  if (launches) *launches += 1;
  return e == cudaSuccess ? 0 : -1;
}

}  // namespace spd
