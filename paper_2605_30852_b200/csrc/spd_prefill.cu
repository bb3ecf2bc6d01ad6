// spd_prefill.cu — batched prefill: the step BEFORE the path.
//
// PAPER.md:158 excludes prefill from the timed region; the decode kernel can run a prompt (one token enters per
// cycle), but that streams every layer's weights once per prompt token.  Prefill is the one genuine contraction of the
// scope — M = prompt tokens — so here it runs layer by layer over a chunk of the prompt as GEMMs on the 5th-generation
// tensor cores: tcgen05.mma (one elected thread issues), operands staged in shared memory by TMA
// (cp.async.bulk.tensor, 128-byte swizzle), accumulators in TMEM, read back with tcgen05.ld for the epilogue.
//
// Numeric contract (C-2.17): weights bf16, activations fp32.  An fp32 activation x is represented EXACTLY as three bf16
// parts, x = hi + mid + lo (hi = RNE(x), mid = RNE(x - hi), lo = x - hi - mid: 3 x 8 = 24 mantissa bits); all three
// multiply the exact bf16 weights into the SAME fp32 accumulator (three MMAs per k step), so every product is exact and
// the only difference from the decode path's GEMV is the order / rounding of the fp32 accumulation.  (Two parts — 16
// mantissa bits, 2^-17 per term — were measured first: K/V rounding flips and hidden-state error 10-15x those of the
// GEMV path on the small test models; with three parts they are the same.)  K/V rows are rounded to bf16 (RNE) when
// appended.
//
// Per layer and chunk of <= kChunk tokens (positions p0 .. p0 + M - 1):
//   k_pf_norm_split   X = RMSNorm(H; g) -> (hi, mid, lo)                       [M, d]
//   k_pf_gemm         Y = X . [Wq; Wk; Wv]^T                               [M, qd + 2 kd]      tcgen05
//   k_pf_rope_append  q -> RoPE -> Q fp32; k -> RoPE -> bf16 cache row; v -> bf16 cache row
//   k_pf_attention    causal GQA attention of the chunk over cache rows 0 .. pos -> (hi, mid, lo) [M, qd]
//   k_pf_gemm         Y = att . Wo^T;  k_pf_residual  H += Y
//   k_pf_norm_split   X = RMSNorm(H; g2);  k_pf_gemm  Y = X . [Wg; Wu]^T;  k_pf_silu_split  act = silu(g) * u -> (hi, mid, lo)
//   k_pf_gemm         Y = act . Wd^T;  k_pf_residual  H += Y
// then Hfin[p0 + t] = H[t]; the first token comes from the decode kernel's MODE_PREFILL_FINAL cycle (one pass over E).
#include <cuda.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include "spd_engine.h"
#include "spd_kernels.cuh"

namespace spd {

constexpr bool kPrefillAttnMma = true;    // prefill attention on mma.sync (false: the fp32 CUDA-core kernel)
constexpr int kGemmBM = 128;              // tokens per tile (TMEM lanes)
constexpr int kGemmBN = 256;              // output features per tile (TMEM fp32 columns)
constexpr int kGemmBK = 64;               // bf16 elements per k block = one 128-byte swizzle row
constexpr int kGemmStages = 2;
constexpr int kGemmThreads = 192;         // warp 0: TMA producer, warp 1: MMA issuer + TMEM owner, warps 2..5: epilogue
constexpr int kGemmStageBytes = (3 * kGemmBM + kGemmBN) * kGemmBK * 2;   // A hi + A mid + A lo + B = 80 KB
constexpr int kGemmSmem = kGemmStages * kGemmStageBytes + 1024 /*alignment*/ + 256 /*barriers*/;

// ------------------------------------------------------------------ PTX wrappers ------------------------------
__device__ __forceinline__ uint32_t pf_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void pf_mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(pf_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void pf_mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(pf_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void pf_mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok = 0;
  while (!ok) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(pf_smem_u32(bar)), "r"(parity) : "memory");
  }
}
__device__ __forceinline__ void pf_tma_load_2d(void *dst, const CUtensorMap *tmap, int c0, int c1, uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(pf_smem_u32(dst)), "l"(tmap), "r"(c0), "r"(c1), "r"(pf_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// D[tmem] (+)= A[smem desc] . B[smem desc]^T, bf16 x bf16 -> fp32, issued by ONE thread for the CTA
__device__ __forceinline__ void tc_mma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// mbarrier arrive when every tcgen05 operation issued so far by this thread has completed
__device__ __forceinline__ void tc_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(pf_smem_u32(bar)) : "memory");
}
// 32 lanes x 32 consecutive fp32 columns of TMEM -> 32 registers per thread (thread = lane)
__device__ __forceinline__ void tc_ld_32x32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

// Shared-memory matrix descriptor of a K-major tile whose rows are 128 bytes (64 bf16), 128-byte swizzled as TMA
// wrote them: start address (>> 4), stride between 8-row groups = 1024 bytes (>> 4), descriptor version 1 (sm_100),
// layout type 2 = SWIZZLE_128B.  The leading-dimension offset is unused for swizzled K-major operands.
__device__ __forceinline__ uint64_t tc_smem_desc(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3ffffu) >> 4);            // bits [0, 14)
  d |= (uint64_t)1 << 16;                                  // leading byte offset (ignored), bits [16, 30)
  d |= (uint64_t)(1024 >> 4) << 32;                        // stride byte offset, bits [32, 46)
  d |= (uint64_t)1 << 46;                                  // version, bits [46, 48)
  d |= (uint64_t)2 << 61;                                  // layout type, bits [61, 64)
  return d;
}
// Instruction descriptor of kind::f16: D fp32, A and B bf16, both K-major, M x N tile.
__host__ __device__ constexpr uint32_t tc_idesc_bf16(int M, int N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// ------------------------------------------------------------------ the GEMM ----------------------------------
// Y[m, col0 + n] = sum_k (Xhi[m, k] + Xlo[m, k]) * W_seg[n, k] for up to three weight matrices (segments) that share X:
// blockIdx.x runs over the 256-row tiles of the segments back to back, blockIdx.y over 128-token tiles.
struct GemmArgs {
  CUtensorMap a_hi, a_mid, a_lo;   // [rows >= M, K] bf16, box {64, 128}
  CUtensorMap b[3];                // [N_seg, K] bf16, box {64, 256}
  int seg_tiles[3];                // 256-row tiles of each segment (0: unused)
  int seg_n[3];                    // rows of each segment
  int seg_col0[3];                 // first output column of each segment
  int M, K, ldy;
  float *y;                        // [M, ldy] fp32
};

__global__ void __launch_bounds__(kGemmThreads, 1) k_pf_gemm(const __grid_constant__ GemmArgs A) {
  extern __shared__ uint8_t pf_smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>(((uintptr_t)pf_smem_raw + 1023) & ~(uintptr_t)1023);   // swizzle atoms: 1024-byte aligned
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + kGemmStages * kGemmStageBytes);
  uint64_t *empty = full + kGemmStages;
  uint64_t *tmem_full = empty + kGemmStages;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tmem_full + 1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int seg = 0, tile = blockIdx.x;
  while (seg < 2 && tile >= A.seg_tiles[seg]) { tile -= A.seg_tiles[seg]; ++seg; }
  const int n0 = tile * kGemmBN, m0 = blockIdx.y * kGemmBM;
  const int nkb = A.K / kGemmBK;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kGemmStages; ++s) { pf_mbar_init(&full[s], 1); pf_mbar_init(&empty[s], 1); }
    pf_mbar_init(tmem_full, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {   // TMEM: 256 fp32 columns x 128 lanes for the accumulator tile
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(pf_smem_u32(tmem_slot)), "r"((uint32_t)kGemmBN) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_d = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {   // ===== TMA producer =====
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % kGemmStages, it = kb / kGemmStages;
        pf_mbar_wait(&empty[s], (it & 1) ^ 1);
        uint8_t *st = smem + (size_t)s * kGemmStageBytes;
        pf_mbar_expect_tx(&full[s], kGemmStageBytes);
        pf_tma_load_2d(st, &A.a_hi, kb * kGemmBK, m0, &full[s]);
        pf_tma_load_2d(st + kGemmBM * 128, &A.a_mid, kb * kGemmBK, m0, &full[s]);
        pf_tma_load_2d(st + 2 * kGemmBM * 128, &A.a_lo, kb * kGemmBK, m0, &full[s]);
        pf_tma_load_2d(st + 3 * kGemmBM * 128, &A.b[seg], kb * kGemmBK, n0, &full[s]);
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {   // ===== MMA issuer =====
      constexpr uint32_t idesc = tc_idesc_bf16(kGemmBM, kGemmBN);
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % kGemmStages, it = kb / kGemmStages;
        pf_mbar_wait(&full[s], it & 1);
        tc_fence_after();
        const uint32_t a_hi = pf_smem_u32(smem + (size_t)s * kGemmStageBytes);
        const uint32_t a_mid = a_hi + kGemmBM * 128, a_lo = a_hi + 2 * kGemmBM * 128, b = a_hi + 3 * kGemmBM * 128;
#pragma unroll
        for (int k = 0; k < kGemmBK / 16; ++k) {      // UMMA_K = 16 bf16 = 32 bytes inside the 128-byte swizzle row
          const uint64_t bd = tc_smem_desc(b + k * 32);
          tc_mma_bf16(tmem_d, tc_smem_desc(a_hi + k * 32), bd, idesc, (kb | k) ? 1u : 0u);
          tc_mma_bf16(tmem_d, tc_smem_desc(a_mid + k * 32), bd, idesc, 1u);
          tc_mma_bf16(tmem_d, tc_smem_desc(a_lo + k * 32), bd, idesc, 1u);
        }
        tc_commit(&empty[s]);                         // the slot is free once these MMAs have read it
      }
      tc_commit(tmem_full);                           // the accumulator tile is complete
    }
  } else {             // ===== epilogue: TMEM -> registers -> Y (a warp owns the 32 TMEM lanes 32 * (warp % 4) ..) =====
    pf_mbar_wait(tmem_full, 0);
    tc_fence_after();
    const int lg = warp & 3;
    const int m = m0 + lg * 32 + lane;
    const int nseg = A.seg_n[seg];
    float *yrow = A.y + (size_t)m * A.ldy + A.seg_col0[seg] + n0;
    for (int c = 0; c < kGemmBN; c += 32) {
      if (n0 + c >= nseg) break;                      // uniform over the warp
      float v[32];
      tc_ld_32x32(tmem_d + ((uint32_t)(lg * 32) << 16) + (uint32_t)c, v);
      if (m < A.M) {
        if (n0 + c + 32 <= nseg) {
#pragma unroll
          for (int i = 0; i < 32; i += 4) *reinterpret_cast<float4 *>(yrow + c + i) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
        } else {
          for (int i = 0; i < 32; ++i) if (n0 + c + i < nseg) yrow[c + i] = v[i];
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"((uint32_t)kGemmBN) : "memory");
  }
}

// ------------------------------------------------------------------ the skinny GEMM (M = a few rows) ------------
// The paper PDM's per-cycle products (spd_pdm.cu): up to 48 activation rows against a weight matrix that has to be
// STREAMED once — HBM-bound like the GEMVs of the cycle kernel, but with M = n + 1 rows per weight tile.  The operands
// swap roles: the 128 x 64 weight tile is the MMA's A operand (weight rows = TMEM lanes), the activation rows — three
// exact bf16 parts of NB <= 48 rows — are the B operand (N = NB), so a 16 KB weight tile is multiplied into every row
// while it sits in shared memory, 8 stages (176 KB) of TMA loads are in flight per SM, and K is split over gridDim.y so
// that narrow matrices still fill 148 SMs.  Output: partial sums part[ks][row][column]; k_pf_skinny_reduce adds them in
// ks order (deterministic) into the destination (optionally on top of the residual).
constexpr int kSkMaxStages = 8;
constexpr int kSkMaxNB = 48;
// a stage = the 16 KB weight tile + three NB x 128-byte activation tiles: 8 stages of 22 KB at NB = 16 (176 KB in flight),
// 7 x 28 KB at NB = 32, 6 x 34 KB at NB = 48
__host__ __device__ constexpr int sk_stage_bytes(int NB) { return kGemmBM * 128 + 3 * NB * 128; }
__host__ __device__ constexpr int sk_stages(int NB) { return NB <= 16 ? 8 : (NB <= 32 ? 7 : 6); }

struct SkinnyArgs {
  CUtensorMap w[3];                // [N_seg, K] bf16, box {64, 128}
  CUtensorMap x[3];                // the three bf16 parts of the activation rows: [48, K], box {64, NB}
  int seg_tiles[3], seg_n[3], seg_col0[3];
  int K, NB, ldp, ksplit;          // ldp = columns of one partial row (sum of the segments' rows)
  float *part;                     // [gridDim.y][NB][ldp]
};

__device__ __forceinline__ void tc_ld_32x16(uint32_t taddr, float (&v)[16]) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}

// PERSISTENT: gridDim.x <= #SMs CTAs walk the work items (weight tile, K split) item = blockIdx.x, + gridDim.x, ...; the
// TMA producer streams across item boundaries without draining the ring, the MMA thread alternates between two TMEM
// accumulators so the epilogue of one item (TMEM -> partial sums) overlaps the next item's MMAs.
__global__ void __launch_bounds__(kGemmThreads, 1) k_pf_gemm_skinny(const __grid_constant__ SkinnyArgs A) {
  extern __shared__ uint8_t pf_smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>(((uintptr_t)pf_smem_raw + 1023) & ~(uintptr_t)1023);
  const int NB = A.NB, kSkStages = sk_stages(NB), kSkStageBytes = sk_stage_bytes(NB);
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + kSkStages * kSkStageBytes);
  uint64_t *empty = full + kSkMaxStages;
  uint64_t *tmem_full = empty + kSkMaxStages;          // [2]
  uint64_t *tmem_empty = tmem_full + 2;                // [2]
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tmem_empty + 2);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tiles = A.seg_tiles[0] + A.seg_tiles[1] + A.seg_tiles[2];
  const int n_items = tiles * A.ksplit;
  const int nkb_all = A.K / kGemmBK, per = (nkb_all + A.ksplit - 1) / A.ksplit;
  const uint32_t stage_tx = (uint32_t)(kGemmBM * 128 + 3 * NB * 128);

  if (threadIdx.x == 0) {
    for (int s = 0; s < kSkStages; ++s) { pf_mbar_init(&full[s], 1); pf_mbar_init(&empty[s], 1); }
    for (int a = 0; a < 2; ++a) { pf_mbar_init(&tmem_full[a], 1); pf_mbar_init(&tmem_empty[a], 4); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(pf_smem_u32(tmem_slot)), "r"(128u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  // item -> (segment, weight tile, K range)
  auto decode = [&](int item, int &seg, int &n0, int &kb0, int &nkb) {
    int tile = item / A.ksplit;
    const int ks = item - tile * A.ksplit;
    seg = 0;
    while (seg < 2 && tile >= A.seg_tiles[seg]) { tile -= A.seg_tiles[seg]; ++seg; }
    n0 = tile * kGemmBM;
    kb0 = ks * per;
    nkb = max(0, min(nkb_all, kb0 + per) - kb0);
    return ks;
  };

  if (warp == 0) {
    if (lane == 0) {   // ===== TMA producer: one continuous stream over this CTA's items =====
      uint32_t q = 0;
      for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        int seg, n0, kb0, nkb;
        decode(item, seg, n0, kb0, nkb);
        for (int i = 0; i < nkb; ++i, ++q) {
          const int s = q % kSkStages, it = q / kSkStages, kb = kb0 + i;
          pf_mbar_wait(&empty[s], (it & 1) ^ 1);
          uint8_t *st = smem + (size_t)s * kSkStageBytes;
          pf_mbar_expect_tx(&full[s], stage_tx);
          pf_tma_load_2d(st, &A.w[seg], kb * kGemmBK, n0, &full[s]);
#pragma unroll
          for (int p = 0; p < 3; ++p) pf_tma_load_2d(st + kGemmBM * 128 + p * NB * 128, &A.x[p], kb * kGemmBK, 0, &full[s]);
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {   // ===== MMA issuer: two accumulators, alternating per item =====
      const uint32_t idesc = tc_idesc_bf16(kGemmBM, NB);
      uint32_t q = 0;
      int n_mine = 0;
      for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++n_mine) {
        int seg, n0, kb0, nkb;
        decode(item, seg, n0, kb0, nkb);
        const int acc = n_mine & 1, use = n_mine >> 1;
        pf_mbar_wait(&tmem_empty[acc], (use & 1) ^ 1);   // the epilogue drained this accumulator (first use: passes)
        tc_fence_after();
        const uint32_t tmem_d = tmem_base + (uint32_t)(acc * 64);
        for (int i = 0; i < nkb; ++i, ++q) {
          const int s = q % kSkStages, it = q / kSkStages;
          pf_mbar_wait(&full[s], it & 1);
          tc_fence_after();
          const uint32_t a = pf_smem_u32(smem + (size_t)s * kSkStageBytes), b = a + kGemmBM * 128;
#pragma unroll
          for (int k = 0; k < kGemmBK / 16; ++k) {
            const uint64_t ad = tc_smem_desc(a + k * 32);
#pragma unroll
            for (int p = 0; p < 3; ++p)
              tc_mma_bf16(tmem_d, ad, tc_smem_desc(b + p * NB * 128 + k * 32), idesc, (i | k | p) ? 1u : 0u);
          }
          tc_commit(&empty[s]);
        }
        tc_commit(&tmem_full[acc]);
      }
    }
  } else {             // ===== epilogue: TMEM -> split-K partial sums =====
    const int lg = warp & 3;
    int n_mine = 0;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x, ++n_mine) {
      int seg, n0, kb0, nkb;
      const int ks = decode(item, seg, n0, kb0, nkb);
      const int acc = n_mine & 1, use = n_mine >> 1;
      pf_mbar_wait(&tmem_full[acc], use & 1);
      tc_fence_after();
      const int n = n0 + lg * 32 + lane;               // this thread's weight row = output column
      const bool in = n < A.seg_n[seg];
      float *prow = A.part + ((size_t)ks * NB) * A.ldp + A.seg_col0[seg] + n;
      for (int c = 0; c < NB; c += 16) {
        float v[16];
        tc_ld_32x16(tmem_base + (uint32_t)(acc * 64) + ((uint32_t)(lg * 32) << 16) + (uint32_t)c, v);
#pragma unroll
        for (int r = 0; r < 16; ++r)
          if (in) prow[(size_t)(c + r) * A.ldp] = nkb > 0 ? v[r] : 0.f;
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(pf_smem_u32(&tmem_empty[acc])) : "memory");
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(128u) : "memory");
  }
}

// dst[r][c] (+)= sum over ks (in order) of part[ks][r][c], r < *rows_ptr (clamped to NB), c < ncol
__global__ void k_pf_skinny_reduce(const float *part, int ksplit, int NB, int ldp, const int *rows_ptr, int rows_fixed,
                                   float *dst, int ldd, int ncol, int residual) {
  const int rows = min(NB, rows_fixed > 0 ? rows_fixed : *rows_ptr);
  const size_t n = (size_t)rows * ncol;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t r = i / ncol, c = i - r * ncol;
    float v = 0.f;
    for (int ks = 0; ks < ksplit; ++ks) v += part[((size_t)ks * NB + r) * ldp + c];
    float *d = dst + r * ldd + c;
    *d = residual ? *d + v : v;
  }
}

// ------------------------------------------------------------------ elementwise kernels ------------------------
// x = hi + mid + lo exactly (finite x; each residual is exact in fp32 and the last one fits 8 mantissa bits)
struct Split3 { uint16_t hi, mid, lo; };
__device__ __forceinline__ Split3 pf_split(float x) {
  Split3 s;
  s.hi = f32_to_bf16(x);
  const float r1 = x - bf16_to_f32(s.hi);
  s.mid = f32_to_bf16(r1);
  s.lo = f32_to_bf16(r1 - bf16_to_f32(s.mid));
  return s;
}

// H[t] = E[tok[p0 + t]] (token entry, a0)
__global__ void k_pf_embed(const uint16_t *embed, const int32_t *tokens, int p0, int d, float *H) {
  const int t = blockIdx.x;
  const uint16_t *e = embed + (size_t)tokens[p0 + t] * d;
  for (int i = threadIdx.x; i < d; i += blockDim.x) H[(size_t)t * d + i] = bf16_to_f32(e[i]);
}

// X = RMSNorm(H[t]; gain) -> bf16 hi / mid / lo rows (a1.1 / a1.6).  One CTA per token; the sum of squares uses the
// decode path's block_rms_scale tree.
__global__ void k_pf_norm_split(const float *H, const uint16_t *gain, int d, float eps, uint16_t *x3, size_t plane) {
  __shared__ float red[33];
  const int t = blockIdx.x;
  const float *h = H + (size_t)t * d;
  const float r = block_rms_scale(h, d, eps, red);
  for (int i = threadIdx.x; i < d; i += blockDim.x) {
    const Split3 sp = pf_split(h[i] * r * bf16_to_f32(gain[i]));
    const size_t o = (size_t)t * d + i;
    x3[o] = sp.hi; x3[plane + o] = sp.mid; x3[2 * plane + o] = sp.lo;
  }
}

// Y row = [q (qd) | k (kd) | v (kd)]: RoPE (C-2.14, angles in double) on q and k; q -> Q fp32; k, v -> bf16 cache rows
// at position p0 + t (a1.3).  One CTA per token.
__global__ void k_pf_rope_append(const float *Y, int ldy, DevPtrs P, int layer, int p0, float *Q) {
  const Dims &D = P.dim;
  __shared__ float2 cs[64];
  const int t = blockIdx.x, pos = p0 + t, half = D.hd / 2, qd = D.Hq * D.hd, kd = D.Hkv * D.hd;
  if (threadIdx.x < half) {
    double s_, c_;
    sincos((double)pos * P.inv_freq[threadIdx.x], &s_, &c_);
    cs[threadIdx.x] = make_float2((float)c_, (float)s_);
  }
  __syncthreads();
  const float *y = Y + (size_t)t * ldy;
  for (int j = threadIdx.x; j < (D.Hq + D.Hkv) * half; j += blockDim.x) {
    const int hh = j / half, i = j - hh * half;
    const float2 c = cs[i];
    if (hh < D.Hq) {
      const float a = y[hh * D.hd + i], b = y[hh * D.hd + i + half];
      float *q = Q + (size_t)t * qd + hh * D.hd;
      q[i] = a * c.x - b * c.y;
      q[i + half] = b * c.x + a * c.y;
    } else {
      const int kh = hh - D.Hq;
      const float a = y[qd + kh * D.hd + i], b = y[qd + kh * D.hd + i + half];
      uint16_t *dst = P.kv + kv_offset(D, layer, 0, kh) + (size_t)pos * D.hd;
      dst[i] = f32_to_bf16(a * c.x - b * c.y);
      dst[i + half] = f32_to_bf16(b * c.x + a * c.y);
    }
  }
  for (int j = threadIdx.x; j < kd; j += blockDim.x) {
    const int kh = j / D.hd, i = j - kh * D.hd;
    P.kv[kv_offset(D, layer, 1, kh) + (size_t)pos * D.hd + i] = f32_to_bf16(y[qd + kd + j]);
  }
}

// H += Y (residual, a1.5 / a1.8)
__global__ void k_pf_residual(float *H, const float *Y, int ldy, int d, int M) {
  const size_t n = (size_t)M * d;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t t = i / d, c = i - t * d;
    H[i] += Y[t * ldy + c];
  }
}

// act = silu(gate) * up -> bf16 hi / mid / lo (a1.7); Y row = [gate (F) | up (F)]
__global__ void k_pf_silu_split(const float *Y, int ldy, int F, int M, uint16_t *x3, size_t plane) {
  const size_t n = (size_t)M * F;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t t = i / F, c = i - t * F;
    const Split3 sp = pf_split(silu_mul(Y[t * ldy + c], Y[t * ldy + F + c]));
    x3[i] = sp.hi; x3[plane + i] = sp.mid; x3[2 * plane + i] = sp.lo;
  }
}

// NEXT-1: H^layer of the paper PDM's anchor set for the chunk's positions: anch[p0 + t][ai] = H[t]
__global__ void k_pf_store_anchor(const float *H, float *anch, int p0, int d, int M, int m, int ai) {
  const size_t n = (size_t)M * d;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t t = i / d, c = i - t * d;
    anch[((size_t)(p0 + t) * m + ai) * d + c] = H[i];
  }
}

// Hfin[p0 + t] = H[t]
__global__ void k_pf_store_hfin(const float *H, float *hfin, int p0, int d, int M) {
  const size_t n = (size_t)M * d;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    hfin[(size_t)p0 * d + i] = H[i];
}

// fp32 matrix -> bf16 hi / mid / lo (spd_op_gemm's input split)
__global__ void k_pf_split(const float *x, size_t n, uint16_t *x3, size_t plane) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const Split3 sp = pf_split(x[i]);
    x3[i] = sp.hi; x3[plane + i] = sp.mid; x3[2 * plane + i] = sp.lo;
  }
}

// ------------------------------------------------------------------ causal prefill attention (a1.4) ------------
// One CTA = one kv head x a block of TQ = 64 / G chunk tokens: R = 64 query rows (token-major, row = tq * G + g), all
// of them reading the same K/V rows.  Cache rows 0 .. pos (causal incl. self) are visited in tiles of 64 rows, widened
// to fp32 in shared memory; scores, online softmax (running max / sum per row) and P.V in fp32 on the CUDA cores —
// 4 flop per K/V byte at M = 1 is the decode path's problem; at prefill the GEMMs dominate.
// Thread (ty, tx) = (tid / 16, tid % 16) owns score rows 4 ty .. 4 ty + 3 x columns tx, tx + 16, tx + 32, tx + 48 and
// output rows 4 ty .. 4 ty + 3 x head-dim elements tx * HD/16 ..; every sum runs in a fixed order.
template <int HD>
__global__ void __launch_bounds__(256, 1) k_pf_attention(DevPtrs P, int layer, int p0, int M, const float *Q,
                                                         uint16_t *x3, size_t plane) {
  constexpr int R = 64, TK = 64, LDK = HD + 4, EPT = HD / 16;
  const Dims &D = P.dim;
  const int G = D.Hq / D.Hkv, TQ = R / G, qd = D.Hq * HD;
  extern __shared__ float pf_att_smem[];
  float *Qs = pf_att_smem;               // [R][LDK]
  float *Ks = Qs + R * LDK;              // [TK][LDK]
  float *Vs = Ks + TK * LDK;             // [TK][LDK]
  float *Ss = Vs + TK * LDK;             // [R][TK + 1]
  float *m_s = Ss + R * (TK + 1);        // [R] running max
  float *l_s = m_s + R;                  // [R] running sum
  float *c_s = l_s + R;                  // [R] correction of this tile
  const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
  const int kvh = blockIdx.y, t0 = blockIdx.x * TQ;
  const float scale = 1.0f / sqrtf((float)HD);
  for (int i = tid; i < R * (HD / 4); i += 256) {          // Q rows of this block (zero for tokens beyond M)
    const int r = i / (HD / 4), c4 = i - r * (HD / 4);
    const int t = t0 + r / G, g = r % G;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (t < M) v = *reinterpret_cast<const float4 *>(Q + (size_t)t * qd + (size_t)(kvh * G + g) * HD + 4 * c4);
    *reinterpret_cast<float4 *>(Qs + r * LDK + 4 * c4) = v;
  }
  if (tid < R) { m_s[tid] = -INFINITY; l_s[tid] = 0.f; }
  float acc[4][EPT];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int e = 0; e < EPT; ++e) acc[i][e] = 0.f;
  const int last_pos = p0 + min(t0 + TQ, M) - 1;            // the newest row any token of the block attends to
  const uint16_t *kc = P.kv + kv_offset(D, layer, 0, kvh), *vc = P.kv + kv_offset(D, layer, 1, kvh);
  for (int r0 = 0; r0 <= last_pos; r0 += TK) {
    __syncthreads();                                         // the previous tile is consumed (and Qs / m / l are written)
    for (int i = tid; i < TK * (HD / 8); i += 256) {         // 16-byte chunks of K and V rows -> fp32
      const int r = i / (HD / 8), c8 = i - r * (HD / 8);
      uint4 kw = make_uint4(0u, 0u, 0u, 0u), vw = kw;
      if (r0 + r <= last_pos) {
        kw = *reinterpret_cast<const uint4 *>(kc + (size_t)(r0 + r) * HD + 8 * c8);
        vw = *reinterpret_cast<const uint4 *>(vc + (size_t)(r0 + r) * HD + 8 * c8);
      }
      float *kd = Ks + r * LDK + 8 * c8, *vd = Vs + r * LDK + 8 * c8;
      *reinterpret_cast<float4 *>(kd) = make_float4(bf16_lo(kw.x), bf16_hi(kw.x), bf16_lo(kw.y), bf16_hi(kw.y));
      *reinterpret_cast<float4 *>(kd + 4) = make_float4(bf16_lo(kw.z), bf16_hi(kw.z), bf16_lo(kw.w), bf16_hi(kw.w));
      *reinterpret_cast<float4 *>(vd) = make_float4(bf16_lo(vw.x), bf16_hi(vw.x), bf16_lo(vw.y), bf16_hi(vw.y));
      *reinterpret_cast<float4 *>(vd + 4) = make_float4(bf16_lo(vw.z), bf16_hi(vw.z), bf16_lo(vw.w), bf16_hi(vw.w));
    }
    __syncthreads();
    // ---- scores of the tile: s[i][j] = q[4 ty + i] . k[tx + 16 j], scaled, causally masked -> Ss ----
    {
      float s[4][4];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s[i][j] = 0.f;
#pragma unroll 4
      for (int k = 0; k < HD; k += 4) {
        float4 qv[4], kv4[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) qv[i] = *reinterpret_cast<const float4 *>(Qs + (4 * ty + i) * LDK + k);
#pragma unroll
        for (int j = 0; j < 4; ++j) kv4[j] = *reinterpret_cast<const float4 *>(Ks + (tx + 16 * j) * LDK + k);
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            s[i][j] = fmaf(qv[i].x, kv4[j].x, s[i][j]); s[i][j] = fmaf(qv[i].y, kv4[j].y, s[i][j]);
            s[i][j] = fmaf(qv[i].z, kv4[j].z, s[i][j]); s[i][j] = fmaf(qv[i].w, kv4[j].w, s[i][j]);
          }
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int r = 4 * ty + i, pos = p0 + t0 + r / G;     // this query row's position
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int c = tx + 16 * j;
          Ss[r * (TK + 1) + c] = (r0 + c <= pos) ? s[i][j] * scale : -INFINITY;
        }
      }
    }
    __syncthreads();
    // ---- online softmax: 4 threads per row, 16 columns each ----
    {
      const int r = tid >> 2, part = tid & 3;
      float *srow = Ss + r * (TK + 1) + 16 * part;
      float mx = -INFINITY;
#pragma unroll
      for (int c = 0; c < 16; ++c) mx = fmaxf(mx, srow[c]);
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
      const float m_old = m_s[r], m_new = fmaxf(m_old, mx);
      float sum = 0.f;
#pragma unroll
      for (int c = 0; c < 16; ++c) {
        const float pr = (m_new == -INFINITY) ? 0.f : expf(srow[c] - m_new);   // a fully masked row (token beyond M) stays 0
        srow[c] = pr;
        sum += pr;
      }
      sum += __shfl_xor_sync(0xffffffffu, sum, 1);
      sum += __shfl_xor_sync(0xffffffffu, sum, 2);
      __syncwarp();
      if (part == 0) {
        const float corr = (m_old == -INFINITY) ? 0.f : expf(m_old - m_new);
        c_s[r] = corr;
        l_s[r] = fmaf(l_s[r], corr, sum);
        m_s[r] = m_new;
      }
    }
    __syncthreads();
    // ---- O = O * corr + P . V ----
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float corr = c_s[4 * ty + i];
#pragma unroll
      for (int e = 0; e < EPT; ++e) acc[i][e] *= corr;
    }
#pragma unroll 4
    for (int c = 0; c < TK; ++c) {
      float vv[EPT];
#pragma unroll
      for (int e = 0; e < EPT; e += 4) {
        const float4 t4 = *reinterpret_cast<const float4 *>(Vs + c * LDK + tx * EPT + e);
        vv[e] = t4.x; vv[e + 1] = t4.y; vv[e + 2] = t4.z; vv[e + 3] = t4.w;
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float pr = Ss[(4 * ty + i) * (TK + 1) + c];
#pragma unroll
        for (int e = 0; e < EPT; ++e) acc[i][e] = fmaf(pr, vv[e], acc[i][e]);
      }
    }
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = 4 * ty + i, t = t0 + r / G, g = r % G;
    if (t >= M) continue;
    const float l = l_s[r];
    const size_t o = (size_t)t * qd + (size_t)(kvh * G + g) * HD + tx * EPT;
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
      const Split3 sp = pf_split(acc[i][e] / l);
      x3[o + e] = sp.hi; x3[plane + o + e] = sp.mid; x3[2 * plane + o + e] = sp.lo;
    }
  }
}

// ------------------------------------------------------------------ prefill attention on the tensor cores -------
// Same work split as k_pf_attention (one CTA = one kv head x 64 / G chunk tokens = 64 query rows, cache rows visited in
// tiles of 64), but scores and P.V run as mma.sync.m16n8k16 (bf16 x bf16 -> fp32): warp w owns query rows 16 w .. 16 w + 15
// and keeps Q (as bf16 hi + lo parts), the score / probability fragments and the 16 x HD output tile in registers
// (flash-attention-2 layout: the score fragment of a thread IS the A fragment of P.V); K and V tiles stay bf16 in shared
// memory, 16-byte chunks XOR-swizzled by (row & 7) so ldmatrix / ldmatrix.trans are bank-conflict-free.  q and the
// probabilities are fp32 by contract (C-2.17): each is split into bf16 hi + lo (16 mantissa bits, products with the exact
// bf16 K / V accumulate in fp32) — the representation the decode kernel's tensor-core attention already uses.
__device__ __forceinline__ void pf_ldsm4(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void pf_ldsm4t(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void pf_mma(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void pf_split2(float x0, float x1, uint32_t &hi, uint32_t &lo) {
  const uint16_t h0 = f32_to_bf16(x0), h1 = f32_to_bf16(x1);
  const uint16_t l0 = f32_to_bf16(x0 - bf16_to_f32(h0)), l1 = f32_to_bf16(x1 - bf16_to_f32(h1));
  hi = (uint32_t)h0 | ((uint32_t)h1 << 16);
  lo = (uint32_t)l0 | ((uint32_t)l1 << 16);
}

template <int HD>
__global__ void __launch_bounds__(128, 2) k_pf_attention_mma(DevPtrs P, int layer, int p0, int M, const float *Q,
                                                             uint16_t *x3, size_t plane) {
  constexpr int TK = 64, KS = HD / 16, NT = HD / 8, CPR = HD / 8;      // k steps of Q.K^T, n tiles of P.V, 16-byte chunks per row
  const Dims &D = P.dim;
  const int G = D.Hq / D.Hkv, TQ = 64 / G, qd = D.Hq * HD;
  __shared__ __align__(128) uint16_t Ks[TK * HD];
  __shared__ __align__(128) uint16_t Vs[TK * HD];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
  const int mi = lane >> 3, mr = lane & 7;                             // ldmatrix: this lane addresses row mr of matrix mi
  const int kvh = blockIdx.y, t0 = blockIdx.x * TQ;
  // this thread's two query rows (of the CTA's 64): r_lo = 16 warp + g, r_hi = r_lo + 8; row = tq * G + head-in-group
  const int r_lo = 16 * warp + g, r_hi = r_lo + 8;
  const int tok_lo = t0 + r_lo / G, tok_hi = t0 + r_hi / G;
  const int hq_lo = kvh * G + r_lo % G, hq_hi = kvh * G + r_hi % G;
  const int pos_lo = p0 + tok_lo, pos_hi = p0 + tok_hi;
  uint32_t qh[KS][4], ql[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    float2 a = make_float2(0.f, 0.f), b = a, c = a, d = a;
    if (tok_lo < M) {
      const float *q = Q + (size_t)tok_lo * qd + (size_t)hq_lo * HD + 16 * ks + 2 * t;
      a = *reinterpret_cast<const float2 *>(q); c = *reinterpret_cast<const float2 *>(q + 8);
    }
    if (tok_hi < M) {
      const float *q = Q + (size_t)tok_hi * qd + (size_t)hq_hi * HD + 16 * ks + 2 * t;
      b = *reinterpret_cast<const float2 *>(q); d = *reinterpret_cast<const float2 *>(q + 8);
    }
    pf_split2(a.x, a.y, qh[ks][0], ql[ks][0]); pf_split2(b.x, b.y, qh[ks][1], ql[ks][1]);
    pf_split2(c.x, c.y, qh[ks][2], ql[ks][2]); pf_split2(d.x, d.y, qh[ks][3], ql[ks][3]);
  }
  float o[NT][4];
#pragma unroll
  for (int j = 0; j < NT; ++j) { o[j][0] = o[j][1] = o[j][2] = o[j][3] = 0.f; }
  float m_lo = -INFINITY, m_hi = -INFINITY, l_lo = 0.f, l_hi = 0.f;
  const float scale = 1.0f / sqrtf((float)HD);
  const int last_pos = p0 + min(t0 + TQ, M) - 1;
  const uint16_t *kc = P.kv + kv_offset(D, layer, 0, kvh), *vc = P.kv + kv_offset(D, layer, 1, kvh);
  const uint32_t ks_base = pf_smem_u32(Ks), vs_base = pf_smem_u32(Vs);
  for (int r0 = 0; r0 <= last_pos; r0 += TK) {
    __syncthreads();                                                   // the previous tile is consumed
    for (int i = tid; i < TK * CPR; i += 128) {                        // 16-byte chunks, swizzled by (row & 7)
      const int r = i / CPR, c = i - r * CPR;
      uint4 kw = make_uint4(0u, 0u, 0u, 0u), vw = kw;
      if (r0 + r <= last_pos) {
        kw = *reinterpret_cast<const uint4 *>(kc + (size_t)(r0 + r) * HD + 8 * c);
        vw = *reinterpret_cast<const uint4 *>(vc + (size_t)(r0 + r) * HD + 8 * c);
      }
      const int o16 = r * CPR + (c ^ (r & 7));
      reinterpret_cast<uint4 *>(Ks)[o16] = kw;
      reinterpret_cast<uint4 *>(Vs)[o16] = vw;
    }
    __syncthreads();
    // ---- S = Q . K^T for this warp's 16 rows x 64 cache rows: 8 n tiles, hi and lo parts of q ----
    float s[8][4];
#pragma unroll
    for (int j = 0; j < 8; ++j) { s[j][0] = s[j][1] = s[j][2] = s[j][3] = 0.f; }
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) {                                   // two n tiles (16 cache rows) per ldmatrix.x4
      const int krow = 16 * jj + (mi >> 1) * 8 + mr;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        const int cc = 2 * ks + (mi & 1);
        uint32_t b[4];
        pf_ldsm4(b, ks_base + (uint32_t)((krow * CPR + (cc ^ (krow & 7))) * 16));
        pf_mma(s[2 * jj], qh[ks], b[0], b[1]); pf_mma(s[2 * jj], ql[ks], b[0], b[1]);
        pf_mma(s[2 * jj + 1], qh[ks], b[2], b[3]); pf_mma(s[2 * jj + 1], ql[ks], b[2], b[3]);
      }
    }
    // ---- scale, causal mask, online softmax (rows g and g + 8 of the warp; a row's 64 columns live in one quad) ----
    float mx_lo = -INFINITY, mx_hi = -INFINITY;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int c0 = r0 + 8 * j + 2 * t;
      s[j][0] = c0 <= pos_lo ? s[j][0] * scale : -INFINITY;
      s[j][1] = c0 + 1 <= pos_lo ? s[j][1] * scale : -INFINITY;
      s[j][2] = c0 <= pos_hi ? s[j][2] * scale : -INFINITY;
      s[j][3] = c0 + 1 <= pos_hi ? s[j][3] * scale : -INFINITY;
      mx_lo = fmaxf(mx_lo, fmaxf(s[j][0], s[j][1]));
      mx_hi = fmaxf(mx_hi, fmaxf(s[j][2], s[j][3]));
    }
    mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 1)); mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 2));
    mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 1)); mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 2));
    const float mn_lo = fmaxf(m_lo, mx_lo), mn_hi = fmaxf(m_hi, mx_hi);
    const float cr_lo = m_lo == -INFINITY ? 0.f : expf(m_lo - mn_lo), cr_hi = m_hi == -INFINITY ? 0.f : expf(m_hi - mn_hi);
    float sum_lo = 0.f, sum_hi = 0.f;
    uint32_t ph[4][4], pl[4][4];                                       // A fragments of P.V, one per 16 cache rows
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const float e0 = mn_lo == -INFINITY ? 0.f : expf(s[j][0] - mn_lo), e1 = mn_lo == -INFINITY ? 0.f : expf(s[j][1] - mn_lo);
      const float e2 = mn_hi == -INFINITY ? 0.f : expf(s[j][2] - mn_hi), e3 = mn_hi == -INFINITY ? 0.f : expf(s[j][3] - mn_hi);
      sum_lo += e0 + e1; sum_hi += e2 + e3;
      // n tile j of S = k rows 8 j .. 8 j + 7 of P.V: tile 2 kk -> a0 (row g), a1 (row g + 8); tile 2 kk + 1 -> a2, a3
      pf_split2(e0, e1, ph[j >> 1][(j & 1) * 2], pl[j >> 1][(j & 1) * 2]);
      pf_split2(e2, e3, ph[j >> 1][(j & 1) * 2 + 1], pl[j >> 1][(j & 1) * 2 + 1]);
    }
    sum_lo += __shfl_xor_sync(0xffffffffu, sum_lo, 1); sum_lo += __shfl_xor_sync(0xffffffffu, sum_lo, 2);
    sum_hi += __shfl_xor_sync(0xffffffffu, sum_hi, 1); sum_hi += __shfl_xor_sync(0xffffffffu, sum_hi, 2);
    l_lo = fmaf(l_lo, cr_lo, sum_lo); l_hi = fmaf(l_hi, cr_hi, sum_hi);
    m_lo = mn_lo; m_hi = mn_hi;
#pragma unroll
    for (int j = 0; j < NT; ++j) { o[j][0] *= cr_lo; o[j][1] *= cr_lo; o[j][2] *= cr_hi; o[j][3] *= cr_hi; }
    // ---- O += P . V: k = the tile's 64 cache rows (4 k steps), n = head dims (NT tiles), V through ldmatrix.trans ----
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) {
      const int vrow = 16 * kk + (mi & 1) * 8 + mr;
#pragma unroll
      for (int jj = 0; jj < NT / 2; ++jj) {
        const int cc = 2 * jj + (mi >> 1);
        uint32_t b[4];
        pf_ldsm4t(b, vs_base + (uint32_t)((vrow * CPR + (cc ^ (vrow & 7))) * 16));
        pf_mma(o[2 * jj], ph[kk], b[0], b[1]); pf_mma(o[2 * jj], pl[kk], b[0], b[1]);
        pf_mma(o[2 * jj + 1], ph[kk], b[2], b[3]); pf_mma(o[2 * jj + 1], pl[kk], b[2], b[3]);
      }
    }
  }
  // ---- out = O / l as three exact bf16 parts (the O projection's GEMM input) ----
#pragma unroll
  for (int j = 0; j < NT; ++j) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int tok = h ? tok_hi : tok_lo;
      if (tok >= M) continue;
      const float l = h ? l_hi : l_lo;
      const size_t ob = (size_t)tok * qd + (size_t)(h ? hq_hi : hq_lo) * HD + 8 * j + 2 * t;
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const Split3 sp = pf_split(o[j][2 * h + e] / l);
        x3[ob + e] = sp.hi; x3[plane + ob + e] = sp.mid; x3[2 * plane + ob + e] = sp.lo;
      }
    }
  }
}

// ------------------------------------------------------------------ host side ----------------------------------
typedef CUresult (*PfEncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                               const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PfEncodeFn pf_encoder() {
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  return (PfEncodeFn)fn;
}

// bf16 matrix [rows, K] row-major -> tensor map with boxes of 64 columns (128 bytes, swizzled) x box_rows rows
static int pf_make_map(PfEncodeFn enc, CUtensorMap *tm, const void *base, int rows, int K, int box_rows) {
  cuuint64_t gdim[2] = {(cuuint64_t)K, (cuuint64_t)rows};
  cuuint64_t gstr[1] = {(cuuint64_t)K * 2};
  cuuint32_t box[2] = {(cuuint32_t)kGemmBK, (cuuint32_t)box_rows}, estr[2] = {1, 1};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), gdim, gstr, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? 0 : -1;
}

static int pf_launch_gemm(PfEncodeFn enc, const uint16_t *x3, size_t plane, int x_rows, int M, int K,
                          const uint16_t *const *w, const int *w_rows, int nseg, float *y, int ldy, cudaStream_t st,
                          long long *launches) {
  GemmArgs A;
  memset(&A, 0, sizeof A);
  if (pf_make_map(enc, &A.a_hi, x3, x_rows, K, kGemmBM) || pf_make_map(enc, &A.a_mid, x3 + plane, x_rows, K, kGemmBM) ||
      pf_make_map(enc, &A.a_lo, x3 + 2 * plane, x_rows, K, kGemmBM))
    return -1;
  int tiles = 0, col = 0;
  for (int s = 0; s < nseg; ++s) {
    if (pf_make_map(enc, &A.b[s], w[s], w_rows[s], K, kGemmBN)) return -1;
    A.seg_tiles[s] = (w_rows[s] + kGemmBN - 1) / kGemmBN;
    A.seg_n[s] = w_rows[s];
    A.seg_col0[s] = col;
    col += w_rows[s];
    tiles += A.seg_tiles[s];
  }
  A.M = M; A.K = K; A.ldy = ldy; A.y = y;
  dim3 grid(tiles, (M + kGemmBM - 1) / kGemmBM);
  k_pf_gemm<<<grid, kGemmThreads, kGemmSmem, st>>>(A);
  if (launches) *launches += 1;
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

// Skinny GEMM launcher: x3 = three bf16 planes of [48][K] rows (plane stride in elements), rows on the device
// (rows_ptr) or fixed.  part: scratch of >= ksplit * NB * ncol floats.
int skinny_gemm(const uint16_t *x3, size_t plane, int K, int NB, const uint16_t *const *w, const int *w_rows, int nseg,
                float *part, size_t part_floats, const int *rows_ptr, int rows_fixed, float *dst, int ldd, int residual,
                cudaStream_t st, long long *launches, int *ksplit_out) {
  static PfEncodeFn enc = nullptr;
  static bool attr = false;
  if (!enc) enc = pf_encoder();
  if (!enc || K % kGemmBK || NB % 16 || NB < 16 || NB > kSkMaxNB) return -1;
  if (!attr) {
    if (cudaFuncSetAttribute(k_pf_gemm_skinny, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024) != cudaSuccess) return -1;
    attr = true;
  }
  const int sk_smem = sk_stages(NB) * sk_stage_bytes(NB) + 1024 + 256;
  SkinnyArgs A;
  memset(&A, 0, sizeof A);
  int tiles = 0, col = 0;
  for (int s = 0; s < nseg; ++s) {
    if (pf_make_map(enc, &A.w[s], w[s], w_rows[s], K, kGemmBM)) return -1;
    A.seg_tiles[s] = (w_rows[s] + kGemmBM - 1) / kGemmBM;
    A.seg_n[s] = w_rows[s];
    A.seg_col0[s] = col;
    col += w_rows[s];
    tiles += A.seg_tiles[s];
  }
  for (int p = 0; p < 3; ++p)
    if (pf_make_map(enc, &A.x[p], x3 + p * plane, kSkMaxNB, K, NB)) return -1;
  const int nkb = K / kGemmBK;
  // K split: work items of >= 8 k-blocks (>= 176 KB) whose count fills whole waves of the persistent grid
  static int sms = 0;
  if (!sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); if (sms < 1) sms = 148; }
  int ksplit = 1;
  double best = -1.0;
  for (int k = 1; k <= 16 && nkb / k >= 8; ++k) {
    if ((size_t)k * NB * col > part_floats) break;
    const int items = tiles * k, waves = (items + sms - 1) / sms;
    const double eff = (double)items / ((double)waves * sms) - 0.01 * k;     // fuller waves first, then fewer partial sums
    if (eff > best) { best = eff; ksplit = k; }
  }
  if ((size_t)ksplit * NB * col > part_floats) return -1;
  A.K = K; A.NB = NB; A.ldp = col; A.part = part; A.ksplit = ksplit;
  const int grid = tiles * ksplit < sms ? tiles * ksplit : sms;
  k_pf_gemm_skinny<<<grid, kGemmThreads, sk_smem, st>>>(A);
  if (ksplit_out) {                                   // the caller reduces the partial sums itself (fused epilogues)
    *ksplit_out = ksplit;
    if (launches) *launches += 1;
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
  }
  const int rb = (int)(((size_t)NB * col + 255) / 256);
  k_pf_skinny_reduce<<<rb < 1184 ? rb : 1184, 256, 0, st>>>(part, ksplit, NB, col, rows_ptr, rows_fixed, dst, ldd, col, residual);
  if (launches) *launches += 2;
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

bool prefill_supported(const Dims &D) {
  const int qd = D.Hq * D.hd;
  const int G = D.Hq / D.Hkv;
  return D.d % kGemmBK == 0 && qd % kGemmBK == 0 && D.F % kGemmBK == 0 && (D.hd == 64 || D.hd == 128) &&
         (G == 1 || G == 2 || G == 4 || G == 8) && D.d % 8 == 0;
}

int prefill_chunk_tokens(const Dims &D) {
  int c = ((D.max_seq + kGemmBM - 1) / kGemmBM) * kGemmBM;
  return c < kPrefillChunk ? c : kPrefillChunk;
}

int prefill_create(const DevPtrs &P, const uint16_t *const *const *src, PrefillPlan *plan) {
  memset(plan, 0, sizeof *plan);
  const Dims &D = P.dim;
  if (!prefill_supported(D) || !P.pf_H || D.L > kPrefillMaxLayers) return -1;
  PfEncodeFn enc = pf_encoder();
  if (!enc) return -1;
  static bool attr_done = false;
  if (!attr_done) {
    if (cudaFuncSetAttribute(k_pf_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem) != cudaSuccess ||
        cudaFuncSetAttribute(k_pf_attention<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, 120 * 1024) != cudaSuccess ||
        cudaFuncSetAttribute(k_pf_attention<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, 120 * 1024) != cudaSuccess) {
      cudaGetLastError();
      return -1;
    }
    attr_done = true;
  }
  for (int i = 0; i < 9; ++i)
    for (int l = 0; l < D.L; ++l) plan->w[i][l] = src[i][l];
  plan->available = 1;
  return 0;
}

// Runs positions [0, n_tokens) through all layers (KV rows appended, Hfin written).  Tokens are in P.pf_tokens.
// One stack of decoder layers over the prompt, chunk by chunk.  Target: rows start as embeddings, the paper PDM's anchors
// are captured on the way, Hfin is written.  PDM (fc_full != nullptr): rows start as the full-depth features
// g^n = FC_{m-1} . Concat(H^b0 .. H^b(m-1)) (Eq. 4; P.anch IS the [position, m d] fp32 matrix of those concatenations),
// the layers / cache are the PDM's (P.kv points at its cache), nothing else is written.
static int prefill_stack(const DevPtrs &P, const uint16_t *const (*w)[kPrefillMaxLayers], int n_layers, const uint16_t *fc_full,
                         int n_tokens, cudaStream_t st, long long *launches) {
  PfEncodeFn enc = pf_encoder();
  if (!enc) return -1;
  const Dims &D = P.dim;
  const int qd = D.Hq * D.hd, kd = D.Hkv * D.hd, Mc = P.pf_chunk;
  const int G = D.Hq / D.Hkv, TQ = 64 / G;
  const size_t att_smem = (size_t)(3 * 64 * (D.hd + 4) + 64 * 65 + 3 * 64) * sizeof(float);
  long long cnt = 0;
  for (int p0 = 0; p0 < n_tokens; p0 += Mc) {
    const int M = n_tokens - p0 < Mc ? n_tokens - p0 : Mc;
    const int eb = (int)(((size_t)M * D.F + 255) / 256 < 4096 ? ((size_t)M * D.F + 255) / 256 : 4096);
    if (fc_full) {
      const int K5 = P.pdm_m * D.d;
      k_pf_split<<<2048, 256, 0, st>>>(P.anch + (size_t)p0 * K5, (size_t)M * K5, P.pf_x3, P.pf_plane);
      const uint16_t *wf[1] = {fc_full};
      const int nf[1] = {D.d};
      if (pf_launch_gemm(enc, P.pf_x3, P.pf_plane, Mc, M, K5, wf, nf, 1, P.pf_H, D.d, st, &cnt)) return -1;
    } else {
      k_pf_embed<<<M, 256, 0, st>>>(P.embed, P.pf_tokens, p0, D.d, P.pf_H);
    }
    ++cnt;
    for (int l = 0; l < n_layers; ++l) {
      // spd_weights order: 0 attn_norm 1 wq 2 wk 3 wv 4 wo 5 mlp_norm 6 w_gate 7 w_up 8 w_down
      if (P.paper_pdm && !fc_full)
        for (int ai = 0; ai < P.pdm_m; ++ai)
          if (P.pdm_anchor[ai] == l) { k_pf_store_anchor<<<eb, 256, 0, st>>>(P.pf_H, P.anch, p0, D.d, M, P.pdm_m, ai); ++cnt; }
      k_pf_norm_split<<<M, 256, 0, st>>>(P.pf_H, w[0][l], D.d, D.eps, P.pf_x3, P.pf_plane);
      const uint16_t *wqkv[3] = {w[1][l], w[2][l], w[3][l]};
      const int nqkv[3] = {qd, kd, kd};
      if (pf_launch_gemm(enc, P.pf_x3, P.pf_plane, Mc, M, D.d, wqkv, nqkv, 3, P.pf_Y, qd + 2 * kd, st, &cnt)) return -1;
      k_pf_rope_append<<<M, 256, 0, st>>>(P.pf_Y, qd + 2 * kd, P, l, p0, P.pf_Q);
      dim3 ag((M + TQ - 1) / TQ, D.Hkv);
      if (kPrefillAttnMma) {
        if (D.hd == 128) k_pf_attention_mma<128><<<ag, 128, 0, st>>>(P, l, p0, M, P.pf_Q, P.pf_x3, P.pf_plane);
        else k_pf_attention_mma<64><<<ag, 128, 0, st>>>(P, l, p0, M, P.pf_Q, P.pf_x3, P.pf_plane);
      } else if (D.hd == 128) k_pf_attention<128><<<ag, 256, att_smem, st>>>(P, l, p0, M, P.pf_Q, P.pf_x3, P.pf_plane);
      else k_pf_attention<64><<<ag, 256, att_smem, st>>>(P, l, p0, M, P.pf_Q, P.pf_x3, P.pf_plane);
      const uint16_t *wo[1] = {w[4][l]};
      const int no[1] = {D.d};
      if (pf_launch_gemm(enc, P.pf_x3, P.pf_plane, Mc, M, qd, wo, no, 1, P.pf_Y, D.d, st, &cnt)) return -1;
      k_pf_residual<<<eb, 256, 0, st>>>(P.pf_H, P.pf_Y, D.d, D.d, M);
      k_pf_norm_split<<<M, 256, 0, st>>>(P.pf_H, w[5][l], D.d, D.eps, P.pf_x3, P.pf_plane);
      const uint16_t *wgu[2] = {w[6][l], w[7][l]};
      const int ngu[2] = {D.F, D.F};
      if (pf_launch_gemm(enc, P.pf_x3, P.pf_plane, Mc, M, D.d, wgu, ngu, 2, P.pf_Y, 2 * D.F, st, &cnt)) return -1;
      k_pf_silu_split<<<eb, 256, 0, st>>>(P.pf_Y, 2 * D.F, D.F, M, P.pf_x3, P.pf_plane);
      const uint16_t *wd[1] = {w[8][l]};
      if (pf_launch_gemm(enc, P.pf_x3, P.pf_plane, Mc, M, D.F, wd, no, 1, P.pf_Y, D.d, st, &cnt)) return -1;
      k_pf_residual<<<eb, 256, 0, st>>>(P.pf_H, P.pf_Y, D.d, D.d, M);
      cnt += 7;
    }
    if (!fc_full) { k_pf_store_hfin<<<eb, 256, 0, st>>>(P.pf_H, P.hfin, p0, D.d, M); ++cnt; }
  }
  if (launches) *launches += cnt;
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int prefill_run(const DevPtrs &P, const PrefillPlan &plan, int n_tokens, cudaStream_t st, long long *launches) {
  if (!plan.available) return -1;
  return prefill_stack(P, plan.w, P.dim.L, nullptr, n_tokens, st, launches);
}

// The paper PDM's full-depth rows of positions 0 .. n_tokens - 1 (its prefill): the same tensor-core GEMMs and prefill
// attention over ITS layers and ITS cache.  Needs the batched-prefill scratch (P.pf_*) sized for K = m d.
int prefill_pdm_rows(const DevPtrs &P, const uint16_t *const (*w)[kPrefillMaxLayers], int n_layers, uint16_t *pdm_kv,
                     const uint16_t *fc_full, int n_tokens, cudaStream_t st, long long *launches) {
  const Dims &D = P.dim;
  if (!prefill_supported(D) || !P.pf_H || (size_t)P.pf_chunk * P.pdm_m * D.d > P.pf_plane) return -1;
  DevPtrs Q = P;
  Q.kv = pdm_kv;
  return prefill_stack(Q, w, n_layers, fc_full, n_tokens, st, launches);
}

// spd_op_gemm: Y[M, N] = X[M, K] . W[N, K]^T with the prefill GEMM (X fp32 -> bf16 hi + mid + lo, exact).  scratch: 3 * M * K bf16.
int prefill_op_gemm(const float *x, const uint16_t *w, int M, int N, int K, float *y, void *scratch, cudaStream_t st) {
  if (K % kGemmBK || M < 1 || N < 1 || N % 4) return -1;
  PfEncodeFn enc = pf_encoder();
  if (!enc) return -1;
  if (cudaFuncSetAttribute(k_pf_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem) != cudaSuccess) return -1;
  uint16_t *x3 = (uint16_t *)scratch;
  const size_t plane = (size_t)M * K;
  k_pf_split<<<1024, 256, 0, st>>>(x, plane, x3, plane);
  const uint16_t *ws[1] = {w};
  const int ns[1] = {N};
  return pf_launch_gemm(enc, x3, plane, M, M, K, ws, ns, 1, y, N, st, nullptr);
}

}  // namespace spd
