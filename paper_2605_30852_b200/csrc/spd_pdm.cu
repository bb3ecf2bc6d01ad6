// spd_pdm.cu — the paper's Pipeline Draft Module on the device.
//
// PAPER.md:71 "an L_s-layer Transformer decoder with an independent LM head"; :91-100 Eq. 3-4: anchors B (b_0 = 0;
// [0, 8, 16, 24, 31] for L = 32), l_max(k) = min(L, k L/n), f(k) = max{i | b_i <= l_max(k)},
// g_t^k = FC_f(k)(Concat(H_t^b0 .. H_t^bf(k))); :102-107 Eq. 5 warm-up layout; :115 pre-step features; :139 reduced
// vocabulary head; :299 "caching appends only the trailing (n+1) refreshed features each step".
//
// One draft = a short kernel sequence on the cycle's stream BEFORE the cycle kernel (pre-step state, no dependency on
// the cycle's forward):  k_pdm_begin (which rows: positions F .. p_new, their depths; F := c) -> k_pdm_features (Eq. 4,
// one GEMV per row against FC_f(k)) -> per PDM layer: RMSNorm, QKV, RoPE + bf16 append into the PDM's own cache (rows are
// REwritten: in-flight features deepen every cycle), split-KV attention, O + residual, RMSNorm, gate/up + SiLU.mul,
// down + residual -> RMSNorm + head GEMV over the reduced vocabulary -> argmax -> vocab_map -> the token the controller
// of the cycle kernel enters into stage 0.  M = rows <= n + 1 vectors share every weight row that is streamed (the
// M = 2 head pass of the cycle kernel generalised); a row's result never depends on which other rows share the pass.
// The paper hides this work on a dedicated GPU; on one GPU its bytes come out of the same HBM, so it is
// reported as what it costs.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include "../../include/spd.h"
#include "spd_engine.h"
#include "spd_kernels.cuh"

namespace spd {

struct PdmRun {                       // written by k_pdm_begin, read by every other kernel of the draft
  int32_t first, rows, final_len;     // rows = positions first .. first + rows - 1; final_len = F
  int32_t depth[kPdmMaxRows];         // completed stages k of each row's token (n: committed)
  int32_t f[kPdmMaxRows];             // Eq. 3
  int32_t hbuf[kPdmMaxRows];          // in-flight rows: hidden buffer of the token (its current residual stream); else -1
};

struct PdmPtrs {
  int32_t Ls, Vs;
  PdmRun *run;
  float *G, *X, *XN, *Y, *Q, *ATT, *ACT;      // [kPdmMaxRows][d | d | d | max(qd + 2 kd, 2 F) | qd | qd | F]
  float *part_o;                      // [kPdmMaxRows][Hq][nsplit][hd]
  float2 *part_ml;
  uint16_t *x3;                       // [3][48][max(d, qd, F)] the GEMM input rows as three exact bf16 parts (skinny GEMM)
  size_t plane;                       // elements per part
  float *part;                        // split-K partial sums of the skinny GEMM
  size_t part_floats;
  int32_t use_tc;                     // 1: tcgen05 skinny GEMM, 0: CUDA-core M-row GEMV
  float2 *rope;                       // [kPdmMaxRows][64] (cos, sin) of the run's positions: computed once per draft
  float *ss_part;                     // [kPdmMaxRows][64] per-256-column partial sums of squares of a row (deferred RMSNorm)
  float *logits, *z;                  // [Vs], [d]
  float *cand_val;                    // [kPdmCand]
  int32_t *cand_idx;
  uint16_t *kv;                       // the PDM's own cache: [L_s][K|V][kv head][max_seq][hd] bf16
  const uint16_t *const *fc;          // device table of the m FC matrices (selected per row by f(k))
  const uint16_t *final_norm, *head;
  const int32_t *vocab_map;
};
constexpr int kPdmCand = 128;

// ------------------------------------------------------------------ which rows ---------------------------------
// fixed_rows > 0: PDM prefill chunk (committed positions, depth n); else the cycle's rows from the device state.
__global__ void k_pdm_begin(DevPtrs P, PdmPtrs PD, int fixed_first, int fixed_rows) {
  if (threadIdx.x != 0) return;
  const Dims &D = P.dim;
  PdmRun *R = PD.run;
  const StepState *st = P.st;
  int first, rows;
  if (fixed_rows > 0) { first = fixed_first; rows = fixed_rows; }
  else if (st->mode != MODE_SPD || !st->occ[0]) { R->rows = 0; return; }
  else { first = R->final_len; rows = st->pos[0] - first + 1; }
  if (rows < 1 || rows > kPdmMaxRows) { P.st->err = 2; R->rows = 0; return; }
  for (int r = 0; r < rows; ++r) {
    const int q = first + r;
    int k = D.n, hb = -1;
    if (fixed_rows <= 0 && q >= st->c) {          // in flight: depth = stages completed BEFORE this cycle's forward
      k = st->pos[0] - q;
      if (k < 0 || k >= D.n || !st->occ[k] || st->pos[k] != q) { P.st->err = 2; R->rows = 0; return; }
      hb = st->hbuf[k];
    }
    const int lmax = min(D.L, k * D.per);
    int f = 0;
    for (int i = 0; i < P.pdm_m; ++i)
      if (P.pdm_anchor[i] <= lmax) f = i;
    R->depth[r] = k; R->f[r] = f; R->hbuf[r] = hb;
  }
  R->first = first; R->rows = rows;
  if (fixed_rows <= 0) R->final_len = st->c;       // rows below c were built at depth n: final
}

__global__ void k_pdm_set_final(PdmPtrs PD, int final_len, int only_lower) {
  if (!only_lower || PD.run->final_len > final_len) PD.run->final_len = final_len;
}

// ------------------------------------------------------------------ Eq. 4: g = FC_f . Concat(anchors) ------------
// grid (ceil(d / 8), kPdmMaxRows); a warp per output element.  An in-flight token's deepest eligible anchor
// H^{k L/n} is the residual stream it currently holds (k = 0: the embedding row).
__global__ void k_pdm_features(DevPtrs P, PdmPtrs PD) {
  const Dims &D = P.dim;
  const PdmRun *R = PD.run;
  const int r = blockIdx.y;
  if (r >= R->rows) return;
  const int o = blockIdx.x * 8 + (threadIdx.x >> 5);
  if (o >= D.d) return;
  const int f = R->f[r], q = R->first + r, k = R->depth[r], hb = R->hbuf[r];
  const uint16_t *wrow = PD.fc[f] + (size_t)o * (f + 1) * D.d;
  float acc = 0.f;
  for (int i = 0; i <= f; ++i) {
    const float *src = (hb >= 0 && P.pdm_anchor[i] == k * D.per) ? P.h + (size_t)hb * D.d
                                                                 : P.anch + ((size_t)q * P.pdm_m + i) * D.d;
    acc += warp_dot_row(wrow + (size_t)i * D.d, src, D.d);
  }
  if ((threadIdx.x & 31) == 0) { PD.X[(size_t)r * D.d + o] = acc; PD.G[(size_t)r * D.d + o] = acc; }
}

// fp32 -> three bf16 parts, x = hi + mid + lo exactly; written to row r of the skinny GEMM's input planes (row stride K)
__device__ __forceinline__ void pdm_put3(const PdmPtrs &PD, int r, int K, int i, float x) {
  const uint16_t hi = f32_to_bf16(x);
  const float r1 = x - bf16_to_f32(hi);
  const uint16_t mid = f32_to_bf16(r1);
  const uint16_t lo = f32_to_bf16(r1 - bf16_to_f32(mid));
  const size_t o = (size_t)r * K + i;
  PD.x3[o] = hi; PD.x3[PD.plane + o] = mid; PD.x3[2 * PD.plane + o] = lo;
}

// XN[r] = RMSNorm(X[r]; gain); grid kPdmMaxRows.  last_only: only the last row (head input, final norm), into PD.z.
__global__ void k_pdm_norm(DevPtrs P, PdmPtrs PD, const uint16_t *gain, int last_only) {
  __shared__ float red[33];
  const PdmRun *R = PD.run;
  const Dims &D = P.dim;
  int r = blockIdx.x;
  if (last_only) { if (r != 0 || R->rows < 1) return; r = R->rows - 1; }
  else if (r >= R->rows) return;
  const uint16_t *g = last_only ? PD.final_norm : gain;
  float *out = last_only ? PD.z : PD.XN + (size_t)r * D.d;
  block_rmsnorm(PD.X + (size_t)r * D.d, g, D.d, D.eps, out, red);
  if (PD.use_tc) {
    __syncthreads();
    for (int i = threadIdx.x; i < D.d; i += blockDim.x) pdm_put3(PD, last_only ? 0 : r, D.d, i, out[i]);
  }
}

// ------------------------------------------------------------------ M-row GEMV ----------------------------------
// Y[r][col0_s + n] (+)= W_s[n] . X[r] for every row r of the run and up to three weight matrices (segments) that share X.
// The x rows live in REGISTERS: thread t of a CTA owns the 8-element chunks t and t + 256 of a 4096-column K pass for up
// to 8 x rows; the CTA then streams its `wr` weight rows once per pass — a weight row's 4096-column slice is one 8 KB
// coalesced read by the 256 threads, multiplied into every x row while in registers (the M = 2 head pass of the cycle
// kernel generalised) — so the x traffic from L2 is M / (2 wr) of the weight traffic and nothing in the main loop waits on
// shared memory.  Per (weight row, x row): one fp32 FMA chain per thread over its chunks, the warp xor tree, the warp
// partials of all passes added in (pass, warp) order by one thread: a value depends only on (weight row, x row), never
// on which other rows share the pass.
constexpr int kRgRows = 8;               // x rows per pass over the weights
constexpr int kRgMaxWr = 32;             // weight rows per CTA
struct RowsGemv {
  const uint16_t *w[3];
  int n[3], col0[3];
  int nseg, K, ldx, ldy, residual, last_only, wr;
  const float *x;
  float *y;
};

__global__ void __launch_bounds__(256, 1) k_pdm_rows_gemv(PdmPtrs PD, RowsGemv A) {
  __shared__ float part[8][kRgMaxWr][kRgRows];        // [warp][weight row][x row]
  const PdmRun *R = PD.run;
  int rows = R->rows;
  if (rows < 1) return;
  if (A.last_only) rows = 1;                          // x and y are single vectors (the head: x = PD.z)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, wr = A.wr;
  int n0 = blockIdx.x * wr, seg = 0;                  // first of this CTA's weight rows
  while (seg < A.nseg) {
    const int padded = (A.n[seg] + wr - 1) / wr * wr;
    if (n0 < padded) break;
    n0 -= padded; ++seg;
  }
  if (seg >= A.nseg) return;
  const int nrow = A.n[seg], nw = min(wr, nrow - n0), nchunk = A.K >> 3;
  const uint4 *wbase = reinterpret_cast<const uint4 *>(A.w[seg] + (size_t)n0 * A.K);
  for (int rb = 0; rb < rows; rb += kRgRows) {
    const int nr = min(kRgRows, rows - rb);
    for (int i = tid; i < 8 * kRgMaxWr * kRgRows; i += 256) (&part[0][0][0])[i] = 0.f;
    __syncthreads();
    for (int k0 = 0; k0 < nchunk; k0 += 512) {        // K passes of 512 chunks
      float4 xr[kRgRows][4];                          // [x row][chunk 0: a, b; chunk 1: a, b]
      const int c0 = k0 + tid, c1 = k0 + 256 + tid;
      const bool v0 = c0 < nchunk, v1 = c1 < nchunk;
#pragma unroll
      for (int r = 0; r < kRgRows; ++r) {
        const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
        xr[r][0] = xr[r][1] = xr[r][2] = xr[r][3] = z;
        if (r < nr) {
          const float4 *xp = reinterpret_cast<const float4 *>(A.x + (size_t)(rb + r) * A.ldx);
          if (v0) { xr[r][0] = xp[2 * c0]; xr[r][1] = xp[2 * c0 + 1]; }
          if (v1) { xr[r][2] = xp[2 * c1]; xr[r][3] = xp[2 * c1 + 1]; }
        }
      }
#pragma unroll 4
      for (int j = 0; j < nw; ++j) {
        const uint4 *wp = wbase + (size_t)j * nchunk;
        const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
        const uint4 w0 = v0 ? __ldg(wp + c0) : z4, w1 = v1 ? __ldg(wp + c1) : z4;
        float acc[kRgRows];
#pragma unroll
        for (int r = 0; r < kRgRows; ++r) {
          float a = 0.f;
          if (r < nr) {
            a = fmaf(bf16_lo(w0.x), xr[r][0].x, a); a = fmaf(bf16_hi(w0.x), xr[r][0].y, a);
            a = fmaf(bf16_lo(w0.y), xr[r][0].z, a); a = fmaf(bf16_hi(w0.y), xr[r][0].w, a);
            a = fmaf(bf16_lo(w0.z), xr[r][1].x, a); a = fmaf(bf16_hi(w0.z), xr[r][1].y, a);
            a = fmaf(bf16_lo(w0.w), xr[r][1].z, a); a = fmaf(bf16_hi(w0.w), xr[r][1].w, a);
            a = fmaf(bf16_lo(w1.x), xr[r][2].x, a); a = fmaf(bf16_hi(w1.x), xr[r][2].y, a);
            a = fmaf(bf16_lo(w1.y), xr[r][2].z, a); a = fmaf(bf16_hi(w1.y), xr[r][2].w, a);
            a = fmaf(bf16_lo(w1.z), xr[r][3].x, a); a = fmaf(bf16_hi(w1.z), xr[r][3].y, a);
            a = fmaf(bf16_lo(w1.w), xr[r][3].z, a); a = fmaf(bf16_hi(w1.w), xr[r][3].w, a);
          }
          acc[r] = a;
        }
#pragma unroll
        for (int r = 0; r < kRgRows; ++r) {
          if (r < nr) {
            const float v = warp_sum(acc[r]);
            if (lane == 0) part[warp][j][r] += v;     // this lane's own slot: passes accumulate in order
          }
        }
      }
    }
    __syncthreads();
    for (int i = tid; i < nw * nr; i += 256) {
      const int j = i / nr, r = i - j * nr;
      float v = 0.f;
#pragma unroll
      for (int w = 0; w < 8; ++w) v += part[w][j][r];
      float *dst = A.y + (size_t)(rb + r) * A.ldy + A.col0[seg] + n0 + j;
      *dst = A.residual ? *dst + v : v;
    }
    __syncthreads();
  }
}

// (cos, sin)(pos * theta_i) of the run's rows, angles in double (C-2.14): once per draft, shared by the L_s layers.
__global__ void k_pdm_rope_table(DevPtrs P, PdmPtrs PD) {
  const PdmRun *R = PD.run;
  const int r = blockIdx.x;
  if (r >= R->rows || (int)threadIdx.x >= P.dim.hd / 2) return;
  double s_, c_;
  sincos((double)(R->first + r) * P.inv_freq[threadIdx.x], &s_, &c_);
  PD.rope[r * 64 + threadIdx.x] = make_float2((float)c_, (float)s_);
}

// Y row = [q | k | v]: RoPE (C-2.14) on q and k; q -> Q; k, v -> bf16 rows of the PDM cache at the row's position
// (REwritten every cycle for in-flight positions).  grid kPdmMaxRows.
__global__ void k_pdm_rope_append(DevPtrs P, PdmPtrs PD, int layer) {
  const Dims &D = P.dim;
  const PdmRun *R = PD.run;
  __shared__ float2 cs[64];
  const int r = blockIdx.x;
  if (r >= R->rows) return;
  const int pos = R->first + r, half = D.hd / 2, qd = D.Hq * D.hd, kd = D.Hkv * D.hd, ldy = qd + 2 * kd;
  if (threadIdx.x < half) cs[threadIdx.x] = PD.rope[r * 64 + threadIdx.x];
  __syncthreads();
  const float *y = PD.Y + (size_t)r * ldy;
  for (int j = threadIdx.x; j < (D.Hq + D.Hkv) * half; j += blockDim.x) {
    const int hh = j / half, i = j - hh * half;
    const float2 c = cs[i];
    if (hh < D.Hq) {
      const float a = y[hh * D.hd + i], b = y[hh * D.hd + i + half];
      float *q = PD.Q + (size_t)r * qd + hh * D.hd;
      q[i] = a * c.x - b * c.y;
      q[i + half] = b * c.x + a * c.y;
    } else {
      const int kh = hh - D.Hq;
      const float a = y[qd + kh * D.hd + i], b = y[qd + kh * D.hd + i + half];
      uint16_t *dst = PD.kv + kv_offset(D, layer, 0, kh) + (size_t)pos * D.hd;
      dst[i] = f32_to_bf16(a * c.x - b * c.y);
      dst[i + half] = f32_to_bf16(b * c.x + a * c.y);
    }
  }
  for (int j = threadIdx.x; j < kd; j += blockDim.x) {
    const int kh = j / D.hd, i = j - kh * D.hd;
    PD.kv[kv_offset(D, layer, 1, kh) + (size_t)pos * D.hd + i] = f32_to_bf16(y[qd + kd + j]);
  }
}

// Split-KV attention of every row over the PDM cache rows 0 .. pos (fixed 128-row splits merged in split order, as the
// target's): grid (split, kv head, kPdmMaxRows), one warp per q head of the group.  Written for memory-level
// parallelism (a draft has few rows, so a warp must keep many loads in flight) with coalesced rows: scores — HD/8 lanes
// share a K row (one 16-byte chunk each, q chunk in registers), 32/(HD/8) rows per load instruction, 8 instructions in
// flight, a 4- or 3-step xor tree per row; softmax over the split with the scores parked in shared memory; P.V with 8 V
// rows in flight (lane = HD/32 head-dim elements).  Fixed order per (row, head, split): batch-invariant.
template <int HD>
__global__ void k_pdm_attn_partial(DevPtrs P, PdmPtrs PD, int layer) {
  constexpr int EPL = HD / 32, LPR = HD / 8, RPI = 32 / LPR, U = 8;
  __shared__ float ps[8][kAttnSplit];
  const Dims &D = P.dim;
  const PdmRun *R = PD.run;
  const int r = blockIdx.z;
  if (r >= R->rows) return;
  const int T = R->first + r + 1, split = blockIdx.x, t0 = split * kAttnSplit;
  if (t0 >= T) return;
  const int t1 = min(T, t0 + kAttnSplit), kvh = blockIdx.y, group = D.Hq / D.Hkv;
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int hq = kvh * group + w;
  const uint16_t *kc = PD.kv + kv_offset(D, layer, 0, kvh), *vc = PD.kv + kv_offset(D, layer, 1, kvh);
  const int sub = lane / LPR, hl = lane % LPR;            // which row of an instruction's RPI rows, which chunk of it
  const float4 qa = *reinterpret_cast<const float4 *>(PD.Q + ((size_t)r * D.Hq + hq) * HD + 8 * hl);
  const float4 qb = *reinterpret_cast<const float4 *>(PD.Q + ((size_t)r * D.Hq + hq) * HD + 8 * hl + 4);
  const float scale = 1.0f / sqrtf((float)HD);
  const int nrows = t1 - t0;
  for (int i0 = 0; i0 < kAttnSplit; i0 += RPI * U) {
    uint4 kw[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int i = i0 + RPI * u + sub;
      kw[u] = make_uint4(0u, 0u, 0u, 0u);
      if (i < nrows) kw[u] = __ldg(reinterpret_cast<const uint4 *>(kc + (size_t)(t0 + i) * HD) + hl);
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      float a = bf16_lo(kw[u].x) * qa.x;
      a = fmaf(bf16_hi(kw[u].x), qa.y, a); a = fmaf(bf16_lo(kw[u].y), qa.z, a); a = fmaf(bf16_hi(kw[u].y), qa.w, a);
      a = fmaf(bf16_lo(kw[u].z), qb.x, a); a = fmaf(bf16_hi(kw[u].z), qb.y, a);
      a = fmaf(bf16_lo(kw[u].w), qb.z, a); a = fmaf(bf16_hi(kw[u].w), qb.w, a);
#pragma unroll
      for (int o = LPR / 2; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
      const int i = i0 + RPI * u + sub;
      if (hl == 0) ps[w][i] = i < nrows ? a * scale : -INFINITY;
    }
  }
  __syncwarp();
  float sc[kAttnSplit / 32], m = -INFINITY;
#pragma unroll
  for (int j = 0; j < kAttnSplit / 32; ++j) { sc[j] = ps[w][lane + 32 * j]; m = fmaxf(m, sc[j]); }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  __syncwarp();
  float l = 0.f;
#pragma unroll
  for (int j = 0; j < kAttnSplit / 32; ++j) {
    const float pr = sc[j] == -INFINITY ? 0.f : expf(sc[j] - m);
    ps[w][lane + 32 * j] = pr;
    l += pr;
  }
  l = warp_sum(l);
  __syncwarp();
  float acc[EPL];
#pragma unroll
  for (int e = 0; e < EPL; ++e) acc[e] = 0.f;
#pragma unroll 8
  for (int i = 0; i < nrows; ++i) {
    const uint16_t *vr = vc + (size_t)(t0 + i) * HD + lane * EPL;
    const float pr = ps[w][i];
    if constexpr (EPL == 4) {
      const uint2 vw = __ldg(reinterpret_cast<const uint2 *>(vr));
      acc[0] = fmaf(pr, bf16_lo(vw.x), acc[0]); acc[1] = fmaf(pr, bf16_hi(vw.x), acc[1]);
      acc[2] = fmaf(pr, bf16_lo(vw.y), acc[2]); acc[3] = fmaf(pr, bf16_hi(vw.y), acc[3]);
    } else {
      const uint32_t vw = __ldg(reinterpret_cast<const uint32_t *>(vr));
      acc[0] = fmaf(pr, bf16_lo(vw), acc[0]); acc[1] = fmaf(pr, bf16_hi(vw), acc[1]);
    }
  }
  const size_t slot = ((size_t)r * D.Hq + hq) * P.nsplit_max + split;
#pragma unroll
  for (int e = 0; e < EPL; ++e) PD.part_o[slot * HD + lane * EPL + e] = acc[e];
  if (lane == 0) PD.part_ml[slot] = make_float2(m, l);
}

// grid (q head, kPdmMaxRows); block = hd threads
__global__ void k_pdm_attn_merge(DevPtrs P, PdmPtrs PD) {
  const Dims &D = P.dim;
  const PdmRun *R = PD.run;
  const int r = blockIdx.y, hq = blockIdx.x;
  if (r >= R->rows) return;
  const int nsplit = (R->first + r + kAttnSplit) / kAttnSplit;
  const size_t slot = ((size_t)r * D.Hq + hq) * P.nsplit_max;
  const float v = attn_merge_elem(PD.part_o + slot * D.hd, PD.part_ml + slot, nsplit, D.hd, threadIdx.x);
  PD.ATT[((size_t)r * D.Hq + hq) * D.hd + threadIdx.x] = v;
  if (PD.use_tc) pdm_put3(PD, r, D.Hq * D.hd, hq * D.hd + threadIdx.x, v);
}

// ACT[r] = silu(gate) * up; Y row = [gate (F) | up (F)]
__global__ void k_pdm_silu(DevPtrs P, PdmPtrs PD) {
  const Dims &D = P.dim;
  const int r = blockIdx.y;
  if (r >= PD.run->rows) return;
  const float *y = PD.Y + (size_t)r * 2 * D.F;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < D.F; i += gridDim.x * blockDim.x) {
    const float v = silu_mul(y[i], y[D.F + i]);
    PD.ACT[(size_t)r * D.F + i] = v;
    if (PD.use_tc) pdm_put3(PD, r, D.F, i, v);
  }
}

// argmax (max value, lowest index) of the reduced-vocabulary logits -> the drafted TARGET token id.
__global__ void k_pdm_argmax_cand(PdmPtrs PD) {
  __shared__ float sv[32];
  __shared__ int si[32];
  if (PD.run->rows < 1) return;
  const int V = PD.Vs, chunk = (V + gridDim.x - 1) / gridDim.x;
  const int lo = blockIdx.x * chunk, hi = min(V, lo + chunk);
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  for (int i = lo + threadIdx.x; i < hi; i += blockDim.x) {
    const float v = PD.logits[i];
    if (cand_better(v, i, bv, bi)) { bv = v; bi = i; }
  }
  for (int o = 16; o > 0; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (cand_better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
  }
  if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = bv; si[threadIdx.x >> 5] = bi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w)
      if (cand_better(sv[w], si[w], bv, bi)) { bv = sv[w]; bi = si[w]; }
    PD.cand_val[blockIdx.x] = bv;
    PD.cand_idx[blockIdx.x] = lo < hi ? bi : -1;
  }
}
__global__ void k_pdm_argmax_final(DevPtrs P, PdmPtrs PD) {
  if (threadIdx.x != 0 || PD.run->rows < 1) return;
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  for (int i = 0; i < kPdmCand; ++i)
    if (PD.cand_idx[i] >= 0 && cand_better(PD.cand_val[i], PD.cand_idx[i], bv, bi)) { bv = PD.cand_val[i]; bi = PD.cand_idx[i]; }
  *P.pdm_draft = PD.vocab_map[bi];
}

// ------------------------------------------------------------------ fused epilogues of the skinny GEMM -----------
// The skinny GEMM leaves split-K partial sums part[ks][row][column].  RMSNorm is DEFERRED so that no kernel has to see a
// whole row before the product: y = W . (x * rs * g) = rs * (W . (x * g)) with the scalar rs = rsqrt(mean(x^2) + eps).
// The kernel that PRODUCES a residual row writes the three bf16 parts of x * g_next and the row's sum of squares as
// per-256-column partials (fixed block tree); the kernel that CONSUMES the next product adds those partials in order
// and multiplies by rs.  One draft layer is then 10 launches instead of 17.
__device__ __forceinline__ float pdm_row_rs(const PdmPtrs &PD, const Dims &D, int r) {
  float ss = 0.f;
  const int nb = (D.d + 255) / 256;
  for (int b = 0; b < nb; ++b) ss += PD.ss_part[r * 64 + b];
  return 1.0f / sqrtf(ss / (float)D.d + D.eps);
}
// block-wide sum of `v` over 256 threads in a fixed order -> ss_part[r][blockIdx.x] (thread 0)
__device__ __forceinline__ void pdm_block_sumsq(const PdmPtrs &PD, int r, float v) {
  __shared__ float red[8];
  v = warp_sum(v);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    float t = 0.f;
    for (int w = 0; w < 8; ++w) t += red[w];
    PD.ss_part[r * 64 + blockIdx.x] = t;
  }
}
// (a) after the features: x3 = parts(X * g), sum-of-squares partials.  grid (ceil(d / 256), kPdmMaxRows), 256 threads
__global__ void __launch_bounds__(256) k_pdm_prep(DevPtrs P, PdmPtrs PD, const uint16_t *gain) {
  const Dims &D = P.dim;
  const int r = blockIdx.y, c = blockIdx.x * 256 + threadIdx.x;
  if (r >= PD.run->rows) return;
  float x = 0.f;
  if (c < D.d) {
    x = PD.X[(size_t)r * D.d + c];
    pdm_put3(PD, r, D.d, c, x * bf16_to_f32(gain[c]));
  }
  pdm_block_sumsq(PD, r, x * x);
}
// (b) O / DOWN: X[r] += sum of the partials; x3 = parts(X * g_next); sum-of-squares partials.  same grid
__global__ void __launch_bounds__(256) k_pdm_reduce_res(DevPtrs P, PdmPtrs PD, int ksplit, int NB, const uint16_t *gain_next) {
  const Dims &D = P.dim;
  const int r = blockIdx.y, c = blockIdx.x * 256 + threadIdx.x;
  if (r >= PD.run->rows) return;
  float x = 0.f;
  if (c < D.d) {
    float v = 0.f;
    for (int ks = 0; ks < ksplit; ++ks) v += PD.part[((size_t)ks * NB + r) * D.d + c];
    x = PD.X[(size_t)r * D.d + c] + v;
    PD.X[(size_t)r * D.d + c] = x;
    pdm_put3(PD, r, D.d, c, x * bf16_to_f32(gain_next[c]));
  }
  pdm_block_sumsq(PD, r, x * x);
}
// (c) gate / up: ACT[r] = silu(rs * sum_gate) * (rs * sum_up) and its parts.  grid (ceil(F / 256), kPdmMaxRows)
__global__ void k_pdm_reduce_silu(DevPtrs P, PdmPtrs PD, int ksplit, int NB) {
  const Dims &D = P.dim;
  const int r = blockIdx.y, c = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= PD.run->rows || c >= D.F) return;
  const float rs = pdm_row_rs(PD, D, r);
  float g = 0.f, u = 0.f;
  for (int ks = 0; ks < ksplit; ++ks) {
    const float *p = PD.part + ((size_t)ks * NB + r) * 2 * D.F;
    g += p[c]; u += p[D.F + c];
  }
  const float v = silu_mul(g * rs, u * rs);
  PD.ACT[(size_t)r * D.F + c] = v;
  pdm_put3(PD, r, D.F, c, v);
}
// (d) QKV: y = rs * sum; RoPE (C-2.14) on q and k; q -> Q; k, v -> bf16 rows of the PDM cache.  grid kPdmMaxRows
__global__ void k_pdm_rope_append_red(DevPtrs P, PdmPtrs PD, int layer, int ksplit, int NB) {
  const Dims &D = P.dim;
  const PdmRun *R = PD.run;
  __shared__ float2 cs[64];
  const int r = blockIdx.x;
  if (r >= R->rows) return;
  const int pos = R->first + r, half = D.hd / 2, qd = D.Hq * D.hd, kd = D.Hkv * D.hd, ldy = qd + 2 * kd;
  if (threadIdx.x < half) cs[threadIdx.x] = PD.rope[r * 64 + threadIdx.x];
  __syncthreads();
  const float rs = pdm_row_rs(PD, D, r);
  auto y = [&](int col) {
    float v = 0.f;
    for (int ks = 0; ks < ksplit; ++ks) v += PD.part[((size_t)ks * NB + r) * ldy + col];
    return v * rs;
  };
  for (int j = threadIdx.x; j < (D.Hq + D.Hkv) * half; j += blockDim.x) {
    const int hh = j / half, i = j - hh * half;
    const float2 c = cs[i];
    if (hh < D.Hq) {
      const float a = y(hh * D.hd + i), b = y(hh * D.hd + i + half);
      float *q = PD.Q + (size_t)r * qd + hh * D.hd;
      q[i] = a * c.x - b * c.y;
      q[i + half] = b * c.x + a * c.y;
    } else {
      const int kh = hh - D.Hq;
      const float a = y(qd + kh * D.hd + i), b = y(qd + kh * D.hd + i + half);
      uint16_t *dst = PD.kv + kv_offset(D, layer, 0, kh) + (size_t)pos * D.hd;
      dst[i] = f32_to_bf16(a * c.x - b * c.y);
      dst[i + half] = f32_to_bf16(b * c.x + a * c.y);
    }
  }
  for (int j = threadIdx.x; j < kd; j += blockDim.x) {
    const int kh = j / D.hd, i = j - kh * D.hd;
    PD.kv[kv_offset(D, layer, 1, kh) + (size_t)pos * D.hd + i] = f32_to_bf16(y(qd + kd + j));
  }
}
// (e) the head: logits = rs * sum for the run's LAST row
__global__ void k_pdm_reduce_logits(DevPtrs P, PdmPtrs PD, int ksplit, int NB) {
  const int rows = PD.run->rows, c = blockIdx.x * blockDim.x + threadIdx.x;
  if (rows < 1 || c >= PD.Vs) return;
  const int r = rows - 1;
  const float rs = pdm_row_rs(PD, P.dim, r);
  float v = 0.f;
  for (int ks = 0; ks < ksplit; ++ks) v += PD.part[((size_t)ks * NB + r) * PD.Vs + c];
  PD.logits[c] = v * rs;
}

// ------------------------------------------------------------------ host side ----------------------------------
struct PdmPlan {
  PdmPtrs PD;
  int Ls, Vs;
  const uint16_t *fc_full;                   // FC_{m-1}: the full-depth rule (k = n)
  int NB;                                    // activation rows per skinny-GEMM tile: n + 1 rounded up to 16
  const uint16_t *w[9][kPrefillMaxLayers];   // host copy of the per-layer device pointers
};

static size_t pdm_carve(const Dims &D, int Ls, int Vs, int m, int nsplit, void *base, PdmPtrs *PD, float **anch,
                        int32_t **draft) {
  char *b = (char *)base;
  size_t off = 0;
  auto take = [&](size_t bytes) { off = (off + 255) & ~(size_t)255; void *p = b ? b + off : nullptr; off += bytes; return p; };
  const size_t R = kPdmMaxRows, qd = (size_t)D.Hq * D.hd, kd = (size_t)D.Hkv * D.hd;
  const size_t ymax = qd + 2 * kd > 2 * (size_t)D.F ? qd + 2 * kd : 2 * (size_t)D.F;
  PdmPtrs Q;
  memset(&Q, 0, sizeof Q);
  Q.Ls = Ls; Q.Vs = Vs;
  Q.run = (PdmRun *)take(sizeof(PdmRun));
  Q.G = (float *)take(R * D.d * 4); Q.X = (float *)take(R * D.d * 4); Q.XN = (float *)take(R * D.d * 4);
  Q.Y = (float *)take(R * ymax * 4); Q.Q = (float *)take(R * qd * 4); Q.ATT = (float *)take(R * qd * 4);
  Q.ACT = (float *)take(R * D.F * 4);
  Q.part_o = (float *)take(R * D.Hq * nsplit * D.hd * 4);
  Q.part_ml = (float2 *)take(R * D.Hq * nsplit * 8);
  const size_t xmax = (size_t)D.d > qd ? ((size_t)D.d > (size_t)D.F ? D.d : D.F) : (qd > (size_t)D.F ? qd : D.F);
  const size_t nmax = ymax > (size_t)Vs ? ymax : (size_t)Vs;
  Q.plane = 48 * xmax;
  Q.x3 = (uint16_t *)take(3 * Q.plane * 2);
  Q.part_floats = 16 * 48 * nmax;                     // ksplit <= 16, NB <= 48
  Q.part = (float *)take(Q.part_floats * 4);
  Q.rope = (float2 *)take(R * 64 * 8);
  Q.ss_part = (float *)take(R * 64 * 4);
  Q.logits = (float *)take((size_t)Vs * 4); Q.z = (float *)take((size_t)D.d * 4);
  Q.cand_val = (float *)take(kPdmCand * 4); Q.cand_idx = (int32_t *)take(kPdmCand * 4);
  Q.fc = (const uint16_t *const *)take(8 * sizeof(void *));
  int32_t *dr = (int32_t *)take(64);
  float *an = (float *)take((size_t)D.max_seq * m * D.d * 4);
  if (PD) *PD = Q;
  if (anch) *anch = an;
  if (draft) *draft = dr;
  return (off + 255) & ~(size_t)255;
}

int pdm_anchor_set(int L, int32_t *b) {
  int cand[5] = {0, L / 4, L / 2, (3 * L) / 4, L - 1}, m = 0;
  for (int i = 0; i < 5; ++i)
    if (m == 0 || cand[i] > b[m - 1]) b[m++] = cand[i];
  return m;
}

size_t pdm_kv_bytes(const Dims &D, int Ls) { return (size_t)Ls * 2 * D.Hkv * D.max_seq * D.hd * sizeof(uint16_t); }
size_t pdm_work_bytes(const Dims &D, int Ls, int Vs) {
  int32_t b[8];
  const int m = pdm_anchor_set(D.L, b);
  return pdm_carve(D, Ls, Vs, m, (D.max_seq + kAttnSplit - 1) / kAttnSplit, nullptr, nullptr, nullptr, nullptr);
}

PdmPlan *pdm_create(DevPtrs *P, const spd_pdm_weights *w, void *kv, void *work, cudaStream_t st) {
  const Dims &D = P->dim;
  if (w->n_layers < 1 || w->n_layers > kPrefillMaxLayers || w->vocab < 1 || w->vocab > D.V) return nullptr;
  PdmPlan *plan = (PdmPlan *)calloc(1, sizeof(PdmPlan));
  if (!plan) return nullptr;
  int32_t b[8];
  const int m = pdm_anchor_set(D.L, b);
  float *anch;
  int32_t *draft;
  const size_t bytes = pdm_carve(D, w->n_layers, w->vocab, m, P->nsplit_max, work, &plan->PD, &anch, &draft);
  plan->Ls = w->n_layers; plan->Vs = w->vocab;
  plan->NB = (D.n + 1 + 15) / 16 * 16;
  plan->PD.use_tc = prefill_supported(D) && plan->NB <= 48 ? 1 : 0;
  plan->PD.kv = (uint16_t *)kv;
  plan->PD.final_norm = w->final_norm; plan->PD.head = w->head; plan->PD.vocab_map = w->vocab_map;
  const uint16_t *const *src[9] = {w->attn_norm, w->wq, w->wk, w->wv, w->wo, w->mlp_norm, w->w_gate, w->w_up, w->w_down};
  for (int i = 0; i < 9; ++i)
    for (int l = 0; l < w->n_layers; ++l) {
      if (!src[i][l]) { free(plan); return nullptr; }
      plan->w[i][l] = src[i][l];
    }
  for (int i = 0; i < m; ++i)
    if (!w->fc[i]) { free(plan); return nullptr; }
  plan->fc_full = w->fc[m - 1];
  if (cudaMemsetAsync(work, 0, bytes - (size_t)D.max_seq * m * D.d * 4, st) != cudaSuccess ||
      cudaMemcpyAsync((void *)plan->PD.fc, w->fc, sizeof(void *) * m, cudaMemcpyHostToDevice, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess) {
    free(plan);
    return nullptr;
  }
  P->paper_pdm = 1; P->pdm_m = m;
  for (int i = 0; i < m; ++i) P->pdm_anchor[i] = b[i];
  P->anch = anch; P->pdm_draft = draft;
  return plan;
}

void pdm_destroy(PdmPlan *plan) { free(plan); }

static int pdm_launch_gemv(const PdmPlan *pl, const uint16_t *const *w, const int *n, int nseg, int K, const float *x, int ldx,
                           float *y, int ldy, int residual, int last_only, cudaStream_t st) {
  RowsGemv A;
  memset(&A, 0, sizeof A);
  int total = 0, col = 0, nmax = 0;
  for (int s = 0; s < nseg; ++s) nmax = n[s] > nmax ? n[s] : nmax;
  const int wr = nmax >= 8192 ? 32 : 16;              // weight rows per CTA: >= 256 CTAs for the narrow matrices
  for (int s = 0; s < nseg; ++s) {
    A.w[s] = w[s]; A.n[s] = n[s]; A.col0[s] = col;
    col += n[s];
    total += (n[s] + wr - 1) / wr;
  }
  A.wr = wr;
  A.nseg = nseg; A.K = K; A.ldx = ldx; A.ldy = ldy; A.residual = residual; A.last_only = last_only; A.x = x; A.y = y;
  k_pdm_rows_gemv<<<total, 256, 0, st>>>(pl->PD, A);
  return 0;
}

// The kernels of one draft after k_pdm_begin (shared by the cycle and the PDM prefill): tensor-core products with the
// fused epilogues above.
static void pdm_enqueue_body_tc(const DevPtrs &P, const PdmPlan *pl, bool head, cudaStream_t st, long long *cnt) {
  const Dims &D = P.dim;
  const PdmPtrs &PD = pl->PD;
  const int R = kPdmMaxRows, qd = D.Hq * D.hd, kd = D.Hkv * D.hd, group = D.Hq / D.Hkv, NB = pl->NB;
  const dim3 gd((D.d + 255) / 256, R);
  int ks = 1;
  auto gemm = [&](const uint16_t *const *w, const int *n, int nseg, int K) {
    skinny_gemm(PD.x3, PD.plane, K, NB, w, n, nseg, PD.part, PD.part_floats, nullptr, 0, nullptr, 0, 0, st, cnt, &ks);
  };
  k_pdm_rope_table<<<R, 64, 0, st>>>(P, PD); ++*cnt;
  k_pdm_features<<<dim3((D.d + 7) / 8, R), 256, 0, st>>>(P, PD); ++*cnt;
  k_pdm_prep<<<gd, 256, 0, st>>>(P, PD, pl->w[0][0]); ++*cnt;                // the first layer's attention norm (deferred)
  const int nd[1] = {D.d};
  for (int l = 0; l < pl->Ls; ++l) {
    const uint16_t *wqkv[3] = {pl->w[1][l], pl->w[2][l], pl->w[3][l]};
    const int nqkv[3] = {qd, kd, kd};
    gemm(wqkv, nqkv, 3, D.d);
    k_pdm_rope_append_red<<<R, 256, 0, st>>>(P, PD, l, ks, NB); ++*cnt;
    dim3 ga(P.nsplit_max, D.Hkv, R);
    if (D.hd == 128) k_pdm_attn_partial<128><<<ga, group * 32, 0, st>>>(P, PD, l);
    else k_pdm_attn_partial<64><<<ga, group * 32, 0, st>>>(P, PD, l);
    ++*cnt;
    k_pdm_attn_merge<<<dim3(D.Hq, R), D.hd, 0, st>>>(P, PD); ++*cnt;
    const uint16_t *wo[1] = {pl->w[4][l]};
    gemm(wo, nd, 1, qd);
    k_pdm_reduce_res<<<gd, 256, 0, st>>>(P, PD, ks, NB, pl->w[5][l]); ++*cnt;
    const uint16_t *wgu[2] = {pl->w[6][l], pl->w[7][l]};
    const int ngu[2] = {D.F, D.F};
    gemm(wgu, ngu, 2, D.d);
    k_pdm_reduce_silu<<<dim3((D.F + 255) / 256, R), 256, 0, st>>>(P, PD, ks, NB); ++*cnt;
    const uint16_t *wd[1] = {pl->w[8][l]};
    gemm(wd, nd, 1, D.F);
    // ... + residual, and the NEXT product's norm (deferred): the next layer's attention norm, or the final norm before the head
    k_pdm_reduce_res<<<gd, 256, 0, st>>>(P, PD, ks, NB, l + 1 < pl->Ls ? pl->w[0][l + 1] : PD.final_norm); ++*cnt;
  }
  if (head) {
    const uint16_t *wh[1] = {PD.head};
    const int nv[1] = {pl->Vs};
    gemm(wh, nv, 1, D.d);
    k_pdm_reduce_logits<<<(pl->Vs + 255) / 256, 256, 0, st>>>(P, PD, ks, NB); ++*cnt;
    k_pdm_argmax_cand<<<kPdmCand, 256, 0, st>>>(PD); ++*cnt;
    k_pdm_argmax_final<<<1, 32, 0, st>>>(P, PD); ++*cnt;
  }
}

static void pdm_enqueue_body(const DevPtrs &P, const PdmPlan *pl, bool head, cudaStream_t st, long long *cnt) {
  if (pl->PD.use_tc) { pdm_enqueue_body_tc(P, pl, head, st, cnt); return; }
  // CUDA-core fallback (shapes the tensor path does not take): one kernel per operation, M-row GEMV
  const Dims &D = P.dim;
  const PdmPtrs &PD = pl->PD;
  const int R = kPdmMaxRows, qd = D.Hq * D.hd, kd = D.Hkv * D.hd, group = D.Hq / D.Hkv;
  k_pdm_rope_table<<<R, 64, 0, st>>>(P, PD); ++*cnt;
  k_pdm_features<<<dim3((D.d + 7) / 8, R), 256, 0, st>>>(P, PD); ++*cnt;
  for (int l = 0; l < pl->Ls; ++l) {
    k_pdm_norm<<<R, 1024, 0, st>>>(P, PD, pl->w[0][l], 0); ++*cnt;
    const uint16_t *wqkv[3] = {pl->w[1][l], pl->w[2][l], pl->w[3][l]};
    const int nqkv[3] = {qd, kd, kd};
    pdm_launch_gemv(pl, wqkv, nqkv, 3, D.d, PD.XN, D.d, PD.Y, qd + 2 * kd, 0, 0, st); ++*cnt;
    k_pdm_rope_append<<<R, 256, 0, st>>>(P, PD, l); ++*cnt;
    dim3 ga(P.nsplit_max, D.Hkv, R);
    if (D.hd == 128) k_pdm_attn_partial<128><<<ga, group * 32, 0, st>>>(P, PD, l);
    else k_pdm_attn_partial<64><<<ga, group * 32, 0, st>>>(P, PD, l);
    ++*cnt;
    k_pdm_attn_merge<<<dim3(D.Hq, R), D.hd, 0, st>>>(P, PD); ++*cnt;
    const uint16_t *wo[1] = {pl->w[4][l]};
    const int nd[1] = {D.d};
    pdm_launch_gemv(pl, wo, nd, 1, qd, PD.ATT, qd, PD.X, D.d, 1, 0, st); ++*cnt;
    k_pdm_norm<<<R, 1024, 0, st>>>(P, PD, pl->w[5][l], 0); ++*cnt;
    const uint16_t *wgu[2] = {pl->w[6][l], pl->w[7][l]};
    const int ngu[2] = {D.F, D.F};
    pdm_launch_gemv(pl, wgu, ngu, 2, D.d, PD.XN, D.d, PD.Y, 2 * D.F, 0, 0, st); ++*cnt;
    k_pdm_silu<<<dim3((D.F + 255) / 256, R), 256, 0, st>>>(P, PD); ++*cnt;
    const uint16_t *wd[1] = {pl->w[8][l]};
    pdm_launch_gemv(pl, wd, nd, 1, D.F, PD.ACT, D.F, PD.X, D.d, 1, 0, st); ++*cnt;
  }
  if (head) {
    k_pdm_norm<<<1, 256, 0, st>>>(P, PD, nullptr, 1); ++*cnt;
    const uint16_t *wh[1] = {PD.head};
    const int nv[1] = {pl->Vs};
    pdm_launch_gemv(pl, wh, nv, 1, D.d, PD.z, D.d, PD.logits, pl->Vs, 0, 1, st); ++*cnt;
    k_pdm_argmax_cand<<<kPdmCand, 256, 0, st>>>(PD); ++*cnt;
    k_pdm_argmax_final<<<1, 32, 0, st>>>(P, PD); ++*cnt;
  }
}

// The draft of one cycle, enqueued in front of the cycle kernel.
int pdm_enqueue_draft(const DevPtrs &P, const PdmPlan *pl, cudaStream_t st, long long *launches) {
  long long cnt = 0;
  k_pdm_begin<<<1, 32, 0, st>>>(P, pl->PD, 0, 0); ++cnt;
  pdm_enqueue_body(P, pl, true, st, &cnt);
  if (launches) *launches += cnt;
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

// After the target's prefill: the full-depth rows of positions 0 .. n_tokens - 1, then F = n_tokens.
int pdm_prefill(const DevPtrs &P, const PdmPlan *pl, int n_tokens, int batched, cudaStream_t st, long long *launches) {
  long long cnt = 0;
  // tensor-core path: the same GEMMs and prefill attention as the target's batched prefill, over the PDM's layers
  if (batched && prefill_pdm_rows(P, pl->w, pl->Ls, pl->PD.kv, pl->fc_full, n_tokens, st, &cnt) == 0) {
    k_pdm_set_final<<<1, 1, 0, st>>>(pl->PD, n_tokens, 0); ++cnt;
    if (launches) *launches += cnt;
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
  }
  cudaGetLastError();
  const int RB = pl->PD.use_tc ? (pl->NB < 32 ? pl->NB : 32) : 32;
  for (int p0 = 0; p0 < n_tokens; p0 += RB) {
    const int rows = n_tokens - p0 < RB ? n_tokens - p0 : RB;
    k_pdm_begin<<<1, 32, 0, st>>>(P, pl->PD, p0, rows); ++cnt;
    pdm_enqueue_body(P, pl, false, st, &cnt);
  }
  k_pdm_set_final<<<1, 1, 0, st>>>(pl->PD, n_tokens, 0); ++cnt;
  if (launches) *launches += cnt;
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int pdm_rollback(const PdmPlan *pl, int new_len, cudaStream_t st) {
  k_pdm_set_final<<<1, 1, 0, st>>>(pl->PD, new_len, 1);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

// what: 0 logits [Vs], 1 last row's hidden state [d], 2 run header int32[3] (first, rows, F), 3 features G [rows][d]
// (index = rows), 4 / 5 K / V rows of PDM layer `index` ([rows][Hkv*hd], rows = bytes / row size)
int pdm_debug_read(const DevPtrs &P, const PdmPlan *pl, int what, int index, void *out, size_t bytes) {
  const Dims &D = P.dim;
  const PdmPtrs &PD = pl->PD;
  PdmRun run;
  if (cudaMemcpy(&run, PD.run, sizeof run, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
  if (what == 0) return bytes == (size_t)pl->Vs * 4 && cudaMemcpy(out, PD.logits, bytes, cudaMemcpyDeviceToHost) == cudaSuccess ? 0 : -1;
  if (what == 1) {
    if (bytes != (size_t)D.d * 4 || run.rows < 1) return -1;
    return cudaMemcpy(out, PD.X + (size_t)(run.rows - 1) * D.d, bytes, cudaMemcpyDeviceToHost) == cudaSuccess ? 0 : -1;
  }
  if (what == 2) {
    if (bytes != 12) return -1;
    int32_t h[3] = {run.first, run.rows, run.final_len};
    memcpy(out, h, 12);
    return 0;
  }
  if (what == 3) {
    if (index != run.rows || bytes != (size_t)run.rows * D.d * 4) return -1;
    return cudaMemcpy(out, PD.G, bytes, cudaMemcpyDeviceToHost) == cudaSuccess ? 0 : -1;
  }
  if (what == 4 || what == 5) {
    const size_t rowb = (size_t)D.Hkv * D.hd * 2;
    if (index < 0 || index >= pl->Ls || bytes % rowb || bytes / rowb > (size_t)D.max_seq) return -1;
    const size_t rows = bytes / rowb;
    for (int hh = 0; hh < D.Hkv && rows; ++hh)
      if (cudaMemcpy2D((char *)out + (size_t)hh * D.hd * 2, rowb, PD.kv + kv_offset(D, index, what == 5, hh), (size_t)D.hd * 2,
                       (size_t)D.hd * 2, rows, cudaMemcpyDeviceToHost) != cudaSuccess)
        return -1;
    return 0;
  }
  return -1;
}

}  // namespace spd
