// spd_kernels.cuh — device functions of the individual operations (plain pointers) and the
// controller kernels (step begin / end) used by both engines.
#pragma once
#include "spd_dev.cuh"

namespace spd {

// ---------------------------------------------------------------------------------------------
// RMSNorm, block-wide: out[i] = x[i] * (1/sqrt(mean(x^2)+eps)) * gain[i].  Fixed reduction tree
// (per-thread strided sum -> warp xor-tree -> warp partials added in order) so the value depends
// only on (x, blockDim).  `red` is >= 33 floats of shared memory.
__device__ __forceinline__ float block_rms_scale(const float *x, int d, float eps, float *red) {
  float ss = 0.f;
  for (int i = threadIdx.x; i < d; i += blockDim.x) { float v = x[i]; ss = fmaf(v, v, ss); }
  ss = warp_sum(ss);
  int nw = (blockDim.x + 31) >> 5;
  __syncthreads();                      // protect `red` against a previous use
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  __syncthreads();
  if (threadIdx.x == 0) {
    float t = 0.f;
    for (int w = 0; w < nw; ++w) t += red[w];
    red[32] = 1.0f / sqrtf(t / (float)d + eps);
  }
  __syncthreads();
  return red[32];
}

__device__ __forceinline__ void block_rmsnorm(const float *x, const uint16_t *gain, int d, float eps,
                                              float *out, float *red) {
  float r = block_rms_scale(x, d, eps, red);
  for (int i = threadIdx.x; i < d; i += blockDim.x) out[i] = x[i] * r * bf16_to_f32(gain[i]);
}

// ---------------------------------------------------------------------------------------------
// One weight row (bf16, k % 8 == 0) dotted with an fp32 vector by one warp.  Lane l takes the
// 8-element chunks l, l+32, ...; fp32 FMA chain per lane, then the xor-tree.  All lanes return the sum.
__device__ __forceinline__ float warp_dot_row(const uint16_t *__restrict__ w, const float *__restrict__ x, int k) {
  const uint4 *wp = reinterpret_cast<const uint4 *>(w);
  const float4 *xp = reinterpret_cast<const float4 *>(x);
  int lane = threadIdx.x & 31;
  int nchunk = k >> 3;
  float a0 = 0.f, a1 = 0.f;
  int c = lane;
  for (; c + 32 < nchunk; c += 64) {
    uint4 w0 = __ldg(wp + c), w1 = __ldg(wp + c + 32);
    float4 x0 = xp[2 * c], x1 = xp[2 * c + 1], y0 = xp[2 * (c + 32)], y1 = xp[2 * (c + 32) + 1];
    a0 = fmaf(bf16_lo(w0.x), x0.x, a0); a0 = fmaf(bf16_hi(w0.x), x0.y, a0);
    a0 = fmaf(bf16_lo(w0.y), x0.z, a0); a0 = fmaf(bf16_hi(w0.y), x0.w, a0);
    a0 = fmaf(bf16_lo(w0.z), x1.x, a0); a0 = fmaf(bf16_hi(w0.z), x1.y, a0);
    a0 = fmaf(bf16_lo(w0.w), x1.z, a0); a0 = fmaf(bf16_hi(w0.w), x1.w, a0);
    a1 = fmaf(bf16_lo(w1.x), y0.x, a1); a1 = fmaf(bf16_hi(w1.x), y0.y, a1);
    a1 = fmaf(bf16_lo(w1.y), y0.z, a1); a1 = fmaf(bf16_hi(w1.y), y0.w, a1);
    a1 = fmaf(bf16_lo(w1.z), y1.x, a1); a1 = fmaf(bf16_hi(w1.z), y1.y, a1);
    a1 = fmaf(bf16_lo(w1.w), y1.z, a1); a1 = fmaf(bf16_hi(w1.w), y1.w, a1);
  }
  for (; c < nchunk; c += 32) {
    uint4 w0 = __ldg(wp + c);
    float4 x0 = xp[2 * c], x1 = xp[2 * c + 1];
    a0 = fmaf(bf16_lo(w0.x), x0.x, a0); a0 = fmaf(bf16_hi(w0.x), x0.y, a0);
    a0 = fmaf(bf16_lo(w0.y), x0.z, a0); a0 = fmaf(bf16_hi(w0.y), x0.w, a0);
    a0 = fmaf(bf16_lo(w0.z), x1.x, a0); a0 = fmaf(bf16_hi(w0.z), x1.y, a0);
    a0 = fmaf(bf16_lo(w0.w), x1.z, a0); a0 = fmaf(bf16_hi(w0.w), x1.w, a0);
  }
  return warp_sum(a0 + a1);
}

__device__ __forceinline__ float silu_mul(float g, float u) { return g / (1.0f + expf(-g)) * u; }

// ---------------------------------------------------------------------------------------------
// Attention partial for one (kv head, split): the `group` q heads that share the kv head, one warp
// each.  Lane l holds head-dim elements [l*EPL, (l+1)*EPL), EPL = HD/32.  Rows [t0, t1) of K/V
// ([rows][HD] bf16).  Online softmax in fp32; writes unnormalised o, running max m and sum l.
template <int HD>
__device__ __forceinline__ void attn_partial_warp(const float *__restrict__ qh, const uint16_t *__restrict__ kc,
                                                  const uint16_t *__restrict__ vc, int t0, int t1,
                                                  float *__restrict__ o_out, float2 *__restrict__ ml_out) {
  constexpr int EPL = HD / 32;
  int lane = threadIdx.x & 31;
  const float scale = 1.0f / sqrtf((float)HD);
  float qv[EPL], acc[EPL];
#pragma unroll
  for (int e = 0; e < EPL; ++e) { qv[e] = __ldcg(qh + lane * EPL + e); acc[e] = 0.f; }   // q comes from other CTAs
  float m = -INFINITY, l = 0.f;
  for (int t = t0; t < t1; t += 4) {
    float s[4];
    float kv_[4][EPL];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      float part = 0.f;
      if (t + r < t1) {
        const uint16_t *kr = kc + (size_t)(t + r) * HD + lane * EPL;
        if constexpr (EPL == 4) {
          uint2 w = *reinterpret_cast<const uint2 *>(kr);
          part = fmaf(bf16_lo(w.x), qv[0], part); part = fmaf(bf16_hi(w.x), qv[1], part);
          part = fmaf(bf16_lo(w.y), qv[2], part); part = fmaf(bf16_hi(w.y), qv[3], part);
        } else {
          uint32_t w = *reinterpret_cast<const uint32_t *>(kr);
          part = fmaf(bf16_lo(w), qv[0], part); part = fmaf(bf16_hi(w), qv[1], part);
        }
        const uint16_t *vr = vc + (size_t)(t + r) * HD + lane * EPL;
        if constexpr (EPL == 4) {
          uint2 w = *reinterpret_cast<const uint2 *>(vr);
          kv_[r][0] = bf16_lo(w.x); kv_[r][1] = bf16_hi(w.x); kv_[r][2] = bf16_lo(w.y); kv_[r][3] = bf16_hi(w.y);
        } else {
          uint32_t w = *reinterpret_cast<const uint32_t *>(vr);
          kv_[r][0] = bf16_lo(w); kv_[r][1] = bf16_hi(w);
        }
      } else {
#pragma unroll
        for (int e = 0; e < EPL; ++e) kv_[r][e] = 0.f;
      }
      s[r] = part;
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) s[r] = warp_sum(s[r]) * scale;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      if (t + r < t1) {
        float mn = fmaxf(m, s[r]);
        float corr = expf(m - mn);       // exp(-inf) = 0 on the first row
        float p = expf(s[r] - mn);
        l = fmaf(l, corr, p);
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = fmaf(acc[e], corr, p * kv_[r][e]);
        m = mn;
      }
    }
  }
#pragma unroll
  for (int e = 0; e < EPL; ++e) o_out[lane * EPL + e] = acc[e];
  if (lane == 0) *ml_out = make_float2(m, l);
}

// Merge of the splits of one q head, in split order (fixed): out = sum_j o_j e^(m_j-M) / sum_j l_j e^(m_j-M).
// Called by HD threads (thread e owns element e) or strided.
__device__ __forceinline__ float attn_merge_elem(const float *__restrict__ part_o, const float2 *__restrict__ part_ml,
                                                 int nsplit, int hd, int e) {
  float M = -INFINITY;
  for (int j = 0; j < nsplit; ++j) M = fmaxf(M, part_ml[j].x);
  float L = 0.f, o = 0.f;
  for (int j = 0; j < nsplit; ++j) {
    float w = expf(part_ml[j].x - M);
    L = fmaf(part_ml[j].y, w, L);
    o = fmaf(part_o[(size_t)j * hd + e], w, o);
  }
  return o / L;
}

// ---------------------------------------------------------------------------------------------
// Controller, first part of a cycle (one thread): fill / p_new, what runs, cycle counter, the
// forced-acceptance draw (C-2.19).
__device__ __forceinline__ void controller_begin(const DevPtrs &P) {
  StepState *st = P.st;
  int n = P.dim.n, fill = 0;
  for (int k = 0; k < n; ++k) fill += st->occ[k];
  st->fill = fill;
  st->p_new = st->occ[0] ? st->pos[0] : -1;
  st->run_pdm = st->mode == MODE_SPD && !P.paper_pdm;   // the paper's PDM runs in its own kernels before the cycle
  st->run_verify = (st->mode == MODE_SPD && st->occ[n - 1]) || st->mode == MODE_PREFILL_FINAL;
  st->forced_now = 0;
  if (st->mode == MODE_SPD) {
    st->K += 1;
    P.cycle_ts[2 * ((st->K - 1) % kResultRing)] = globaltimer_ns();   // entry stamp of cycle K (SPD_DBG_CYCLE_TIMES)
    if (st->forced_on) {
      unsigned long long draw = splitmix64(st->forced_seed + (unsigned long long)st->K) >> 11;
      int ti = st->p_new + 1 - st->prompt_len;
      if (draw < st->forced_thresh && ti >= 0 && ti < st->n_truth) st->forced_now = 1;
    }
  }
}

// RoPE table of this cycle: (cos, sin)(pos_k * theta_i) in double, rounded to fp32 (C-2.14).
__device__ __forceinline__ void rope_table_fill(const DevPtrs &P, int tid, int nthreads) {
  int half = P.dim.hd / 2;
  for (int i = tid; i < P.dim.n * half; i += nthreads) {
    int k = i / half, j = i - k * half;
    if (!P.st->occ[k]) continue;
    double ang = (double)P.st->pos[k] * P.inv_freq[j];
    double s, c;
    sincos(ang, &s, &c);
    P.rope[i] = make_float2((float)c, (float)s);
  }
}

// ---------------------------------------------------------------------------------------------
// Sampling verification (NEXT-2).  All of it runs in the controller CTA at the end of a cycle.

// S-6: u(seed, K, j) = (splitmix64(seed + 3 K + j) >> 40) * 2^-24.
__device__ __forceinline__ float samp_uniform(unsigned long long seed, long long K, int j) {
  return (float)(splitmix64(seed + 3ull * (unsigned long long)K + (unsigned long long)j) >> 40) * (1.0f / 16777216.0f);
}

// S-2: the top_k entries of logits[0..V) in the order (value descending, index ascending), listed in ascending
// token id with p = softmax(l / T) over them.  Whole CTA (>= 64 threads); `out` is global or shared memory.
//   1. tau = the k-th best argmax candidate: the candidates are distinct entries, so at least k logits are
//      >= tau and every top-k entry is;  2. one scan keeps the entries >= tau (about k .. 2k of them for
//      near-i.i.d. logits);  3. each survivor's rank among the survivors decides membership.
//   If fewer than k candidates exist or more than kSampCap entries survive (heavy ties, adversarial logits):
//   k exact rounds of "best entry after the previous one".
struct TopkSmem {   // shared-memory scratch of topk_dist (the caller says where it lives)
  double e[kMaxTopK];
  float sel_v[kMaxTopK], red_v[32], tau;
  int sel_i[kMaxTopK], red_i[32], cnt, nvalid;
  float sv[kSampCap];               // the survivors, staged for the all-pairs ranking
  int si[kSampCap];
};
//   0. (fused engine) the head pass itself listed every logit >= a guessed threshold (the previous cycle's k-th
//      value minus a margin) while the value was in a register: if that list holds between k and kSampCap
//      entries it contains the whole top-k and replaces steps 1-2 (no second pass over the logits); otherwise
//      the scan runs.  pre_cnt < 0: no such list.  *next_guess receives the threshold for the next cycle.
struct TopkPre {
  const float *val;
  const int32_t *idx;
  int cnt;
};
__device__ __forceinline__ void topk_dist(const float *logits, int V, const float *cand_val, const int32_t *cand_idx,
                                          int ncand, int top_k, float temperature, float *surv_val,
                                          int32_t *surv_idx, SampleDist *out, int32_t *exact_rounds, TopkSmem *ts,
                                          TopkPre pre = TopkPre{nullptr, nullptr, -1}, int32_t *prefiltered = nullptr,
                                          float *next_guess = nullptr) {
  float &s_tau = ts->tau;
  float *s_sel_v = ts->sel_v, *s_red_v = ts->red_v;
  double *s_e = ts->e;
  int &s_cnt = ts->cnt, &s_nvalid = ts->nvalid;
  int *s_sel_i = ts->sel_i, *s_red_i = ts->red_i;
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nt >> 5;
  const int k = min(min(top_k, V), kMaxTopK);
  if (tid == 0) { s_tau = -INFINITY; s_cnt = 0; s_nvalid = 0; }
  __syncthreads();
  const bool use_pre = pre.cnt >= k && pre.cnt <= kSampCap;
  if (use_pre) {
    if (tid == 0 && prefiltered) *prefiltered += 1;
    surv_val = const_cast<float *>(pre.val);
    surv_idx = const_cast<int32_t *>(pre.idx);
  }
  for (int i = tid; i < (use_pre ? 0 : ncand); i += nt) {
    const int ix = cand_idx[i];
    if (ix < 0) continue;
    const float v = cand_val[i];
    int better = 0;
    for (int j = 0; j < ncand; ++j) {
      const int jx = cand_idx[j];
      if (jx >= 0 && cand_better(cand_val[j], jx, v, ix)) ++better;
    }
    atomicAdd(&s_nvalid, 1);
    if (better == k - 1) s_tau = v;
  }
  __syncthreads();
  bool exact = !use_pre && s_nvalid < k && V > kSampCap;
  if (!exact) {
    const float tau = s_nvalid < k ? -INFINITY : s_tau;
    auto keep = [&](float v, int i) {
      if (v >= tau) {
        const int pos = atomicAdd(&s_cnt, 1);
        if (pos < kSampCap) { surv_val[pos] = v; surv_idx[pos] = i; }
      }
    };
    // the vector sits in L2: 8 independent 16-byte loads per thread and round keep the one scanning SM busy
    constexpr int U = 8;
    const int n4 = use_pre ? 0 : ((reinterpret_cast<uintptr_t>(logits) & 15) == 0 ? V >> 2 : 0);
    const float4 *l4 = reinterpret_cast<const float4 *>(logits);
    for (int base = 0; base < n4; base += nt * U) {
      float4 v[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int i = base + u * nt + tid;
        if (i < n4) v[u] = __ldcg(l4 + i);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int i = base + u * nt + tid;
        if (i < n4) { keep(v[u].x, 4 * i); keep(v[u].y, 4 * i + 1); keep(v[u].z, 4 * i + 2); keep(v[u].w, 4 * i + 3); }
      }
    }
    for (int i = 4 * n4 + tid; i < (use_pre ? 0 : V); i += nt) keep(__ldcg(logits + i), i);
    __syncthreads();
    const int m = use_pre ? pre.cnt : s_cnt;
    if (m > kSampCap) exact = true;
    else {
      for (int i = tid; i < m; i += nt) { ts->sv[i] = __ldcg(surv_val + i); ts->si[i] = __ldcg(surv_idx + i); }
      __syncthreads();
      for (int i = tid; i < m; i += nt) {
        const float v = ts->sv[i];
        const int ix = ts->si[i];
        int better = 0;
        for (int j = 0; j < m; ++j) better += cand_better(ts->sv[j], ts->si[j], v, ix) ? 1 : 0;
        if (better < k) { s_sel_v[better] = v; s_sel_i[better] = ix; }
      }
    }
  }
  if (exact) {   // uniform over the CTA: s_nvalid, s_cnt are shared
    if (tid == 0 && exact_rounds) *exact_rounds += 1;
    float pv = INFINITY;
    int pi = -1;
    for (int r = 0; r < k; ++r) {
      float bv = -INFINITY;
      int bi = 0x7fffffff;
      for (int i = tid; i < V; i += nt) {
        const float v = __ldcg(logits + i);
        if (cand_better(pv, pi, v, i) && cand_better(v, i, bv, bi)) { bv = v; bi = i; }   // after the previous pick
      }
      for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (cand_better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
      }
      if (lane == 0) { s_red_v[warp] = bv; s_red_i[warp] = bi; }
      __syncthreads();
      if (tid == 0) {
        for (int w = 1; w < nwarp; ++w)
          if (cand_better(s_red_v[w], s_red_i[w], bv, bi)) { bv = s_red_v[w]; bi = s_red_i[w]; }
        s_sel_v[r] = bv; s_sel_i[r] = bi;
      }
      __syncthreads();
      pv = s_sel_v[r]; pi = s_sel_i[r];
    }
  }
  __syncthreads();
  // ascending token id, then softmax((l - max) / T): exponentials and their sum in fp64, p rounded to fp32
  float lv = 0.f;
  int rank = 0, ix = 0;
  if (tid < k) {
    ix = s_sel_i[tid]; lv = s_sel_v[tid];
    for (int j = 0; j < k; ++j) rank += s_sel_i[j] < ix ? 1 : 0;
  }
  const float mx = s_sel_v[0];
  if (tid == 0 && next_guess) {   // next cycle's list threshold: this cycle's k-th value minus a margin that follows the
    // LOCAL spacing of the order statistics (rank k/2 to rank k), not the maximum: a peaked distribution (one
    // dominant logit) must not drag the threshold below the bulk, or every logit would be listed
    const float kth = s_sel_v[k - 1];
    *next_guess = kth - fmaxf(1.25f * (s_sel_v[(k - 1) / 2] - kth), 0.1f + 0.05f * fabsf(kth));
  }
  __syncthreads();
  if (tid < k) {
    out->id[rank] = ix;
    s_e[rank] = exp(((double)lv - (double)mx) / (double)temperature);
  }
  __syncthreads();
  if (tid < k) {
    double Z = 0.0;
    for (int j = 0; j < k; ++j) Z += s_e[j];
    out->p[tid] = (float)(s_e[tid] / Z);
  }
  if (tid == 0) out->k = k;
  __syncthreads();
}

// Shared-memory working set of the sampler in the controller CTA.
struct SampSmem {
  TopkSmem tk;
  SampleDist qd, pt, qs;            // this cycle's draft / target distributions, the judged token's stored one
  double w[kMaxTopK];               // residual weights max(0, P - Q) over P's support
  int ctl[12];                      // controller_end's CTA-wide scalars
};
__device__ __forceinline__ double dist_prob(const SampleDist *D, int token) {
  for (int i = 0; i < D->k; ++i)
    if (D->id[i] == token) return (double)D->p[i];
  return 0.0;
}
// S-3: inverse CDF over weights in list order, fp64: the smallest i with u * W < w_0 + .. + w_i.
__device__ __forceinline__ int pick_index(const double *w, int k, double u) {
  double W = 0.0;
  for (int i = 0; i < k; ++i) W += w[i];
  double c = 0.0;
  int last = -1;
  for (int i = 0; i < k; ++i) {
    c += w[i];
    if (w[i] > 0.0) last = i;
    if (u * W < c) return i;
  }
  return last;
}
__device__ __forceinline__ int sample_cdf(const SampleDist *D, double u) {
  double W = 0.0;
  for (int i = 0; i < D->k; ++i) W += (double)D->p[i];
  double c = 0.0;
  int last = -1;
  for (int i = 0; i < D->k; ++i) {
    c += (double)D->p[i];
    if (D->p[i] > 0.f) last = i;
    if (u * W < c) return D->id[i];
  }
  return D->id[last];
}
// The replacement of a rejected token: drawn from norm(max(0, P - Q)); w = those
// weights over P's support (computed by the CTA in parallel), all zero -> P itself.
__device__ __forceinline__ int sample_residual(const SampleDist *Pt, const double *w, double u) {
  double W = 0.0;
  for (int i = 0; i < Pt->k; ++i) W += w[i];
  if (W > 0.0) return Pt->id[pick_index(w, Pt->k, u)];
  return sample_cdf(Pt, u);
}

// Controller, last part of a cycle (one CTA, >= 32 threads): reduce the argmax candidates, verify,
// accept / reject + rollback, shift the pipeline, enter the next token, record.
// Needs >= 64 threads.  `ncand` candidates per head (verify = row 0, PDM = row 1 of cand_val/cand_idx).
// `sm`: shared-memory scratch for the sampler (may be nullptr when P.sampling == 0).
// `with_lists`: the head pass filled the threshold lists (fused engine).
__device__ __forceinline__ void controller_end(const DevPtrs &P, int ncand, SampSmem *sm, bool with_lists = false) {
  // CTA-wide scalars of the controller live in the caller's scratch (no static shared memory: the fused kernels' dynamic
  // segment is 1024-byte aligned and has no room for a padded static one)
  int &s_y = sm->ctl[0], &s_draft = sm->ctl[1], &s_exit_buf = sm->ctl[2], &s_exit_pos = sm->ctl[3], &s_enter_tok = sm->ctl[4],
      &s_enter_buf = sm->ctl[5], &s_do_exit = sm->ctl[6], &s_do_enter = sm->ctl[7], &s_keep_q = sm->ctl[8], &s_stamp = sm->ctl[9];
  StepState *st = P.st;
  const Dims &D = P.dim;
  int n = D.n;
  SampleState *ss = P.samp;
  const bool sampling = P.sampling != 0;
  if (sampling) {   // filtered distributions of this cycle's PDM and exit logits (the heads kept the full vectors)
    if (threadIdx.x == 0) { ss->rec.exact_rounds = 0; ss->rec.prefiltered = 0; sm->qd.k = 0; sm->pt.k = 0; sm->qs.k = 0; }
    __syncthreads();
    // head-pass lists (fused engine; row 0 = verify, row 1 = PDM); the reference engine has none
    const int cnt_v = with_lists ? __ldcg(&ss->pre_cnt[0]) : -1, cnt_p = with_lists ? __ldcg(&ss->pre_cnt[1]) : -1;
    if (st->run_pdm)
      topk_dist(P.logits_p, D.V, P.cand_val + kMaxCand, P.cand_idx + kMaxCand, ncand, ss->top_k, ss->temperature,
                P.samp_val, P.samp_idx, &sm->qd, &ss->rec.exact_rounds, &sm->tk,
                TopkPre{P.pre_val + kSampCap, P.pre_idx + kSampCap, cnt_p}, &ss->rec.prefiltered, &ss->tau_guess[1]);
    if (st->run_verify)
      topk_dist(P.logits_v, D.V, P.cand_val, P.cand_idx, ncand, ss->top_k, ss->temperature, P.samp_val, P.samp_idx,
                &sm->pt, &ss->rec.exact_rounds, &sm->tk, TopkPre{P.pre_val, P.pre_idx, cnt_v}, &ss->rec.prefiltered,
                &ss->tau_guess[0]);
    if (threadIdx.x < 2) ss->pre_cnt[threadIdx.x] = 0;
    // the judged token's stored distribution (n = 1: the draft of this very cycle, C-2.12) and the residual
    // weights, which depend on P and Q only — ready before thread 0 takes the decisions
    const bool judging = st->mode == MODE_SPD && st->occ[n - 1];
    constexpr int DW = (int)(sizeof(SampleDist) / 4);
    if (judging) {
      const int32_t *src = n > 1 ? reinterpret_cast<const int32_t *>(&ss->q[st->hbuf[n - 2]])
                                 : reinterpret_cast<const int32_t *>(&sm->qd);
      for (int i = threadIdx.x; i < DW; i += blockDim.x) reinterpret_cast<int32_t *>(&sm->qs)[i] = src[i];
    }
    for (int i = threadIdx.x; i < DW; i += blockDim.x) {   // the record of this cycle (SPD_DBG_SAMPLE)
      reinterpret_cast<int32_t *>(&ss->rec.draft)[i] = reinterpret_cast<const int32_t *>(&sm->qd)[i];
      reinterpret_cast<int32_t *>(&ss->rec.target)[i] = reinterpret_cast<const int32_t *>(&sm->pt)[i];
    }
    __syncthreads();
    if (judging && sm->qs.k == 0) {   // in flight since before sampling was switched on: a deterministic draft, Q one-hot
      __syncthreads();
      if (threadIdx.x == 0) { sm->qs.k = 1; sm->qs.id[0] = st->tok[n - 2]; sm->qs.p[0] = 1.f; }
      __syncthreads();
    }
    if (judging && (int)threadIdx.x < sm->pt.k) {
      const double r = (double)sm->pt.p[threadIdx.x] - dist_prob(&sm->qs, sm->pt.id[threadIdx.x]);
      sm->w[threadIdx.x] = r > 0.0 ? r : 0.0;
    }
    __syncthreads();
  }
  if (threadIdx.x < 64) {
    // warp 0 = verify, warp 1 = PDM; lowest index among equal maxima ((value, index) is a total order,
    // so the result does not depend on the reduction shape)
    int which = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float bv = -INFINITY;
    int bi = 0x7fffffff;
    for (int i = lane; i < ncand; i += 32) {
      float v = P.cand_val[which * kMaxCand + i];
      int ix = P.cand_idx[which * kMaxCand + i];
      if (ix >= 0 && cand_better(v, ix, bv, bi)) { bv = v; bi = ix; }
    }
    for (int o = 16; o > 0; o >>= 1) {
      float ov = __shfl_xor_sync(0xffffffffu, bv, o);
      int oi = __shfl_xor_sync(0xffffffffu, bi, o);
      if (cand_better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
    }
    if (lane == 0) { if (which == 0) s_y = bi; else s_draft = bi; }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int mode = st->mode;
    int exited = st->occ[n - 1];
    int y = s_y, draft = s_draft;
    StepResult r;
    r.step_index = (int)st->K; r.fill = st->fill; r.exited = 0; r.accepted = 0; r.emitted_token = -1;
    r.draft_token = -1; r.draft_forced = 0; r.discarded = 0;
    s_do_exit = 0; s_do_enter = 0; s_keep_q = 0;
    s_stamp = mode == MODE_SPD ? (r.step_index - 1) % kResultRing : -1;
    if (sampling) {
      ss->rec.u_draft = ss->rec.u_accept = ss->rec.u_resid = -1.f;
      ss->rec.succ_token = -1; ss->rec.succ_q = ss->rec.succ_p = 0.f;
      if (mode == MODE_SPD) {                 // x^ ~ Q_t (S-3, j = 0)
        ss->rec.u_draft = samp_uniform(ss->seed, st->K, 0);
        draft = sample_cdf(&sm->qd, (double)ss->rec.u_draft);
      } else if (mode == MODE_PREFILL_FINAL) {   // the first token is drawn from P as well (j = 2, K = 0)
        ss->rec.u_resid = samp_uniform(ss->seed, 0, 2);
        y = sample_cdf(&sm->pt, (double)ss->rec.u_resid);
      }
    }
    s_exit_buf = st->hbuf[n - 1]; s_exit_pos = st->pos[n - 1];
    int enter_tok = -1, enter_pos = -1;
    bool flush = false;
    if (mode == MODE_SPD) {
      if (P.paper_pdm) draft = *P.pdm_draft;        // NEXT-1: drafted by spd_pdm.cu's kernels on the pre-step state
      if (st->forced_now) { draft = P.truth[st->p_new + 1 - st->prompt_len]; r.draft_forced = 1; }
      r.draft_token = draft;
      if (exited) {
        s_do_exit = 1;
        st->c = st->pos[n - 1] + 1;
        st->N += 1;
        r.exited = 1;
        int succ = n > 1 ? st->tok[n - 2] : draft;   // the token one stage behind (C-2.12 for n = 1)
        bool ok = succ == y;                         // greedy: exact argmax match
        if (sampling) {                              // sampling: standard rejection sampling
          const double qx = dist_prob(&sm->qs, succ), px = dist_prob(&sm->pt, succ);
          ss->rec.succ_token = succ; ss->rec.succ_q = (float)qx; ss->rec.succ_p = (float)px;
          ss->rec.u_accept = samp_uniform(ss->seed, st->K, 1);
          ok = (double)ss->rec.u_accept * qx < px;
          if (ok) y = succ;
          else {                                     // the replacement ~ norm(max(0, P - Q)) (j = 2)
            ss->rec.u_resid = samp_uniform(ss->seed, st->K, 2);
            y = sample_residual(&sm->pt, sm->w, (double)ss->rec.u_resid);
          }
        }
        r.emitted_token = y;
        if (ok) {
          r.accepted = 1;
          enter_tok = draft; enter_pos = st->p_new + 1;
          s_keep_q = sampling;
        } else {
          r.discarded = st->fill - 1;
          for (int l = 0; l < D.L; ++l) if (P.len[l] > st->c) P.len[l] = st->c;   // truncate
          flush = true;
          enter_tok = y; enter_pos = st->c;                                       // reseed; draft dropped
        }
      } else {
        enter_tok = draft; enter_pos = st->p_new + 1;
        s_keep_q = sampling;
      }
    } else if (mode == MODE_PREFILL) {
      if (exited) { s_do_exit = 1; st->c = st->pos[n - 1] + 1; }
      if (st->pf_next < st->pf_n) { enter_tok = P.pf_tokens[st->pf_next]; enter_pos = st->pf_next; st->pf_next += 1; }
    } else if (mode == MODE_PREFILL_FINAL) {
      flush = true;
      enter_tok = y; enter_pos = st->c;
      st->mode = MODE_SPD; st->K = 0; st->N = 1;
      r.emitted_token = y;
    }
    // shift depth k -> k+1; the buffer ids rotate so the exiting token's buffer receives the entrant
    int freebuf = st->hbuf[n - 1];
    for (int k = n - 1; k > 0; --k) {
      st->occ[k] = flush ? 0 : st->occ[k - 1];
      st->pos[k] = st->pos[k - 1]; st->tok[k] = st->tok[k - 1]; st->hbuf[k] = st->hbuf[k - 1];
    }
    st->hbuf[0] = freebuf;
    st->occ[0] = enter_tok >= 0;
    st->pos[0] = enter_pos; st->tok[0] = enter_tok;
    s_do_enter = enter_tok >= 0; s_enter_tok = enter_tok; s_enter_buf = freebuf;
    r.committed_len = st->c;
    if (mode == MODE_SPD) P.results[(r.step_index - 1) % kResultRing] = r;
    else if (mode == MODE_PREFILL_FINAL) P.results[0] = r;
  }
  __syncthreads();
  if (s_keep_q) {      // the entering draft keeps the distribution it was drawn from, filed under its hidden buffer
    const int32_t *src = reinterpret_cast<const int32_t *>(&sm->qd);
    int32_t *dst = reinterpret_cast<int32_t *>(&ss->q[s_enter_buf]);
    for (int i = threadIdx.x; i < (int)(sizeof(SampleDist) / 4); i += blockDim.x) dst[i] = src[i];
  }
  int d = D.d;   // d % 8 == 0
  if (s_do_exit) {     // Hfin[e.pos] = e.h  (C-2.4) — read before the buffer is reused below
    const float4 *src = reinterpret_cast<const float4 *>(P.h + (size_t)s_exit_buf * d);
    float4 *dst = reinterpret_cast<float4 *>(P.hfin + (size_t)s_exit_pos * d);
    for (int i = threadIdx.x; i < (d >> 2); i += blockDim.x) dst[i] = src[i];
  }
  __syncthreads();
  if (s_do_enter) {    // token entry: h = E[tok] (k = 0 is the embedding-level input)
    const uint2 *e = reinterpret_cast<const uint2 *>(P.embed + (size_t)s_enter_tok * d);
    float4 *dst = reinterpret_cast<float4 *>(P.h + (size_t)s_enter_buf * d);
    for (int i = threadIdx.x; i < (d >> 2); i += blockDim.x) {
      uint2 w = e[i];
      dst[i] = make_float4(bf16_lo(w.x), bf16_hi(w.x), bf16_lo(w.y), bf16_hi(w.y));
    }
  }
  __syncthreads();
  if (threadIdx.x == 0 && s_stamp >= 0) P.cycle_ts[2 * s_stamp + 1] = globaltimer_ns();   // the cycle's state is final
}

}  // namespace spd
