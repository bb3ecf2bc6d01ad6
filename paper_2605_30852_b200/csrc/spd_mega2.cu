// spd_mega2.cu — the fused persistent engine with MULTIPLEXED STAGE CHAINS (SPD_OPT_ENGINE = 2): one cooperative kernel
// per SPD cycle, the building blocks of spd_mega.cu (spd_mega_dev.cuh: tile ring, gemv_stream, head_stream, attention
// items, fused epilogues — same mappings, same summation orders), a different schedule.
//
// Why (measured on the one-chain engine, profiles/r02_k_spd_cycle_full.md): while tiles are consumed every GEMV phase runs
// at 7.4-7.7 TB/s, but a CTA serves ONE stage, so at each of the 5 L/n phase boundaries it sits in the group barrier
// (3-9 us: tail skew of one unit + the release / acquire chain) and then stages the next activation vector (1-2 us).
// An SM's bandwidth is bound by the bytes it keeps in flight (176 KB of ring), so nobody else can use what it leaves
// idle: 30 us per pass = 11 % of the 9b_n4 cycle, 19 % of the 4b_n4 cycle.
//
// Schedule here:
//   * the a active stages are grouped in pairs (one triple when a is odd) and a CTA serves ALL chains of its group in
//     turn: visit (phase p, chain 0), (p, chain 1), (p + 1, chain 0), ...  The phase p + 1 of a chain depends on its
//     phase p — which every CTA of the group finished one visit earlier: by the time it is needed the barrier has long
//     opened, and the skew of one visit is absorbed by the dynamic unit claims of the next (nobody waits in between).
//   * a STAGER (2 warps) runs one visit ahead of the consumers: it polls the dependency (ld.acquire on the group's
//     counter), copies the next visit's activation vector L2 -> shared memory (RMSNorm fused: every lane holds its 16
//     float4 and their gains in registers, one L2 round trip), and hands the buffer over through an mbarrier.  Consumers
//     never touch global memory for their inputs and never poll a global counter.
//   * two 24 KB activation buffers alternate between visits.  W_down is therefore streamed as TWO phases over the two
//     K parts of the repacked matrix (residual += part a, then += part b: a fixed order), so no visit needs more than
//     24 KB: 6 phases per pass (QKV, ATTN, O, GATEUP, DOWN_A, DOWN_B).  The ring keeps its 11 slots.  A CTA streams
//     DOWN_B for exactly the units it claimed in DOWN_A, so the two residual updates of a row are local and ordered and
//     DOWN_B has no dependency on other CTAs' DOWN_A.
//   * attention visits use their buffer as scratch; an item's q (G heads, 2 KB) arrives through the ring behind its K/V tiles.
//   * PDM phase (visit 0) and LM head (last visit) are the one-chain engine's (foreground staging, whole buffer).
// Results do not depend on the grouping: every row's dot product, every attention split and every merge keep their fixed
// mapping and order (batch invariance as in spd_mega.cu).  DOWN differs from the one-chain engine by the point where the
// residual is added (h + a, then + b, instead of h + (a + b)): the same products, one more fp32 rounding.
#include "spd_mega_dev.cuh"

namespace spd {

constexpr int kXHalf = kXFloats / 2;                      // floats per activation buffer (24 KB)
constexpr int kStagerThreads = 64;
constexpr int kThreads2 = kConsumerThreads + 32 + kStagerThreads + 32;   // 8 consumer warps, producer, 2 stager warps, publisher
// (12 warps = 3 per SM sub-partition: the most that leaves the consumers their 168 registers)
constexpr int kMaxChains = kMega2MaxChains;               // stage chains a CTA serves at most
constexpr int kPhasesPerPass = 6;
// W_down's second K part (DOWN_B) is streamed for the SAME units a CTA claimed in DOWN_A: both residual updates of a row
// then happen in one CTA, in program order, and DOWN_B needs no cross-CTA dependency on DOWN_A (its input, the second half
// of the SwiGLU vector, is complete since GATEUP).  A CTA stops claiming at kDnCap units; the rest of its group takes them.
constexpr int kDnCap = 96;

enum Phase2 { P2_QKV = 0, P2_ATTN = 1, P2_O = 2, P2_GU = 3, P2_DNA = 4, P2_DNB = 5 };

// Per-cycle schedule, computed identically by every CTA from the device state.
struct Sched2 {
  int mode, n_act, run_pdm, run_verify, p_new, c;
  unsigned int occ_mask;
  int pos[kMaxStages], hbuf[kMaxStages];
  int m;                                        // chains of this CTA's group (0: no stage is active)
  int gsize;                                    // CTAs in this CTA's group
  int lead;                                     // this CTA does the once-per-stage bookkeeping of its chains
  int exit_gsize;                               // CTAs in the group that serves stage n - 1 (0: that stage is empty)
  int pdm_slot, pdm_idx;
  int stage[kMaxChains];
  int attn_ns[kMaxChains], attn_total[kMaxChains], attn_nonfinal[kMaxChains];
};

struct Visit {
  int kind;                                     // 0 PDM, 1 layer phase, 2 LM head
  int p;                                        // global phase index: 0 PDM, 1 + 6 pass + type, np - 1 head
  int type, pass, j;                            // layer visits: Phase2, pass, chain
};

__device__ __forceinline__ Visit visit_decode(int v, int nv, int np, int m) {
  Visit x;
  x.type = 0; x.pass = 0; x.j = 0;
  if (v == 0) { x.kind = 0; x.p = 0; }
  else if (v == nv - 1) { x.kind = 2; x.p = np - 1; }
  else {
    const int w = v - 1, pl = w / m;
    x.kind = 1; x.j = w - pl * m; x.pass = pl / kPhasesPerPass; x.type = pl - x.pass * kPhasesPerPass; x.p = 1 + pl;
  }
  return x;
}

// What a visit streams for this CTA (pure function of the schedule: producer, stager and consumers agree).
struct Work2 {
  int job, U, nc;                               // job < 0: nothing to stream
  const uint8_t *base;
  unsigned int *ctr;
};

__device__ __forceinline__ Work2 work_desc(const Visit &x, const Sched2 &S, const MegaLayout &ML, const Dims &D,
                                           unsigned int *claim) {
  Work2 w;
  w.job = -1; w.U = 0; w.nc = 0; w.base = nullptr; w.ctr = claim + (size_t)x.p * kMaxStages;
  if (x.kind == 0) {
    if (!S.run_pdm) return w;
    w.job = S.pdm_slot; w.U = ML.u_pdm; w.nc = ML.nc_d;
    w.base = ML.repack + ML.off_pdm + (unsigned long long)w.job * ML.pdm_job_bytes;
  } else if (x.kind == 2) {
    if (!S.run_pdm && !S.run_verify) return w;
    w.job = 0; w.U = ML.u_head; w.nc = ML.nc_d;
    w.base = ML.repack + ML.off_head;
  } else {
    const int k = S.stage[x.j];
    w.job = k;
    if (x.type == P2_ATTN) { w.U = S.attn_total[x.j]; }
    else {
      const uint8_t *lb = ML.repack + (unsigned long long)(k * D.per + x.pass) * ML.layer_bytes;
      if (x.type == P2_QKV) { w.U = ML.u_qkv; w.nc = ML.nc_d; w.base = lb; }
      else if (x.type == P2_O) { w.U = ML.u_o; w.nc = ML.nc_qd; w.base = lb + ML.off_o; }
      else if (x.type == P2_GU) { w.U = ML.u_gu; w.nc = ML.nc_d; w.base = lb + ML.off_gu; }
      else if (x.type == P2_DNA) { w.U = ML.u_dn; w.nc = ML.nc_fa; w.base = lb + ML.off_dn; }
      else { w.nc = ML.nc_f - ML.nc_fa; w.U = w.nc > 0 ? ML.u_dn : 0; w.base = lb + ML.off_dnb; }
    }
  }
  w.ctr += w.job;
  return w;
}

// Clock stamps are filed per VISIT; slot kProfPhases - 1 holds the kernel's entry / exit stamps, later visits are not recorded.
__device__ __forceinline__ void vstamp(const DevPtrs &P, int cta, int v, int stamp) {
  if (v < kProfPhases - 1) prof_stamp(P, cta, v, stamp);
}
__device__ __forceinline__ void stager_sync() { asm volatile("bar.sync 2, 64;" ::: "memory"); }

// What a visit's inputs depend on (stager): polled with ld.acquire by one lane per stager warp.
struct Dep {
  const unsigned int *c0, *c1;                  // counters (nullptr: none)
  unsigned int t0, t1;                          // targets
};
__device__ __forceinline__ void dep_wait(const Dep &dp, int st) {
  if ((st & 31) == 0) {
    if (dp.c0) while (ld_acquire_u32(dp.c0) < dp.t0) {}
    if (dp.c1) while (ld_acquire_u32(dp.c1) < dp.t1) {}
  }
  __syncwarp();
}

// Stager: waits for the dependency, then K fp32 values (K % 4 == 0) from global (ld.global.cg, written by other CTAs) -> dst,
// zero padding up to kpad.  gain != nullptr: RMSNorm (x * r * gain, r from the sum of squares of the 64 lanes in a fixed
// order); `raw_out` (anchor capture of the paper PDM) receives the unscaled values.  `st` = stager thread 0..63.
// The SM's L2 port is saturated by the weight stream, so a round trip costs 2-3 us: the gains (weights: they do not depend
// on anything) are fetched BEFORE the dependency wait and parked in the unused tail of the buffer, and all of a lane's
// x loads are in flight at once, so a staging is dependency + one round trip.
__device__ __noinline__ void stager_copy(const Dep &dp, const float *src, float *dst, int K, int kpad, const uint16_t *gain,
                                            float eps, float *raw_out, float *sred, int st) {
  const float4 *s4 = reinterpret_cast<const float4 *>(src);
  float4 *d4 = reinterpret_cast<float4 *>(dst);
  const int n4 = K >> 2;
  constexpr int R = 16;                          // float4 per lane and round: 4096 floats per round
  if (gain == nullptr) {
    dep_wait(dp, st);
    for (int base = st; base < n4; base += kStagerThreads * R) {
      float4 v[R];
#pragma unroll
      for (int i = 0; i < R; ++i) { const int idx = base + kStagerThreads * i; if (idx < n4) v[i] = __ldcg(s4 + idx); }
#pragma unroll
      for (int i = 0; i < R; ++i) { const int idx = base + kStagerThreads * i; if (idx < n4) d4[idx] = v[i]; }
    }
  } else if (n4 <= kStagerThreads * R && kpad * 4 + K * 2 <= kXHalf * 4) {
    const uint2 *g2 = reinterpret_cast<const uint2 *>(gain);
    uint2 *gs = reinterpret_cast<uint2 *>(dst + kpad);    // this lane's gains, parked behind the vector
    {
      uint2 g[R];
#pragma unroll
      for (int i = 0; i < R; ++i) { const int idx = st + kStagerThreads * i; if (idx < n4) g[i] = __ldg(g2 + idx); }
      dep_wait(dp, st);
#pragma unroll
      for (int i = 0; i < R; ++i) { const int idx = st + kStagerThreads * i; if (idx < n4) gs[idx] = g[i]; }
    }
    float4 v[R];
    float ss = 0.f;
#pragma unroll
    for (int i = 0; i < R; ++i) {
      const int idx = st + kStagerThreads * i;
      v[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (idx < n4) v[i] = __ldcg(s4 + idx);
    }
#pragma unroll
    for (int i = 0; i < R; ++i) {
      ss = fmaf(v[i].x, v[i].x, ss); ss = fmaf(v[i].y, v[i].y, ss); ss = fmaf(v[i].z, v[i].z, ss); ss = fmaf(v[i].w, v[i].w, ss);
    }
    if (raw_out) {
      float4 *r4 = reinterpret_cast<float4 *>(raw_out);
#pragma unroll
      for (int i = 0; i < R; ++i) { const int idx = st + kStagerThreads * i; if (idx < n4) r4[idx] = v[i]; }
    }
    ss = warp_sum(ss);
    if ((st & 31) == 0) sred[st >> 5] = ss;
    stager_sync();
    const float r = 1.0f / sqrtf((sred[0] + sred[1]) / (float)K + eps);
#pragma unroll
    for (int i = 0; i < R; ++i) {
      const int idx = st + kStagerThreads * i;
      if (idx < n4) {
        const uint2 g = gs[idx];                 // written by this lane
        float4 o;
        o.x = v[i].x * r * bf16_lo(g.x); o.y = v[i].y * r * bf16_hi(g.x);
        o.z = v[i].z * r * bf16_lo(g.y); o.w = v[i].w * r * bf16_hi(g.y);
        d4[idx] = o;
      }
    }
    stager_sync();                               // sred is rewritten by the next normalising visit
  } else {                                       // wide models: raw copy, then scale in place
    dep_wait(dp, st);
    const uint2 *g2 = reinterpret_cast<const uint2 *>(gain);
    float ss = 0.f;
    for (int idx = st; idx < n4; idx += kStagerThreads) {
      const float4 v = __ldcg(s4 + idx);
      d4[idx] = v;
      if (raw_out) reinterpret_cast<float4 *>(raw_out)[idx] = v;
      ss = fmaf(v.x, v.x, ss); ss = fmaf(v.y, v.y, ss); ss = fmaf(v.z, v.z, ss); ss = fmaf(v.w, v.w, ss);
    }
    ss = warp_sum(ss);
    if ((st & 31) == 0) sred[st >> 5] = ss;
    stager_sync();
    const float r = 1.0f / sqrtf((sred[0] + sred[1]) / (float)K + eps);
    for (int idx = st; idx < n4; idx += kStagerThreads) {
      float4 v = d4[idx];
      const uint2 g = __ldg(g2 + idx);
      v.x = v.x * r * bf16_lo(g.x); v.y = v.y * r * bf16_hi(g.x);
      v.z = v.z * r * bf16_lo(g.y); v.w = v.w * r * bf16_hi(g.y);
      d4[idx] = v;
    }
    stager_sync();
  }
  for (int i = K + st; i < kpad; i += kStagerThreads) dst[i] = 0.f;
}

__device__ __forceinline__ void red_release_cta_shared_add(unsigned int *p, unsigned int v) {
  asm volatile("red.release.cta.shared::cta.add.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned int ld_acquire_cta_shared(const unsigned int *p) {
  unsigned int v;
  asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}

__global__ void __launch_bounds__(kThreads2, 1) k_spd_cycle2(DevPtrs P, MegaLayout ML, const __grid_constant__ CUtensorMap kv_tmap) {
  extern __shared__ __align__(1024) uint8_t smem[];   // ring slots must be 1024-byte aligned (128-byte swizzle)
  uint8_t *ring = smem;                                                  // kStages * 16 KB
  float *xs = reinterpret_cast<float *>(smem + kStages * kTileBytes);    // 2 buffers of kXHalf floats
  uint64_t *full = reinterpret_cast<uint64_t *>(xs + kXFloats);          // [kStages]
  uint64_t *empty = full + kStages;                                      // [kStages]
  uint64_t *xfull = empty + kStages;                                     // [2] buffer b holds the visit's inputs
  uint64_t *xempty = xfull + 2;                                          // [2] the consumers are done with buffer b
  float *red = reinterpret_cast<float *>(xempty + 2);                    // [16]
  float *cbest_v = red + 16;                                             // [2][8]
  int *cbest_i = reinterpret_cast<int *>(cbest_v + 16);                  // [2][8]
  int *meta = cbest_i + 16;                                              // [kStages] slot tags (+ padding to 16)
  float *gpart = reinterpret_cast<float *>(meta + 16);                   // [2][8][8] warp partials of a unit
  float *sred = gpart + 128;                                             // [3] stager: warp sums of squares
  unsigned int *vdone = reinterpret_cast<unsigned int *>(sred + 3);      // [1] visits the consumers have finished
  unsigned short *dnl = reinterpret_cast<unsigned short *>(sred + 4);    // [kMaxChains][kDnCap] W_down units this CTA claimed
  Sched2 *Sp = reinterpret_cast<Sched2 *>(dnl + kMaxChains * kDnCap);

  const Dims &D = P.dim;
  const int cta = blockIdx.x, ncta = gridDim.x;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int np = 2 + kPhasesPerPass * D.per;
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
    Sched2 &S = *Sp;
    S.mode = st->mode; S.c = st->c;
    int act[kMaxStages];
    int a = 0;
    S.occ_mask = 0u;
    for (int k = 0; k < D.n; ++k) {
      S.pos[k] = st->pos[k]; S.hbuf[k] = st->hbuf[k];
      if (st->occ[k]) { S.occ_mask |= 1u << k; act[a++] = k; }
    }
    S.n_act = a;
    S.p_new = st->occ[0] ? st->pos[0] : -1;
    S.run_pdm = st->mode == MODE_SPD && !P.paper_pdm;
    S.run_verify = (st->mode == MODE_SPD && st->occ[D.n - 1]) || st->mode == MODE_PREFILL_FINAL;
    // Groups: shares r = cta mod a; the a shares (= active stages, ascending) are cut into ng = ceil(a / chains) runs of
    // a / ng or a / ng + 1 consecutive shares, and the CTAs of a run serve all of its stages as chains.  A dependent visit
    // of a chain is m - 1 visits behind its producer: with m = 4 the barrier latency (skew of one visit + release /
    // acquire + the stager's copy, ~8 us) is covered even by the short visits (ATTN, O, DOWN parts: 5-6 us each).
    S.m = 0; S.gsize = 0; S.lead = 0; S.exit_gsize = 0;
    if (a > 0) {
      const int cm = max(1, min(ML.chains, kMaxChains));
      const int ng = (a + cm - 1) / cm, gb = a / ng, grem = a % ng;
      const int r = cta % a;
      int g = 0, first = 0;
      while (first + gb + (g < grem ? 1 : 0) <= r) { first += gb + (g < grem ? 1 : 0); ++g; }
      const int last = first + gb + (g < grem ? 1 : 0) - 1;               // shares (= chains) of this CTA's group
      S.m = last - first + 1;
      for (int j = 0; j < S.m; ++j) {
        const int k = act[first + j];
        S.stage[j] = k;
        S.attn_ns[j] = (S.pos[k] + kAttnSplit) / kAttnSplit;               // ceil((pos + 1) / split)
        S.attn_total[j] = D.Hkv * S.attn_ns[j];
        S.attn_nonfinal[j] = D.Hkv * (S.attn_ns[j] - 1);
      }
      for (int rr = first; rr <= last; ++rr) S.gsize += ncta / a + (rr < ncta % a ? 1 : 0);
      S.lead = cta == first;                                               // the lowest CTA of the group
      if (st->occ[D.n - 1]) {                                              // stage n - 1 = act[a - 1]: the last group
        const int f2 = a - (gb + (ng - 1 < grem ? 1 : 0));
        for (int rr = f2; rr <= a - 1; ++rr) S.exit_gsize += ncta / a + (rr < ncta % a ? 1 : 0);
      }
    }
    S.pdm_slot = cta % D.n;
    S.pdm_idx = cta / D.n;
    for (int s = 0; s < kStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); }
    for (int b = 0; b < 2; ++b) { mbar_init(&xfull[b], kStagerThreads); mbar_init(&xempty[b], 1); }
    *vdone = 0u;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const Sched2 &S = *Sp;
  const unsigned long long launch = ld_acquire_u64(bar_launch);
  if (cta == 0 && tid == 0) controller_begin(P);   // writes only fields no other CTA reads in this kernel
  if (P.prof_on && tid == 0 && cta < kProfCtas) {
    unsigned long long *pr = P.prof + ((size_t)cta * kProfPhases + (kProfPhases - 1)) * kProfStamps;
    pr[0] = (unsigned long long)clock64(); pr[1] = globaltimer_ns();
  }
  __syncthreads();
  const int RPS = kTileBytes / (D.hd * 2);         // K/V rows per ring slot
  const int m = S.m;
  const int nv = 2 + (m > 0 ? kPhasesPerPass * D.per * m : 0);

  if (warp == 8) {
    // =========================== producer: claim and stream every visit's work, running ahead =====
    if (lane == 0) {
      uint64_t pol_w, pol_kv;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_w));
      asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol_kv));
      uint32_t seq = 0;
      int dn_cnt[kMaxChains];
      for (int j = 0; j < kMaxChains; ++j) dn_cnt[j] = 0;
      for (int v = 0; v < nv; ++v) {
        const Visit x = visit_decode(v, nv, np, m);
        const Work2 w = work_desc(x, S, ML, D, P.claim);
        if (x.kind == 1 && x.type == P2_DNB) {
          bool first = true;
          for (int i = 0; i < dn_cnt[x.j] && w.nc > 0; ++i) {     // the units of this CTA's DOWN_A visit, in the same order
            const int u = dnl[x.j * kDnCap + i];
            const uint8_t *src = w.base + (unsigned long long)u * w.nc * kTileBytes;
            for (int t = 0; t < w.nc; ++t, ++seq, src += kTileBytes) {
              uint32_t slot = seq % kStages, itn = seq / kStages;
              mbar_wait(&empty[slot], (itn & 1) ^ 1);
              meta[slot] = u;
              mbar_expect_tx(&full[slot], kTileBytes);
              tma_load_1d(ring + (size_t)slot * kTileBytes, src, kTileBytes, &full[slot], pol_w);
              if (first) { vstamp(P, cta, v, 3); first = false; }
            }
          }
          vstamp(P, cta, v, 4);
        } else if (w.job >= 0 && w.U > 0) {
          unsigned int next = atomicAdd(w.ctr, 1u);
          if (x.kind == 1 && x.type == P2_ATTN) {
            const int k = w.job;
            bool first = true, kv_ready = false;
            while (next < (unsigned int)w.U) {
              AttnItem it;
              attn_decode(k, S.attn_ns[x.j], S.attn_nonfinal[x.j], S.pos[k], (int)next, it);
              const int item = (int)next;
              next = atomicAdd(w.ctr, 1u);
              auto wait_qkv = [&]() {   // this pass's QKV phase of the group: q of the stage and the row it appended
                if (!kv_ready) {
                  const unsigned int target = (unsigned int)(x.p - 1) * (unsigned int)S.gsize;
                  while (ld_acquire_u32(gbar + 32 * k) < target) {}
                  fence_proxy_async();
                  kv_ready = true;
                }
              };
              if (item >= S.attn_nonfinal[x.j]) wait_qkv();   // the last split holds the appended row
              const int layer = k * D.per + x.pass;
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
                  if (first) { vstamp(P, cta, v, 3); first = false; }
                }
              }
              {   // the item's q (G heads, fp32, contiguous) rides the ring too: no consumer ever waits on an L2 round trip
                wait_qkv();
                const int G = D.Hq / D.Hkv;
                const uint32_t slot = seq % kStages, itn = seq / kStages;
                const uint32_t bytes = (uint32_t)(G * D.hd * 4);
                mbar_wait(&empty[slot], (itn & 1) ^ 1);
                meta[slot] = item;
                mbar_expect_tx(&full[slot], bytes);
                tma_load_1d(ring + (size_t)slot * kTileBytes, P.q + ((size_t)k * D.Hq + (size_t)it.kvh * G) * D.hd, bytes, &full[slot],
                            pol_kv);
                ++seq;
              }
            }
          } else {
            bool first = true;
            const bool is_dna = x.kind == 1 && x.type == P2_DNA;
            int ndn = 0;
            while (next < (unsigned int)w.U) {
              const int u = (int)next;
              if (is_dna) dnl[x.j * kDnCap + ndn++] = (unsigned short)u;
              next = (is_dna && ndn == kDnCap) ? (unsigned int)w.U   // full list: leave the rest to the group
                                               : atomicAdd(w.ctr, 1u);   // claim ahead: its latency hides behind this unit's tiles
              const uint8_t *src = w.base + (unsigned long long)u * w.nc * kTileBytes;
              for (int i = 0; i < w.nc; ++i, ++seq, src += kTileBytes) {
                uint32_t slot = seq % kStages, itn = seq / kStages;
                mbar_wait(&empty[slot], (itn & 1) ^ 1);
                meta[slot] = u;
                mbar_expect_tx(&full[slot], kTileBytes);
                tma_load_1d(ring + (size_t)slot * kTileBytes, src, kTileBytes, &full[slot], pol_w);
                if (first) { vstamp(P, cta, v, 3); first = false; }
              }
            }
            if (is_dna) dn_cnt[x.j] = ndn;
          }
          vstamp(P, cta, v, 4);
        }
        // END slot: closes the visit for the consumers
        uint32_t slot = seq % kStages, itn = seq / kStages;
        mbar_wait(&empty[slot], (itn & 1) ^ 1);
        meta[slot] = kEndMark;
        mbar_arrive(&full[slot]);
        ++seq;
      }
    }
  } else if (warp == 11) {
    // =========================== publisher: release the consumers' finished visits to the other CTAs =====
    // (one release at gpu scope after the consumers' CTA barrier + their release on `vdone`: cumulative over what that
    // ordered before it.  A release waits until the CTA's writes are visible, 2-3 us under the weight stream: here it
    // delays nobody.)
    if (lane == 0) {
      for (int v = 0; v < nv; ++v) {
        while (ld_acquire_cta_shared(vdone) <= (unsigned int)v) {}
        const Visit x = visit_decode(v, nv, np, m);
        if (m == 1 && !(x.kind == 1 && x.type == P2_DNA)) continue;   // one chain: released by the consumers (see below)
        if (x.kind == 2) red_release_add_u64(bar_count, 1ull);
        else if (x.kind == 0) { if (S.run_pdm) red_release_add_u32(pdm_done, 1u); }
        else red_release_add_u32(gbar + 32 * S.stage[x.j], 1u);
      }
    }
  } else if (warp > 8) {
    // =========================== stager: dependencies + activation vectors, one visit ahead =====
    const int st = tid - (kConsumerThreads + 32);
    for (int v = 0; v < nv; ++v) {
      const int b = v & 1, kk = v >> 1;
      if (kk >= 1) mbar_wait(&xempty[b], (kk - 1) & 1);     // the consumers are done with visit v - 2
      const Visit x = visit_decode(v, nv, np, m);
      // ---- the producers of this visit's inputs.  Chains are independent: a layer visit waits only for the previous
      //      phase of its own stage's group; the first O phase, the first to overwrite a residual stream, also waits until
      //      every CTA has read its pre-step PDM slot vector; the LM head waits for the exit stage's group and for the
      //      PDM partial products --------------------------------------------------------------------------------
      Dep dp;
      dp.c0 = dp.c1 = nullptr; dp.t0 = dp.t1 = 0u;
      if (x.kind == 2) {
        if (S.run_verify && S.exit_gsize > 0) { dp.c0 = gbar + 32 * (D.n - 1); dp.t0 = (unsigned int)(np - 2) * (unsigned int)S.exit_gsize; }
        if (S.run_pdm) { dp.c1 = pdm_done; dp.t1 = (unsigned int)ncta; }
      } else if (x.kind == 1) {
        // DOWN_B reads the second half of the SwiGLU vector (complete since GATEUP) and updates only rows this CTA updated
        // in DOWN_A: it waits for GATEUP (two phases back), not for DOWN_A
        const int back = x.type == P2_DNB ? 2 : 1;
        if (x.p >= 2) { dp.c0 = gbar + 32 * S.stage[x.j]; dp.t0 = (unsigned int)(x.p - back) * (unsigned int)S.gsize; }
        if (x.p == 1 + P2_O && S.run_pdm) { dp.c1 = pdm_staged; dp.t1 = (unsigned int)ncta; }
      }
      if (x.kind == 1 && x.type != P2_ATTN) {
        const int k = S.stage[x.j];
        const int layer = k * D.per + x.pass;
        float *dst = xs + b * kXHalf;
        if (x.type == P2_QKV || x.type == P2_GU) {
          const float *h = P.h + (size_t)S.hbuf[k] * D.d;
          const uint16_t *g = x.type == P2_QKV ? P.attn_norm[layer] : P.mlp_norm[layer];
          float *raw = nullptr;
          if (x.type == P2_QKV && S.lead) {        // NEXT-1: H^layer of the paper PDM's anchor set (the raw residual stream)
            const int ai = anchor_index(P, layer);
            if (ai >= 0 && S.pos[k] < D.max_seq) raw = P.anch + ((size_t)S.pos[k] * P.pdm_m + ai) * D.d;
          }
          float2 cs = make_float2(1.f, 0.f);       // RoPE table entry of the chain's position (C-2.14): the double-precision
          if (x.type == P2_QKV && st < D.hd / 2) { //   sincos (1-2 us for a 64-lane table) runs while the dependency is still open
            double s_, c_;
            sincos((double)S.pos[k] * P.inv_freq[st], &s_, &c_);
            cs = make_float2((float)c_, (float)s_);
          }
          stager_copy(dp, h, dst, D.d, ML.nc_d * kTileCols, g, D.eps, raw, sred, st);
          if (x.type == P2_QKV && st < D.hd / 2)   // stored behind the vector (the parked gains are dead: every stager thread
            reinterpret_cast<float2 *>(dst + ML.nc_d * kTileCols)[st] = cs;   // has passed stager_copy's last barrier)
          if (x.type == P2_QKV && S.lead && st == 0) {
            // causality / capacity precondition of the KV append, and the new length (one CTA per stage)
            const int pos = S.pos[k];
            if (P.len[layer] != pos || pos >= D.max_seq) P.st->err = 1;
            else P.len[layer] = pos + 1;
          }
        } else if (x.type == P2_O) {
          const int K = D.Hq * D.hd;
          stager_copy(dp, P.att + (size_t)k * K, dst, K, ML.nc_qd * kTileCols, nullptr, 0.f, nullptr, sred, st);
        } else {
          const int ka = min(ML.nc_fa * kTileCols, D.F);
          if (x.type == P2_DNA)
            stager_copy(dp, P.act + (size_t)k * D.F, dst, ka, ML.nc_fa * kTileCols, nullptr, 0.f, nullptr, sred, st);
          else if (ML.nc_f > ML.nc_fa)
            stager_copy(dp, P.act + (size_t)k * D.F + ka, dst, D.F - ka, (ML.nc_f - ML.nc_fa) * kTileCols, nullptr, 0.f, nullptr,
                        sred, st);
          else dep_wait(dp, st);
        }
      } else {
        dep_wait(dp, st);
      }
      mbar_arrive(&xfull[b]);                      // release: this thread's part of the buffer (and the dependency) is in place
    }
  } else {
    // =========================== consumers ======================================================
    uint32_t seq = 0;
    const int G = D.Hq / D.Hkv;
    for (int v = 0; v < nv; ++v) {
      const int b = v & 1;
      const Visit x = visit_decode(v, nv, np, m);
      mbar_wait(&xfull[b], (v >> 1) & 1);          // inputs staged, dependencies satisfied
      if (tid == 0) {
        vstamp(P, cta, v, 0);
        if (P.prof_on && cta < kProfCtas && v < kProfPhases - 1) P.prof[((size_t)cta * kProfPhases + v) * kProfStamps + 5] = globaltimer_ns();
      }
      const Work2 w = work_desc(x, S, ML, D, P.claim);
      float *xb = xs + b * kXHalf;
      if (x.kind == 1 && x.type == P2_ATTN) {
        const int j = x.j, k = S.stage[j];
        if (tid == 0) vstamp(P, cta, v, 1);
        // ---- split-KV decode attention (as in spd_mega.cu; scratch = this visit's buffer, q read per item) ----
        int *done_list = reinterpret_cast<int *>(xb + 10 * G * kAttnSplit);   // [kAttnDoneMax] item ids
        int *merge_cnt = done_list + kAttnDoneMax;                            // [1]
        int *merge_list = merge_cnt + 1;                                      // [kAttnDoneMax * 8] (item slot, head)
        int n_done = 0;
        bool more = true;
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
            attn_decode(k, S.attn_ns[j], S.attn_nonfinal[j], S.pos[k], item, it);
            const int nk = (it.rows + RPS - 1) / RPS;
            for (int jj = 1; jj <= 2 * nk; ++jj) mbar_wait(&full[(seq + jj) % kStages], ((seq + jj) / kStages) & 1);
            const int qslot = (int)((seq + 2 * nk) % kStages);      // K slots, V slots, then the q slot
            const float *qsm = reinterpret_cast<const float *>(ring + (size_t)qslot * kTileBytes);
            if (ML.attn_mma && it.rows == kAttnSplit) {
              if (G == 4) attn_item_mma<4>(P, it, ring, seq, xb, empty, nullptr, qsm, qslot);
              else if (G == 2) attn_item_mma<2>(P, it, ring, seq, xb, empty, nullptr, qsm, qslot);
              else attn_item_mma<1>(P, it, ring, seq, xb, empty, nullptr, qsm, qslot);
            } else if (D.hd == 128) attn_item_g<128>(P, it, ring, seq, nk, xb, empty, G, qsm, qslot);
            else attn_item_g<64>(P, it, ring, seq, nk, xb, empty, G, qsm, qslot);
            seq += 2 * nk + 1;
            if (tid == 0) done_list[n_done] = item;
            ++n_done;
          }
          if (n_done == kAttnDoneMax || (!more && n_done > 0)) {
            if (tid == 0) *merge_cnt = 0;
            __threadfence();                       // this CTA's partial outputs, before their completion counts
            consumer_sync();
            for (int e = tid; e < n_done * G; e += kConsumerThreads) {
              AttnItem it;
              attn_decode(k, S.attn_ns[j], S.attn_nonfinal[j], S.pos[k], done_list[e / G], it);
              const int hq = it.kvh * G + e % G;
              if (atomicAdd(&P.att_cnt[it.stage * D.Hq + hq], 1) == it.nsplit - 1) merge_list[atomicAdd(merge_cnt, 1)] = e;
            }
            consumer_sync();
            const int nm = *merge_cnt;
            if (nm > 0) {
              __threadfence();
              for (int mm = warp; mm < nm; mm += 8) {   // the last split of a q head to finish merges them (fixed split order)
                const int e = merge_list[mm];
                AttnItem it;
                attn_decode(k, S.attn_ns[j], S.attn_nonfinal[j], S.pos[k], done_list[e / G], it);
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
      } else if (x.kind == 1) {
        if (tid == 0) vstamp(P, cta, v, 1);
        const int t = x.type == P2_QKV ? PH_QKV : x.type == P2_O ? PH_O : x.type == P2_GU ? PH_GATEUP : PH_DOWN;
        gemv_stream(P, S, t, w.job, x.pass, w.nc, ring, full, empty, meta, xb, gpart, seq,
                    reinterpret_cast<const float2 *>(xb + ML.nc_d * kTileCols));   // QKV: the stager's RoPE table
        if (x.type == P2_QKV) fence_proxy_async();   // the appended K/V rows are read by TMA (async proxy) next
      } else {
        // ---- PDM phase / LM head: staged by the consumers themselves (whole buffer), as in spd_mega.cu ----
        const int k = w.job;
        if (k >= 0) {
          const int K = D.d;
          if (x.kind == 0) {
            // slot j = k: pre-step state of the token at depth j, else Hfin[p_new - j], else zero (Eq. 5)
            int q = S.p_new - k;
            const float *src = ((S.occ_mask >> k) & 1u) ? P.h + (size_t)S.hbuf[k] * D.d
                                                        : (q >= 0 ? P.hfin + (size_t)q * D.d : nullptr);
            if (src) stage_copy(src, xs, K);
            else for (int i = tid; i < K; i += kConsumerThreads) xs[i] = 0.f;
            consumer_sync();
            if (tid == 0) { __threadfence(); atomicAdd(pdm_staged, 1u); }   // the pre-step state has been read
            if (S.pdm_idx == 0)               // kept for the parity tests (SPD_DBG_PDM_FEAT)
              for (int i = tid; i < K; i += kConsumerThreads) P.feat[(size_t)k * D.d + i] = xs[i];
          } else {  // LM head: verify input at xs[0..d), PDM input at xs[kXHalf ..)
            if (S.run_verify) {
              const float *h = S.mode == MODE_PREFILL_FINAL ? P.hfin + (size_t)(S.c - 1) * D.d
                                                            : P.h + (size_t)S.hbuf[D.n - 1] * D.d;
              float ss = consumer_sum(stage_copy(h, xs, D.d), red);
              stage_scale(xs, P.final_norm, D.d, 1.0f / sqrtf(ss / (float)D.d + D.eps));
            }
            if (S.run_pdm) {
              float *xp = xs + kXHalf;
              float4 *xp4w = reinterpret_cast<float4 *>(xp);
              float ss = 0.f;
              for (int i = tid; i < (D.d >> 2); i += kConsumerThreads) {   // u = sum_j W_p[:, block j] f_j, j ascending
                float4 u = make_float4(0.f, 0.f, 0.f, 0.f);
                for (int jj = 0; jj < D.n; ++jj) {
                  float4 vv = __ldcg(reinterpret_cast<const float4 *>(P.pdm_part + (size_t)jj * D.d) + i);
                  u.x += vv.x; u.y += vv.y; u.z += vv.z; u.w += vv.w;
                }
                xp4w[i] = u;
                if (cta == 0) reinterpret_cast<float4 *>(P.pdm_u)[i] = u;    // kept for the parity tests (SPD_DBG_PDM_PRENORM)
                ss = fmaf(u.x, u.x, ss); ss = fmaf(u.y, u.y, ss); ss = fmaf(u.z, u.z, ss); ss = fmaf(u.w, u.w, ss);
              }
              ss = consumer_sum(ss, red);
              stage_scale(xp, P.pdm_norm, D.d, 1.0f / sqrtf(ss / (float)D.d + D.eps));
            }
          }
          const int kpad = w.nc * kTileCols;
          for (int i = K + tid; i < kpad; i += kConsumerThreads) xs[i] = 0.f;
          if (x.kind == 2) for (int i = K + tid; i < kpad; i += kConsumerThreads) xs[kXHalf + i] = 0.f;
        }
        consumer_sync();
        if (tid == 0) vstamp(P, cta, v, 1);
        if (k < 0) {                               // nothing to stream: one END slot, read by every warp
          const uint32_t slot = seq % kStages;
          mbar_wait(&full[slot], (seq / kStages) & 1);
          __syncwarp();
          if (lane == 0) mbar_arrive(&empty[slot]);
          ++seq;
        } else if (x.kind == 2) {
          const bool do_v = S.run_verify, do_p = S.run_pdm;
          if (w.nc <= 4) head_stream<1>(P, w.nc, do_v, do_p, ring, full, empty, meta, xs, seq, cbest_v, cbest_i);
          else if (w.nc <= 8) head_stream<2>(P, w.nc, do_v, do_p, ring, full, empty, meta, xs, seq, cbest_v, cbest_i);
          else head_stream<3>(P, w.nc, do_v, do_p, ring, full, empty, meta, xs, seq, cbest_v, cbest_i);
          consumer_sync();
          if (tid < 2) {                           // CTA-level candidates -> global
            float bv = -INFINITY;
            int bi = 0x7fffffff;
            for (int ww = 0; ww < 8; ++ww)
              if (cand_better(cbest_v[tid * 8 + ww], cbest_i[tid * 8 + ww], bv, bi)) { bv = cbest_v[tid * 8 + ww]; bi = cbest_i[tid * 8 + ww]; }
            P.cand_val[tid * kMaxCand + cta] = bv;
            P.cand_idx[tid * kMaxCand + cta] = bi == 0x7fffffff ? -1 : bi;
          }
        } else {
          gemv_stream(P, S, PH_PDM, k, 0, w.nc, ring, full, empty, meta, xs, gpart, seq, nullptr);
        }
      }
      // ---- hand the buffer back to the stager and the visit's outputs to the publisher ------------------------
      if (tid == 0) vstamp(P, cta, v, 2);
      consumer_sync();
      if (tid == 0) {
        mbar_arrive(&xempty[b]);
        red_release_cta_shared_add(vdone, 1u);     // the publisher takes it from here ...
        if (m == 1 && !(x.kind == 1 && x.type == P2_DNA)) {
          // ... except with a single chain (one active stage): the next visit depends on this one (DOWN_B on DOWN_A excepted),
          // so nothing is gained by the hand-over
          if (x.kind == 2) red_release_add_u64(bar_count, 1ull);
          else if (x.kind == 0) { if (S.run_pdm) red_release_add_u32(pdm_done, 1u); }
          else red_release_add_u32(gbar + 32 * S.stage[x.j], 1u);
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
    for (int i = tid; i < np * kMaxStages; i += kThreads2) P.claim[i] = 0u;  // every producer is done claiming
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

// ------------------------------------------------------------------ host side ------------------
static int mega2_smem_bytes() {
  return kStages * kTileBytes + kXFloats * 4 + 2 * kStages * 8 + 4 * 8 + 16 * 4 + 32 * 4 + 16 * 4 + 128 * 4 +
         4 * 4 + kMaxChains * kDnCap * 2 + (int)sizeof(Sched2);   // sred[3] + vdone, dnl
}

// Shares the one-chain engine's plan (repacked weights, layout, K/V tensor map); adds only the launch geometry.
int mega2_create(const DevPtrs &P, const MegaPlan &base, Mega2Plan *plan) {
  const Dims &D = P.dim;
  plan->available = 0;
  if (!base.available) return -1;
  MegaLayout ML;
  memcpy(&ML, base.layout, sizeof ML);
  const int G = D.Hq / D.Hkv, qd = D.Hq * D.hd;
  // every visit's vector and the attention scratch (+ its completion lists) must fit one 24 KB buffer; the claim /
  // profile tables hold 2 + 6 L/n phases
  int sms = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (kDnCap * (sms / kMaxStages) < ML.u_dn || ML.u_dn > 65535) return -1;   // DOWN_A claims are capped per CTA (kDnCap)
  if (ML.nc_d * kTileCols + 2 * 64 > kXHalf || D.hd > 128 || qd > kXHalf || ML.nc_fa * kTileCols > kXHalf || G > 4 ||
      10 * G * kAttnSplit + kAttnDoneMax * 9 + 1 > kXHalf || 2 + kPhasesPerPass * D.per > kClaimPhases) return -1;
  const int smem = mega2_smem_bytes();
  if (cudaFuncSetAttribute(k_spd_cycle2, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  int occ = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_spd_cycle2, kThreads2, smem) != cudaSuccess || occ < 1) {
    cudaGetLastError();
    return -1;
  }
  plan->smem_bytes = smem;
  plan->chains = D.n > 8 ? 3 : kMega2DefaultChains;   // measured: 2 at n = 4 and 8, 3 at n = 16
  plan->available = 1;
  return 0;
}

int mega2_enqueue_step(const DevPtrs &P, const MegaPlan &base, const Mega2Plan &plan, cudaStream_t sm, long long *launches) {
  if (!plan.available || !base.available) return -1;
  MegaLayout ML;
  memcpy(&ML, base.layout, sizeof ML);
  ML.chains = plan.chains;
  DevPtrs Pc = P;
  CUtensorMap tm;
  memcpy(&tm, base.kv_tmap, sizeof tm);
  void *args[] = {(void *)&Pc, (void *)&ML, (void *)&tm};
  cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_spd_cycle2, dim3(base.n_cta), dim3(kThreads2), args,
                                              (size_t)plan.smem_bytes, sm);
  if (launches) *launches += 1;
  return e == cudaSuccess ? 0 : -1;
}

}  // namespace spd
