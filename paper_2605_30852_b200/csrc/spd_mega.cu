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
#include "spd_mega_dev.cuh"

namespace spd {

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
              const uint8_t *src = w.base + (unsigned long long)u * w.nc1 * kTileBytes;
              for (int i = 0; i < w.nc; ++i, ++seq, src += kTileBytes) {
                if (i == w.nc1) src = w.base2 + (unsigned long long)u * (w.nc - w.nc1) * kTileBytes;   // W_down: second K part
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
  ML->chains = 0;
  ML->nc_fa = (ML->nc_f + 1) / 2;                  // W_down as two K parts (spd_mega_dev.cuh)
  ML->off_dnb = ML->off_dn + (unsigned long long)ML->u_dn * ML->nc_fa * kTileBytes;
  ML->layer_bytes = b_qkv + b_o + b_gu + b_dn;
  ML->pdm_job_bytes = (unsigned long long)ML->u_pdm * ML->nc_d * kTileBytes;
  ML->off_pdm = ML->layer_bytes * D.L;
  ML->off_head = ML->off_pdm + ML->pdm_job_bytes * D.n;
  *total = ML->off_head + (unsigned long long)ML->u_head * ML->nc_d * kTileBytes;
}

static bool mega_supported(const Dims &D) {
  int qd = D.Hq * D.hd;
  int G = D.Hq / D.Hkv;
  // 2 + 5 * (L / n) phases must fit the claim-counter table (P.claim is [kClaimPhases][kMaxStages]) and the profile table
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
    {   // W_down: columns [0, ka) and [ka, F) as two unit arrays
      const int ka = ML.nc_fa * kTileCols < D.F ? ML.nc_fa * kTileCols : D.F;
      k_repack<<<RB, RT, 0, stream>>>((uint16_t *)(lb + ML.off_dn), ML.u_dn, ML.nc_fa, RM_PLAIN, src[8][l], nullptr, nullptr,
                                      D.d, 0, 0, ka, D.F, 0, D.hd);
      if (ML.nc_f > ML.nc_fa)
        k_repack<<<RB, RT, 0, stream>>>((uint16_t *)(lb + ML.off_dnb), ML.u_dn, ML.nc_f - ML.nc_fa, RM_PLAIN, src[8][l], nullptr,
                                        nullptr, D.d, 0, 0, D.F - ka, D.F, ka, D.hd);
    }
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
