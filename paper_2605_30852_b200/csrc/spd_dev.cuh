// spd_dev.cuh — device-side state, buffer map and small helpers shared by the library's kernels.
// (CUDA path only; nothing here is used by, or taken from, oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace spd {

constexpr int kMaxStages = 32;
constexpr int kAttnSplit = 128;     // KV rows per attention split — fixed, so a token's result never
                                    // depends on n, slot, fill or history (batch invariance)
constexpr int kResultRing = 1024;   // device ring of step results (spd_step_many batch limit)
constexpr int kMaxCand = 256;       // per-CTA argmax candidates of the LM-head pass
// Synchronisation words of the fused engine (DevPtrs::bar), one 128-byte line each: [0] finished-CTA count,
// [32] launch count, [kBarGroup0 + 32 k] arrivals of stage k's CTA group, then two PDM counters.
constexpr int kBarGroup0 = 64;
constexpr int kBarWords = kBarGroup0 + 32 * (kMaxStages + 2);
// Optional per-phase clock stamps of the fused kernel (SPD_OPT_PHASE_PROFILE): [cta][phase][stamp]
constexpr int kProfCtas = 160, kProfPhases = 168, kProfStamps = 6;
constexpr int kClaimPhases = 200;   // rows of the work-claim table: 2 + 6 * (L / n) phases of a cycle (engine 2 at L = 32, n = 1: 194)

// Sampling verification ("under sampling we apply standard rejection
// sampling", :141 "T=1 ... top-k=50 and top-p=1.0"; readings S-1..S-9 of DESIGN.md).
constexpr int kMaxTopK = 64;        // largest top_k
constexpr int kSampCap = 2048;      // survivors of the threshold scan (above that: exact k-round selection)

// A filtered distribution: support in ascending token id, fp32 probabilities (S-2).
struct SampleDist {
  int32_t k;
  int32_t id[kMaxTopK];
  float p[kMaxTopK];
};
// What the sampler of the last cycle saw and decided (SPD_DBG_SAMPLE).
struct SampleRecord {
  SampleDist draft;                  // Q_t of this cycle's PDM
  SampleDist target;                 // P of this cycle's exit (or of the prefill's final head)
  float u_draft, u_accept, u_resid;  // S-6 uniforms (-1: not drawn)
  int32_t succ_token;                // the judged token, its stored draft probability and its target probability
  float succ_q, succ_p;
  int32_t exact_rounds;              // how many of the two selections took the exact k-round path
  int32_t prefiltered;               // ... and how many used the head pass's threshold list (no scan)
};
struct SampleState {
  int32_t on, top_k;
  float temperature;
  int32_t pad_;
  unsigned long long seed;
  int32_t pre_cnt[2];                // entries the head pass listed this cycle (0 verify, 1 PDM); may exceed kSampCap
  float tau_guess[2];                // the list threshold of the next head pass (+inf: none yet)
  SampleDist q[kMaxStages];          // indexed by hidden-buffer id: the distribution the token living there was drawn from
  SampleRecord rec;
};

enum Mode : int32_t { MODE_IDLE = 0, MODE_SPD = 1, MODE_PREFILL = 2, MODE_PREFILL_FINAL = 3 };

struct StepResult {
  int32_t step_index, fill, exited, accepted, emitted_token, draft_token, draft_forced, discarded,
      committed_len;
};

// Device-resident controller state: the in-flight pipeline indexed by depth k (= stage), the
// committed length, counters and the forced-acceptance rule.  Updated only by the step's last kernel,
// so steps can be enqueued back to back without the host.
struct StepState {
  int32_t mode;
  int32_t c;                         // committed length
  int32_t occ[kMaxStages];           // stage k holds a token
  int32_t pos[kMaxStages];
  int32_t tok[kMaxStages];
  int32_t hbuf[kMaxStages];          // which hidden-state buffer that token lives in
  long long K, N;                    // cycles / emitted tokens since prefill
  int32_t prompt_len;
  int32_t forced_on, n_truth;
  unsigned long long forced_thresh, forced_seed;
  int32_t pf_next, pf_n;             // prefill progress
  int32_t err;                       // sticky device-side check (causality / capacity)
  // per-step scratch written by the step's first kernel
  int32_t run_pdm, run_verify, fill, p_new, forced_now;
  int32_t pad_;
};

struct Dims {
  int32_t d, L, n, Hq, Hkv, hd, F, V, max_seq, per;   // per = L / n
  float eps;
};

// Everything a kernel needs, passed by value.
struct DevPtrs {
  Dims dim;
  StepState *st;
  int32_t *len;                      // [L] valid KV rows
  float *h;                          // [n][d]   hidden state buffers (indexed by hbuf)
  float *x;                          // [n][d]   normed activations
  float *act;                        // [n][F]   SwiGLU output silu(gate)*up
  float *q;                          // [n][Hq*hd]
  float *kvtmp;                      // [n][2*Hkv*hd] fp32 k, v before RoPE/rounding (reference engine)
  float *att;                        // [n][Hq*hd]
  float *part_o;                     // [n][Hq][nsplit][hd]
  float2 *part_ml;                   // [n][Hq][nsplit]
  int32_t *att_cnt;                  // [n][Hq] split-completion counters (fused engine)
  float *feat;                       // [n][d]   PDM slot vectors
  float *pdm_part;                   // [n][d]   per-slot partial products of W_p (fused engine)
  float *pdm_u;                      // [d]
  float *xv, *xp;                    // [d] verify / PDM head inputs
  float *logits_v, *logits_p;        // [V]
  float *cand_val;                   // [2][kMaxCand]
  int32_t *cand_idx;                 // [2][kMaxCand]
  float2 *rope;                      // [n][hd/2] (cos, sin) for this step's positions
  double *inv_freq;                  // [hd/2] base^(-2i/hd), computed on the host in double
  float *hfin;                       // [max_seq][d]
  int32_t *truth;                    // [max_seq]
  int32_t *pf_tokens;                // [max_seq]
  StepResult *results;               // [kResultRing]
  unsigned long long *cycle_ts;      // [kResultRing][2] %globaltimer (ns) when the cycle's controller began / ended, filed like results
  unsigned int *bar;                 // grid-barrier words (fused engine)
  unsigned int *claim;               // [kClaimPhases][kMaxStages] work-claim counters of one cycle (fused engine)
  uint16_t *kv;                      // K/V cache
  const uint16_t *embed, *final_norm, *pdm_proj, *pdm_norm;
  const uint16_t *const *attn_norm, *const *wq, *const *wk, *const *wv, *const *wo, *const *mlp_norm,
      *const *w_gate, *const *w_up, *const *w_down;   // device arrays of [L] device pointers
  int32_t debug_logits;
  int32_t sampling;                  // kernel parameter: 1 = sampling verification (the head keeps full logit vectors)
  SampleState *samp;
  float *samp_val;                   // [kSampCap] survivors of the top-k threshold scan
  int32_t *samp_idx;                 // [kSampCap]
  float *pre_val;                    // [2][kSampCap] logits >= tau_guess listed by the fused head pass
  int32_t *pre_idx;                  // [2][kSampCap]
  // the paper's Pipeline Draft Module (spd_pdm.cu, NEXT-1); paper_pdm == 0: the simplified PDM of BASELINE.json
  int32_t paper_pdm;
  int32_t pdm_m;                     // anchors
  int32_t pdm_anchor[8];             // B = [0, L/4, L/2, 3L/4, L-1]
  float *anch;                       // [max_seq][m][d] H_pos^{b_i}: the residual stream entering layer b_i
  int32_t *pdm_draft;                // the token the paper's PDM drafted for this cycle
  // batched prefill scratch (spd_prefill.cu), sized for pf_chunk tokens
  float *pf_H;                       // [pf_chunk][d] residual streams of the chunk
  float *pf_Q;                       // [pf_chunk][Hq*hd] q after RoPE
  float *pf_Y;                       // [pf_chunk][max(Hq*hd + 2 Hkv*hd, 2 F, d)] GEMM output
  uint16_t *pf_x3;                   // [3][pf_chunk * max(d, Hq*hd, F)] bf16 hi / mid / lo parts of the GEMM input
  size_t pf_plane;                   // elements per part
  int32_t pf_chunk;
  int32_t nsplit_max;
  unsigned long long *prof;          // [kProfCtas][kProfPhases][kProfStamps] clock stamps (fused engine)
  int32_t prof_on;
};

__host__ __device__ inline size_t kv_head_stride(const Dims &d) { return (size_t)d.max_seq * d.hd; }
// K (which=0) or V (which=1) rows of (layer, kv head): [max_seq][hd] bf16
__host__ __device__ inline size_t kv_offset(const Dims &d, int layer, int which, int kvh) {
  return (((size_t)layer * 2 + which) * d.Hkv + kvh) * kv_head_stride(d);
}

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }
__device__ __forceinline__ float bf16_to_f32(uint16_t b) { return __uint_as_float((uint32_t)b << 16); }
// fp32 -> bf16 round-to-nearest-even (finite values)
__device__ __forceinline__ uint16_t f32_to_bf16(float f) {
  uint32_t u = __float_as_uint(f);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

// Anchor index of `layer` in the paper PDM's anchor set, or -1.
__device__ __forceinline__ int anchor_index(const DevPtrs &P, int layer) {
  if (!P.paper_pdm) return -1;
  for (int i = 0; i < P.pdm_m; ++i)
    if (P.pdm_anchor[i] == layer) return i;
  return -1;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__device__ __forceinline__ unsigned long long splitmix64(unsigned long long x) {
  unsigned long long z = x + 0x9e3779b97f4a7c15ull;
  z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
  z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
  return z ^ (z >> 31);
}

// (value, index) ordering of the greedy argmax: larger value wins, equal values -> lower index.
__device__ __forceinline__ bool cand_better(float v, int i, float bv, int bi) {
  return v > bv || (v == bv && i < bi);
}

}  // namespace spd
