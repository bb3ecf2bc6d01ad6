// spd_engine.h — host-side entry points of the engines (internal to the library).
#pragma once
#include "spd_dev.cuh"

namespace spd {

// Reference engine: enqueue all kernels of one cycle (main stream + PDM branch on `sp`).
int ref_enqueue_step(const DevPtrs &P, cudaStream_t sm, cudaStream_t sp, cudaEvent_t ev_fork, cudaEvent_t ev_join,
                     long long *launches);

// Fused persistent engine (spd_mega.cu).
struct MegaPlan {
  const uint16_t *repack;   // streaming layout of all layer weights + W_p (device)
  int n_cta;                // persistent grid size (one CTA per SM)
  int smem_bytes;
  int available;
  unsigned long long layout[24];   // opaque MegaLayout (offsets of the repacked matrices)
  alignas(64) unsigned char kv_tmap[128];   // CUtensorMap over the K/V cache (128-byte-swizzled 64 x 64 boxes)
  int has_kv_tmap;          // 0: the driver entry point is missing -> attention stays on the scalar path
};
size_t mega_repack_bytes(const Dims &D);
// src: the nine host tables of per-layer device pointers in spd_weights order.  Returns 0 on success.
int mega_create(const DevPtrs &P, const uint16_t *const *const *src, void *repack, size_t repack_bytes,
                cudaStream_t stream, MegaPlan *plan);
int mega_enqueue_step(const DevPtrs &P, const MegaPlan &plan, cudaStream_t sm, long long *launches);

// Fused persistent engine with multiplexed stage chains (spd_mega2.cu): the same repacked weights, layout and K/V tensor map
// (MegaPlan), its own launch geometry.
#ifndef SPD_DEFAULT_FUSED_ENGINE
#define SPD_DEFAULT_FUSED_ENGINE 2
#endif
constexpr int kMega2DefaultChains = 2, kMega2MaxChains = 4;
struct Mega2Plan {
  int smem_bytes;
  int available;
  int chains;               // stage chains per CTA (SPD_OPT_CHAINS)
};
int mega2_create(const DevPtrs &P, const MegaPlan &base, Mega2Plan *plan);
int mega2_enqueue_step(const DevPtrs &P, const MegaPlan &base, const Mega2Plan &plan, cudaStream_t sm, long long *launches);


// Batched tensor-core prefill (spd_prefill.cu).
constexpr int kPrefillChunk = 1024;      // prompt tokens per pass over the layers (scratch is sized for it)
constexpr int kPrefillMaxLayers = 128;
struct PrefillPlan {
  int available;
  const uint16_t *w[9][kPrefillMaxLayers];   // host copy of the per-layer device pointers, spd_weights order
};
bool prefill_supported(const Dims &D);
int prefill_chunk_tokens(const Dims &D);
int prefill_create(const DevPtrs &P, const uint16_t *const *const *src, PrefillPlan *plan);
// Positions [0, n_tokens) of P.pf_tokens through all layers: K/V rows appended, Hfin written.  Returns 0 on success.
int prefill_run(const DevPtrs &P, const PrefillPlan &plan, int n_tokens, cudaStream_t st, long long *launches);
int prefill_pdm_rows(const DevPtrs &P, const uint16_t *const (*w)[kPrefillMaxLayers], int n_layers, uint16_t *pdm_kv,
                     const uint16_t *fc_full, int n_tokens, cudaStream_t st, long long *launches);
int skinny_gemm(const uint16_t *x3, size_t plane, int K, int NB, const uint16_t *const *w, const int *w_rows, int nseg,
                float *part, size_t part_floats, const int *rows_ptr, int rows_fixed, float *dst, int ldd, int residual,
                cudaStream_t st, long long *launches, int *ksplit_out = nullptr);
int prefill_op_gemm(const float *x, const uint16_t *w, int M, int N, int K, float *y, void *scratch, cudaStream_t st);


// The paper's Pipeline Draft Module (spd_pdm.cu).
constexpr int kPdmMaxRows = 40;          // >= kMaxStages + 1 rows per draft (n + 1)
struct PdmPlan;
}  // namespace spd
struct spd_pdm_weights;
namespace spd {
int pdm_anchor_set(int L, int32_t *b);
size_t pdm_kv_bytes(const Dims &D, int Ls);
size_t pdm_work_bytes(const Dims &D, int Ls, int Vs);
PdmPlan *pdm_create(DevPtrs *P, const ::spd_pdm_weights *w, void *kv, void *work, cudaStream_t st);
void pdm_destroy(PdmPlan *plan);
int pdm_enqueue_draft(const DevPtrs &P, const PdmPlan *pl, cudaStream_t st, long long *launches);
int pdm_prefill(const DevPtrs &P, const PdmPlan *pl, int n_tokens, int batched, cudaStream_t st, long long *launches);
int pdm_rollback(const PdmPlan *pl, int new_len, cudaStream_t st);
int pdm_debug_read(const DevPtrs &P, const PdmPlan *pl, int what, int index, void *out, size_t bytes);

}  // namespace spd
