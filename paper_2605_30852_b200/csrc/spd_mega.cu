// spd_mega.cu — fused persistent engine (placeholder until the kernel lands: reports "not available",
// the library then runs the reference engine).
#include "spd_engine.h"

namespace spd {
size_t mega_repack_bytes(const Dims &) { return 256; }
int mega_create(const DevPtrs &, const uint16_t *const *const *, void *, size_t, cudaStream_t, MegaPlan *plan) {
  if (plan) plan->available = 0;
  return -1;
}
int mega_enqueue_step(const DevPtrs &, const MegaPlan &, cudaStream_t, long long *) { return -1; }
}  // namespace spd
