// fused.cu -- variant 1 of K2: the fused sliding-window collide-stream kernel (placeholder
// until the kernel lands; the two-pass variant in collide.cu is the default meanwhile).
#include "d3q27.cuh"

namespace hhrr {
cudaError_t launch_fused(hhrr_lattice* L, const PhysF& ph, const BodiesF& bo) {
  (void)L; (void)ph; (void)bo;
  return cudaErrorNotSupported;
}
}  // namespace hhrr
