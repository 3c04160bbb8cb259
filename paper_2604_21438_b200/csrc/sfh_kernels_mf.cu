// sfh_kernels_mf.cu — the stage kernels (sfh_stage.cuh) instantiated WITH mass-flux export: every walker also
// writes the mass flux of its faces to StageParams::mf, which the passive-scalar kernels consume (eq. 12-13,
// PAPER.md:80-88; reading R32).  A translation unit of its own so that the two sets compile in parallel.
#include "sfh_stage.cuh"

namespace sfh {

cudaError_t configure_stage_kernels_mf() { return configure_stage_kernels<true>(); }

cudaError_t launch_stage_mf(int stage, const TensorMaps& tm, const StageParams& p, int sms, cudaStream_t st) {
  return launch_stage_impl<true>(stage, tm, p, sms, st);
}

}  // namespace sfh
