// sfh_kernels.cu — host side of the stage kernels (sfh_stage.cuh): the instantiations WITHOUT mass-flux export.
// Those with it (meshes that carry passive scalars) are compiled in sfh_kernels_mf.cu.
#include "sfh_stage.cuh"

namespace sfh {

cudaError_t configure_stage_kernels_mf();
cudaError_t launch_stage_mf(int stage, const TensorMaps& tm, const StageParams& p, int sms, cudaStream_t st);

// Raises the dynamic shared-memory limit of the stage kernels and returns the SM count of the current
// device (the persistent grid is one CTA per SM).
cudaError_t configure_kernels(int* sm_count) {
  cudaError_t e;
  if ((e = configure_stage_kernels<false>()) != cudaSuccess || (e = configure_stage_kernels_mf()) != cudaSuccess) return e;
  int dev = 0, sms = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess ||
      (e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
    return e;
  *sm_count = sms > 0 ? sms : 1;
  return cudaSuccess;
}

cudaError_t launch_stage(int stage, const TensorMaps& tm, const StageParams& p, int sms, cudaStream_t st) {
  return p.mf ? launch_stage_mf(stage, tm, p, sms, st) : launch_stage_impl<false>(stage, tm, p, sms, st);
}

}  // namespace sfh
