// Shared-memory staged fp32 Dslash stencil (tmw_dslash_stage.cuh), 3 right-hand-side columns per thread.
#include "tmw_dslash_stage.cuh"

namespace tmw {
template <int NR> cudaError_t launch_dslash_stage_nr(const DslashArgs<float>& a, int ng, int epi, int clover, const StageGeom& sg, cudaStream_t s);
template <> cudaError_t launch_dslash_stage_nr<3>(const DslashArgs<float>& a, int ng, int epi, int clover, const StageGeom& sg, cudaStream_t s) {
  if (ng == 12) return launch_stage_epi<12, 3>(a, epi, clover, sg, s);
  if (ng == 18) return launch_stage_epi<18, 3>(a, epi, clover, sg, s);
  return cudaErrorInvalidValue;
}
}  // namespace tmw
