// Shared-memory staged fp32 Dslash stencil (tmw_dslash_stage.cuh), one right-hand-side column per thread.
#include "tmw_dslash_stage.cuh"

namespace tmw {
template <int NR> cudaError_t launch_dslash_stage_nr(const DslashArgs<float>& a, int ng, int epi, int clover, const StageGeom& sg, cudaStream_t s);
template <> cudaError_t launch_dslash_stage_nr<1>(const DslashArgs<float>& a, int ng, int epi, int clover, const StageGeom& sg, cudaStream_t s) {
  if (ng == 12) return launch_stage_epi<12, 1>(a, epi, clover, sg, s);
  if (ng == 18) return launch_stage_epi<18, 1>(a, epi, clover, sg, s);
  return cudaErrorInvalidValue;
}
template <> cudaError_t launch_dslash_stage_nr<2>(const DslashArgs<float>& a, int ng, int epi, int clover, const StageGeom& sg, cudaStream_t s);
template <> cudaError_t launch_dslash_stage_nr<3>(const DslashArgs<float>& a, int ng, int epi, int clover, const StageGeom& sg, cudaStream_t s);

cudaError_t launch_dslash_stage(const DslashArgs<float>& a, int ng, int epi, int clover, int nr, const StageGeom& sg, cudaStream_t s) {
  switch (nr) {
    case 1: return launch_dslash_stage_nr<1>(a, ng, epi, clover, sg, s);
    case 2: return launch_dslash_stage_nr<2>(a, ng, epi, clover, sg, s);
    case 3: return launch_dslash_stage_nr<3>(a, ng, epi, clover, sg, s);
  }
  return cudaErrorInvalidValue;
}
int stage_max_threads(int nr) { return nr == 3 ? (int)StageTune<3>::MAXT : (int)StageTune<1>::MAXT; }
}  // namespace tmw
