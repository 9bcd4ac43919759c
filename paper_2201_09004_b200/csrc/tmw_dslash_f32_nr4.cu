// fp32 Dslash stencil with 4 right-hand-side columns per thread; 12-real gauge only.
#include "tmw_dslash_impl.cuh"

namespace tmw {
template <int NR> cudaError_t launch_dslash_f32_nr(const DslashArgs<float>& a, int ng, int epi, int clover, cudaStream_t s);
template <> cudaError_t launch_dslash_f32_nr<4>(const DslashArgs<float>& a, int ng, int epi, int clover, cudaStream_t s) {
  if (ng == 12) return launch_epi<float, 12, 4>(a, epi, clover, s);
  if (ng == 18) return launch_epi<float, 18, 4>(a, epi, clover, s);
  return cudaErrorInvalidValue;
}
}  // namespace tmw
