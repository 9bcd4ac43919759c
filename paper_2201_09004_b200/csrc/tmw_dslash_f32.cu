// fp32 instantiations of the Dslash stencil (12-real reconstructed and 18-real gauge), one column per thread, and the
// dispatcher over columns per thread (the NR = 2, 3, 4 instantiations live in tmw_dslash_f32_nr*.cu).
#include "tmw_dslash_impl.cuh"

namespace tmw {
template <int NR> cudaError_t launch_dslash_f32_nr(const DslashArgs<float>& a, int ng, int epi, int clover, cudaStream_t s);
template <> cudaError_t launch_dslash_f32_nr<1>(const DslashArgs<float>& a, int ng, int epi, int clover, cudaStream_t s) {
  if (ng == 12) return launch_epi<float, 12, 1>(a, epi, clover, s);
  if (ng == 18) return launch_epi<float, 18, 1>(a, epi, clover, s);
  return cudaErrorInvalidValue;
}
template <> cudaError_t launch_dslash_f32_nr<2>(const DslashArgs<float>& a, int ng, int epi, int clover, cudaStream_t s);
template <> cudaError_t launch_dslash_f32_nr<3>(const DslashArgs<float>& a, int ng, int epi, int clover, cudaStream_t s);
template <> cudaError_t launch_dslash_f32_nr<4>(const DslashArgs<float>& a, int ng, int epi, int clover, cudaStream_t s);

cudaError_t launch_dslash(const DslashArgs<float>& a, int ng, int epi, int clover, int nr, cudaStream_t s) {
  switch (nr) {
    case 1: return launch_dslash_f32_nr<1>(a, ng, epi, clover, s);
    case 2: return launch_dslash_f32_nr<2>(a, ng, epi, clover, s);
    case 3: return launch_dslash_f32_nr<3>(a, ng, epi, clover, s);
    case 4: return launch_dslash_f32_nr<4>(a, ng, epi, clover, s);
  }
  return cudaErrorInvalidValue;
}
cudaError_t launch_diag(const Diag<float>& d, const Geom& g, int par, bool clover, int inverse, const void* in, void* out, cudaStream_t s) {
  return launch_diag_t<float>(d, g, par, clover, inverse, in, out, s);
}
}  // namespace tmw
