// fp32 instantiations of the Dslash stencil (12-real reconstructed and 18-real gauge).
#include "tmw_dslash_impl.cuh"

namespace tmw {
cudaError_t launch_dslash(const DslashArgs<float>& a, int ng, int epi, bool clover, cudaStream_t s) {
  if (ng == 12) return launch_epi<float, 12>(a, epi, clover, s);
  if (ng == 18) return launch_epi<float, 18>(a, epi, clover, s);
  return cudaErrorInvalidValue;
}
cudaError_t launch_diag(const Diag<float>& d, const Geom& g, int par, bool clover, int inverse, const void* in, void* out, cudaStream_t s) {
  return launch_diag_t<float>(d, g, par, clover, inverse, in, out, s);
}
}  // namespace tmw
