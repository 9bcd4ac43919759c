// fp64 instantiations of the Dslash stencil (18-real gauge), used by the fp64 outer residual of the reliable
// updates, the full-lattice apply and the TMW_DOUBLE solver. One column per thread (255 registers already).
#include "tmw_dslash_impl.cuh"

namespace tmw {
cudaError_t launch_dslash(const DslashArgs<double>& a, int ng, int epi, int clover, int nr, cudaStream_t s) {
  (void)nr;
  if (ng == 18) return launch_epi<double, 18, 1>(a, epi, clover, s);
  return cudaErrorInvalidValue;
}
cudaError_t launch_diag(const Diag<double>& d, const Geom& g, int par, bool clover, int inverse, const void* in, void* out, cudaStream_t s) {
  return launch_diag_t<double>(d, g, par, clover, inverse, in, out, s);
}
}  // namespace tmw
