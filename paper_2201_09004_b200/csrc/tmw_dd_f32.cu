// fp32 instantiations of the domain-decomposition passes of the stencil: interior (dslash_kernel with
// DD = 1), exterior (dslash_ext_kernel) and the face pack, for 12-real and 18-real gauge storage.
#include "tmw_dslash_impl.cuh"

namespace tmw {
cudaError_t launch_dslash_dd(const DslashArgs<float>& a, int ng, int epi, int clover, int pass, cudaStream_t s) {
  if (ng == 12) return launch_dd_epi<float, 12>(a, epi, clover, pass, s);
  if (ng == 18) return launch_dd_epi<float, 18>(a, epi, clover, pass, s);
  return cudaErrorInvalidValue;
}
cudaError_t launch_face_pack(const DslashArgs<float>& a, int ng, void* const (&send)[2][2], cudaStream_t s) {
  if (ng == 12) return launch_face_pack_t<float, 12>(a, send, s);
  if (ng == 18) return launch_face_pack_t<float, 18>(a, send, s);
  return cudaErrorInvalidValue;
}
}  // namespace tmw
