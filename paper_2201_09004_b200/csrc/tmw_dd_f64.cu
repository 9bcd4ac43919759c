// fp64 instantiations of the domain-decomposition passes of the stencil, and the kernel that cuts a
// domain's packed fields out of the whole-lattice ones.
#include "tmw_dslash_impl.cuh"

namespace tmw {
// packed field of a domain <- the same field of the whole lattice (any 16-byte vector type): vector (k, cb) of the domain
// is vector (k, cbg) of the global field, cbg the checkerboard index of the same site in the global lattice
__global__ void __launch_bounds__(128) extract_planes_kernel(const Geom g, int nplanes, int64_t gVh, const uint4* __restrict__ src, uint4* dst) {
  const int cb = blockIdx.x * 128 + threadIdx.x;
  if (cb >= g.Vh) return;
  const int xh = cb % g.Lh;
  int q = cb / g.Lh;
  const int y = q % g.L;
  q /= g.L;
  const int z = q % g.Lz, t = q / g.Lz;
  const int64_t cbg = xh + (int64_t)g.Lh * (y + (int64_t)g.L * ((z + g.oz) + (int64_t)g.L * (t + g.ot)));
  for (int k = 0; k < nplanes; k++) dst[(int64_t)k * g.Vh + cb] = src[k * gVh + cbg];
}

cudaError_t launch_dslash_dd(const DslashArgs<double>& a, int ng, int epi, int clover, int pass, cudaStream_t s) {
  if (ng == 18) return launch_dd_epi<double, 18>(a, epi, clover, pass, s);
  return cudaErrorInvalidValue;
}
cudaError_t launch_face_pack(const DslashArgs<double>& a, int ng, void* const (&send)[2][2], cudaStream_t s) {
  if (ng == 18) return launch_face_pack_t<double, 18>(a, send, s);
  return cudaErrorInvalidValue;
}
cudaError_t launch_extract_planes(const Geom& g, int nplanes, int64_t gVh, const void* src, void* dst, cudaStream_t s) {
  extract_planes_kernel<<<(g.Vh + 127) / 128, 128, 0, s>>>(g, nplanes, gVh, (const uint4*)src, (uint4*)dst);
  return cudaGetLastError();
}
}  // namespace tmw
