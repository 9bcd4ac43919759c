// Persistent fp32 Dslash stencil with the links prefetched through a shared-memory ring (tmw_dslash_ring.cuh), 1 column(s) per thread.
#include "tmw_dslash_ring.cuh"

namespace tmw {
cudaError_t launch_dslash_ring_nr1(const DslashArgs<float>& a, int epi, int clover, cudaStream_t s) { return launch_ring_epi<1>(a, epi, clover, s); }
cudaError_t launch_dslash_ring_nr2(const DslashArgs<float>& a, int epi, int clover, cudaStream_t s);
cudaError_t launch_dslash_ring_nr3(const DslashArgs<float>& a, int epi, int clover, cudaStream_t s);
cudaError_t launch_dslash_ring_nr4(const DslashArgs<float>& a, int epi, int clover, cudaStream_t s);
cudaError_t launch_dslash_ring(const DslashArgs<float>& a, int epi, int clover, int nr, cudaStream_t s) {
  switch (nr) {
    case 1: return launch_dslash_ring_nr1(a, epi, clover, s);
    case 2: return launch_dslash_ring_nr2(a, epi, clover, s);
    case 3: return launch_dslash_ring_nr3(a, epi, clover, s);
    case 4: return launch_dslash_ring_nr4(a, epi, clover, s);
  }
  return cudaErrorInvalidValue;
}
}  // namespace tmw
