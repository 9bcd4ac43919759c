// Persistent fp32 Dslash stencil with the links prefetched through a shared-memory ring (tmw_dslash_ring.cuh), 3 column(s) per thread.
#include "tmw_dslash_ring.cuh"

namespace tmw {
cudaError_t launch_dslash_ring_nr3(const DslashArgs<float>& a, int epi, int clover, cudaStream_t s) { return launch_ring_epi<3>(a, epi, clover, s); }
}  // namespace tmw
