// Persistent fp32 Dslash stencil with the links prefetched through a shared-memory ring (tmw_dslash_ring.cuh), 4 column(s) per thread.
#include "tmw_dslash_ring.cuh"

namespace tmw {
cudaError_t launch_dslash_ring_nr4(const DslashArgs<float>& a, int epi, int clover, cudaStream_t s) { return launch_ring_epi<4>(a, epi, clover, s); }
}  // namespace tmw
