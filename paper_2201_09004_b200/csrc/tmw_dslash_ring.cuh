// tmw_dslash_ring.cuh — the fp32 Dslash stencil as a persistent kernel whose LINKS arrive through a per-thread ring in
// shared memory (hopping part of PAPER.md:62 Eq. (2)).
//
// Why: the multi-column launches are bound by load latency with 12 warps per SM, and the loads that always
// come from DRAM are the links (each link is used by exactly one site). Here a CTA walks over site blocks (grid-stride), and
// while it works on one site block every thread already has the 8 links of ITS site of the NEXT block in flight: 16-byte
// cp.async copies (LDGSTS, no registers) into slots of shared memory that only this thread reads, so no barrier is needed —
// cp.async.wait_group orders a thread's own copies. The slot pair of direction mu is refilled as soon as the two hops of
// that direction are done, i.e. one whole site (thousands of cycles) ahead of its use. The neighbour spinors still come
// by LDG (seven of their eight reads hit L1/L2). 12-real links only: 8 links x 3 planes x 16 B x 128 threads = 48 KB per CTA.
#pragma once
#include "tmw_dslash_impl.cuh"
#include "tmw_dslash_stage.cuh"  // cp_async16

namespace tmw {

enum { RING_BLOCK = 128 };

// slot (l, k) of this thread: link l = 2*mu + (0 forward | 1 backward), plane k < 3
__device__ __forceinline__ float4* ring_slot(float4* ring, int l, int k) { return ring + (l * 3 + k) * RING_BLOCK + threadIdx.x; }

template <int MU> __device__ __forceinline__ void ring_fetch(const DslashArgs<float>& a, float4* ring, int cb, int cb_bwd) {
  const int64_t Vh = a.g.Vh;
  const float4* uf = (const float4*)a.U[a.par] + (int64_t)MU * 3 * Vh + cb;
  const float4* ub = (const float4*)a.U[1 - a.par] + (int64_t)MU * 3 * Vh + cb_bwd;
#pragma unroll
  for (int k = 0; k < 3; k++) {
    cp_async16(ring_slot(ring, 2 * MU, k), uf + k * Vh);
    cp_async16(ring_slot(ring, 2 * MU + 1, k), ub + k * Vh);
  }
}
__device__ __forceinline__ void ring_link(float4* ring, int l, cx<float> (&U)[9]) {
  float g[12];
#pragma unroll
  for (int k = 0; k < 3; k++) {
    const float4 q = *ring_slot(ring, l, k);
    g[4 * k] = q.x; g[4 * k + 1] = q.y; g[4 * k + 2] = q.z; g[4 * k + 3] = q.w;
  }
#pragma unroll
  for (int i = 0; i < 6; i++) U[i] = mk<float>(g[2 * i], g[2 * i + 1]);
  U[6] = conj(U[1] * U[5] - U[2] * U[4]);
  U[7] = conj(U[2] * U[3] - U[0] * U[5]);
  U[8] = conj(U[0] * U[4] - U[1] * U[3]);
}

// the two hops of direction MU for the NR columns of this thread, links from the ring
template <int MU, int NR> __device__ __forceinline__ void ring_hops(const DslashArgs<float>& a, const Nbr& n, float4* ring, const int (&cofs)[NR], float (&acc)[NR][24],
                                                                      float2 (&acc2)[(NR + 1) / 2][24]) {
  const int64_t Vh = a.g.Vh;
#pragma unroll
  for (int dir = 0; dir < 2; dir++) {
    cx<float> U[9];
    ring_link(ring, 2 * MU + dir, U);
    const int nb = dir ? n.bwd[MU] : n.fwd[MU];
    const float bc = (MU == 3 && (dir ? n.wrap_tb : n.wrap_tf)) ? -1.f : 1.f;
    const float sig = dir ? -a.sig : a.sig;
    if constexpr (TMW_PACK2 && NR % 2 == 0) {
      LinkPairs P;
      link_pairs(U, bc, P);
#pragma unroll
      for (int p = 0; p < NR / 2; p++) {
        float psiA[24], psiB[24];
        load_reals<24>(a.in, Vh, nb + cofs[2 * p], psiA);
        load_reals<24>(a.in, Vh, nb + cofs[2 * p + 1], psiB);
        if (dir) hop2<MU, false>(psiA, psiB, P, sig, acc2[p]);
        else hop2<MU, true>(psiA, psiB, P, sig, acc2[p]);
      }
    } else {
#pragma unroll
      for (int j = 0; j < NR; j++) {
        float psi[24];
        load_reals<24>(a.in, Vh, nb + cofs[j], psi);
        if (dir) hop<float, MU, false>(psi, U, sig, bc, acc[j]);
        else hop<float, MU, true>(psi, U, sig, bc, acc[j]);
      }
    }
  }
}

// work item w = group + ngroups * site block (as blockIdx.x of dslash_kernel); nwork items, grid-stride over them
template <int EPI, int CLOVER, int NR, int MINB>
__global__ void __launch_bounds__(RING_BLOCK, MINB) dslash_ring_kernel(const DslashArgs<float> a, int nwork) {
  extern __shared__ float4 ring[];
  if (a.skip && *a.skip) return;
  int w = blockIdx.x;
  if (w >= nwork) return;
  Site s;
  bool active;
  {
    const int sblock = a.ngroups > 1 ? w / a.ngroups : w;
    active = thread_site<RING_BLOCK>(a.g, sblock, s);
  }
  Nbr n = neighbours(a.g, a.par, s);
  if (active) {
    ring_fetch<0>(a, ring, s.cb, n.bwd[0]);
    ring_fetch<1>(a, ring, s.cb, n.bwd[1]);
    ring_fetch<2>(a, ring, s.cb, n.bwd[2]);
    ring_fetch<3>(a, ring, s.cb, n.bwd[3]);
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  for (;;) {
    const int grp = a.ngroups > 1 ? w % a.ngroups : 0;
    const int wn = w + gridDim.x;
    const bool have_next = wn < nwork;
    Site sn = s;
    bool active_n = false;
    if (have_next) active_n = thread_site<RING_BLOCK>(a.g, a.ngroups > 1 ? wn / a.ngroups : wn, sn);
    const Nbr nn = neighbours(a.g, a.par, sn);
    int colj[NR], cofs[NR];
    bool valid[NR];
#pragma unroll
    for (int j = 0; j < NR; j++) {
      const int slot = grp * NR + j;
      valid[j] = slot < a.ncol;
      colj[j] = a.col[valid[j] ? slot : a.ncol - 1];
      cofs[j] = colj[j] * a.cstride;
    }
    float o[NR][24], r2[NR][3];
    float2 o2[(NR + 1) / 2][24];
#pragma unroll
    for (int j = 0; j < NR; j++)
#pragma unroll
      for (int i = 0; i < 24; i++) o[j][i] = 0.f;
#pragma unroll
    for (int p = 0; p < (NR + 1) / 2; p++)
#pragma unroll
      for (int i = 0; i < 24; i++) o2[p][i] = make_float2(0.f, 0.f);
    asm volatile("cp.async.wait_group 0;" ::: "memory");  // this thread's links of the current site are in its slots
    if (active) ring_hops<0, NR>(a, n, ring, cofs, o, o2);
    if (active_n) ring_fetch<0>(a, ring, sn.cb, nn.bwd[0]);
    if (active) ring_hops<1, NR>(a, n, ring, cofs, o, o2);
    if (active_n) ring_fetch<1>(a, ring, sn.cb, nn.bwd[1]);
    if (active) ring_hops<2, NR>(a, n, ring, cofs, o, o2);
    if (active_n) ring_fetch<2>(a, ring, sn.cb, nn.bwd[2]);
    if (active) ring_hops<3, NR>(a, n, ring, cofs, o, o2);
    if (active_n) ring_fetch<3>(a, ring, sn.cb, nn.bwd[3]);
    asm volatile("cp.async.commit_group;" ::: "memory");
    if (active) {
      if constexpr (TMW_PACK2 && NR % 2 == 0) {
#pragma unroll
        for (int p = 0; p < NR / 2; p++)
#pragma unroll
          for (int i = 0; i < 24; i++) { o[2 * p][i] = o2[p][i].x; o[2 * p + 1][i] = o2[p][i].y; }
      }
      dslash_epilogue<float, 12, EPI, CLOVER, NR, false>(a, s.cb, cofs, valid, o, r2);
      if (!stored_in_site<EPI, CLOVER>()) {
        if (a.g5) {
#pragma unroll
          for (int j = 0; j < NR; j++)
#pragma unroll
            for (int i = 12; i < 24; i++) o[j][i] = -o[j][i];
        }
#pragma unroll
        for (int j = 0; j < NR; j++)
          if (valid[j] && a.out) store_reals_s<24>(a.out, a.g.Vh, s.cb + cofs[j], o[j]);
      }
    }
    if (a.red_mode != 0) {  // uniform across the grid
      site_reductions<float, NR, RING_BLOCK>(a, s, active, cofs, colj, valid, o, r2);
      __syncthreads();  // the reduction's shared scratch is written again by the next site block of this CTA
    }
    if (!have_next) break;
    w = wn;
    s = sn;
    n = nn;
    active = active_n;
  }
}

template <int NR> struct RingTune;
template <> struct RingTune<1> { enum { MINB = 4 }; };
template <> struct RingTune<2> { enum { MINB = 3 }; };
template <> struct RingTune<3> { enum { MINB = 3 }; };
template <> struct RingTune<4> { enum { MINB = 2 }; };

template <int EPI, int CLOVER, int NR> static cudaError_t launch_ring_one(DslashArgs<float> a, cudaStream_t s) {
  const size_t smem = (size_t)8 * 3 * RING_BLOCK * sizeof(float4);
  auto kern = dslash_ring_kernel<EPI, CLOVER, NR, RingTune<NR>::MINB>;
  // resident CTAs per SM and the SM count, per device (the shared-memory attribute belongs to (function, device) as well)
  enum { MAXDEV = 64 };
  static int ctas_cache[MAXDEV] = {0}, sms_cache[MAXDEV] = {0};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAXDEV) return cudaErrorInvalidDevice;
  if (!ctas_cache[dev]) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int n = 0, m = 0;
    e = cudaDeviceGetAttribute(&m, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, RING_BLOCK, smem);
    if (e != cudaSuccess) return e;
    sms_cache[dev] = m;
    ctas_cache[dev] = n < 1 ? 1 : n;
  }
  const int ctas_per_sm = ctas_cache[dev], sms = sms_cache[dev];
  a.ngroups = (a.ncol + NR - 1) / NR;
  const int nwork = ((a.g.Vh + RING_BLOCK - 1) / RING_BLOCK) * a.ngroups;
  const int grid = nwork < sms * ctas_per_sm ? nwork : sms * ctas_per_sm;
  kern<<<grid, RING_BLOCK, smem, s>>>(a, nwork);
  return cudaGetLastError();
}
template <int NR> static cudaError_t launch_ring_epi(const DslashArgs<float>& a, int epi, int clover, cudaStream_t s) {
  switch (epi) {
    case EPI_HOP: return launch_ring_one<EPI_HOP, CL_NONE, NR>(a, s);
    case EPI_AINV_HOP:
      if (clover == CL_TWISTED) return launch_ring_one<EPI_AINV_HOP, CL_TWISTED, NR>(a, s);
      return clover ? launch_ring_one<EPI_AINV_HOP, CL_CLOVER, NR>(a, s) : launch_ring_one<EPI_AINV_HOP, CL_NONE, NR>(a, s);
    case EPI_A_XPAY: return clover ? launch_ring_one<EPI_A_XPAY, CL_CLOVER, NR>(a, s) : launch_ring_one<EPI_A_XPAY, CL_NONE, NR>(a, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace tmw
