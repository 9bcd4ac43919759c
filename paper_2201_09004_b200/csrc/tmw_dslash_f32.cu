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
// The memory floor of the hopping kernel's access pattern (tmw_time_kernel, TMW_K_HOP32_LOADONLY): the same 8 neighbour
// spinors (6 float4 each), 8 links (NG/4 float4 each, same cache policy), one 6-float4 store per site, same indices and
// launch shape, but the loaded vectors are only added up.
template <int NG> __global__ void __launch_bounds__(128, 4) hop_loadonly_kernel(const DslashArgs<float> a) {
  Site s;
  if (!thread_site<128>(a.g, blockIdx.x, s)) return;
  const Nbr n = neighbours(a.g, a.par, s);
  const int NPG = Planes<float, NG>::N;
  const int64_t Vh = a.g.Vh;
  float4 acc[6];
#pragma unroll
  for (int k = 0; k < 6; k++) acc[k] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
  for (int mu = 0; mu < 4; mu++) {
#pragma unroll
    for (int dir = 0; dir < 2; dir++) {
      const int nb = dir ? n.bwd[mu] : n.fwd[mu];
      const float4* u = (const float4*)a.U[dir ? 1 - a.par : a.par] + (int64_t)mu * NPG * Vh + (dir ? nb : s.cb);
      const float4* p = (const float4*)a.in + nb;
#pragma unroll
      for (int k = 0; k < NPG; k++) {
        const float4 q = ldv_s(u + k * Vh);
        acc[k].x += q.x; acc[k].y += q.y; acc[k].z += q.z; acc[k].w += q.w;
      }
#pragma unroll
      for (int k = 0; k < 6; k++) {
        const float4 q = ldv(p + k * Vh);
        acc[k].x += q.x; acc[k].y += q.y; acc[k].z += q.z; acc[k].w += q.w;
      }
    }
  }
#pragma unroll
  for (int k = 0; k < 6; k++) stv_s((float4*)a.out + k * Vh + s.cb, acc[k]);
}
cudaError_t launch_hop_loadonly(const DslashArgs<float>& a, int ng, cudaStream_t s) {
  const unsigned grid = (unsigned)((a.g.Vh + 127) / 128);
  if (ng == 12) hop_loadonly_kernel<12><<<grid, 128, 0, s>>>(a);
  else hop_loadonly_kernel<18><<<grid, 128, 0, s>>>(a);
  return cudaGetLastError();
}
// The fp32 ALU ceiling (tmw_time_kernel, TMW_K_FFMA_PROBE / TMW_K_FFMA2_PROBE): 16 independent FMA chains per thread in
// registers, as scalar FFMA or as 8 packed FFMA2 pairs; enough resident warps (8 CTAs of 256 threads per SM) to fill the pipe.
template <int PACKED> __global__ void __launch_bounds__(256) ffma_probe_kernel(float* out, float a0, float b0, int iters) {
  float x[16];
#pragma unroll
  for (int i = 0; i < 16; i++) x[i] = threadIdx.x * 0.001f + i;
  const float a = a0 + threadIdx.x * 1e-9f, b = b0 + threadIdx.x * 1e-9f;
  if (PACKED == 0) {
    for (int it = 0; it < iters; it++) {
#pragma unroll
      for (int i = 0; i < 16; i++) x[i] = fmaf(x[i], a, b);
    }
  } else {
    const float2 aa = make_float2(a, a), bb = make_float2(b, b);
    float2 y[8];
#pragma unroll
    for (int i = 0; i < 8; i++) y[i] = make_float2(x[2 * i], x[2 * i + 1]);
    for (int it = 0; it < iters; it++) {
#pragma unroll
      for (int i = 0; i < 8; i++) y[i] = TMW_FMA2(y[i], aa, bb);
    }
#pragma unroll
    for (int i = 0; i < 8; i++) { x[2 * i] = y[i].x; x[2 * i + 1] = y[i].y; }
  }
  float sum = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) sum += x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = sum;
}
cudaError_t launch_ffma_probe(int packed, int fmas_per_thread, int sms, float* sink, cudaStream_t s) {
  if (packed) ffma_probe_kernel<1><<<sms * 8, 256, 0, s>>>(sink, 1.0001f, 0.5f, fmas_per_thread / 16);
  else ffma_probe_kernel<0><<<sms * 8, 256, 0, s>>>(sink, 1.0001f, 0.5f, fmas_per_thread / 16);
  return cudaGetLastError();
}
cudaError_t launch_diag(const Diag<float>& d, const Geom& g, int par, bool clover, int inverse, const void* in, void* out, cudaStream_t s) {
  return launch_diag_t<float>(d, g, par, clover, inverse, in, out, s);
}
}  // namespace tmw
