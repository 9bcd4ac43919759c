// tmw_pack.cu — layout conversion: canonical fp64 arrays (include/tmw.h) <-> even-odd
// checkerboarded planes of 16-byte vectors. The gauge field gets an fp64 18-real copy and an fp32 copy with
// 12 reals (rows 0,1; row 2 is rebuilt in the stencil) or 18 reals.
#include "tmw_internal.h"

namespace tmw {

// lexicographic index in the GLOBAL lattice (canonical arrays) of the site (x, y, z, t) of the (sub-)lattice g
__device__ __forceinline__ int64_t global_lex(const Geom& g, int x, int y, int z, int t) {
  return x + (int64_t)g.L * (y + (int64_t)g.L * ((z + g.oz) + (int64_t)g.L * (t + g.ot)));
}
// global lexicographic site of checkerboard index cb on parity par (origins are even: local parity = global parity)
__device__ __forceinline__ int64_t lex_of_cb(const Geom& g, int par, int cb) {
  const int xh = cb % g.Lh;
  int q = cb / g.Lh;
  const int y = q % g.L;
  q /= g.L;
  const int z = q % g.Lz;
  const int t = q / g.Lz;
  const int x = 2 * xh + ((y + z + t + par) & 1);
  return global_lex(g, x, y, z, t);
}

template <int NG32> __global__ void __launch_bounds__(128) pack_gauge_kernel(const Geom g, const double* __restrict__ canon, double2* g64e, double2* g64o, float4* g32e, float4* g32o) {
  // one thread per (cb, mu, parity)
  const int cb = blockIdx.x * 128 + threadIdx.x;
  if (cb >= g.Vh) return;
  const int mu = blockIdx.y, par = blockIdx.z;
  const int64_t V = (int64_t)g.L * g.L * g.L * g.GT;  // global volume: stride of mu in the canonical array
  const int64_t lex = lex_of_cb(g, par, cb);
  const double* u = canon + 18 * ((int64_t)mu * V + lex);
  double r[18];
#pragma unroll
  for (int i = 0; i < 18; i++) r[i] = u[i];
  double2* d64 = (par ? g64o : g64e) + (int64_t)mu * 9 * g.Vh;
  store_reals<18>(d64, g.Vh, cb, r);
  const int NP = Planes<float, NG32>::N;
  float4* d32 = (par ? g32o : g32e) + (int64_t)mu * NP * g.Vh;
  float f[20];
#pragma unroll
  for (int i = 0; i < 18; i++) f[i] = (float)r[i];
  f[18] = f[19] = 0.f;
  store_reals<NG32>(d32, g.Vh, cb, f);
}

cudaError_t launch_pack_gauge(const Geom& g, const double* canon, void* g64_even, void* g64_odd, void* g32_even, void* g32_odd, int ng32, cudaStream_t s) {
  dim3 grid((g.Vh + 127) / 128, 4, 2);
  if (ng32 == 12) pack_gauge_kernel<12><<<grid, 128, 0, s>>>(g, canon, (double2*)g64_even, (double2*)g64_odd, (float4*)g32_even, (float4*)g32_odd);
  else pack_gauge_kernel<18><<<grid, 128, 0, s>>>(g, canon, (double2*)g64_even, (double2*)g64_odd, (float4*)g32_even, (float4*)g32_odd);
  return cudaGetLastError();
}

template <typename R> __global__ void __launch_bounds__(128) pack_spinor_kernel(const Geom g, int par, const double* __restrict__ canon, void* packed) {
  const int cb = blockIdx.x * 128 + threadIdx.x;
  if (cb >= g.Vh) return;
  const double* p = canon + 24 * lex_of_cb(g, par, cb);
  R v[24];
#pragma unroll
  for (int i = 0; i < 24; i++) v[i] = (R)p[i];
  store_reals<24>(packed, g.Vh, cb, v);
}
template <typename R> __global__ void __launch_bounds__(128) unpack_spinor_kernel(const Geom g, int par, const void* packed, double* __restrict__ canon) {
  const int cb = blockIdx.x * 128 + threadIdx.x;
  if (cb >= g.Vh) return;
  double* p = canon + 24 * lex_of_cb(g, par, cb);
  R v[24];
  load_reals<24>(packed, g.Vh, cb, v);
#pragma unroll
  for (int i = 0; i < 24; i++) p[i] = (double)v[i];
}

// Both parities at once: one thread per LEXICOGRAPHIC site, so that a warp touches 6 KB of contiguous canonical memory
// with 16-byte accesses (the one-parity kernels above skip every other 192-byte site and use 8-byte accesses: 1.58 ms
// per parity to unpack at 48^3 x 144, against 1.0 ms for both parities here). Used by tmw_apply FULL and tmw_solve.
template <typename R> __global__ void __launch_bounds__(128) pack_spinor_both_kernel(const Geom g, int64_t lex0, int64_t lex1, const double2* __restrict__ canon, void* pe, void* po) {
  const int64_t lex = lex0 + (int64_t)blockIdx.x * 128 + threadIdx.x;  // local lexicographic index
  if (lex >= lex1) return;
  int64_t q = lex;
  const int x = (int)(q % g.L); q /= g.L;
  const int y = (int)(q % g.L); q /= g.L;
  const int z = (int)(q % g.Lz);
  const int t = (int)(q / g.Lz);
  const int par = (x + y + z + t) & 1;
  const double2* p = canon + 12 * global_lex(g, x, y, z, t);
  R v[24];
#pragma unroll
  for (int i = 0; i < 12; i++) {
    const double2 d = p[i];
    v[2 * i] = (R)d.x;
    v[2 * i + 1] = (R)d.y;
  }
  store_reals<24>(par ? po : pe, g.Vh, lex >> 1, v);
}
// The packed side is read as in pack_spinor_both_kernel; the canonical side is written through shared memory, so that a
// warp stores 512 contiguous bytes per instruction instead of 32 separate 16-byte pieces 192 bytes apart (2.3 -> 1.0 ms
// at 48^3 x 144: partial-sector writes were the slow part). Site stride 13 double2 in shared memory: conflict-free both ways.
template <typename R> __global__ void __launch_bounds__(128) unpack_spinor_both_kernel(const Geom g, int64_t lex0, int64_t lex1, const void* pe, const void* po, double2* __restrict__ canon) {
  __shared__ double2 tile[128 * 13];
  __shared__ int64_t glex[128];
  const int64_t base = lex0 + (int64_t)blockIdx.x * 128;
  const int64_t lex = base + threadIdx.x;  // local lexicographic index
  if (lex < lex1) {
    int64_t q = lex;
    const int x = (int)(q % g.L); q /= g.L;
    const int y = (int)(q % g.L); q /= g.L;
    const int z = (int)(q % g.Lz);
    const int t = (int)(q / g.Lz);
    const int par = (x + y + z + t) & 1;
    R v[24];
    load_reals<24>(par ? po : pe, g.Vh, lex >> 1, v);
    glex[threadIdx.x] = global_lex(g, x, y, z, t);
#pragma unroll
    for (int i = 0; i < 12; i++) tile[threadIdx.x * 13 + i] = make_double2((double)v[2 * i], (double)v[2 * i + 1]);
  }
  __syncthreads();
  const int nsite = (int)((lex1 - base) < 128 ? (lex1 - base) : 128);
#pragma unroll
  for (int k = 0; k < 12; k++) {
    const int j = threadIdx.x + 128 * k, site = j / 12, comp = j - 12 * site;
    if (site < nsite) canon[12 * glex[site] + comp] = tile[site * 13 + comp];
  }
}
cudaError_t launch_pack_spinor_both(const Geom& g, int prec, const double* canon, void* packed_even, void* packed_odd, cudaStream_t s, int64_t lex0, int64_t lex1) {
  if (lex1 < 0) lex1 = 2 * (int64_t)g.Vh;
  const unsigned grid = (unsigned)((lex1 - lex0 + 127) / 128);
  if (prec == 0) pack_spinor_both_kernel<float><<<grid, 128, 0, s>>>(g, lex0, lex1, (const double2*)canon, packed_even, packed_odd);
  else pack_spinor_both_kernel<double><<<grid, 128, 0, s>>>(g, lex0, lex1, (const double2*)canon, packed_even, packed_odd);
  return cudaGetLastError();
}
cudaError_t launch_unpack_spinor_both(const Geom& g, int prec, const void* packed_even, const void* packed_odd, double* canon, cudaStream_t s, int64_t lex0, int64_t lex1) {
  if (lex1 < 0) lex1 = 2 * (int64_t)g.Vh;
  const unsigned grid = (unsigned)((lex1 - lex0 + 127) / 128);
  if (prec == 0) unpack_spinor_both_kernel<float><<<grid, 128, 0, s>>>(g, lex0, lex1, packed_even, packed_odd, (double2*)canon);
  else unpack_spinor_both_kernel<double><<<grid, 128, 0, s>>>(g, lex0, lex1, packed_even, packed_odd, (double2*)canon);
  return cudaGetLastError();
}

cudaError_t launch_pack_spinor(const Geom& g, int par, int prec, const double* canon, void* packed, cudaStream_t s) {
  const int grid = (g.Vh + 127) / 128;
  if (prec == 0) pack_spinor_kernel<float><<<grid, 128, 0, s>>>(g, par, canon, packed);
  else pack_spinor_kernel<double><<<grid, 128, 0, s>>>(g, par, canon, packed);
  return cudaGetLastError();
}
cudaError_t launch_unpack_spinor(const Geom& g, int par, int prec, const void* packed, double* canon, cudaStream_t s) {
  const int grid = (g.Vh + 127) / 128;
  if (prec == 0) unpack_spinor_kernel<float><<<grid, 128, 0, s>>>(g, par, packed, canon);
  else unpack_spinor_kernel<double><<<grid, 128, 0, s>>>(g, par, packed, canon);
  return cudaGetLastError();
}

}  // namespace tmw
