// tmw_dslash_impl.cuh — the Dslash stencil kernel (Eq. (2) hopping part with the
// fused mass/twist/clover epilogues of Eq. (2)-(3)) and the site-local diagonal kernel. Included by
// tmw_dslash_f32.cu and tmw_dslash_f64.cu with TMW_REAL defined.
#pragma once
#include "tmw_internal.h"

namespace tmw {

// block-level sum of up to 3 doubles per thread, one atomicAdd per block and value
template <int NV, int BLOCK> __device__ __forceinline__ void block_reduce_atomic(double (&v)[NV], double* dst) {
  __shared__ double sm[NV][BLOCK / 32];
#pragma unroll
  for (int k = 0; k < NV; k++) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], off);
  }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < NV; k++) sm[k][w] = v[k];
  }
  __syncthreads();
  if (threadIdx.x < NV) {
    double s = 0;
#pragma unroll
    for (int i = 0; i < BLOCK / 32; i++) s += sm[threadIdx.x][i];
    atomicAdd(dst + threadIdx.x, s);
  }
}

template <typename R, int NG, int EPI, bool CLOVER, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_kernel(const DslashArgs<R> a) {
  const int cb = blockIdx.x * BLOCK + threadIdx.x;
  const bool active = cb < a.g.Vh;
  R o[24], ax[24];
  if (active) {
    dslash_site<R, NG, EPI, CLOVER>(a, cb, o, ax);
    store_reals_s<24>(a.out, a.g.Vh, cb, o);
  }
  if (a.red_mode != 0) {  // uniform across the grid
    double v[3] = {0, 0, 0};
    if (active) {
      if (a.red_mode == 1) {
        R d[24];
        load_reals<24>(a.dotv, a.g.Vh, cb, d);
        R re = 0, im = 0;
#pragma unroll
        for (int i = 0; i < 12; i++) {  // conj(d) * o
          re += d[2 * i] * o[2 * i] + d[2 * i + 1] * o[2 * i + 1];
          im += d[2 * i] * o[2 * i + 1] - d[2 * i + 1] * o[2 * i];
        }
        v[0] = re;
        v[1] = im;
      } else if (EPI >= 2) {
        R re = 0, im = 0, nn = 0;
#pragma unroll
        for (int i = 0; i < 12; i++) {  // conj(o) * ax, |o|^2
          re += o[2 * i] * ax[2 * i] + o[2 * i + 1] * ax[2 * i + 1];
          im += o[2 * i] * ax[2 * i + 1] - o[2 * i + 1] * ax[2 * i];
          nn += o[2 * i] * o[2 * i] + o[2 * i + 1] * o[2 * i + 1];
        }
        v[0] = re;
        v[1] = im;
        v[2] = nn;
      }
    }
    block_reduce_atomic<3, BLOCK>(v, a.red);
  }
}

template <typename R, bool CLOVER, bool INV, int BLOCK> __global__ void __launch_bounds__(BLOCK) diag_kernel(const Diag<R> d, const Geom g, int par, const void* in, void* out) {
  const int cb = blockIdx.x * BLOCK + threadIdx.x;
  if (cb >= g.Vh) return;
  R v[24], o[24];
  load_reals<24>(in, g.Vh, cb, v);
  if (INV) apply_Ainv<R, CLOVER>(d, par, g.Vh, cb, v, o);
  else apply_A<R, CLOVER>(d, par, g.Vh, cb, v, o);
  store_reals<24>(out, g.Vh, cb, o);
}

template <typename R> struct Tune;
template <> struct Tune<float> { enum { BLOCK = 128, MINB = 4 }; };
template <> struct Tune<double> { enum { BLOCK = 128, MINB = 2 }; };

template <typename R, int NG, int EPI, bool CLOVER> static cudaError_t launch_one(const DslashArgs<R>& a, cudaStream_t s) {
  const int B = Tune<R>::BLOCK;
  const int grid = (a.g.Vh + B - 1) / B;
  dslash_kernel<R, NG, EPI, CLOVER, B, Tune<R>::MINB><<<grid, B, 0, s>>>(a);
  return cudaGetLastError();
}

template <typename R, int NG> static cudaError_t launch_epi(const DslashArgs<R>& a, int epi, bool clover, cudaStream_t s) {
  switch (epi) {
    case EPI_HOP: return launch_one<R, NG, EPI_HOP, false>(a, s);
    case EPI_AINV_HOP: return clover ? launch_one<R, NG, EPI_AINV_HOP, true>(a, s) : launch_one<R, NG, EPI_AINV_HOP, false>(a, s);
    case EPI_A_XPAY: return clover ? launch_one<R, NG, EPI_A_XPAY, true>(a, s) : launch_one<R, NG, EPI_A_XPAY, false>(a, s);
    case EPI_XPAY: return launch_one<R, NG, EPI_XPAY, false>(a, s);
    case EPI_AINV_XPAY: return clover ? launch_one<R, NG, EPI_AINV_XPAY, true>(a, s) : launch_one<R, NG, EPI_AINV_XPAY, false>(a, s);
  }
  return cudaErrorInvalidValue;
}

template <typename R> static cudaError_t launch_diag_t(const Diag<R>& d, const Geom& g, int par, bool clover, int inverse, const void* in, void* out, cudaStream_t s) {
  const int B = 128;
  const int grid = (g.Vh + B - 1) / B;
  if (clover) {
    if (inverse) diag_kernel<R, true, true, B><<<grid, B, 0, s>>>(d, g, par, in, out);
    else diag_kernel<R, true, false, B><<<grid, B, 0, s>>>(d, g, par, in, out);
  } else {
    if (inverse) diag_kernel<R, false, true, B><<<grid, B, 0, s>>>(d, g, par, in, out);
    else diag_kernel<R, false, false, B><<<grid, B, 0, s>>>(d, g, par, in, out);
  }
  return cudaGetLastError();
}

}  // namespace tmw
