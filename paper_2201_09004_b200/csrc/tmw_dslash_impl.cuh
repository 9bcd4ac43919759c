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

template <typename R, int NG, int EPI, int CLOVER, int NR, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_kernel(const DslashArgs<R> a) {
  typedef typename Vec16<R>::T V;
  // blockIdx.x = group + ngroups * site block: the CTAs that share the links of a site block are launched together
  int sblock = blockIdx.x, grp = 0;
  if (a.ngroups > 1) {
    sblock = blockIdx.x / a.ngroups;
    grp = blockIdx.x - sblock * a.ngroups;
  }
  Site s;
  const bool active = thread_site<BLOCK>(a.g, sblock, s);
  int colj[NR], cofs[NR];
  bool valid[NR];
#pragma unroll
  for (int j = 0; j < NR; j++) {
    const int slot = grp * NR + j;
    valid[j] = slot < a.ncol;  // a ragged last group recomputes the last column and drops the result
    colj[j] = a.col[valid[j] ? slot : a.ncol - 1];
    cofs[j] = colj[j] * a.cstride;
  }
  R o[NR][24], r2[NR][3];
  if (active) {
    // one column per thread: nobody else reads this thread's links and clover blocks (evict-first); with more columns the
    // other column groups of a site block find them in L2
    dslash_site<R, NG, EPI, CLOVER, NR, NR == 1>(a, s, cofs, valid, o, r2);
    if (!stored_in_site<EPI, CLOVER>()) {
      if (a.g5) {  // uniform across the grid
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
#pragma unroll
    for (int j = 0; j < NR; j++) {
      double v[7] = {0, 0, 0, 0, 0, 0, 0};
      if (active && valid[j]) {
        if (a.red_mode == 1) {
          R d[24];
          load_reals<24>(a.dotv, a.g.Vh, s.cb + cofs[j], d);
          R re = 0, im = 0;
#pragma unroll
          for (int i = 0; i < 12; i++) {  // conj(d) * o
            re += d[2 * i] * o[j][2 * i] + d[2 * i + 1] * o[j][2 * i + 1];
            im += d[2 * i] * o[j][2 * i + 1] - d[2 * i + 1] * o[j][2 * i];
          }
          v[0] = re;
          v[1] = im;
        } else if (a.red_mode == 3) {  // |dotv - o|^2: the residual norm of the final check, o itself is not kept
          R d[24];
          load_reals<24>(a.dotv, a.g.Vh, s.cb + cofs[j], d);
          R nn = 0;
#pragma unroll
          for (int i = 0; i < 24; i++) nn += (d[i] - o[j][i]) * (d[i] - o[j][i]);
          v[2] = nn;
        } else {
          v[0] = r2[j][0];
          v[1] = r2[j][1];
          v[2] = r2[j][2];
          if (a.red_mode == 4) {  // also <dotv, o> and <dotv, aux> (aux is re-read: it was consumed chirality by chirality)
            R d[24], x[24];
            load_reals<24>(a.dotv, a.g.Vh, s.cb + cofs[j], d);
            R re = 0, im = 0;
#pragma unroll
            for (int i = 0; i < 12; i++) {
              re += d[2 * i] * o[j][2 * i] + d[2 * i + 1] * o[j][2 * i + 1];
              im += d[2 * i] * o[j][2 * i + 1] - d[2 * i + 1] * o[j][2 * i];
            }
            v[3] = re;
            v[4] = im;
            load_reals<24>(a.aux, a.g.Vh, s.cb + cofs[j], x);
            re = 0;
            im = 0;
#pragma unroll
            for (int i = 0; i < 12; i++) {
              re += d[2 * i] * x[2 * i] + d[2 * i + 1] * x[2 * i + 1];
              im += d[2 * i] * x[2 * i + 1] - d[2 * i + 1] * x[2 * i];
            }
            v[5] = re;
            v[6] = im;
          }
        }
      }
      if (j > 0) __syncthreads();  // the shared scratch of block_reduce_atomic is reused
      double* dst = a.red + (int64_t)colj[j] * a.red_stride;
      if (a.red_mode == 4) {
        block_reduce_atomic<7, BLOCK>(v, dst);
      } else {
        double v3[3] = {v[0], v[1], v[2]};
        block_reduce_atomic<3, BLOCK>(v3, dst);
      }
    }
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

// launch shape per precision and columns per thread (128 threads x 4 CTAs/SM = 128 registers for the
// single-column fp32 kernel; more columns per thread need the accumulators of all of them in registers)
template <typename R, int NR> struct Tune;
template <> struct Tune<float, 1> { enum { BLOCK = 128, MINB = 4 }; };
template <> struct Tune<float, 2> { enum { BLOCK = 128, MINB = 3 }; };
template <> struct Tune<float, 3> { enum { BLOCK = 128, MINB = 3 }; };
template <> struct Tune<float, 4> { enum { BLOCK = 128, MINB = 2 }; };
template <> struct Tune<double, 1> { enum { BLOCK = 128, MINB = 2 }; };

template <typename R, int NG, int EPI, int CLOVER, int NR> static cudaError_t launch_one(DslashArgs<R> a, cudaStream_t s) {
  const int B = Tune<R, NR>::BLOCK;
  a.ngroups = (a.ncol + NR - 1) / NR;
  dim3 grid;
  if (a.g.tiled) grid = dim3((unsigned)(a.g.ntx * a.g.nty * a.ngroups), (unsigned)(a.g.Lz >> a.g.lz), (unsigned)(a.g.T >> a.g.lt));
  else grid = dim3((unsigned)(((a.g.Vh + B - 1) / B) * a.ngroups), 1, 1);
  dslash_kernel<R, NG, EPI, CLOVER, NR, B, Tune<R, NR>::MINB><<<grid, B, 0, s>>>(a);
  return cudaGetLastError();
}

// clover: CL_NONE | CL_CLOVER | CL_TWISTED; only the kernels that apply A^{-1} have a separate twisted instantiation
template <typename R, int NG, int NR> static cudaError_t launch_epi(const DslashArgs<R>& a, int epi, int clover, cudaStream_t s) {
  switch (epi) {
    case EPI_HOP: return launch_one<R, NG, EPI_HOP, CL_NONE, NR>(a, s);
    case EPI_AINV_HOP:
      if (clover == CL_TWISTED) return launch_one<R, NG, EPI_AINV_HOP, CL_TWISTED, NR>(a, s);
      return clover ? launch_one<R, NG, EPI_AINV_HOP, CL_CLOVER, NR>(a, s) : launch_one<R, NG, EPI_AINV_HOP, CL_NONE, NR>(a, s);
    case EPI_A_XPAY: return clover ? launch_one<R, NG, EPI_A_XPAY, CL_CLOVER, NR>(a, s) : launch_one<R, NG, EPI_A_XPAY, CL_NONE, NR>(a, s);
    case EPI_XPAY: return launch_one<R, NG, EPI_XPAY, CL_NONE, NR>(a, s);
    case EPI_AINV_XPAY:
      if (clover == CL_TWISTED) return launch_one<R, NG, EPI_AINV_XPAY, CL_TWISTED, NR>(a, s);
      return clover ? launch_one<R, NG, EPI_AINV_XPAY, CL_CLOVER, NR>(a, s) : launch_one<R, NG, EPI_AINV_XPAY, CL_NONE, NR>(a, s);
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
