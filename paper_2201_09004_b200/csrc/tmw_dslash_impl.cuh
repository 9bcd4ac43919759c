// tmw_dslash_impl.cuh — the Dslash stencil kernel (Eq. (2) hopping part with the
// fused mass/twist/clover epilogues of Eq. (2)-(3)) and the site-local diagonal kernel. Included by
// tmw_dslash_f32.cu and tmw_dslash_f64.cu with TMW_REAL defined.
#pragma once
#include "tmw_internal.h"

namespace tmw {

// block-level sum of up to 3 doubles per thread, one atomicAdd per block and value
// BLOCK = 0: the block size is blockDim.x (a multiple of 32, at most 256) instead of a compile-time constant
template <int NV, int BLOCK> __device__ __forceinline__ void block_reduce_atomic(double (&v)[NV], double* dst) {
  __shared__ double sm[NV][BLOCK ? BLOCK / 32 : 8];
  const int nwarps = BLOCK ? BLOCK / 32 : (int)(blockDim.x >> 5);
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
    for (int i = 0; i < (BLOCK ? BLOCK / 32 : 8); i++)
      if (i < nwarps) s += sm[threadIdx.x][i];
    atomicAdd(dst + threadIdx.x, s);
  }
}

// The fused reductions of a stencil launch (DslashArgs::red_mode) for the NR column slots of this thread: o = the output
// spinors, r2 = what dslash_epilogue accumulated; `contributes` = this thread holds a finished site. Block-uniform.
template <typename R, int NR, int BLOCK>
__device__ __forceinline__ void site_reductions(const DslashArgs<R>& a, const Site& s, bool contributes, const int (&cofs)[NR], const int (&colj)[NR],
                                                const bool (&valid)[NR], R (&o)[NR][24], R (&r2)[NR][3]) {
#pragma unroll
  for (int j = 0; j < NR; j++) {
    double v[7] = {0, 0, 0, 0, 0, 0, 0};
    if (contributes && valid[j]) {
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

// DD = 0: the stencil on the whole lattice. DD = 1: interior pass on one domain of a domain-decomposed context (sites on a
// cut are left raw for dslash_ext_kernel, see dslash_site).
template <typename R, int NG, int EPI, int CLOVER, int NR, int BLOCK, int MINB, int DD>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_kernel(const DslashArgs<R> a) {
  typedef typename Vec16<R>::T V;
  if (a.skip && *a.skip) return;
  // blockIdx.x = group + ngroups * site block: the CTAs that share the links of a site block are launched together
  int sblock = blockIdx.x, grp = 0;
  if (a.ngroups > 1) {
    sblock = blockIdx.x / a.ngroups;
    grp = blockIdx.x - sblock * a.ngroups;
  }
  Site s;
  const bool active = thread_site<BLOCK>(a.g, sblock + a.sb0, s) && s.cb < a.cb_end;
  int colj[NR], cofs[NR];
  bool valid[NR];
#pragma unroll
  for (int j = 0; j < NR; j++) {
    const int slot = grp * NR + j;
    valid[j] = slot < a.ncol;  // a ragged last group recomputes the last column and drops the result
    colj[j] = a.col[valid[j] ? slot : a.ncol - 1];
    cofs[j] = colj[j] * a.cstride;
  }
  if (DD == 0 && a.pf_blocks > 0 && grp == 0 && !a.g.tiled) {  // the first column group of a site block prefetches for a later block
    Site sp;
    if (thread_site<BLOCK>(a.g, sblock + a.sb0 + a.pf_blocks, sp) && sp.cb < a.cb_end) {
      const Nbr np = neighbours(a.g, a.par, sp);
      const int NPG = Planes<R, NG>::N;
#pragma unroll
      for (int mu = 0; mu < 4; mu++) {
        const V* uf = (const V*)a.U[a.par] + (int64_t)mu * NPG * a.g.Vh + sp.cb;
        const V* ub = (const V*)a.U[1 - a.par] + (int64_t)mu * NPG * a.g.Vh + np.bwd[mu];
#pragma unroll
        for (int k = 0; k < NPG; k++) {
          asm volatile("prefetch.global.L2 [%0];" ::"l"(uf + (int64_t)k * a.g.Vh));
          asm volatile("prefetch.global.L2 [%0];" ::"l"(ub + (int64_t)k * a.g.Vh));
        }
      }
    }
  }
  R o[NR][24], r2[NR][3];
  bool raw = false;
  if (active) {
    // one column per thread: nobody else reads this thread's links and clover blocks (evict-first); with more columns the
    // other column groups of a site block find them in L2
    raw = dslash_site<R, NG, EPI, CLOVER, NR, NR == 1, DD>(a, s, cofs, valid, o, r2);
    if (!raw && !stored_in_site<EPI, CLOVER>()) {
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
  if (a.red_mode != 0) site_reductions<R, NR, BLOCK>(a, s, active && !raw, cofs, colj, valid, o, r2);  // uniform across the grid
}

// ---- domain decomposition (SURVEY §8(f4); the paper's multi-GPU runs: PAPER.md:52, :71-76 "Nodes", :315) ----
// Face pack: for every cut of the domain and both sides, the half spinors the neighbours need (DDArgs), from the
// input spinor a.in (parity 1 - a.par). blockIdx.y = 2 * direction + side (0: first slice -> the neighbour BEHIND, its "hi"
// ghost, projected only; 1: last slice -> the neighbour AHEAD, its "lo" ghost, projected and multiplied by U^dag);
// blockIdx.z = column slot. send[d][side]: same layout as DDArgs::ghost.
template <typename R> struct FaceOut {
  void* send[2][2];
};
template <typename R, int NG, int MU, int SIDE> __device__ __forceinline__ void face_pack_site(const DslashArgs<R>& a, int cb, int cofs, cx<R> (&w)[6]) {
  typedef typename Vec16<R>::T V;
  R psi[24];
  load_reals<24>(a.in, a.g.Vh, cb + cofs, psi);
  if (SIDE == 0) {
    project_half<R, MU>(psi, a.sig, w);
  } else {
    cx<R> h[6], U[9];
    project_half<R, MU>(psi, -a.sig, h);
    load_link<R, NG, true>((const V*)a.U[1 - a.par] + (int64_t)MU * Planes<R, NG>::N * a.g.Vh, a.g.Vh, cb, U);
    su3_mul_half<R, false>(U, h, w);
  }
}
template <typename R, int NG, int BLOCK> __global__ void __launch_bounds__(BLOCK) face_pack_kernel(const DslashArgs<R> a, const FaceOut<R> fo) {
  typedef typename Vec16<R>::T V;
  const int d = blockIdx.y >> 1, side = blockIdx.y & 1;
  if (!a.dd.part[d] || (a.skip && *a.skip)) return;
  const int f = blockIdx.x * BLOCK + threadIdx.x;
  if (f >= a.dd.nface[d]) return;
  const int col = a.col[blockIdx.z];
  const int xh = f % a.g.Lh;
  int q = f / a.g.Lh;
  const int y = q % a.g.L;
  q /= a.g.L;  // t (z cut) or z (t cut)
  const int z = d == 0 ? (side ? a.g.Lz - 1 : 0) : q;
  const int t = d == 0 ? q : (side ? a.g.T - 1 : 0);
  const int cb = xh + a.g.Lh * (y + a.g.L * (z + a.g.Lz * t));
  cx<R> w[6];
  if (d == 0) {
    if (side == 0) face_pack_site<R, NG, 2, 0>(a, cb, col * a.cstride, w);
    else face_pack_site<R, NG, 2, 1>(a, cb, col * a.cstride, w);
  } else {
    if (side == 0) face_pack_site<R, NG, 3, 0>(a, cb, col * a.cstride, w);
    else face_pack_site<R, NG, 3, 1>(a, cb, col * a.cstride, w);
  }
  R v[12];
#pragma unroll
  for (int i = 0; i < 6; i++) { v[2 * i] = w[i].re; v[2 * i + 1] = w[i].im; }
  store_reals<12>((V*)fo.send[d][side] + (int64_t)col * a.dd.gstride[d], a.dd.nface[d], f, v);
}

// Exterior pass: one thread per output site on a cut. The raw sum of the hops inside the domain (left in `out` by the
// interior pass) + the hop terms that arrived in the ghost buffers -> epilogue, store, fused reductions.
// Sites: first the two z-cut planes (z = 0, Lz-1: all xh, y, t), then the two t-cut planes without the sites already in
// the z-cut planes. blockIdx.y = column slot.
template <typename R, int NG, int MU> __device__ __forceinline__ void ghost_hops(const DslashArgs<R>& a, const Site& s, bool lo, bool hi, int f, int col, R* acc) {
  typedef typename Vec16<R>::T V;
  const int d = MU - 2;
  if (lo) {  // backward hop, finished by the sender: (1 - sig g_mu) U^dag psi
    R v[12];
    load_reals<12>((const V*)a.dd.ghost[d][0] + (int64_t)col * a.dd.gstride[d], a.dd.nface[d], f, v);
    cx<R> w[6];
#pragma unroll
    for (int i = 0; i < 6; i++) w[i] = mk<R>(a.dd.bc[d][0] * v[2 * i], a.dd.bc[d][0] * v[2 * i + 1]);
    recon_acc<R, MU>(w, -a.sig, acc);
  }
  if (hi) {  // forward hop: U_mu(x) times the projected half spinor of the neighbour
    R v[12];
    load_reals<12>((const V*)a.dd.ghost[d][1] + (int64_t)col * a.dd.gstride[d], a.dd.nface[d], f, v);
    cx<R> h[6], w[6], U[9];
#pragma unroll
    for (int i = 0; i < 6; i++) h[i] = mk<R>(a.dd.bc[d][1] * v[2 * i], a.dd.bc[d][1] * v[2 * i + 1]);
    load_link<R, NG, true>((const V*)a.U[a.par] + (int64_t)MU * Planes<R, NG>::N * a.g.Vh, a.g.Vh, s.cb, U);
    su3_mul_half<R, true>(U, h, w);
    recon_acc<R, MU>(w, a.sig, acc);
  }
}
template <typename R, int NG, int EPI, int CLOVER, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_ext_kernel(const DslashArgs<R> a) {
  if (a.skip && *a.skip) return;
  const Geom& g = a.g;
  const int zplane = g.Lh * g.L * g.T;                          // sites of one z-cut plane
  const int nzb = a.dd.part[0] ? 2 * zplane : 0;
  const int z0 = a.dd.part[0] ? 1 : 0, nzint = g.Lz - 2 * z0;    // z range of the t-cut planes
  const int tplane = g.Lh * g.L * nzint;
  const int ntb = a.dd.part[1] ? 2 * tplane : 0;
  int e = blockIdx.x * BLOCK + threadIdx.x;
  const bool active = e < nzb + ntb;
  Site s;
  s.xh = s.y = s.z = s.t = s.cb = 0;
  if (active) {
    if (e < nzb) {
      const int side = e >= zplane;
      e -= side * zplane;
      s.xh = e % g.Lh;
      e /= g.Lh;
      s.y = e % g.L;
      s.t = e / g.L;
      s.z = side ? g.Lz - 1 : 0;
    } else {
      e -= nzb;
      const int side = e >= tplane;
      e -= side * tplane;
      s.xh = e % g.Lh;
      e /= g.Lh;
      s.y = e % g.L;
      s.z = z0 + e / g.L;
      s.t = side ? g.T - 1 : 0;
    }
    s.cb = s.xh + g.Lh * (s.y + g.L * (s.z + g.Lz * s.t));
  }
  int colj[1], cofs[1];
  bool valid[1] = {true};
  colj[0] = a.col[blockIdx.y];
  cofs[0] = colj[0] * a.cstride;
  R o[1][24], r2[1][3];
  if (active) {
    load_reals<24>(a.out, g.Vh, s.cb + cofs[0], o[0]);
    const Nbr n = neighbours(g, a.par, s);
    if (a.dd.part[0]) ghost_hops<R, NG, 2>(a, s, n.wrap_zb, n.wrap_zf, s.xh + g.Lh * (s.y + g.L * s.t), colj[0], o[0]);
    if (a.dd.part[1]) ghost_hops<R, NG, 3>(a, s, n.wrap_tb, n.wrap_tf, s.xh + g.Lh * (s.y + g.L * s.z), colj[0], o[0]);
    dslash_epilogue<R, NG, EPI, CLOVER, 1, true>(a, s.cb, cofs, valid, o, r2);
    if (!stored_in_site<EPI, CLOVER>()) {
      if (a.g5) {
#pragma unroll
        for (int i = 12; i < 24; i++) o[0][i] = -o[0][i];
      }
      store_reals_s<24>(a.out, g.Vh, s.cb + cofs[0], o[0]);
    }
  }
  if (a.red_mode != 0) site_reductions<R, 1, BLOCK>(a, s, active, cofs, colj, valid, o, r2);
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
  else grid = dim3((unsigned)(((a.cb_end - a.sb0 * B + B - 1) / B) * a.ngroups), 1, 1);
  dslash_kernel<R, NG, EPI, CLOVER, NR, B, Tune<R, NR>::MINB, 0><<<grid, B, 0, s>>>(a);
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

// ---- launchers of the domain-decomposition passes (one column per thread; a.ncol columns through blockIdx) ----
template <typename R, int NG, int EPI, int CLOVER> static cudaError_t launch_dd_one(DslashArgs<R> a, int pass, cudaStream_t s) {
  const int B = Tune<R, 1>::BLOCK;
  if (pass == 0) {  // interior
    a.ngroups = a.ncol;
    dslash_kernel<R, NG, EPI, CLOVER, 1, B, Tune<R, 1>::MINB, 1><<<dim3((unsigned)(((a.g.Vh + B - 1) / B) * a.ngroups), 1, 1), B, 0, s>>>(a);
  } else {  // exterior
    const int z0 = a.dd.part[0] ? 1 : 0;
    const int nb = (a.dd.part[0] ? 2 * a.g.Lh * a.g.L * a.g.T : 0) + (a.dd.part[1] ? 2 * a.g.Lh * a.g.L * (a.g.Lz - 2 * z0) : 0);
    if (nb > 0) dslash_ext_kernel<R, NG, EPI, CLOVER, B, Tune<R, 1>::MINB><<<dim3((unsigned)((nb + B - 1) / B), (unsigned)a.ncol, 1), B, 0, s>>>(a);
  }
  return cudaGetLastError();
}
template <typename R, int NG> static cudaError_t launch_dd_epi(const DslashArgs<R>& a, int epi, int clover, int pass, cudaStream_t s) {
  switch (epi) {
    case EPI_HOP: return launch_dd_one<R, NG, EPI_HOP, CL_NONE>(a, pass, s);
    case EPI_AINV_HOP:
      if (clover == CL_TWISTED) return launch_dd_one<R, NG, EPI_AINV_HOP, CL_TWISTED>(a, pass, s);
      return clover ? launch_dd_one<R, NG, EPI_AINV_HOP, CL_CLOVER>(a, pass, s) : launch_dd_one<R, NG, EPI_AINV_HOP, CL_NONE>(a, pass, s);
    case EPI_A_XPAY: return clover ? launch_dd_one<R, NG, EPI_A_XPAY, CL_CLOVER>(a, pass, s) : launch_dd_one<R, NG, EPI_A_XPAY, CL_NONE>(a, pass, s);
    case EPI_XPAY: return launch_dd_one<R, NG, EPI_XPAY, CL_NONE>(a, pass, s);
    case EPI_AINV_XPAY:
      if (clover == CL_TWISTED) return launch_dd_one<R, NG, EPI_AINV_XPAY, CL_TWISTED>(a, pass, s);
      return clover ? launch_dd_one<R, NG, EPI_AINV_XPAY, CL_CLOVER>(a, pass, s) : launch_dd_one<R, NG, EPI_AINV_XPAY, CL_NONE>(a, pass, s);
  }
  return cudaErrorInvalidValue;
}
template <typename R, int NG> static cudaError_t launch_face_pack_t(const DslashArgs<R>& a, void* const (&send)[2][2], cudaStream_t s) {
  FaceOut<R> fo;
  for (int d = 0; d < 2; d++)
    for (int k = 0; k < 2; k++) fo.send[d][k] = send[d][k];
  const int nf = a.dd.nface[0] > a.dd.nface[1] ? a.dd.nface[0] : a.dd.nface[1];
  face_pack_kernel<R, NG, 128><<<dim3((unsigned)((nf + 127) / 128), 4, (unsigned)a.ncol), 128, 0, s>>>(a, fo);
  return cudaGetLastError();
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
