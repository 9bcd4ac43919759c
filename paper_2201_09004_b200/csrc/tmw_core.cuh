// tmw_core.cuh — per-site arithmetic of the twisted-mass Wilson(-clover) operator (arXiv:2201.09004 Eqs. (1)-(3),
// PAPER.md:58-67) for the CUDA kernels of libtmw.so: packed-layout loads/stores, spin projection to half
// spinors, SU(3) multiply with 12-real reconstruction, packed Hermitian 6x6 clover blocks, fused epilogues.
// This header is private to csrc/ and shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define TMW_HD __host__ __device__ __forceinline__

namespace tmw {

// ---------------------------------------------------------------------------------------------------------
// geometry of one parity of an L^3 x T lattice; cb = (x/2) + Lh*(y + L*(z + L*t))
// ---------------------------------------------------------------------------------------------------------
// A Geom describes either the whole lattice or one domain of a domain-decomposed context: a sub-lattice
// of extents L x L x Lz x T (x, y never split) whose site (x, y, z, t) is the global site (x, y, z + oz, t + ot); oz and ot
// are even, so local and global parity agree. For the whole lattice Lz = L, oz = ot = 0.
struct Geom {
  int L, T, Lh;    // x, y extent; t extent; L/2
  int Lz;          // z extent
  int oz, ot;      // origin of the domain in the global lattice (canonical-layout conversion only)
  int GT;          // global t extent (canonical-layout conversion only)
  int Vh;          // sites per parity (< 2^31)
  int sy, sz, st;  // cb strides of +1 in y, z, t
  // Thread -> site mapping of the stencil kernels. tiled = 0: CTA b covers cb in [b*BLOCK, (b+1)*BLOCK).
  // tiled = 1: a CTA covers a 4-D tile of 2^lx (in xh) x 2^ly x 2^lz x 2^lt = BLOCK sites, so that most neighbour
  // spinors of the tile are shared between its threads and hit in L1; tiles are ordered xh, y (blockIdx.x),
  // z (blockIdx.y), t (blockIdx.z), i.e. the sweep through the lattice is the same as in cb order.
  int tiled;
  int lx, ly, lz, lt;
  int ntx, nty;    // tiles along xh and y
  // Sweep order of the 1-D mapping (tiled = 0). zc = 0: site blocks in cb order, i.e. time slice after time slice. zc > 0
  // (a divisor of Lz with Lh*L*zc a multiple of the CTA size): the lattice is cut into Lz/zc slabs in z and the blocks go
  // through ALL time slices of one slab before the next slab, so that the -t / +t neighbours of a block are re-read
  // after 2*Lh*L*zc sites instead of 2*Lh*L*Lz: with many right-hand-side columns per launch a whole time slice of
  // every column no longer fits in L2 between the two reads. nbzt = CTAs per (slab, time slice).
  int zc, nbzt;
};

// coordinates of one site of a parity: x = 2*xh + ((y + z + t + par) & 1)
struct Site {
  int xh, y, z, t, cb;
};

// site of this thread; sblock = blockIdx.x stripped of the right-hand-side group (see dslash_kernel)
template <int BLOCK> __device__ __forceinline__ bool thread_site(const Geom& g, int sblock, Site& s) {
  const int tid = threadIdx.x;
  if (g.tiled) {
    const int by = sblock / g.ntx, bx = sblock - by * g.ntx;
    s.xh = (bx << g.lx) | (tid & ((1 << g.lx) - 1));
    int q = tid >> g.lx;
    s.y = (by << g.ly) | (q & ((1 << g.ly) - 1));
    q >>= g.ly;
    s.z = ((int)blockIdx.y << g.lz) | (q & ((1 << g.lz) - 1));
    q >>= g.lz;
    s.t = ((int)blockIdx.z << g.lt) | q;
    s.cb = s.xh + g.Lh * (s.y + g.L * (s.z + g.L * s.t));
    return true;
  }
  if (g.zc) {  // slab-major, then t, then the blocks of the slab's share of the time slice
    const int q = sblock / g.nbzt, j = sblock - q * g.nbzt;
    const int slab = q / g.T, t = q - slab * g.T;
    sblock = (t * (g.Lz / g.zc) + slab) * g.nbzt + j;
  }
  s.cb = sblock * BLOCK + tid;
  s.xh = s.cb % g.Lh;
  int q = s.cb / g.Lh;
  s.y = q % g.L;
  q /= g.L;
  s.z = q % g.Lz;
  s.t = q / g.Lz;
  return s.cb < g.Vh;
}

// ---------------------------------------------------------------------------------------------------------
// 16-byte vector access. A packed field of NREAL reals per site is stored as planes of 16-byte vectors:
// vector (k, cb) at index k*stride + cb holds reals [k*N, k*N+N) of the site, N = 4 (float) or 2 (double).
// ---------------------------------------------------------------------------------------------------------
template <typename R> struct Vec16;
template <> struct Vec16<float> { typedef float4 T; enum { N = 4 }; };
template <> struct Vec16<double> { typedef double2 T; enum { N = 2 }; };

template <typename R, int NREAL> struct Planes { enum { N = (NREAL + Vec16<R>::N - 1) / Vec16<R>::N }; };

TMW_HD float4 ldv(const float4* p) {
#ifdef __CUDA_ARCH__
  return __ldg(p);
#else
  return *p;
#endif
}
TMW_HD double2 ldv(const double2* p) {
#ifdef __CUDA_ARCH__
  return __ldg(p);
#else
  return *p;
#endif
}

// Loads of data that a kernel touches exactly once (links, clover blocks): TMW_LD_STREAM selects the cache policy
//   0: ld.global.nc (same as the spinor loads)   1: ld.global.cs (evict-first)   2: ld.global.nc.L1::no_allocate
#ifndef TMW_LD_STREAM
#define TMW_LD_STREAM 1  // measured on B200: -0.7 % hop, -2 % K2 vs ld.global.nc
#endif
// Stores of the stencil output: TMW_ST_STREAM 0: st.global   1: st.global.cs (evict-first)
#ifndef TMW_ST_STREAM
#define TMW_ST_STREAM 0
#endif
TMW_HD float4 ldv_s(const float4* p) {
#if defined(__CUDA_ARCH__) && TMW_LD_STREAM == 1
  return __ldcs(p);
#elif defined(__CUDA_ARCH__) && TMW_LD_STREAM == 2
  float4 q;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(q.x), "=f"(q.y), "=f"(q.z), "=f"(q.w) : "l"(p));
  return q;
#else
  return ldv(p);
#endif
}
TMW_HD double2 ldv_s(const double2* p) {
#if defined(__CUDA_ARCH__) && TMW_LD_STREAM == 1
  return __ldcs(p);
#elif defined(__CUDA_ARCH__) && TMW_LD_STREAM == 2
  double2 q;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(q.x), "=d"(q.y) : "l"(p));
  return q;
#else
  return ldv(p);
#endif
}
TMW_HD void stv_s(float4* p, float4 q) {
#if defined(__CUDA_ARCH__) && TMW_ST_STREAM == 1
  __stcs(p, q);
#else
  *p = q;
#endif
}
TMW_HD void stv_s(double2* p, double2 q) {
#if defined(__CUDA_ARCH__) && TMW_ST_STREAM == 1
  __stcs(p, q);
#else
  *p = q;
#endif
}

template <int NREAL> TMW_HD void load_reals_s(const void* base, int64_t stride, int64_t idx, float* v) {
  const float4* p = (const float4*)base + idx;
#pragma unroll
  for (int k = 0; k < (NREAL + 3) / 4; k++) {
    float4 q = ldv_s(p + k * stride);
    v[4 * k] = q.x;
    v[4 * k + 1] = q.y;
    if (4 * k + 2 < NREAL) v[4 * k + 2] = q.z;
    if (4 * k + 3 < NREAL) v[4 * k + 3] = q.w;
  }
}
template <int NREAL> TMW_HD void load_reals_s(const void* base, int64_t stride, int64_t idx, double* v) {
  const double2* p = (const double2*)base + idx;
#pragma unroll
  for (int k = 0; k < NREAL / 2; k++) {
    double2 q = ldv_s(p + k * stride);
    v[2 * k] = q.x;
    v[2 * k + 1] = q.y;
  }
}
template <int NREAL> TMW_HD void store_reals_s(void* base, int64_t stride, int64_t idx, const float* v) {
  float4* p = (float4*)base + idx;
#pragma unroll
  for (int k = 0; k < (NREAL + 3) / 4; k++) {
    float4 q;
    q.x = v[4 * k];
    q.y = v[4 * k + 1];
    q.z = (4 * k + 2 < NREAL) ? v[4 * k + 2] : 0.f;
    q.w = (4 * k + 3 < NREAL) ? v[4 * k + 3] : 0.f;
    stv_s(p + k * stride, q);
  }
}
template <int NREAL> TMW_HD void store_reals_s(void* base, int64_t stride, int64_t idx, const double* v) {
  double2* p = (double2*)base + idx;
#pragma unroll
  for (int k = 0; k < NREAL / 2; k++) {
    double2 q;
    q.x = v[2 * k];
    q.y = v[2 * k + 1];
    stv_s(p + k * stride, q);
  }
}

template <int NREAL> TMW_HD void load_reals(const void* base, int64_t stride, int64_t idx, float* v) {
  const float4* p = (const float4*)base + idx;
#pragma unroll
  for (int k = 0; k < (NREAL + 3) / 4; k++) {
    float4 q = ldv(p + k * stride);
    v[4 * k] = q.x;
    v[4 * k + 1] = q.y;
    if (4 * k + 2 < NREAL) v[4 * k + 2] = q.z;
    if (4 * k + 3 < NREAL) v[4 * k + 3] = q.w;
  }
}
template <int NREAL> TMW_HD void load_reals(const void* base, int64_t stride, int64_t idx, double* v) {
  const double2* p = (const double2*)base + idx;
#pragma unroll
  for (int k = 0; k < NREAL / 2; k++) {
    double2 q = ldv(p + k * stride);
    v[2 * k] = q.x;
    v[2 * k + 1] = q.y;
  }
}
template <int NREAL> TMW_HD void store_reals(void* base, int64_t stride, int64_t idx, const float* v) {
  float4* p = (float4*)base + idx;
#pragma unroll
  for (int k = 0; k < (NREAL + 3) / 4; k++) {
    float4 q;
    q.x = v[4 * k];
    q.y = v[4 * k + 1];
    q.z = (4 * k + 2 < NREAL) ? v[4 * k + 2] : 0.f;
    q.w = (4 * k + 3 < NREAL) ? v[4 * k + 3] : 0.f;
    p[k * stride] = q;
  }
}
template <int NREAL> TMW_HD void store_reals(void* base, int64_t stride, int64_t idx, const double* v) {
  double2* p = (double2*)base + idx;
#pragma unroll
  for (int k = 0; k < NREAL / 2; k++) {
    double2 q;
    q.x = v[2 * k];
    q.y = v[2 * k + 1];
    p[k * stride] = q;
  }
}

// ---------------------------------------------------------------------------------------------------------
// complex helpers on (re, im) pairs held in plain arrays: z[2*i] = re, z[2*i+1] = im
// ---------------------------------------------------------------------------------------------------------
template <typename R> struct cx {
  R re, im;
};
template <typename R> TMW_HD cx<R> mk(R re, R im) { cx<R> z; z.re = re; z.im = im; return z; }
template <typename R> TMW_HD cx<R> operator+(cx<R> a, cx<R> b) { return mk<R>(a.re + b.re, a.im + b.im); }
template <typename R> TMW_HD cx<R> operator-(cx<R> a, cx<R> b) { return mk<R>(a.re - b.re, a.im - b.im); }
template <typename R> TMW_HD cx<R> operator*(cx<R> a, cx<R> b) {
  return mk<R>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <typename R> TMW_HD cx<R> conj(cx<R> a) { return mk<R>(a.re, -a.im); }
// acc += a*b
template <typename R> TMW_HD void cmad(cx<R>& acc, cx<R> a, cx<R> b) {
  acc.re += a.re * b.re;
  acc.re -= a.im * b.im;
  acc.im += a.re * b.im;
  acc.im += a.im * b.re;
}
// acc += conj(a)*b
template <typename R> TMW_HD void cmadc(cx<R>& acc, cx<R> a, cx<R> b) {
  acc.re += a.re * b.re;
  acc.re += a.im * b.im;
  acc.im += a.re * b.im;
  acc.im -= a.im * b.re;
}

// ---------------------------------------------------------------------------------------------------------
// SU(3) link from NG stored reals (rows 0,1 [+ row 2]); NG = 12 rebuilds row 2 = conj(row0 x row1)
// ---------------------------------------------------------------------------------------------------------
// STREAM: the link is read by this thread only (evict-first load, TMW_LD_STREAM); otherwise other CTAs (column groups)
// read the same link and it should stay in L2 (plain read-only load)
template <typename R, int NG, bool STREAM> TMW_HD void load_link(const void* base, int64_t stride, int64_t idx, cx<R> (&U)[9]) {
  R g[(NG == 12) ? 12 : 20];
  if (STREAM) load_reals_s<NG>(base, stride, idx, g);
  else load_reals<NG>(base, stride, idx, g);
#pragma unroll
  for (int i = 0; i < NG / 2; i++) U[i] = mk<R>(g[2 * i], g[2 * i + 1]);
  if (NG == 12) {
    U[6] = conj(U[1] * U[5] - U[2] * U[4]);
    U[7] = conj(U[2] * U[3] - U[0] * U[5]);
    U[8] = conj(U[0] * U[4] - U[1] * U[3]);
  }
}

// ---------------------------------------------------------------------------------------------------------
// One hop of Eq. (2): acc += P(U h), with the spin projector 1 + sig*gamma_MU of rank 2 (DeGrand-Rossi basis):
// only rows h0, h1 go through the colour multiply; rows 2, 3 of the result are +-1/+-i multiples of them.
//   MU = x: h0 = p0 + sig*i*p3, h1 = p1 + sig*i*p2, row2 = -sig*i*h1, row3 = -sig*i*h0
//   MU = y: h0 = p0 - sig*p3,   h1 = p1 + sig*p2,   row2 = +sig*h1,   row3 = -sig*h0
//   MU = z: h0 = p0 + sig*i*p2, h1 = p1 - sig*i*p3, row2 = -sig*i*h0, row3 = +sig*i*h1
//   MU = t: h0 = p0 + sig*p2,   h1 = p1 + sig*p3,   row2 = +sig*h0,   row3 = +sig*h1
// FWD: colour matrix U (forward hop, U_mu(x)); else U^dagger (backward hop, U_mu(x-mu)^dagger).
// bc multiplies the whole hop (antiperiodic time boundary: -1 when the hop wraps).
// psi: 24 reals of the neighbour spinor, index 2*(3*spin+colour)+ri. acc: 24 reals.
// ---------------------------------------------------------------------------------------------------------
template <typename R, int MU, bool FWD> TMW_HD void hop(const R* psi, const cx<R> (&U)[9], R sig, R bc, R* acc) {
  cx<R> h[6];  // h[3*s + c], s = 0,1
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const cx<R> p0 = mk<R>(psi[2 * c], psi[2 * c + 1]);
    const cx<R> p1 = mk<R>(psi[6 + 2 * c], psi[6 + 2 * c + 1]);
    const cx<R> p2 = mk<R>(psi[12 + 2 * c], psi[12 + 2 * c + 1]);
    const cx<R> p3 = mk<R>(psi[18 + 2 * c], psi[18 + 2 * c + 1]);
    if (MU == 0) {
      h[c] = mk<R>(p0.re - sig * p3.im, p0.im + sig * p3.re);
      h[3 + c] = mk<R>(p1.re - sig * p2.im, p1.im + sig * p2.re);
    } else if (MU == 1) {
      h[c] = mk<R>(p0.re - sig * p3.re, p0.im - sig * p3.im);
      h[3 + c] = mk<R>(p1.re + sig * p2.re, p1.im + sig * p2.im);
    } else if (MU == 2) {
      h[c] = mk<R>(p0.re - sig * p2.im, p0.im + sig * p2.re);
      h[3 + c] = mk<R>(p1.re + sig * p3.im, p1.im - sig * p3.re);
    } else {
      h[c] = mk<R>(p0.re + sig * p2.re, p0.im + sig * p2.im);
      h[3 + c] = mk<R>(p1.re + sig * p3.re, p1.im + sig * p3.im);
    }
  }
  if (MU == 3) {
#pragma unroll
    for (int i = 0; i < 6; i++) { h[i].re *= bc; h[i].im *= bc; }
  }
#pragma unroll
  for (int s = 0; s < 2; s++) {
#pragma unroll
    for (int a = 0; a < 3; a++) {
      cx<R> w = mk<R>((R)0, (R)0);
#pragma unroll
      for (int b = 0; b < 3; b++) {
        if (FWD) cmad(w, U[3 * a + b], h[3 * s + b]);
        else cmadc(w, U[3 * b + a], h[3 * s + b]);
      }
      // rows 0,1
      acc[2 * (3 * s + a)] += w.re;
      acc[2 * (3 * s + a) + 1] += w.im;
      // rows 2,3
      if (MU == 0) {  // row2 = -sig*i*h1, row3 = -sig*i*h0 : -i*w = (w.im, -w.re)
        const int r = (s == 0) ? 3 : 2;
        acc[2 * (3 * r + a)] += sig * w.im;
        acc[2 * (3 * r + a) + 1] -= sig * w.re;
      } else if (MU == 1) {  // row2 = +sig*h1, row3 = -sig*h0
        if (s == 0) {
          acc[2 * (9 + a)] -= sig * w.re;
          acc[2 * (9 + a) + 1] -= sig * w.im;
        } else {
          acc[2 * (6 + a)] += sig * w.re;
          acc[2 * (6 + a) + 1] += sig * w.im;
        }
      } else if (MU == 2) {  // row2 = -sig*i*h0, row3 = +sig*i*h1
        if (s == 0) {
          acc[2 * (6 + a)] += sig * w.im;
          acc[2 * (6 + a) + 1] -= sig * w.re;
        } else {
          acc[2 * (9 + a)] -= sig * w.im;
          acc[2 * (9 + a) + 1] += sig * w.re;
        }
      } else {  // row2 = +sig*h0, row3 = +sig*h1
        acc[2 * (3 * (s + 2) + a)] += sig * w.re;
        acc[2 * (3 * (s + 2) + a) + 1] += sig * w.im;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// hop<> for TWO right-hand-side columns at once on sm_100a's packed fp32 pairs (FFMA2 / FADD2 / FMUL2: one issue slot,
// two lanes): every per-column quantity is a float2 with .x = column A, .y = column B; the link is shared, so its reals
// are broadcast pairs (u, u). The spin projection stays scalar (its results are written straight into the pair halves);
// the colour multiply accumulates sum u.re h and sum u.im h separately and combines them once per output
// (w = A -+ i B for U / U^dag), so that no negated copies of the link are needed; the reconstruction adds sig*w pairs.
// Per hop and column: 12 scalar + 54 packed instructions instead of 108 scalar ones.
// ---------------------------------------------------------------------------------------------------------
#ifndef TMW_PACK2
#define TMW_PACK2 1
#endif
struct LinkPairs {
  float2 re[9], im[9];  // (u.re, u.re), (u.im, u.im)
};
// bc (the antiperiodic sign of a wrapping t hop) is folded into the broadcast link
__device__ __forceinline__ void link_pairs(const cx<float> (&U)[9], float bc, LinkPairs& P) {
#pragma unroll
  for (int i = 0; i < 9; i++) {
    const float r = bc * U[i].re, m = bc * U[i].im;
    P.re[i] = make_float2(r, r);
    P.im[i] = make_float2(m, m);
  }
}
#if defined(__CUDA_ARCH__) && __CUDA_ARCH__ >= 1000
#define TMW_FMA2(a, b, c) __ffma2_rn((a), (b), (c))
#define TMW_MUL2(a, b) __fmul2_rn((a), (b))
#define TMW_ADD2(a, b) __fadd2_rn((a), (b))
#else
#define TMW_FMA2(a, b, c) make_float2((a).x * (b).x + (c).x, (a).y * (b).y + (c).y)
#define TMW_MUL2(a, b) make_float2((a).x * (b).x, (a).y * (b).y)
#define TMW_ADD2(a, b) make_float2((a).x + (b).x, (a).y + (b).y)
#endif
template <int MU, bool FWD> __device__ __forceinline__ void hop2(const float* psiA, const float* psiB, const LinkPairs& P, float sig, float2* acc) {
  float2 hr[6], hi[6];  // h[3*s + c] of both columns, real and imaginary parts
#pragma unroll
  for (int col = 0; col < 2; col++) {
    const float* psi = col ? psiB : psiA;
#pragma unroll
    for (int c = 0; c < 3; c++) {
      const float p0r = psi[2 * c], p0i = psi[2 * c + 1], p1r = psi[6 + 2 * c], p1i = psi[6 + 2 * c + 1];
      const float p2r = psi[12 + 2 * c], p2i = psi[12 + 2 * c + 1], p3r = psi[18 + 2 * c], p3i = psi[18 + 2 * c + 1];
      float ar, ai, br, bi;  // h[c], h[3 + c]
      if (MU == 0) { ar = p0r - sig * p3i; ai = p0i + sig * p3r; br = p1r - sig * p2i; bi = p1i + sig * p2r; }
      else if (MU == 1) { ar = p0r - sig * p3r; ai = p0i - sig * p3i; br = p1r + sig * p2r; bi = p1i + sig * p2i; }
      else if (MU == 2) { ar = p0r - sig * p2i; ai = p0i + sig * p2r; br = p1r + sig * p3i; bi = p1i - sig * p3r; }
      else { ar = p0r + sig * p2r; ai = p0i + sig * p2i; br = p1r + sig * p3r; bi = p1i + sig * p3i; }
      if (col == 0) { hr[c].x = ar; hi[c].x = ai; hr[3 + c].x = br; hi[3 + c].x = bi; }
      else { hr[c].y = ar; hi[c].y = ai; hr[3 + c].y = br; hi[3 + c].y = bi; }
    }
  }
  const float2 sg = make_float2(sig, sig), nsg = make_float2(-sig, -sig), m1 = make_float2(-1.f, -1.f);
#pragma unroll
  for (int s = 0; s < 2; s++) {
#pragma unroll
    for (int a = 0; a < 3; a++) {
      // A = sum_b u.re h_b, B = sum_b u.im (h_b.im, h_b.re); w = A + i u.im h = (A.re - B.re, A.im + B.im) for U,
      // (A.re + B.re, A.im - B.im) for U^dag (u = U[a][b] or U[b][a])
      const int i0 = FWD ? 3 * a : a, st = FWD ? 1 : 3;
      float2 Ar = TMW_MUL2(P.re[i0], hr[3 * s]), Ai = TMW_MUL2(P.re[i0], hi[3 * s]);
      float2 Br = TMW_MUL2(P.im[i0], hi[3 * s]), Bi = TMW_MUL2(P.im[i0], hr[3 * s]);
#pragma unroll
      for (int b = 1; b < 3; b++) {
        Ar = TMW_FMA2(P.re[i0 + b * st], hr[3 * s + b], Ar);
        Ai = TMW_FMA2(P.re[i0 + b * st], hi[3 * s + b], Ai);
        Br = TMW_FMA2(P.im[i0 + b * st], hi[3 * s + b], Br);
        Bi = TMW_FMA2(P.im[i0 + b * st], hr[3 * s + b], Bi);
      }
      float2 wr, wi;
      if (FWD) { wr = TMW_FMA2(m1, Br, Ar); wi = TMW_ADD2(Ai, Bi); }
      else { wr = TMW_ADD2(Ar, Br); wi = TMW_FMA2(m1, Bi, Ai); }
      float2* o = acc + 2 * (3 * s + a);
      o[0] = TMW_ADD2(o[0], wr);
      o[1] = TMW_ADD2(o[1], wi);
      if (MU == 0) {  // row (s == 0 ? 3 : 2) += -sig * i * w = sig * (w.im, -w.re)
        float2* q = acc + 2 * (3 * (s == 0 ? 3 : 2) + a);
        q[0] = TMW_FMA2(sg, wi, q[0]);
        q[1] = TMW_FMA2(nsg, wr, q[1]);
      } else if (MU == 1) {  // row 3 -= sig * w (s = 0); row 2 += sig * w (s = 1)
        float2* q = acc + 2 * ((s == 0 ? 9 : 6) + a);
        q[0] = TMW_FMA2(s == 0 ? nsg : sg, wr, q[0]);
        q[1] = TMW_FMA2(s == 0 ? nsg : sg, wi, q[1]);
      } else if (MU == 2) {  // row 2 += -sig * i * w (s = 0); row 3 += sig * i * w (s = 1)
        float2* q = acc + 2 * ((s == 0 ? 6 : 9) + a);
        q[0] = TMW_FMA2(s == 0 ? sg : nsg, wi, q[0]);
        q[1] = TMW_FMA2(s == 0 ? nsg : sg, wr, q[1]);
      } else {  // row s + 2 += sig * w
        float2* q = acc + 2 * (3 * (s + 2) + a);
        q[0] = TMW_FMA2(sg, wr, q[0]);
        q[1] = TMW_FMA2(sg, wi, q[1]);
      }
    }
  }
}

// The three stages of hop<> as separate functions, for the domain-decomposed stencil, where the spin
// projection (and, for backward hops, the colour multiply) of a hop that crosses a domain boundary happens on the
// sending side and only the 12 reals of the half spinor travel.
template <typename R, int MU> TMW_HD void project_half(const R* psi, R sig, cx<R> (&h)[6]) {
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const cx<R> p0 = mk<R>(psi[2 * c], psi[2 * c + 1]);
    const cx<R> p1 = mk<R>(psi[6 + 2 * c], psi[6 + 2 * c + 1]);
    const cx<R> p2 = mk<R>(psi[12 + 2 * c], psi[12 + 2 * c + 1]);
    const cx<R> p3 = mk<R>(psi[18 + 2 * c], psi[18 + 2 * c + 1]);
    if (MU == 0) {
      h[c] = mk<R>(p0.re - sig * p3.im, p0.im + sig * p3.re);
      h[3 + c] = mk<R>(p1.re - sig * p2.im, p1.im + sig * p2.re);
    } else if (MU == 1) {
      h[c] = mk<R>(p0.re - sig * p3.re, p0.im - sig * p3.im);
      h[3 + c] = mk<R>(p1.re + sig * p2.re, p1.im + sig * p2.im);
    } else if (MU == 2) {
      h[c] = mk<R>(p0.re - sig * p2.im, p0.im + sig * p2.re);
      h[3 + c] = mk<R>(p1.re + sig * p3.im, p1.im - sig * p3.re);
    } else {
      h[c] = mk<R>(p0.re + sig * p2.re, p0.im + sig * p2.im);
      h[3 + c] = mk<R>(p1.re + sig * p3.re, p1.im + sig * p3.im);
    }
  }
}
// w = U h (FWD) or U^dagger h, for both spin rows of the half spinor
template <typename R, bool FWD> TMW_HD void su3_mul_half(const cx<R> (&U)[9], const cx<R> (&h)[6], cx<R> (&w)[6]) {
#pragma unroll
  for (int s = 0; s < 2; s++)
#pragma unroll
    for (int a = 0; a < 3; a++) {
      cx<R> t = mk<R>((R)0, (R)0);
#pragma unroll
      for (int b = 0; b < 3; b++) {
        if (FWD) cmad(t, U[3 * a + b], h[3 * s + b]);
        else cmadc(t, U[3 * b + a], h[3 * s + b]);
      }
      w[3 * s + a] = t;
    }
}
// acc += the 4-spinor rebuilt from the half spinor w of the projector 1 + sig*gamma_MU (table above hop<>)
template <typename R, int MU> TMW_HD void recon_acc(const cx<R> (&w6)[6], R sig, R* acc) {
#pragma unroll
  for (int s = 0; s < 2; s++)
#pragma unroll
    for (int a = 0; a < 3; a++) {
      const cx<R> w = w6[3 * s + a];
      acc[2 * (3 * s + a)] += w.re;
      acc[2 * (3 * s + a) + 1] += w.im;
      if (MU == 0) {
        const int r = (s == 0) ? 3 : 2;
        acc[2 * (3 * r + a)] += sig * w.im;
        acc[2 * (3 * r + a) + 1] -= sig * w.re;
      } else if (MU == 1) {
        if (s == 0) {
          acc[2 * (9 + a)] -= sig * w.re;
          acc[2 * (9 + a) + 1] -= sig * w.im;
        } else {
          acc[2 * (6 + a)] += sig * w.re;
          acc[2 * (6 + a) + 1] += sig * w.im;
        }
      } else if (MU == 2) {
        if (s == 0) {
          acc[2 * (6 + a)] += sig * w.im;
          acc[2 * (6 + a) + 1] -= sig * w.re;
        } else {
          acc[2 * (9 + a)] -= sig * w.im;
          acc[2 * (9 + a) + 1] += sig * w.re;
        }
      } else {
        acc[2 * (3 * (s + 2) + a)] += sig * w.re;
        acc[2 * (3 * (s + 2) + a) + 1] += sig * w.im;
      }
    }
}

// ---------------------------------------------------------------------------------------------------------
// Packed Hermitian 6x6 block (36 reals: 6 real diagonal, then 15 strictly-lower complex entries row-major,
// entry (i,j), i>j, at 6 + 2*(i*(i-1)/2 + j)) times a 6-vector: out = B v.
// v, out: 12 reals = 6 complex, index i = 3*(spin mod 2) + colour of one chirality.
// ---------------------------------------------------------------------------------------------------------
template <typename R> TMW_HD void herm6_mul(const R* B, const R* v, R* out) {
#pragma unroll
  for (int i = 0; i < 6; i++) {
    R re = B[i] * v[2 * i], im = B[i] * v[2 * i + 1];
#pragma unroll
    for (int j = 0; j < 6; j++) {
      if (j < i) {
        const int k = 6 + 2 * (i * (i - 1) / 2 + j);
        re += B[k] * v[2 * j] - B[k + 1] * v[2 * j + 1];
        im += B[k] * v[2 * j + 1] + B[k + 1] * v[2 * j];
      } else if (j > i) {
        const int k = 6 + 2 * (j * (j - 1) / 2 + i);
        re += B[k] * v[2 * j] + B[k + 1] * v[2 * j + 1];
        im += B[k] * v[2 * j + 1] - B[k + 1] * v[2 * j];
      }
    }
    out[2 * i] = re;
    out[2 * i + 1] = im;
  }
}

// ---------------------------------------------------------------------------------------------------------
// The site-diagonal part A of D and its inverse.
//   A v = C v + i*tw_chi*v   per chirality chi (upper = spins 0,1; lower = spins 2,3)
//   no clover: C = diag (= -(4 + Re m)); clover: C = packed Hermitian block that includes the diagonal.
//   tw_up = -Im m, tw_lo = +Im m for D with the gamma5 twist (C4); signs flip for D^dagger; both = -Im m (D) for
//   the complex-scalar reading.
//   A^{-1}: no clover: complex scalar (inv_re, inv_im_chi) per chirality. Clover, tw = 0: packed C^{-1}.
//   Clover with twist ("complex diagonal part"): (C + i tw)^{-1} = (C - i tw) (C^2 + tw^2)^{-1};
//   the Hermitian (C^2 + tw^2)^{-1} is what `cinv` holds then, and C is read as well.
// ---------------------------------------------------------------------------------------------------------
template <typename R> struct Diag {
  R diag;                 // -(4 + Re m), no-clover case
  R tw_up, tw_lo;         // i*tw added per chirality
  R inv_re, inv_im_up, inv_im_lo;  // no-clover inverse scalars
  int twisted_clover;     // clover && tw != 0
  const void* c[2];       // packed C blocks, per parity: [18 or 36 planes][Vh]
  const void* cinv[2];    // packed inverse blocks (even parity only in practice)
};

// out = A v at site cb of parity par (v, out: 24 reals; may not alias)
template <typename R, bool CLOVER> TMW_HD void apply_A(const Diag<R>& d, int par, int64_t Vh, int64_t cb, const R* v, R* out) {
  if (CLOVER) {
    const int NPB = Planes<R, 36>::N;  // planes per block
#pragma unroll
    for (int b = 0; b < 2; b++) {
      R B[36];
      load_reals_s<36>((const typename Vec16<R>::T*)d.c[par] + (int64_t)b * NPB * Vh, Vh, cb, B);
      herm6_mul(B, v + 12 * b, out + 12 * b);
    }
  } else {
#pragma unroll
    for (int i = 0; i < 24; i++) out[i] = d.diag * v[i];
  }
#pragma unroll
  for (int i = 0; i < 6; i++) {
    out[2 * i] -= d.tw_up * v[2 * i + 1];
    out[2 * i + 1] += d.tw_up * v[2 * i];
    out[12 + 2 * i] -= d.tw_lo * v[12 + 2 * i + 1];
    out[12 + 2 * i + 1] += d.tw_lo * v[12 + 2 * i];
  }
}

// out = A^{-1} v
template <typename R, bool CLOVER> TMW_HD void apply_Ainv(const Diag<R>& d, int par, int64_t Vh, int64_t cb, const R* v, R* out) {
  if (CLOVER) {
    const int NPB = Planes<R, 36>::N;
#pragma unroll
    for (int b = 0; b < 2; b++) {
      R B[36];
      load_reals_s<36>((const typename Vec16<R>::T*)d.cinv[par] + (int64_t)b * NPB * Vh, Vh, cb, B);
      if (!d.twisted_clover) {
        herm6_mul(B, v + 12 * b, out + 12 * b);
      } else {
        R w[12];
        herm6_mul(B, v + 12 * b, w);
        load_reals_s<36>((const typename Vec16<R>::T*)d.c[par] + (int64_t)b * NPB * Vh, Vh, cb, B);
        herm6_mul(B, w, out + 12 * b);
        const R tw = b ? d.tw_lo : d.tw_up;  // (C - i tw) w
#pragma unroll
        for (int i = 0; i < 6; i++) {
          out[12 * b + 2 * i] += tw * w[2 * i + 1];
          out[12 * b + 2 * i + 1] -= tw * w[2 * i];
        }
      }
    }
  } else {
#pragma unroll
    for (int i = 0; i < 6; i++) {
      out[2 * i] = d.inv_re * v[2 * i] - d.inv_im_up * v[2 * i + 1];
      out[2 * i + 1] = d.inv_re * v[2 * i + 1] + d.inv_im_up * v[2 * i];
      out[12 + 2 * i] = d.inv_re * v[12 + 2 * i] - d.inv_im_lo * v[12 + 2 * i + 1];
      out[12 + 2 * i + 1] = d.inv_re * v[12 + 2 * i + 1] + d.inv_im_lo * v[12 + 2 * i];
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// The stencil. Epilogues (h = 1/2 sum of the 8 hops = the hopping block H_{p pbar} applied to `in`):
// ---------------------------------------------------------------------------------------------------------
enum { MAXCOL = 16 };  // most right-hand sides per call

// kind of site-diagonal part a stencil kernel is compiled for: no clover (a complex scalar per chirality), clover, or
// clover with a twist, whose inverse is two factors. A compile-time choice: as a runtime branch the
// two-factor path cost the common K1 kernel 32 bytes of register spills.
enum { CL_NONE = 0, CL_CLOVER = 1, CL_TWISTED = 2 };

enum { EPI_HOP = 0,        // out = h
       EPI_AINV_HOP = 1,   // out = A^{-1} h                      (K1 of the Schur operator)
       EPI_A_XPAY = 2,     // out = A aux + sgn*h                 (K2: sgn = -1; full apply: sgn = +1)
       EPI_XPAY = 3,       // out = aux + sgn*h                   (source preparation)
       EPI_AINV_XPAY = 4   // out = A^{-1} (aux + sgn*h)          (solution reconstruction)
};

// Domain decomposition: what a stencil launch on ONE domain needs to know about its cuts. Directions
// z (index 0) and t (index 1) may be partitioned. ghost[d][0] ("lo") holds, for the output sites at local coordinate 0,
// the finished backward hop term (1 - sig g_mu) U_mu(x-mu)^dag psi(x-mu) as a half spinor (projected AND multiplied by
// the neighbour, who owns that link); ghost[d][1] ("hi") holds, for the sites at the last local coordinate, the
// projected half spinor (1 + sig g_mu) psi(x+mu) of the forward hop (this side multiplies by its own U_mu(x)).
// 12 reals per face site: vector (k, f) of column c at index c*gstride[d] + k*nface[d] + f, k < 12/N planes,
// face index f = xh + Lh*(y + L*t) (z cut) or xh + Lh*(y + L*z) (t cut) — the same on both sides of a cut.
template <typename R> struct DDArgs {
  int part[2];              // is z / t partitioned
  const void* ghost[2][2];  // [direction][lo, hi] receive buffers
  R bc[2][2];               // factor on the ghost term: -1 on the physical (antiperiodic) time boundary, else +1
  int nface[2];             // face sites per parity
  int gstride[2];           // 16-byte vectors per column in a ghost buffer
};

template <typename R> struct DslashArgs {
  const void* in;    // packed spinor, parity 1-par
  void* out;         // packed spinor, parity par
  const void* aux;   // packed spinor, parity par (EPI >= 2)
  const void* U[2];  // packed gauge per parity: [mu][planes][Vh]
  Geom g;
  int par;           // parity of the output sites
  R sig;             // +1 for D, -1 for D^dagger (sign of gamma_mu in the projectors)
  R coef;            // 1/2 * sgn
  int g5;            // multiply the result by gamma5 = diag(1,1,-1,-1) (the fused gamma5 D_w of PAPER.md:315)
  Diag<R> d;
  // fused reductions (kernel wrapper): red_mode 0 none; 1: red[0..1] += <dotv, out>; 2: red[0..1] += <out, aux>, red[2] += <out,out>;
  // 3: red[2] += |dotv - out|^2 (out may then be null: nothing is stored); 4: as 2 plus red[3..4] += <dotv, out>,
  // red[5..6] += <dotv, aux>
  int red_mode;
  const void* dotv;
  double* red;
  // right-hand-side columns (the "12 columns" of PAPER.md:78): slot j of this launch works on column
  // col[j]; in/out/aux/dotv of column c start c*cstride 16-byte vectors after the base pointers, its reduction
  // target red_stride doubles after red. One thread does NR consecutive slots of one site (links and clover blocks
  // are loaded once for the NR columns); CTAs of the ngroups = ceil(ncol/NR) slot groups of one site block are
  // adjacent in blockIdx.x, so the groups after the first find the links in L2.
  int ncol, ngroups;
  // a launch may cover only the site blocks [sb0, ...) up to checkerboard index cb_end (a t-slab of the lattice: the
  // pipelined host-pointer path of tmw_apply); a normal launch has sb0 = 0, cb_end = Vh
  int sb0, cb_end;
  int cstride;  // 16-byte vectors per column; (columns in the buffers) * cstride < 2^31 (checked by the host)
  int red_stride;
  unsigned char col[MAXCOL];
  // launched one iteration ahead of the host's look at the solver scalars: if *skip != 0 the kernel returns at once (the
  // device has decided that the host must act first, tmw_internal.h launch_sc_begin_iter); null: never skipped
  const int* skip;
  // L2 prefetch distance in site blocks (0: off): a thread also issues prefetch.global.L2 for the 8 links of its lane's site in
  // block sblock + pf_blocks, so that the links - the loads of the stencil that always miss to DRAM - are L2 hits when that
  // block's CTA runs (tmw_options.prefetch)
  int pf_blocks;
  DDArgs<R> dd;      // read only by the domain-decomposition kernels (DD != 0)
};

// neighbour checkerboard indices and the time-boundary sign
struct Nbr {
  int fwd[4], bwd[4];
  bool wrap_tf, wrap_tb;  // the +t / -t hop leaves the (local) lattice
  bool wrap_zf, wrap_zb;  // the +z / -z hop leaves the (local) lattice
};
TMW_HD Nbr neighbours(const Geom& g, int par, const Site& s) {
  Nbr n;
  const int xh = s.xh, y = s.y, z = s.z, t = s.t, cb = s.cb;
  const int o = (y + z + t + par) & 1;  // x = 2*xh + o
  // x+1 -> xh + o (wrap to 0), x-1 -> xh + o - 1 (wrap to Lh-1)
  const int xf = xh + o, xb = xh + o - 1;
  n.fwd[0] = cb - xh + (xf == g.Lh ? 0 : xf);
  n.bwd[0] = cb - xh + (xb < 0 ? g.Lh - 1 : xb);
  n.fwd[1] = (y == g.L - 1) ? cb - (g.L - 1) * g.sy : cb + g.sy;
  n.bwd[1] = (y == 0) ? cb + (g.L - 1) * g.sy : cb - g.sy;
  n.wrap_zf = (z == g.Lz - 1);
  n.wrap_zb = (z == 0);
  n.fwd[2] = n.wrap_zf ? cb - (g.Lz - 1) * g.sz : cb + g.sz;
  n.bwd[2] = n.wrap_zb ? cb + (g.Lz - 1) * g.sz : cb - g.sz;
  n.wrap_tf = (t == g.T - 1);
  n.wrap_tb = (t == 0);
  n.fwd[3] = n.wrap_tf ? cb - (g.T - 1) * g.st : cb + g.st;
  n.bwd[3] = n.wrap_tb ? cb + (g.T - 1) * g.st : cb - g.st;
  return n;
}

// DD = 1 (interior pass of a domain): hops that leave the domain through a cut are skipped, the exterior pass adds them
template <typename R, int NG, int MU, int NR, bool STREAM, int DD>
__device__ __forceinline__ void hop_pair(const DslashArgs<R>& a, const Nbr& n, int cb, const int (&cofs)[NR], R (&acc)[NR][24]) {
  const int NPG = Planes<R, NG>::N;
  const int64_t Vh = a.g.Vh;
  typedef typename Vec16<R>::T V;
  bool skip_f = false, skip_b = false;
  if (DD && MU >= 2 && a.dd.part[MU - 2]) {
    skip_f = (MU == 2) ? n.wrap_zf : n.wrap_tf;
    skip_b = (MU == 2) ? n.wrap_zb : n.wrap_tb;
  }
  if (!skip_f) {  // forward: (1 + sig g_mu) U_mu(x) psi(x+mu)
    cx<R> U[9];
    load_link<R, NG, STREAM>((const V*)a.U[a.par] + (int64_t)MU * NPG * Vh, Vh, cb, U);
    const R bc = (MU == 3 && n.wrap_tf) ? (R)-1 : (R)1;
#pragma unroll
    for (int j = 0; j < NR; j++) {
      R psi[24];
      load_reals<24>(a.in, Vh, n.fwd[MU] + cofs[j], psi);
      hop<R, MU, true>(psi, U, a.sig, bc, acc[j]);
    }
  }
  if (!skip_b) {  // backward: (1 - sig g_mu) U_mu(x-mu)^dag psi(x-mu)
    cx<R> U[9];
    load_link<R, NG, STREAM>((const V*)a.U[1 - a.par] + (int64_t)MU * NPG * Vh, Vh, n.bwd[MU], U);
    const R bc = (MU == 3 && n.wrap_tb) ? (R)-1 : (R)1;
#pragma unroll
    for (int j = 0; j < NR; j++) {
      R psi[24];
      load_reals<24>(a.in, Vh, n.bwd[MU] + cofs[j], psi);
      hop<R, MU, false>(psi, U, -a.sig, bc, acc[j]);
    }
  }
}

// hop_pair for NP PAIRS of columns (slots 2p, 2p+1) on packed fp32 pairs: the link is loaded, rebuilt and broadcast once
template <int NG, int MU, int NP, bool STREAM>
__device__ __forceinline__ void hop_pair2(const DslashArgs<float>& a, const Nbr& n, int cb, const int (&cofs)[2 * NP], float2 (&acc)[NP][24]) {
  const int NPG = Planes<float, NG>::N;
  const int64_t Vh = a.g.Vh;
  {  // forward: (1 + sig g_mu) U_mu(x) psi(x+mu)
    cx<float> U[9];
    load_link<float, NG, STREAM>((const float4*)a.U[a.par] + (int64_t)MU * NPG * Vh, Vh, cb, U);
    LinkPairs P;
    link_pairs(U, (MU == 3 && n.wrap_tf) ? -1.f : 1.f, P);
#pragma unroll
    for (int p = 0; p < NP; p++) {
      float psiA[24], psiB[24];
      load_reals<24>(a.in, Vh, n.fwd[MU] + cofs[2 * p], psiA);
      load_reals<24>(a.in, Vh, n.fwd[MU] + cofs[2 * p + 1], psiB);
      hop2<MU, true>(psiA, psiB, P, a.sig, acc[p]);
    }
  }
  {  // backward: (1 - sig g_mu) U_mu(x-mu)^dag psi(x-mu)
    cx<float> U[9];
    load_link<float, NG, STREAM>((const float4*)a.U[1 - a.par] + (int64_t)MU * NPG * Vh, Vh, n.bwd[MU], U);
    LinkPairs P;
    link_pairs(U, (MU == 3 && n.wrap_tb) ? -1.f : 1.f, P);
#pragma unroll
    for (int p = 0; p < NP; p++) {
      float psiA[24], psiB[24];
      load_reals<24>(a.in, Vh, n.bwd[MU] + cofs[2 * p], psiA);
      load_reals<24>(a.in, Vh, n.bwd[MU] + cofs[2 * p + 1], psiB);
      hop2<MU, false>(psiA, psiB, P, -a.sig, acc[p]);
    }
  }
}

// One chirality b (12 reals: spins 2b, 2b+1) of the site-diagonal part, with the block held in registers so that it
// serves several right-hand sides: w = A_b v and w = A_b^{-1} v as in apply_A / apply_Ainv above.
template <typename R, int CLOVER, bool STREAM> TMW_HD void load_block(const void* base, int b, int64_t Vh, int64_t cb, R* B) {
  if (CLOVER) {
    if (STREAM) load_reals_s<36>((const typename Vec16<R>::T*)base + (int64_t)b * Planes<R, 36>::N * Vh, Vh, cb, B);
    else load_reals<36>((const typename Vec16<R>::T*)base + (int64_t)b * Planes<R, 36>::N * Vh, Vh, cb, B);
  }
}
template <typename R, int CLOVER> TMW_HD void half_A(const Diag<R>& d, int b, const R* B, const R* v, R* w) {
  if (CLOVER) {
    herm6_mul(B, v, w);
  } else {
#pragma unroll
    for (int i = 0; i < 12; i++) w[i] = d.diag * v[i];
  }
  const R tw = b ? d.tw_lo : d.tw_up;
#pragma unroll
  for (int i = 0; i < 6; i++) {
    w[2 * i] -= tw * v[2 * i + 1];
    w[2 * i + 1] += tw * v[2 * i];
  }
}
// no clover: the complex scalar inverse; clover: w = Binv v (Binv = C^{-1}, or (C^2 + tw^2)^{-1} when twisted: the
// caller then multiplies by (C - i tw) with half_twfix)
template <typename R, int CLOVER> TMW_HD void half_Ainv(const Diag<R>& d, int b, const R* Binv, const R* v, R* w) {
  if (CLOVER) {
    herm6_mul(Binv, v, w);
  } else {
    const R ii = b ? d.inv_im_lo : d.inv_im_up;
#pragma unroll
    for (int i = 0; i < 6; i++) {
      w[2 * i] = d.inv_re * v[2 * i] - ii * v[2 * i + 1];
      w[2 * i + 1] = d.inv_re * v[2 * i + 1] + ii * v[2 * i];
    }
  }
}
template <typename R> TMW_HD void half_twfix(const Diag<R>& d, int b, const R* C, const R* v, R* w) {  // w = (C - i tw) v
  herm6_mul(C, v, w);
  const R tw = b ? d.tw_lo : d.tw_up;
#pragma unroll
  for (int i = 0; i < 6; i++) {
    w[2 * i] += tw * v[2 * i + 1];
    w[2 * i + 1] -= tw * v[2 * i];
  }
}

// true if dslash_site has already stored the result (the untwisted clover K1)
template <int EPI, int CLOVER> __device__ __forceinline__ constexpr bool stored_in_site() { return EPI == EPI_AINV_HOP && CLOVER == CL_CLOVER; }

// The stencil at one site for NR right-hand sides: on return acc[j] holds the output spinor of column slot j.
// red[j] = {Re, Im <out, aux>, <out, out>} when WANT_RED2 (EPI >= 2), accumulated chirality by chirality.
// is this output site on a cut of its domain (some hop of it arrives through a ghost buffer)?
template <typename R> TMW_HD bool on_cut(const DslashArgs<R>& a, const Nbr& n) {
  return (a.dd.part[0] && (n.wrap_zf || n.wrap_zb)) || (a.dd.part[1] && (n.wrap_tf || n.wrap_tb));
}

template <typename R, int NG, int EPI, int CLOVER, int NR, bool STREAM> __device__ __forceinline__ void dslash_epilogue(const DslashArgs<R>& a, int cb, const int (&cofs)[NR], const bool (&valid)[NR], R (&acc)[NR][24], R (&red2)[NR][3]);

// DD = 0: the whole lattice (or a domain without cuts). DD = 1: interior pass of a domain: returns true for a site on a
// cut, whose hops inside the domain have then been summed and stored RAW (no 1/2, no epilogue) in `out` for the exterior
// pass (dslash_ext_kernel) to finish; such a site takes no part in the fused reductions of this pass.
template <typename R, int NG, int EPI, int CLOVER, int NR, bool STREAM, int DD>
__device__ __forceinline__ bool dslash_site(const DslashArgs<R>& a, const Site& s, const int (&cofs)[NR], const bool (&valid)[NR], R (&acc)[NR][24], R (&red2)[NR][3]) {
  // cofs[j] = column * cstride: the column offset is added to the 32-bit SITE INDEX (the host checks that it fits), so
  // that every load address stays one IMAD.WIDE on a kernel-parameter base pointer, as with a single column
  const Nbr n = neighbours(a.g, a.par, s);
  const int cb = s.cb;
  if constexpr (TMW_PACK2 && sizeof(R) == 4 && NR % 2 == 0 && DD == 0) {
    // an even number of columns per thread: two columns per packed fp32 pair (hop2)
    float2 acc2[NR / 2][24];
#pragma unroll
    for (int p = 0; p < NR / 2; p++)
#pragma unroll
      for (int i = 0; i < 24; i++) acc2[p][i] = make_float2(0.f, 0.f);
    hop_pair2<NG, 0, NR / 2, STREAM>(a, n, cb, cofs, acc2);
    hop_pair2<NG, 1, NR / 2, STREAM>(a, n, cb, cofs, acc2);
    hop_pair2<NG, 2, NR / 2, STREAM>(a, n, cb, cofs, acc2);
    hop_pair2<NG, 3, NR / 2, STREAM>(a, n, cb, cofs, acc2);
#pragma unroll
    for (int p = 0; p < NR / 2; p++)
#pragma unroll
      for (int i = 0; i < 24; i++) { acc[2 * p][i] = acc2[p][i].x; acc[2 * p + 1][i] = acc2[p][i].y; }
  } else {
#pragma unroll
    for (int j = 0; j < NR; j++)
#pragma unroll
      for (int i = 0; i < 24; i++) acc[j][i] = (R)0;
    hop_pair<R, NG, 0, NR, STREAM, DD>(a, n, cb, cofs, acc);
    hop_pair<R, NG, 1, NR, STREAM, DD>(a, n, cb, cofs, acc);
    hop_pair<R, NG, 2, NR, STREAM, DD>(a, n, cb, cofs, acc);
    hop_pair<R, NG, 3, NR, STREAM, DD>(a, n, cb, cofs, acc);
  }
  if (DD && on_cut(a, n)) {
#pragma unroll
    for (int j = 0; j < NR; j++) {
      if (valid[j]) store_reals<24>(a.out, a.g.Vh, cb + cofs[j], acc[j]);
      red2[j][0] = red2[j][1] = red2[j][2] = (R)0;
    }
    return true;
  }
  dslash_epilogue<R, NG, EPI, CLOVER, NR, STREAM>(a, cb, cofs, valid, acc, red2);
  return false;
}

// acc[j] = the summed hops of column slot j at site cb -> the output spinor (1/2, site-diagonal part, aux); see dslash_site
template <typename R, int NG, int EPI, int CLOVER, int NR, bool STREAM>
__device__ __forceinline__ void dslash_epilogue(const DslashArgs<R>& a, int cb, const int (&cofs)[NR], const bool (&valid)[NR], R (&acc)[NR][24], R (&red2)[NR][3]) {
  typedef typename Vec16<R>::T V;
  const int64_t Vh = a.g.Vh;
#pragma unroll
  for (int j = 0; j < NR; j++) {
#pragma unroll
    for (int i = 0; i < 24; i++) acc[j][i] *= a.coef;
    red2[j][0] = red2[j][1] = red2[j][2] = (R)0;
  }
  if (EPI == EPI_HOP) return;
  const int HP = Planes<R, 12>::N;  // planes of one chirality of a spinor
#pragma unroll
  for (int b = 0; b < 2; b++) {
    R B[CLOVER ? 36 : 1];
    if (EPI == EPI_AINV_HOP || EPI == EPI_AINV_XPAY) load_block<R, CLOVER, STREAM>(a.d.cinv[a.par], b, Vh, cb, B);
    else if (EPI == EPI_A_XPAY) load_block<R, CLOVER, STREAM>(a.d.c[a.par], b, Vh, cb, B);
#pragma unroll
    for (int j = 0; j < NR; j++) {
      R* o = acc[j] + 12 * b;
      R ax[12], w[12];
      if (EPI >= 2) load_reals<12>((const V*)a.aux + (int64_t)b * HP * Vh, Vh, cb + cofs[j], ax);
      if (EPI == EPI_AINV_HOP) {
        half_Ainv<R, CLOVER>(a.d, b, B, o, w);
        if (stored_in_site<EPI, CLOVER>()) {
          // K1 has no fused reduction and no gamma5: store this chirality now, so that its accumulators are dead
          // before the block of the other chirality is loaded (the kernel wrapper skips its store, see stored_in_site)
          if (valid[j]) store_reals_s<12>((V*)a.out + (int64_t)b * HP * Vh, Vh, cb + cofs[j], w);
        } else {
#pragma unroll
          for (int i = 0; i < 12; i++) o[i] = w[i];
        }
      } else if (EPI == EPI_A_XPAY) {
        half_A<R, CLOVER>(a.d, b, B, ax, w);
#pragma unroll
        for (int i = 0; i < 12; i++) o[i] += w[i];
      } else if (EPI == EPI_XPAY) {
#pragma unroll
        for (int i = 0; i < 12; i++) o[i] += ax[i];
      } else {
#pragma unroll
        for (int i = 0; i < 12; i++) ax[i] += o[i];
        half_Ainv<R, CLOVER>(a.d, b, B, ax, w);
#pragma unroll
        for (int i = 0; i < 12; i++) o[i] = w[i];
      }
      if (EPI == EPI_A_XPAY || EPI == EPI_XPAY) {
#pragma unroll
        for (int i = 0; i < 6; i++) {  // conj(o) * ax, |o|^2
          red2[j][0] += o[2 * i] * ax[2 * i] + o[2 * i + 1] * ax[2 * i + 1];
          red2[j][1] += o[2 * i] * ax[2 * i + 1] - o[2 * i + 1] * ax[2 * i];
          red2[j][2] += o[2 * i] * o[2 * i] + o[2 * i + 1] * o[2 * i + 1];
        }
      }
    }
    if (CLOVER == CL_TWISTED && (EPI == EPI_AINV_HOP || EPI == EPI_AINV_XPAY)) {
      {  // (C + i tw)^{-1} = (C - i tw)(C^2 + tw^2)^{-1}: second factor, same registers
        load_block<R, CLOVER, STREAM>(a.d.c[a.par], b, Vh, cb, B);
#pragma unroll
        for (int j = 0; j < NR; j++) {
          R* o = acc[j] + 12 * b;
          R w[12];
          half_twfix<R>(a.d, b, B, o, w);
#pragma unroll
          for (int i = 0; i < 12; i++) o[i] = w[i];
        }
      }
    }
  }
}

}  // namespace tmw
