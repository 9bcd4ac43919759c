// tmw_blas.cu — fused BLAS-1 kernels of the BiCGStab recurrences (the "vector operations" of
// PAPER.md:315). Complex scalars (alpha, beta, omega, rho) live on the device in a Scalars block; reductions are
// accumulated in fp64 (per-thread -> warp shuffle -> block -> one atomicAdd per block and value).
// All vectors are packed parity spinors viewed as flat arrays of complex numbers; a work item is a PAIR of
// complex numbers = 4 reals (one float4, or two double2).
// Every kernel is batched over right-hand-side columns: blockIdx.y = slot, column c = cm.col[slot];
// column c of a vector starts c*cs work items after its base pointer and uses the scalar block sc[c]. A single
// solve is the batch {0}.
#include <atomic>

#include "tmw_internal.h"

namespace tmw {

__device__ __forceinline__ void ldp(const float* base, int64_t i, float* v) {
  const float4 q = *((const float4*)base + i);
  v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
}
__device__ __forceinline__ void ldp(const double* base, int64_t i, double* v) {
  const double2 a = *((const double2*)base + 2 * i), b = *((const double2*)base + 2 * i + 1);
  v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}
__device__ __forceinline__ void stp(float* base, int64_t i, const float* v) { *((float4*)base + i) = make_float4(v[0], v[1], v[2], v[3]); }
__device__ __forceinline__ void stp(double* base, int64_t i, const double* v) {
  *((double2*)base + 2 * i) = make_double2(v[0], v[1]);
  *((double2*)base + 2 * i + 1) = make_double2(v[2], v[3]);
}

// Mixed-precision kernels pair an fp32 packed spinor with an fp64 packed spinor. The plane layouts differ: the
// float4 vector (k, cb) holds reals 4k..4k+3 of site cb, which are the double2 vectors (2k, cb) and (2k+1, cb).
// Work item i = k*Vh + cb (a float4 index); the "m" accessors address either precision by that item. With several
// domains back to back in a vector (Vh = sites of ONE domain) item i = (6 d + k)*Vh + cb pairs with the double2
// vectors (12 d + 2k [+1])*Vh + cb = (2q [+1])*Vh + cb, q = i / Vh: the same formula.
__device__ __forceinline__ void ldm(const float* base, int64_t i, int64_t, float* v) { ldp(base, i, v); }
__device__ __forceinline__ void stm(float* base, int64_t i, int64_t, const float* v) { stp(base, i, v); }
__device__ __forceinline__ void ldm(const double* base, int64_t i, int64_t Vh, double* v) {
  const int64_t k = i / Vh, cb = i - k * Vh;
  const double2 a = *((const double2*)base + (2 * k) * Vh + cb), b = *((const double2*)base + (2 * k + 1) * Vh + cb);
  v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}
__device__ __forceinline__ void stm(double* base, int64_t i, int64_t Vh, const double* v) {
  const int64_t k = i / Vh, cb = i - k * Vh;
  *((double2*)base + (2 * k) * Vh + cb) = make_double2(v[0], v[1]);
  *((double2*)base + (2 * k + 1) * Vh + cb) = make_double2(v[2], v[3]);
}

enum { BB = 256 };
// SM count of the current device (asked once per device; 148 = B200 if the query fails)
static int sm_count() {
  enum { MAXDEV = 64 };
  static std::atomic<int> cache[MAXDEV];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAXDEV) return 148;
  int n = cache[dev].load(std::memory_order_relaxed);
  if (n == 0) {
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) n = 148;
    cache[dev].store(n, std::memory_order_relaxed);
  }
  return n;
}
// grid-stride launches: at most 8 CTAs of 256 threads per SM
static inline int blas_grid(int64_t n) {
  int64_t g = (n + BB - 1) / BB;
  const int64_t cap = (int64_t)sm_count() * 8;
  return (int)(g < cap ? (g > 0 ? g : 1) : cap);
}

template <int NV> __device__ __forceinline__ void reduce_atomic(double (&v)[NV], double* const* dst) {
  __shared__ double sm[NV][BB / 32];
#pragma unroll
  for (int k = 0; k < NV; k++)
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], off);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < NV; k++) sm[k][w] = v[k];
  __syncthreads();
  if (threadIdx.x < NV) {
    double s = 0;
#pragma unroll
    for (int i = 0; i < BB / 32; i++) s += sm[threadIdx.x][i];
    atomicAdd(dst[threadIdx.x], s);
  }
}

// ---- scalar phase kernels (one thread) ----
__device__ __forceinline__ void cdiv(const double* a, const double* b, double* q) {  // q = a / b
  const double d = b[0] * b[0] + b[1] * b[1];
  const double re = (a[0] * b[0] + a[1] * b[1]) / d, im = (a[1] * b[0] - a[0] * b[1]) / d;
  q[0] = re; q[1] = im;
}
__global__ void sc_begin_iter_kernel(Scalars* sc0, ColMap cm, int* attn, int check, double delta2) {
  Scalars* sc = sc0 + cm.col[threadIdx.x];
  if (check) {  // does the host have to look at this column before the iteration may go on? (tmw_internal.h)
    long long trip = 0;
    const double rr = sc->rr, rho2 = sc->rho[0] * sc->rho[0] + sc->rho[1] * sc->rho[1];
    if (!isfinite(rr) || !isfinite(rho2)) {
      trip = TRIP_BROKEN;
    } else {
      if (rr <= sc->stop2) trip |= TRIP_CONV;
      if (sc->maxr2 > 0.0 && rr < delta2 * sc->maxr2) trip |= TRIP_RELIABLE;
      if (!(rho2 > sc->brk2 * rr)) trip |= TRIP_BREAKDOWN;
      if (!trip && rr > sc->maxr2) sc->maxr2 = rr;
    }
    sc->trip = trip;
    if (trip) atomicOr(attn, 1);
  }
  __syncthreads();
  if (*(volatile int*)attn) return;  // raised now or by an earlier iteration: leave everything as it is
  sc->rhat_v[0] = sc->rhat_v[1] = 0.0;
  sc->ts[0] = sc->ts[1] = 0.0;
  sc->tt = 0.0;
  sc->rhat_t[0] = sc->rhat_t[1] = 0.0;
  sc->rhat_s[0] = sc->rhat_s[1] = 0.0;
  if (threadIdx.x == 0) attn[1]++;
}
__global__ void sc_alpha_kernel(Scalars* sc0, ColMap cm, const int* skip) {
  if (skip && *skip) return;
  Scalars* sc = sc0 + cm.col[threadIdx.x];
  cdiv(sc->rho, sc->rhat_v, sc->alpha);
}
__global__ void sc_omega_kernel(Scalars* sc0, ColMap cm, const int* skip) {
  if (skip && *skip) return;
  Scalars* sc = sc0 + cm.col[threadIdx.x];
  // <t,t> = 0: s = r - alpha v vanished, x + alpha p is exact at the half step (a source that is an eigenvector, a free
  // field). omega = 0 then makes update_xrp do x += alpha p, r = s (= 0); beta = 0 keeps the next p finite.
  const bool exact = sc->tt == 0.0;
  const double wr = exact ? 0.0 : sc->ts[0] / sc->tt, wi = exact ? 0.0 : sc->ts[1] / sc->tt;
  sc->omega[0] = wr;
  sc->omega[1] = wi;
  sc->rho_old[0] = sc->rho[0];
  sc->rho_old[1] = sc->rho[1];
  // <rhat, r_new> with r_new = s - omega t, from the two dot products the second K2 reduced
  sc->rho[0] = sc->rhat_s[0] - (wr * sc->rhat_t[0] - wi * sc->rhat_t[1]);
  sc->rho[1] = sc->rhat_s[1] - (wr * sc->rhat_t[1] + wi * sc->rhat_t[0]);
  double a[2], b[2];
  cdiv(sc->rho, sc->rho_old, a);
  cdiv(sc->alpha, sc->omega, b);
  sc->beta[0] = exact ? 0.0 : a[0] * b[0] - a[1] * b[1];
  sc->beta[1] = exact ? 0.0 : a[0] * b[1] + a[1] * b[0];
  sc->rr = 0.0;
}
cudaError_t launch_sc_begin_iter(Scalars* sc, const ColMap& cm, int* attn, int check, double delta2, cudaStream_t s) {
  sc_begin_iter_kernel<<<1, cm.n, 0, s>>>(sc, cm, attn, check, delta2);
  return cudaGetLastError();
}
cudaError_t launch_sc_alpha(Scalars* sc, const ColMap& cm, const int* skip, cudaStream_t s) { sc_alpha_kernel<<<1, cm.n, 0, s>>>(sc, cm, skip); return cudaGetLastError(); }
cudaError_t launch_sc_omega(Scalars* sc, const ColMap& cm, const int* skip, cudaStream_t s) { sc_omega_kernel<<<1, cm.n, 0, s>>>(sc, cm, skip); return cudaGetLastError(); }

// ---- vector updates ----
template <typename R> __global__ void __launch_bounds__(BB) update_s_kernel(int64_t n, R* s, const R* r, const R* v, const Scalars* sc, ColMap cm, const int* skip) {
  if (skip && *skip) return;
  const int c = cm.col[blockIdx.y];
  sc += c;
  { const int64_t o = 4 * n * c; s += o; r += o; v += o; }
  const R ar = (R)sc->alpha[0], ai = (R)sc->alpha[1];
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    R rr[4], vv[4], ss[4];
    ldp(r, i, rr); ldp(v, i, vv);
#pragma unroll
    for (int c = 0; c < 2; c++) {
      ss[2 * c] = rr[2 * c] - (ar * vv[2 * c] - ai * vv[2 * c + 1]);
      ss[2 * c + 1] = rr[2 * c + 1] - (ar * vv[2 * c + 1] + ai * vv[2 * c]);
    }
    stp(s, i, ss);
  }
}
template <typename R> __global__ void __launch_bounds__(BB) update_xrp_kernel(int64_t n, R* x, R* r, R* p, const R* s, const R* t, const R* v, Scalars* sc, ColMap cm, const int* skip) {
  if (skip && *skip) return;
  const int c = cm.col[blockIdx.y];
  sc += c;
  { const int64_t o = 4 * n * c; x += o; r += o; p += o; s += o; t += o; v += o; }
  const R ar = (R)sc->alpha[0], ai = (R)sc->alpha[1], wr = (R)sc->omega[0], wi = (R)sc->omega[1], br = (R)sc->beta[0], bi = (R)sc->beta[1];
  double acc[1] = {0};
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    R xx[4], pp[4], ss[4], tt[4], vv[4], rr[4];
    ldp(x, i, xx); ldp(p, i, pp); ldp(s, i, ss); ldp(t, i, tt); ldp(v, i, vv);
    R nn = 0;
#pragma unroll
    for (int k = 0; k < 2; k++) {
      xx[2 * k] += (ar * pp[2 * k] - ai * pp[2 * k + 1]) + (wr * ss[2 * k] - wi * ss[2 * k + 1]);
      xx[2 * k + 1] += (ar * pp[2 * k + 1] + ai * pp[2 * k]) + (wr * ss[2 * k + 1] + wi * ss[2 * k]);
      rr[2 * k] = ss[2 * k] - (wr * tt[2 * k] - wi * tt[2 * k + 1]);
      rr[2 * k + 1] = ss[2 * k + 1] - (wr * tt[2 * k + 1] + wi * tt[2 * k]);
      nn += rr[2 * k] * rr[2 * k] + rr[2 * k + 1] * rr[2 * k + 1];
      const R ur = pp[2 * k] - (wr * vv[2 * k] - wi * vv[2 * k + 1]);
      const R ui = pp[2 * k + 1] - (wr * vv[2 * k + 1] + wi * vv[2 * k]);
      pp[2 * k] = rr[2 * k] + (br * ur - bi * ui);
      pp[2 * k + 1] = rr[2 * k + 1] + (br * ui + bi * ur);
    }
    stp(x, i, xx);
    stp(r, i, rr);
    stp(p, i, pp);
    acc[0] += nn;
  }
  double* dst[1] = {&sc->rr};
  reduce_atomic<1>(acc, dst);
}
template <typename R> __global__ void __launch_bounds__(BB) dot_norm_kernel(int64_t n, const R* a, const R* b, double* out, ColMap cm) {
  const int c = cm.col[blockIdx.y];
  out += 4 * c;
  { const int64_t o = 4 * n * c; if (a) a += o; b += o; }
  double acc[3] = {0, 0, 0};
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    R aa[4] = {0, 0, 0, 0}, bb[4];
    if (a) ldp(a, i, aa);
    ldp(b, i, bb);
    R re = 0, im = 0, nn = 0;
#pragma unroll
    for (int c = 0; c < 2; c++) {
      re += aa[2 * c] * bb[2 * c] + aa[2 * c + 1] * bb[2 * c + 1];
      im += aa[2 * c] * bb[2 * c + 1] - aa[2 * c + 1] * bb[2 * c];
      nn += bb[2 * c] * bb[2 * c] + bb[2 * c + 1] * bb[2 * c + 1];
    }
    acc[0] += re; acc[1] += im; acc[2] += nn;
  }
  double* dst[3] = {out, out + 1, out + 2};
  reduce_atomic<3>(acc, dst);
}
template <typename R> __global__ void __launch_bounds__(BB) acc_y_kernel(int64_t n, int64_t Vh, double* y, R* x, ColMap cm) {
  { const int64_t o = 4 * n * cm.col[blockIdx.y]; y += o; x += o; }
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    R xx[4];
    double yy[4];
    ldm(x, i, Vh, xx); ldm(y, i, Vh, yy);
#pragma unroll
    for (int c = 0; c < 4; c++) { yy[c] += (double)xx[c]; xx[c] = (R)0; }
    stm(y, i, Vh, yy);
    stm(x, i, Vh, xx);
  }
}
template <typename R> __global__ void __launch_bounds__(BB) resid_convert_kernel(int64_t n, int64_t Vh, const double* b, const double* w, double* r64, R* r, const R* rhat, R* p, Scalars* sc, ColMap cm) {
  const int c = cm.col[blockIdx.y];
  sc += c;
  { const int64_t o = 4 * n * c; b += o; if (w) w += o; r64 += o; r += o; rhat += o; if (p) p += o; }
  double acc[3] = {0, 0, 0};
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    double bb[4], ww[4], dd[4];
    R hh[4], rr[4];
    ldm(b, i, Vh, bb); ldm(rhat, i, Vh, hh);
    if (w) ldm(w, i, Vh, ww);
    else ww[0] = ww[1] = ww[2] = ww[3] = 0.0;
#pragma unroll
    for (int c = 0; c < 4; c++) { dd[c] = bb[c] - ww[c]; rr[c] = (R)dd[c]; }
    if (p) {  // p += r_new - r_old
      R ro[4], pp[4];
      ldm(r, i, Vh, ro); ldm(p, i, Vh, pp);
#pragma unroll
      for (int c = 0; c < 4; c++) pp[c] += rr[c] - ro[c];
      stm(p, i, Vh, pp);
    }
    stm(r64, i, Vh, dd);
    stm(r, i, Vh, rr);
#pragma unroll
    for (int c = 0; c < 2; c++) {
      acc[0] += (double)hh[2 * c] * dd[2 * c] + (double)hh[2 * c + 1] * dd[2 * c + 1];
      acc[1] += (double)hh[2 * c] * dd[2 * c + 1] - (double)hh[2 * c + 1] * dd[2 * c];
      acc[2] += dd[2 * c] * dd[2 * c] + dd[2 * c + 1] * dd[2 * c + 1];
    }
  }
  double* dst[3] = {&sc->rho[0], &sc->rho[1], &sc->rr};
  reduce_atomic<3>(acc, dst);
}
template <typename R> __global__ void __launch_bounds__(BB) convert_kernel(int64_t n, int64_t Vh, const double* src, R* dst, ColMap cm) {
  { const int64_t o = 4 * n * cm.col[blockIdx.y]; src += o; dst += o; }
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    double ss[4];
    R dd[4];
    ldm(src, i, Vh, ss);
#pragma unroll
    for (int c = 0; c < 4; c++) dd[c] = (R)ss[c];
    stm(dst, i, Vh, dd);
  }
}
__global__ void __launch_bounds__(BB) sub_norm_kernel(int64_t n, const double* a, const double* b, double* d, double* out, ColMap cm) {
  const int c = cm.col[blockIdx.y];
  out += 4 * c;
  { const int64_t o = 4 * n * c; a += o; b += o; d += o; }
  double acc[1] = {0};
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    double aa[4], bb[4], dd[4];
    ldp(a, i, aa); ldp(b, i, bb);
#pragma unroll
    for (int c = 0; c < 4; c++) { dd[c] = aa[c] - bb[c]; acc[0] += dd[c] * dd[c]; }
    stp(d, i, dd);
  }
  double* dst[1] = {out + 2};
  reduce_atomic<1>(acc, dst);
}

// a += b (fp64, n double2-pair work items per column)
__global__ void __launch_bounds__(BB) add64_kernel(int64_t n, double* a, const double* b, ColMap cm) {
  { const int64_t o = 4 * n * cm.col[blockIdx.y]; a += o; b += o; }
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    double aa[4], bb[4];
    ldp(a, i, aa); ldp(b, i, bb);
#pragma unroll
    for (int c = 0; c < 4; c++) aa[c] += bb[c];
    stp(a, i, aa);
  }
}

// One step of the Clenshaw recursion for a Chebyshev series in X = scale*H + shift:
// out = c*psi + f*(scale*hb + shift*b1) - b2, hb = H b1; out may alias b2. Real coefficients, fp64.
__global__ void __launch_bounds__(BB) clenshaw_kernel(int64_t n, double* out, const double* psi, const double* hb, const double* b1, const double* b2,
                                                      double c, double f, double scale, double shift) {
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    double pp[4], hh[4], u1[4], u2[4], oo[4];
    ldp(psi, i, pp); ldp(hb, i, hh); ldp(b1, i, u1); ldp(b2, i, u2);
#pragma unroll
    for (int k = 0; k < 4; k++) oo[k] = c * pp[k] + f * (scale * hh[k] + shift * u1[k]) - u2[k];
    stp(out, i, oo);
  }
}
cudaError_t launch_clenshaw(int64_t n64, void* out, const void* psi, const void* hb, const void* b1, const void* b2, double c, double f, double scale,
                            double shift, cudaStream_t s) {
  const int64_t np = n64 / 2;
  clenshaw_kernel<<<blas_grid(np), BB, 0, s>>>(np, (double*)out, (const double*)psi, (const double*)hb, (const double*)b1, (const double*)b2, c, f, scale, shift);
  return cudaGetLastError();
}
// dst = c * src (fp64)
__global__ void __launch_bounds__(BB) scale_kernel(int64_t n, double* dst, const double* src, double c) {
  for (int64_t i = (int64_t)blockIdx.x * BB + threadIdx.x; i < n; i += (int64_t)gridDim.x * BB) {
    double v[4];
    ldp(src, i, v);
#pragma unroll
    for (int k = 0; k < 4; k++) v[k] *= c;
    stp(dst, i, v);
  }
}
cudaError_t launch_scale(int64_t n64, void* dst, const void* src, double c, cudaStream_t s) {
  const int64_t np = n64 / 2;
  scale_kernel<<<blas_grid(np), BB, 0, s>>>(np, (double*)dst, (const double*)src, c);
  return cudaGetLastError();
}

// ---- GCR(k) kernels (the paper's "standard GPU inverter with GCR algorithm") ----
// Batched over right-hand-side columns like the BiCGStab kernels: blockIdx.y (vector kernels) or blockIdx.x / threadIdx.x
// (scalar kernels) = slot, column c = cm.col[slot] with its own GcrScalars block gs[c]. Krylov vectors q_j (= Mhat p_j,
// orthogonal, NOT normalised: nq[j] = <q_j,q_j>) and p_j, j < KMAX: vector j of column c starts (j*ncw + c)*n work items
// after the base pointer (ncw = columns the workspace holds), so that the vectors j of all columns are one multi-column
// spinor the stencil can write. x and r of column c start c*n work items after their base pointers.

// dots[2j..2j+1] += <q_j, w> for j < i (w = q_i before orthogonalisation): one pass over w and the i vectors q_j
template <typename R> __global__ void __launch_bounds__(BB) gcr_dots_kernel(int64_t n, int i, int ncw, const R* Q, GcrScalars* gs0, ColMap cm) {
  const int c = cm.col[blockIdx.y];
  GcrScalars* gs = gs0 + c;
  Q += 4 * n * c;
  const R* w = Q + 4 * n * ncw * i;
  double acc[2 * GCR_KMAX];
#pragma unroll
  for (int j = 0; j < 2 * GCR_KMAX; j++) acc[j] = 0.0;
  for (int64_t e = (int64_t)blockIdx.x * BB + threadIdx.x; e < n; e += (int64_t)gridDim.x * BB) {
    R ww[4];
    ldp(w, e, ww);
#pragma unroll
    for (int j = 0; j < GCR_KMAX; j++) {
      if (j < i) {
        R qq[4];
        ldp(Q + 4 * n * ncw * j, e, qq);
        acc[2 * j] += (double)(qq[0] * ww[0] + qq[1] * ww[1] + qq[2] * ww[2] + qq[3] * ww[3]);
        acc[2 * j + 1] += (double)(qq[0] * ww[1] - qq[1] * ww[0] + qq[2] * ww[3] - qq[3] * ww[2]);
      }
    }
  }
  __shared__ double sm[BB / 32];
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  for (int j = 0; j < 2 * i; j++) {
    double v = acc[j];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    if (lane == 0) sm[wp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
      double t = 0;
#pragma unroll
      for (int k = 0; k < BB / 32; k++) t += sm[k];
      atomicAdd(&gs->dots[j], t);
    }
    __syncthreads();
  }
}
// coef_j = dots_j / nq_j (j < i); zero the accumulators of the next two kernels. blockIdx.x = slot, threadIdx.x = j
__global__ void gcr_coef_kernel(int i, GcrScalars* gs0, ColMap cm) {
  GcrScalars* gs = gs0 + cm.col[blockIdx.x];
  const int j = threadIdx.x;
  if (j < i) {
    gs->coef[2 * j] = gs->dots[2 * j] / gs->nq[j];
    gs->coef[2 * j + 1] = gs->dots[2 * j + 1] / gs->nq[j];
    gs->dots[2 * j] = gs->dots[2 * j + 1] = 0.0;
  }
  if (j == 0) { gs->nw = 0.0; gs->g[0] = gs->g[1] = 0.0; gs->rr = 0.0; }
}
// w -= sum_j coef_j q_j (stored as q_i);  p_i = r - sum_j coef_j p_j;  nw += <w,w>;  g += <w,r>
template <typename R> __global__ void __launch_bounds__(BB) gcr_orth_kernel(int64_t n, int i, int ncw, R* Q, R* P, const R* r, GcrScalars* gs0, ColMap cm) {
  const int col = cm.col[blockIdx.y];
  GcrScalars* gs = gs0 + col;
  Q += 4 * n * col;
  P += 4 * n * col;
  r += 4 * n * col;
  R cr[GCR_KMAX], ci[GCR_KMAX];
#pragma unroll
  for (int j = 0; j < GCR_KMAX; j++) {
    cr[j] = j < i ? (R)gs->coef[2 * j] : (R)0;
    ci[j] = j < i ? (R)gs->coef[2 * j + 1] : (R)0;
  }
  double acc[3] = {0, 0, 0};
  R* w = Q + 4 * n * ncw * i;
  R* p = P + 4 * n * ncw * i;
  for (int64_t e = (int64_t)blockIdx.x * BB + threadIdx.x; e < n; e += (int64_t)gridDim.x * BB) {
    R ww[4], pp[4], rr[4];
    ldp(w, e, ww); ldp(r, e, rr);
#pragma unroll
    for (int c = 0; c < 4; c++) pp[c] = rr[c];
#pragma unroll
    for (int j = 0; j < GCR_KMAX; j++) {
      if (j < i) {
        R qq[4], pj[4];
        ldp(Q + 4 * n * ncw * j, e, qq); ldp(P + 4 * n * ncw * j, e, pj);
#pragma unroll
        for (int c = 0; c < 2; c++) {
          ww[2 * c] -= cr[j] * qq[2 * c] - ci[j] * qq[2 * c + 1];
          ww[2 * c + 1] -= cr[j] * qq[2 * c + 1] + ci[j] * qq[2 * c];
          pp[2 * c] -= cr[j] * pj[2 * c] - ci[j] * pj[2 * c + 1];
          pp[2 * c + 1] -= cr[j] * pj[2 * c + 1] + ci[j] * pj[2 * c];
        }
      }
    }
    stp(w, e, ww); stp(p, e, pp);
#pragma unroll
    for (int c = 0; c < 2; c++) {
      acc[0] += (double)(ww[2 * c] * ww[2 * c] + ww[2 * c + 1] * ww[2 * c + 1]);
      acc[1] += (double)(ww[2 * c] * rr[2 * c] + ww[2 * c + 1] * rr[2 * c + 1]);
      acc[2] += (double)(ww[2 * c] * rr[2 * c + 1] - ww[2 * c + 1] * rr[2 * c]);
    }
  }
  double* dst[3] = {&gs->nw, &gs->g[0], &gs->g[1]};
  reduce_atomic<3>(acc, dst);
}
// a = g / nw; nq[i] = nw. threadIdx.x = slot
__global__ void gcr_alpha_kernel(int i, GcrScalars* gs0, ColMap cm) {
  GcrScalars* gs = gs0 + cm.col[threadIdx.x];
  gs->nq[i] = gs->nw;
  gs->a[0] = gs->g[0] / gs->nw;
  gs->a[1] = gs->g[1] / gs->nw;
}
// x += a p_i;  r -= a q_i;  rr += <r,r>
template <typename R> __global__ void __launch_bounds__(BB) gcr_update_kernel(int64_t n, int i, int ncw, R* x, R* r, const R* Q, const R* P, GcrScalars* gs0, ColMap cm) {
  const int col = cm.col[blockIdx.y];
  GcrScalars* gs = gs0 + col;
  x += 4 * n * col;
  r += 4 * n * col;
  const R ar = (R)gs->a[0], ai = (R)gs->a[1];
  const R* w = Q + 4 * n * (ncw * i + col);
  const R* p = P + 4 * n * (ncw * i + col);
  double acc[1] = {0};
  for (int64_t e = (int64_t)blockIdx.x * BB + threadIdx.x; e < n; e += (int64_t)gridDim.x * BB) {
    R xx[4], rr[4], ww[4], pp[4];
    ldp(x, e, xx); ldp(r, e, rr); ldp(w, e, ww); ldp(p, e, pp);
#pragma unroll
    for (int c = 0; c < 2; c++) {
      xx[2 * c] += ar * pp[2 * c] - ai * pp[2 * c + 1];
      xx[2 * c + 1] += ar * pp[2 * c + 1] + ai * pp[2 * c];
      rr[2 * c] -= ar * ww[2 * c] - ai * ww[2 * c + 1];
      rr[2 * c + 1] -= ar * ww[2 * c + 1] + ai * ww[2 * c];
      acc[0] += (double)(rr[2 * c] * rr[2 * c] + rr[2 * c + 1] * rr[2 * c + 1]);
    }
    stp(x, e, xx); stp(r, e, rr);
  }
  double* dst[1] = {&gs->rr};
  reduce_atomic<1>(acc, dst);
}

// n16 = number of 16-byte vectors of R in ONE column; pairs = n16 (float) or n16/2 (double)
template <typename R> static inline int64_t pairs_of(int64_t n16) { return sizeof(R) == 4 ? n16 : n16 / 2; }
static inline dim3 grid_of(int64_t np, const ColMap& cm) { return dim3((unsigned)blas_grid(np), (unsigned)cm.n, 1); }

template <typename R> cudaError_t launch_update_s(int64_t n, void* sv, const void* r, const void* v, const Scalars* sc, const ColMap& cm, const int* skip, cudaStream_t s) {
  const int64_t np = pairs_of<R>(n);
  update_s_kernel<R><<<grid_of(np, cm), BB, 0, s>>>(np, (R*)sv, (const R*)r, (const R*)v, sc, cm, skip);
  return cudaGetLastError();
}
template <typename R> cudaError_t launch_update_xrp(int64_t n, void* x, void* r, void* p, const void* sv, const void* t, const void* v, Scalars* sc, const ColMap& cm, const int* skip, cudaStream_t s) {
  const int64_t np = pairs_of<R>(n);
  update_xrp_kernel<R><<<grid_of(np, cm), BB, 0, s>>>(np, (R*)x, (R*)r, (R*)p, (const R*)sv, (const R*)t, (const R*)v, sc, cm, skip);
  return cudaGetLastError();
}
template <typename R> cudaError_t launch_dot_norm(int64_t n, const void* a, const void* b, double* out, const ColMap& cm, cudaStream_t s) {
  const int64_t np = pairs_of<R>(n);
  dot_norm_kernel<R><<<grid_of(np, cm), BB, 0, s>>>(np, (const R*)a, (const R*)b, out, cm);
  return cudaGetLastError();
}
template <typename R> cudaError_t launch_acc_y(int64_t n64, int64_t vh, void* y64, void* x, const ColMap& cm, cudaStream_t s) {
  const int64_t np = n64 / 2;
  acc_y_kernel<R><<<grid_of(np, cm), BB, 0, s>>>(np, vh, (double*)y64, (R*)x, cm);
  return cudaGetLastError();
}
template <typename R> cudaError_t launch_resid_convert(int64_t n64, int64_t vh, const void* b64, const void* w64, void* r64, void* r, const void* rhat, void* p, Scalars* sc, const ColMap& cm, cudaStream_t s) {
  const int64_t np = n64 / 2;
  resid_convert_kernel<R><<<grid_of(np, cm), BB, 0, s>>>(np, vh, (const double*)b64, (const double*)w64, (double*)r64, (R*)r, (const R*)rhat, (R*)p, sc, cm);
  return cudaGetLastError();
}
template <typename R> cudaError_t launch_convert(int64_t n64, int64_t vh, const void* src64, void* dst, const ColMap& cm, cudaStream_t s) {
  const int64_t np = n64 / 2;
  convert_kernel<R><<<grid_of(np, cm), BB, 0, s>>>(np, vh, (const double*)src64, (R*)dst, cm);
  return cudaGetLastError();
}
cudaError_t launch_sub_norm(int64_t n64, const void* a, const void* b, void* d, double* out, const ColMap& cm, cudaStream_t s) {
  const int64_t np = n64 / 2;
  sub_norm_kernel<<<grid_of(np, cm), BB, 0, s>>>(np, (const double*)a, (const double*)b, (double*)d, out, cm);
  return cudaGetLastError();
}

cudaError_t launch_add64(int64_t n64, void* a, const void* b, const ColMap& cm, cudaStream_t s) {
  const int64_t np = n64 / 2;
  add64_kernel<<<grid_of(np, cm), BB, 0, s>>>(np, (double*)a, (const double*)b, cm);
  return cudaGetLastError();
}

template <typename R> cudaError_t launch_gcr_step(int64_t n16, int i, int ncw, void* Q, void* P, void* x, void* r, GcrScalars* gs, const ColMap& cm, cudaStream_t s) {
  const int64_t np = pairs_of<R>(n16);
  if (i > 0) gcr_dots_kernel<R><<<grid_of(np, cm), BB, 0, s>>>(np, i, ncw, (const R*)Q, gs, cm);
  gcr_coef_kernel<<<cm.n, GCR_KMAX, 0, s>>>(i, gs, cm);
  gcr_orth_kernel<R><<<grid_of(np, cm), BB, 0, s>>>(np, i, ncw, (R*)Q, (R*)P, (const R*)r, gs, cm);
  gcr_alpha_kernel<<<1, cm.n, 0, s>>>(i, gs, cm);
  gcr_update_kernel<R><<<grid_of(np, cm), BB, 0, s>>>(np, i, ncw, (R*)x, (R*)r, (const R*)Q, (const R*)P, gs, cm);
  return cudaGetLastError();
}
template cudaError_t launch_gcr_step<float>(int64_t, int, int, void*, void*, void*, void*, GcrScalars*, const ColMap&, cudaStream_t);
template cudaError_t launch_gcr_step<double>(int64_t, int, int, void*, void*, void*, void*, GcrScalars*, const ColMap&, cudaStream_t);

#define TMW_INST(R)                                                                                                          \
  template cudaError_t launch_update_s<R>(int64_t, void*, const void*, const void*, const Scalars*, const ColMap&, const int*, cudaStream_t);           \
  template cudaError_t launch_update_xrp<R>(int64_t, void*, void*, void*, const void*, const void*, const void*, Scalars*, const ColMap&, const int*, cudaStream_t); \
  template cudaError_t launch_dot_norm<R>(int64_t, const void*, const void*, double*, const ColMap&, cudaStream_t);                         \
  template cudaError_t launch_acc_y<R>(int64_t, int64_t, void*, void*, const ColMap&, cudaStream_t);                                        \
  template cudaError_t launch_resid_convert<R>(int64_t, int64_t, const void*, const void*, void*, void*, const void*, void*, Scalars*, const ColMap&, cudaStream_t); \
  template cudaError_t launch_convert<R>(int64_t, int64_t, const void*, void*, const ColMap&, cudaStream_t);
TMW_INST(float)
TMW_INST(double)

}  // namespace tmw
