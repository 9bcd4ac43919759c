// tmw_clover.cu — clover term of Eq. (3) computed on the device from the gauge field, and its
// inverse ("calculate the entire clover term (and its inverse) ... directly"). SURVEY §8(a) A1, A2.
//
//   F_mu_nu(x) = (Q_mu_nu - Q_mu_nu^dag) / (8i),  Q = sum of the four plaquette leaves around x in the (mu,nu) plane
//   (no trace subtraction; link geometry periodic in all four directions — reading C7), and the site term
//   (c_sw/2) sum_{mu<nu} sigma_mu_nu (x) F_mu_nu is block diagonal in chirality in the DeGrand-Rossi basis:
//     upper (spins 0,1): k [ tau1 (F_yz - F_xt) + tau2 (F_xz + F_yt) + tau3 (F_xy - F_zt) ]
//     lower (spins 2,3): k [ tau1 (F_yz + F_xt) + tau2 (F_xz - F_yt) + tau3 (F_xy + F_zt) ],   k = c_sw/2
//   Each 6x6 Hermitian block (index 3*(spin mod 2) + colour) is stored packed with the real diagonal
//   -(4 + Re m) added: 6 real diagonal + 15 complex strictly-lower entries = 36 reals.
#include "tmw_internal.h"

namespace tmw {

typedef cx<double> zd;

// C = op(A) op(B), op = dagger if the flag is set; 3x3 row-major
template <bool DA, bool DB> __device__ __forceinline__ void mm(const zd* A, const zd* B, zd* C) {
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      zd s = mk<double>(0.0, 0.0);
#pragma unroll
      for (int k = 0; k < 3; k++) {
        const zd a = DA ? conj(A[3 * k + i]) : A[3 * i + k];
        const zd b = DB ? conj(B[3 * j + k]) : B[3 * k + j];
        cmad(s, a, b);
      }
      C[3 * i + j] = s;
    }
}

struct Lat {
  int L, T;
  int64_t V;
};
__device__ __forceinline__ int64_t lex(const Lat& g, const int* c) { return c[0] + (int64_t)g.L * (c[1] + (int64_t)g.L * (c[2] + (int64_t)g.L * c[3])); }
// site c shifted by dm in direction mu and dn in direction nu, periodic
__device__ __forceinline__ int64_t shifted(const Lat& g, const int* c, int mu, int dm, int nu, int dn) {
  int n[4] = {c[0], c[1], c[2], c[3]};
  const int em = (mu == 3) ? g.T : g.L, en = (nu == 3) ? g.T : g.L;
  n[mu] = (n[mu] + dm + em) % em;
  n[nu] = (n[nu] + dn + en) % en;
  return lex(g, n);
}
__device__ __forceinline__ void ld_link(const Lat& g, const double* __restrict__ canon, int mu, int64_t site, zd* U) {
  const double2* p = (const double2*)(canon + 18 * ((int64_t)mu * g.V + site));
#pragma unroll
  for (int i = 0; i < 9; i++) {
    const double2 q = __ldg(p + i);
    U[i] = mk<double>(q.x, q.y);
  }
}

// Q += A op B op C op D with the daggers given; all four links loaded here
template <bool D0, bool D1, bool D2, bool D3>
__device__ __forceinline__ void leaf(const Lat& g, const double* canon, int m0, int64_t s0, int m1, int64_t s1, int m2, int64_t s2, int m3, int64_t s3, zd* Q) {
  zd A[9], B[9], P[9], R2[9];
  ld_link(g, canon, m0, s0, A);
  ld_link(g, canon, m1, s1, B);
  mm<D0, D1>(A, B, P);
  ld_link(g, canon, m2, s2, A);
  mm<false, D2>(P, A, R2);
  ld_link(g, canon, m3, s3, B);
  mm<false, D3>(R2, B, P);
#pragma unroll
  for (int i = 0; i < 9; i++) Q[i] = Q[i] + P[i];
}

__device__ void field_strength(const Lat& g, const double* canon, const int* c, int mu, int nu, zd* F) {
  zd Q[9];
#pragma unroll
  for (int i = 0; i < 9; i++) Q[i] = mk<double>(0.0, 0.0);
  const int64_t x = lex(g, c);
  const int64_t xpm = shifted(g, c, mu, +1, nu, 0), xpn = shifted(g, c, mu, 0, nu, +1);
  const int64_t xmm = shifted(g, c, mu, -1, nu, 0), xmn = shifted(g, c, mu, 0, nu, -1);
  const int64_t xmmpn = shifted(g, c, mu, -1, nu, +1), xmmmn = shifted(g, c, mu, -1, nu, -1), xpmmn = shifted(g, c, mu, +1, nu, -1);
  // U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
  leaf<false, false, true, true>(g, canon, mu, x, nu, xpm, mu, xpn, nu, x, Q);
  // U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
  leaf<false, true, true, false>(g, canon, nu, x, mu, xmmpn, nu, xmm, mu, xmm, Q);
  // U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
  leaf<true, true, false, false>(g, canon, mu, xmm, nu, xmmmn, mu, xmmmn, nu, xmn, Q);
  // U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
  leaf<true, false, false, true>(g, canon, nu, xmn, mu, xmn, nu, xpmmn, mu, x, Q);
  // (Q - Q^dag)/(8i):  z/(8i) = (z.im, -z.re)/8
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      const zd z = Q[3 * i + j] - conj(Q[3 * j + i]);
      F[3 * i + j] = mk<double>(0.125 * z.im, -0.125 * z.re);
    }
}

// pack one chirality block from E1, E2, E3 (3x3 each): k [[E3, E1 - iE2], [E1 + iE2, -E3]] + diag
__device__ __forceinline__ void pack_block(const zd* E1, const zd* E2, const zd* E3, double k, double diag, double* B) {
#pragma unroll
  for (int i = 0; i < 3; i++) {
    B[i] = k * E3[4 * i].re + diag;
    B[3 + i] = -k * E3[4 * i].re + diag;
  }
#pragma unroll
  for (int i = 1; i < 6; i++)
#pragma unroll
    for (int j = 0; j < i; j++) {
      zd e;
      if (i < 3) e = E3[3 * i + j];
      else if (j >= 3) e = mk<double>(-E3[3 * (i - 3) + (j - 3)].re, -E3[3 * (i - 3) + (j - 3)].im);
      else {  // E1 + i E2
        const zd a = E1[3 * (i - 3) + j], b = E2[3 * (i - 3) + j];
        e = mk<double>(a.re - b.im, a.im + b.re);
      }
      const int idx = 6 + 2 * (i * (i - 1) / 2 + j);
      B[idx] = k * e.re;
      B[idx + 1] = k * e.im;
    }
}

__global__ void __launch_bounds__(128) clover_build_kernel(const Geom g, const double* __restrict__ canon, double k, double diag, double2* c64e, double2* c64o, float4* c32e, float4* c32o) {
  const int64_t site = (int64_t)blockIdx.x * 128 + threadIdx.x;
  Lat lt;
  lt.L = g.L;
  lt.T = g.T;
  lt.V = 2 * (int64_t)g.Vh;
  if (site >= lt.V) return;
  int c[4];
  int64_t q = site;
  c[0] = (int)(q % g.L); q /= g.L;
  c[1] = (int)(q % g.L); q /= g.L;
  c[2] = (int)(q % g.L); q /= g.L;
  c[3] = (int)q;
  const int par = (c[0] + c[1] + c[2] + c[3]) & 1;
  const int cb = (int)(site >> 1);
  // planes: xy=0 xz=1 xt=2 yz=3 yt=4 zt=5
  zd Fa[9], Fb[9], E1u[9], E2u[9], E3u[9], E1l[9], E2l[9], E3l[9];
  field_strength(lt, canon, c, 0, 1, Fa);  // xy
  field_strength(lt, canon, c, 2, 3, Fb);  // zt
#pragma unroll
  for (int i = 0; i < 9; i++) { E3u[i] = Fa[i] - Fb[i]; E3l[i] = Fa[i] + Fb[i]; }
  field_strength(lt, canon, c, 0, 2, Fa);  // xz
  field_strength(lt, canon, c, 1, 3, Fb);  // yt
#pragma unroll
  for (int i = 0; i < 9; i++) { E2u[i] = Fa[i] + Fb[i]; E2l[i] = Fa[i] - Fb[i]; }
  field_strength(lt, canon, c, 1, 2, Fa);  // yz
  field_strength(lt, canon, c, 0, 3, Fb);  // xt
#pragma unroll
  for (int i = 0; i < 9; i++) { E1u[i] = Fa[i] - Fb[i]; E1l[i] = Fa[i] + Fb[i]; }
  double B[72];
  pack_block(E1u, E2u, E3u, k, diag, B);
  pack_block(E1l, E2l, E3l, k, diag, B + 36);
  double2* d64 = par ? c64o : c64e;
  float4* d32 = par ? c32o : c32e;
  float Bf[72];
#pragma unroll
  for (int i = 0; i < 72; i++) Bf[i] = (float)B[i];
  store_reals<36>(d64, g.Vh, cb, B);
  store_reals<36>(d64 + (int64_t)18 * g.Vh, g.Vh, cb, B + 36);
  store_reals<36>(d32, g.Vh, cb, Bf);
  store_reals<36>(d32 + (int64_t)9 * g.Vh, g.Vh, cb, Bf + 36);
}

cudaError_t launch_clover_build(const Geom& g, const double* canon_gauge, double c_sw, double diag, void* c64_even, void* c64_odd, void* c32_even, void* c32_odd, cudaStream_t s) {
  const int64_t V = 2 * (int64_t)g.Vh;
  clover_build_kernel<<<(unsigned)((V + 127) / 128), 128, 0, s>>>(g, canon_gauge, 0.5 * c_sw, diag, (double2*)c64_even, (double2*)c64_odd, (float4*)c32_even, (float4*)c32_odd);
  return cudaGetLastError();
}

// ---- inverse of a packed Hermitian block: Gauss-Jordan with partial pivoting on the full complex 6x6 ----
// M = C (tw2 == 0) or C^2 + tw2 (twisted clover: (C + i tw)^{-1} = (C - i tw)(C^2 + tw^2)^{-1}); result Hermitian.
__global__ void __launch_bounds__(64) clover_invert_kernel(const Geom g, const double2* __restrict__ c64, double tw2, double2* inv64, float4* inv32, int* singular) {
  const int idx = blockIdx.x * 64 + threadIdx.x;  // (block b, cb)
  if (idx >= 2 * g.Vh) return;
  const int b = idx / g.Vh, cb = idx % g.Vh;
  double P[36];
  load_reals<36>(c64 + (int64_t)b * 18 * g.Vh, g.Vh, cb, P);
  zd M[6][6], X[6][6];
  double scale = 0;
  for (int i = 0; i < 6; i++) {
    M[i][i] = mk<double>(P[i], 0.0);
    for (int j = 0; j < i; j++) {
      const int k = 6 + 2 * (i * (i - 1) / 2 + j);
      M[i][j] = mk<double>(P[k], P[k + 1]);
      M[j][i] = mk<double>(P[k], -P[k + 1]);
    }
  }
  if (tw2 != 0.0) {
    for (int i = 0; i < 6; i++)
      for (int j = 0; j < 6; j++) {
        zd s = mk<double>(i == j ? tw2 : 0.0, 0.0);
        for (int k = 0; k < 6; k++) cmad(s, M[i][k], M[k][j]);
        X[i][j] = s;
      }
    for (int i = 0; i < 6; i++)
      for (int j = 0; j < 6; j++) M[i][j] = X[i][j];
  }
  for (int i = 0; i < 6; i++)
    for (int j = 0; j < 6; j++) {
      X[i][j] = mk<double>(i == j ? 1.0 : 0.0, 0.0);
      scale = fmax(scale, fabs(M[i][j].re) + fabs(M[i][j].im));
    }
  bool bad = !(scale > 0.0);
  for (int col = 0; col < 6 && !bad; col++) {
    int piv = col;
    double best = M[col][col].re * M[col][col].re + M[col][col].im * M[col][col].im;
    for (int r = col + 1; r < 6; r++) {
      const double a = M[r][col].re * M[r][col].re + M[r][col].im * M[r][col].im;
      if (a > best) { best = a; piv = r; }
    }
    if (!(sqrt(best) > 1e-13 * scale)) { bad = true; break; }
    if (piv != col)
      for (int j = 0; j < 6; j++) {
        zd t = M[col][j]; M[col][j] = M[piv][j]; M[piv][j] = t;
        t = X[col][j]; X[col][j] = X[piv][j]; X[piv][j] = t;
      }
    const zd pinv = mk<double>(M[col][col].re / best, -M[col][col].im / best);
    for (int j = 0; j < 6; j++) { M[col][j] = M[col][j] * pinv; X[col][j] = X[col][j] * pinv; }
    for (int r = 0; r < 6; r++) {
      if (r == col) continue;
      const zd f = M[r][col];
      for (int j = 0; j < 6; j++) { M[r][j] = M[r][j] - f * M[col][j]; X[r][j] = X[r][j] - f * X[col][j]; }
    }
  }
  if (bad) {
    atomicExch(singular, 1);
    for (int i = 0; i < 36; i++) P[i] = 0.0;
  } else {
    for (int i = 0; i < 6; i++) {
      P[i] = X[i][i].re;
      for (int j = 0; j < i; j++) {  // Hermitian part (the exact inverse is Hermitian)
        const int k = 6 + 2 * (i * (i - 1) / 2 + j);
        P[k] = 0.5 * (X[i][j].re + X[j][i].re);
        P[k + 1] = 0.5 * (X[i][j].im - X[j][i].im);
      }
    }
  }
  float Pf[36];
  for (int i = 0; i < 36; i++) Pf[i] = (float)P[i];
  store_reals<36>(inv64 + (int64_t)b * 18 * g.Vh, g.Vh, cb, P);
  store_reals<36>(inv32 + (int64_t)b * 9 * g.Vh, g.Vh, cb, Pf);
}

cudaError_t launch_clover_invert(const Geom& g, const void* c64, double tw2, void* inv64, void* inv32, int* singular, cudaStream_t s) {
  const int n = 2 * g.Vh;
  clover_invert_kernel<<<(n + 63) / 64, 64, 0, s>>>(g, (const double2*)c64, tw2, (double2*)inv64, (float4*)inv32, singular);
  return cudaGetLastError();
}

__global__ void __launch_bounds__(128) clover_export_kernel(const Geom g, const double2* __restrict__ c64, double* dst) {
  const int idx = blockIdx.x * 128 + threadIdx.x;
  if (idx >= 2 * g.Vh) return;
  const int b = idx / g.Vh, cb = idx % g.Vh;
  double P[36];
  load_reals<36>(c64 + (int64_t)b * 18 * g.Vh, g.Vh, cb, P);
  double* o = dst + 72 * (int64_t)cb + 36 * b;
  for (int i = 0; i < 36; i++) o[i] = P[i];
}
cudaError_t launch_clover_export(const Geom& g, const void* c64, double* dst, cudaStream_t s) {
  const int n = 2 * g.Vh;
  clover_export_kernel<<<(n + 127) / 128, 128, 0, s>>>(g, (const double2*)c64, dst);
  return cudaGetLastError();
}

}  // namespace tmw
