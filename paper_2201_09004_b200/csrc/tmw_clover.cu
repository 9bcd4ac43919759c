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
  int L, T, Lh;
  int64_t Vh;
  const double2* U[2];  // packed fp64 gauge per parity: [mu][9 planes][Vh] (tmw_pack.cu)
};
// site code: (lexicographic index << 1) | parity; lex >> 1 is the checkerboard index (L is even)
__device__ __forceinline__ int64_t lex(const Lat& g, const int* c) {
  return ((c[0] + (int64_t)g.L * (c[1] + (int64_t)g.L * (c[2] + (int64_t)g.L * c[3]))) << 1) | ((c[0] + c[1] + c[2] + c[3]) & 1);
}
// site c shifted by dm in direction mu and dn in direction nu, periodic
__device__ __forceinline__ int64_t shifted(const Lat& g, const int* c, int mu, int dm, int nu, int dn) {
  int n[4] = {c[0], c[1], c[2], c[3]};
  const int em = (mu == 3) ? g.T : g.L, en = (nu == 3) ? g.T : g.L;
  n[mu] = (n[mu] + dm + em) % em;
  n[nu] = (n[nu] + dn + en) % en;
  return lex(g, n);
}
// link U_mu at the lexicographic site index: read from the packed (checkerboarded, plane-major) fp64 copy, so that the
// 32 lanes of a warp (consecutive checkerboard sites of one parity) read 512 contiguous bytes per plane. Reading the
// canonical array-of-structures field instead costs 36 L1 wavefronts per warp load instead of 4 and made this kernel
// L1-bound (38.6 ms at 48^3 x 144).
__device__ __forceinline__ void ld_link(const Lat& g, const double* __restrict__, int mu, int64_t site, zd* U) {
  const double2* p = g.U[site & 1] + (int64_t)mu * 9 * g.Vh + (site >> 2);
#pragma unroll
  for (int i = 0; i < 9; i++) {
    const double2 v = __ldg(p + i * g.Vh);
    U[i] = mk<double>(v.x, v.y);
  }
}

// Q += op(A) op(B) op(C) op(D) with the daggers given; all four links loaded here. The product is built row by row:
// v = the first NROW rows of op(A), then v <- v op(B), v <- v op(C), v <- v op(D) (3 x NROW x 9 complex multiply-adds).
// That keeps NROW x 3 + 9 complex numbers live per step instead of three full matrices, so that the next link is in
// flight while the current one is multiplied. NROW = 2 (links known to be SU(3): the context stores 12-real fp32 links):
// the third row of the SU(3) product is conj(row0 x row1), a third fewer multiply-adds.
template <int NROW, bool DAG> __device__ __forceinline__ void vmul(zd (&v)[NROW][3], const zd* M) {
#pragma unroll
  for (int r = 0; r < NROW; r++) {
    zd w[3];
#pragma unroll
    for (int j = 0; j < 3; j++) {
      zd s = mk<double>(0.0, 0.0);
#pragma unroll
      for (int k = 0; k < 3; k++) cmad(s, v[r][k], DAG ? conj(M[3 * j + k]) : M[3 * k + j]);
      w[j] = s;
    }
#pragma unroll
    for (int j = 0; j < 3; j++) v[r][j] = w[j];
  }
}
template <int NROW, bool D0, bool D1, bool D2, bool D3>
__device__ __forceinline__ void leaf(const Lat& g, const double* canon, int m0, int64_t s0, int m1, int64_t s1, int m2, int64_t s2, int m3, int64_t s3, zd* Q) {
  zd A[9], B[9];
  zd v[NROW][3];
  ld_link(g, canon, m0, s0, A);
  ld_link(g, canon, m1, s1, B);
#pragma unroll
  for (int r = 0; r < NROW; r++)
#pragma unroll
    for (int k = 0; k < 3; k++) v[r][k] = D0 ? conj(A[3 * k + r]) : A[3 * r + k];
  ld_link(g, canon, m2, s2, A);
  vmul<NROW, D1>(v, B);
  ld_link(g, canon, m3, s3, B);
  vmul<NROW, D2>(v, A);
  vmul<NROW, D3>(v, B);
#pragma unroll
  for (int r = 0; r < NROW; r++)
#pragma unroll
    for (int k = 0; k < 3; k++) Q[3 * r + k] = Q[3 * r + k] + v[r][k];
  if (NROW == 2) {
    Q[6] = Q[6] + conj(v[0][1] * v[1][2] - v[0][2] * v[1][1]);
    Q[7] = Q[7] + conj(v[0][2] * v[1][0] - v[0][0] * v[1][2]);
    Q[8] = Q[8] + conj(v[0][0] * v[1][1] - v[0][1] * v[1][0]);
  }
}

template <int NROW> __device__ __noinline__ void field_strength(const Lat& g, const double* canon, const int* c, int mu, int nu, zd* F) {
  zd Q[9];
#pragma unroll
  for (int i = 0; i < 9; i++) Q[i] = mk<double>(0.0, 0.0);
  const int64_t x = lex(g, c);
  const int64_t xpm = shifted(g, c, mu, +1, nu, 0), xpn = shifted(g, c, mu, 0, nu, +1);
  const int64_t xmm = shifted(g, c, mu, -1, nu, 0), xmn = shifted(g, c, mu, 0, nu, -1);
  const int64_t xmmpn = shifted(g, c, mu, -1, nu, +1), xmmmn = shifted(g, c, mu, -1, nu, -1), xpmmn = shifted(g, c, mu, +1, nu, -1);
  // U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
  leaf<NROW, false, false, true, true>(g, canon, mu, x, nu, xpm, mu, xpn, nu, x, Q);
  // U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
  leaf<NROW, false, true, true, false>(g, canon, nu, x, mu, xmmpn, nu, xmm, mu, xmm, Q);
  // U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
  leaf<NROW, true, true, false, false>(g, canon, mu, xmm, nu, xmmmn, mu, xmmmn, nu, xmn, Q);
  // U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
  leaf<NROW, true, false, false, true>(g, canon, nu, xmn, mu, xmn, nu, xpmmn, mu, x, Q);
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

// One warp per plane: CTA = 32 consecutive lexicographic sites x 6 planes (192 threads). Thread (site, plane) computes
// the Hermitian F_plane(site) (4 leaves = 12 SU(3) products in fp64) and leaves its 9 independent reals in shared
// memory; warps 0 and 1 then assemble the packed block of chirality 0 / 1 of the 32 sites and store the fp64 and fp32
// copies (one 16-byte vector per lane and plane: coalesced). The earlier one-thread-per-site version kept six field
// strengths and both blocks in one thread (255 registers + 1.9 KB of spills) and ran 4x slower.
//
// Traversal. A site's six field strengths touch the links of its 2-hop neighbourhood in every plane, so the order in
// which the CTAs sweep the lattice decides how often a link comes from DRAM. In plain checkerboard order (all of one
// parity, then the other; the +-t neighbours a whole time slice apart) ncu counted 50.6 GB of DRAM reads at 48^3 x 144
// for a 9.17 GB gauge field. The sweep therefore goes tile by tile: tiles of (all x) x By x Bz x Bt sites (B = the
// largest divisor <= 8 of the extent), inside a tile first the even then the odd sites, each in (xh, y, z, t) order, so
// that everything a tile needs (its own links plus a one-site halo in y, z, t: 1.95x its volume at B = 8) stays in L2
// while the tile is worked on, and the y-neighbour tile comes next.
struct CloverTiles {
  int By, Bz, Bt;   // tile extents in y, z, t
  int nby, nbz;     // tiles along y, z
  int ts;           // sites of one parity in a tile = Lh * By * Bz * Bt
};
enum { CB_SITES = 32 };
#ifndef TMW_CLOVER_MINB
#define TMW_CLOVER_MINB 2
#endif
template <int NROW> __global__ void __launch_bounds__(6 * CB_SITES, TMW_CLOVER_MINB) clover_build_kernel(const Geom g, const CloverTiles tl, const double2* __restrict__ u64e, const double2* __restrict__ u64o, double k, double diag, double2* c64e, double2* c64o, float4* c32e, float4* c32o) {
  __shared__ double Fs[6][9][CB_SITES];  // [plane][re(0,0) re(1,1) re(2,2) re/im(1,0) re/im(2,0) re/im(2,1)][site]
  const int lane = threadIdx.x & 31, plane = threadIdx.x >> 5;
  // position of this lane's site in the sweep: (tile, parity, index inside the tile's parity)
  const int64_t pos = (int64_t)blockIdx.x * CB_SITES + lane;
  const int tile = (int)(pos / (2 * tl.ts));
  int r = (int)(pos - (int64_t)tile * 2 * tl.ts);
  const int par = r / tl.ts;
  r -= par * tl.ts;
  const double* canon = nullptr;
  Lat lt;
  lt.L = g.L;
  lt.T = g.T;
  lt.Lh = g.Lh;
  lt.Vh = g.Vh;
  lt.U[0] = u64e;
  lt.U[1] = u64o;
  const bool active = pos < 2 * (int64_t)g.Vh;
  int c[4] = {0, 0, 0, 0};
  int cb = 0;
  if (active) {
    const int xh = r % g.Lh;
    int q = r / g.Lh;
    c[1] = (tile % tl.nby) * tl.By + q % tl.By; q /= tl.By;
    c[2] = ((tile / tl.nby) % tl.nbz) * tl.Bz + q % tl.Bz; q /= tl.Bz;
    c[3] = (tile / (tl.nby * tl.nbz)) * tl.Bt + q;
    c[0] = 2 * xh + ((c[1] + c[2] + c[3] + par) & 1);
    cb = xh + g.Lh * (c[1] + g.L * (c[2] + g.L * c[3]));
    zd F[9];
    // planes: xy=0 xz=1 xt=2 yz=3 yt=4 zt=5. mu, nu are RUNTIME values (one copy of the 12 unrolled 3x3 products for
    // all six warps): with one specialised copy per plane the kernel was instruction-fetch bound (ncu: stall
    // no_instruction 8.9 per issue, fp64 pipe 24 %).
    const int mu = (plane < 3) ? 0 : (plane < 5 ? 1 : 2);
    const int nu = (plane < 3) ? plane + 1 : (plane < 5 ? plane - 1 : 3);
    field_strength<NROW>(lt, canon, c, mu, nu, F);
    Fs[plane][0][lane] = F[0].re;
    Fs[plane][1][lane] = F[4].re;
    Fs[plane][2][lane] = F[8].re;
    Fs[plane][3][lane] = F[3].re; Fs[plane][4][lane] = F[3].im;
    Fs[plane][5][lane] = F[6].re; Fs[plane][6][lane] = F[6].im;
    Fs[plane][7][lane] = F[7].re; Fs[plane][8][lane] = F[7].im;
  }
  __syncthreads();
  if (plane >= 2 || !active) return;
  // chirality b = plane: upper (b = 0): E1 = F_yz - F_xt, E2 = F_xz + F_yt, E3 = F_xy - F_zt; lower: opposite signs
  const double sg = plane ? 1.0 : -1.0;
  zd E1[9], E2[9], E3[9];
  {
    // rebuild full Hermitian matrices from the 9 reals
    auto herm = [&](int pa, int pb, double sa, double sb, zd* E) {
      double v[9];
#pragma unroll
      for (int i = 0; i < 9; i++) v[i] = sa * Fs[pa][i][lane] + sb * Fs[pb][i][lane];
      E[0] = mk<double>(v[0], 0.0); E[4] = mk<double>(v[1], 0.0); E[8] = mk<double>(v[2], 0.0);
      E[3] = mk<double>(v[3], v[4]); E[1] = mk<double>(v[3], -v[4]);
      E[6] = mk<double>(v[5], v[6]); E[2] = mk<double>(v[5], -v[6]);
      E[7] = mk<double>(v[7], v[8]); E[5] = mk<double>(v[7], -v[8]);
    };
    herm(3, 2, 1.0, sg, E1);    // F_yz -/+ F_xt
    herm(1, 4, 1.0, -sg, E2);   // F_xz +/- F_yt
    herm(0, 5, 1.0, sg, E3);    // F_xy -/+ F_zt
  }
  double B[36];
  pack_block(E1, E2, E3, k, diag, B);
  double2* d64 = (par ? c64o : c64e) + (int64_t)plane * 18 * g.Vh;
  float4* d32 = (par ? c32o : c32e) + (int64_t)plane * 9 * g.Vh;
  float Bf[36];
#pragma unroll
  for (int i = 0; i < 36; i++) Bf[i] = (float)B[i];
  store_reals<36>(d64, g.Vh, cb, B);
  store_reals<36>(d32, g.Vh, cb, Bf);
}

cudaError_t launch_clover_build(const Geom& g, const void* g64_even, const void* g64_odd, double c_sw, double diag, void* c64_even, void* c64_odd, void* c32_even, void* c32_odd, bool su3, cudaStream_t s) {
  const auto tile_extent = [](int n) { int b = 1; for (int d = 2; d <= 8; d++) if (n % d == 0) b = d; return b; };
  CloverTiles tl;
  tl.By = tl.Bz = tile_extent(g.L);
  tl.Bt = tile_extent(g.T);
  tl.nby = tl.nbz = g.L / tl.By;
  tl.ts = g.Lh * tl.By * tl.Bz * tl.Bt;
  const dim3 grid((unsigned)((2 * (int64_t)g.Vh + CB_SITES - 1) / CB_SITES), 1, 1);
  if (su3) clover_build_kernel<2><<<grid, 6 * CB_SITES, 0, s>>>(g, tl, (const double2*)g64_even, (const double2*)g64_odd, 0.5 * c_sw, diag, (double2*)c64_even, (double2*)c64_odd, (float4*)c32_even, (float4*)c32_odd);
  else clover_build_kernel<3><<<grid, 6 * CB_SITES, 0, s>>>(g, tl, (const double2*)g64_even, (const double2*)g64_odd, 0.5 * c_sw, diag, (double2*)c64_even, (double2*)c64_odd, (float4*)c32_even, (float4*)c32_odd);
  return cudaGetLastError();
}

// ---- fallback inverse of a packed Hermitian block: Gauss-Jordan with partial pivoting on the full complex 6x6 (used only
// when the unpivoted factorisation below met a tiny pivot; dynamic row indexing puts M and X in local memory) ----
// M = C (tw2 == 0) or C^2 + tw2 (twisted clover: (C + i tw)^{-1} = (C - i tw)(C^2 + tw^2)^{-1}); result Hermitian.
__global__ void __launch_bounds__(64) clover_invert_pivot_kernel(const Geom g, const double2* __restrict__ c64, double tw2, double2* inv64, float4* inv32, int* singular) {
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

// ---- inverse of a packed Hermitian block by an unpivoted L D L^dag factorisation, fully unrolled so that every index is
// static and the factors live in registers: A = L D L^dag, A^{-1} = L^{-dag} D^{-1} L^{-1}. M = C, or C^2 + tw2 for
// twisted clover ((C + i tw)^{-1} = (C - i tw)(C^2 + tw^2)^{-1}). Without pivoting the factorisation is backward stable
// for DEFINITE blocks only — which is what physical parameters give (|clover term| <= 3 c_sw < 4 + m) — so a pivot of
// the wrong sign or below 1e-6 of the block's scale sets *retry: the host then reruns the field with the pivoted kernel
// above, which alone decides whether a block is singular. ----
__global__ void __launch_bounds__(64) clover_invert_kernel(const Geom g, const double2* __restrict__ c64, double tw2, double2* inv64, float4* inv32, int* retry) {
  const int idx = blockIdx.x * 64 + threadIdx.x;  // (block b, cb)
  if (idx >= 2 * g.Vh) return;
  const int b = idx / g.Vh, cb = idx % g.Vh;
  double P[36];
  load_reals<36>(c64 + (int64_t)b * 18 * g.Vh, g.Vh, cb, P);
  // lower triangle of A: a[i][j], j <= i (diagonal real)
  zd a[6][6];
#pragma unroll
  for (int i = 0; i < 6; i++) {
    a[i][i] = mk<double>(P[i], 0.0);
#pragma unroll
    for (int j = 0; j < 6; j++)
      if (j < i) a[i][j] = mk<double>(P[6 + 2 * (i * (i - 1) / 2 + j)], P[6 + 2 * (i * (i - 1) / 2 + j) + 1]);
  }
  if (tw2 != 0.0) {  // A <- A^2 + tw2 (Hermitian): (A^2)_ij = sum_k A_ik conj(A_jk)
    zd q[6][6];
#pragma unroll
    for (int i = 0; i < 6; i++)
#pragma unroll
      for (int j = 0; j < 6; j++)
        if (j <= i) {
          zd sum = mk<double>(i == j ? tw2 : 0.0, 0.0);
#pragma unroll
          for (int k = 0; k < 6; k++) {
            const zd aik = (k <= i) ? a[i][k] : conj(a[k][i]);
            const zd ajk = (k <= j) ? a[j][k] : conj(a[k][j]);
            cmad(sum, aik, conj(ajk));
          }
          q[i][j] = sum;
        }
#pragma unroll
    for (int i = 0; i < 6; i++)
#pragma unroll
      for (int j = 0; j < 6; j++)
        if (j <= i) a[i][j] = q[i][j];
#pragma unroll
    for (int i = 0; i < 6; i++) a[i][i].im = 0.0;
  }
  double scale = 0.0;
#pragma unroll
  for (int i = 0; i < 6; i++)
#pragma unroll
    for (int j = 0; j < 6; j++)
      if (j <= i) scale = fmax(scale, fabs(a[i][j].re) + fabs(a[i][j].im));
  // in place: a[i][j] (j < i) <- L_ij, d[j] <- D_j
  double d[6], dinv[6];
  bool bad = !(scale > 0.0);
#pragma unroll
  for (int j = 0; j < 6; j++) {
    double dj = a[j][j].re;
#pragma unroll
    for (int k = 0; k < 6; k++)
      if (k < j) dj -= (a[j][k].re * a[j][k].re + a[j][k].im * a[j][k].im) * d[k];
    d[j] = dj;
    // stable only for definite blocks (all pivots of one sign, none tiny): anything else goes to the pivoted kernel
    if (!(fabs(dj) > 1e-6 * scale) || dj * d[0] < 0.0) bad = true;
    dinv[j] = 1.0 / dj;
#pragma unroll
    for (int i = 0; i < 6; i++)
      if (i > j) {
        zd v = a[i][j];
#pragma unroll
        for (int k = 0; k < 6; k++)
          if (k < j) {
            const zd t = a[i][k] * conj(a[j][k]);
            v.re -= t.re * d[k];
            v.im -= t.im * d[k];
          }
        a[i][j] = mk<double>(v.re * dinv[j], v.im * dinv[j]);
      }
  }
  // W = L^{-1} (unit lower), in place column by column: W_ij = -L_ij - sum_{j<k<i} L_ik W_kj
  zd w[6][6];
#pragma unroll
  for (int j = 0; j < 6; j++)
#pragma unroll
    for (int i = 0; i < 6; i++)
      if (i > j) {
        zd v = mk<double>(-a[i][j].re, -a[i][j].im);
#pragma unroll
        for (int k = 0; k < 6; k++)
          if (k > j && k < i) {
            const zd t = a[i][k] * w[k][j];
            v.re -= t.re;
            v.im -= t.im;
          }
        w[i][j] = v;
      }
  // A^{-1}_ij = sum_{k >= i} conj(W_ki) W_kj / D_k  (i >= j; W_kk = 1)
  if (bad) {
    atomicExch(retry, 1);
    return;
  }
#pragma unroll
  for (int i = 0; i < 6; i++) {
#pragma unroll
    for (int j = 0; j < 6; j++)
      if (j <= i) {
        zd sum = mk<double>(0.0, 0.0);
#pragma unroll
        for (int k = 0; k < 6; k++)
          if (k >= i) {
            const zd wki = (k == i) ? mk<double>(1.0, 0.0) : w[k][i];
            const zd wkj = (k == j) ? mk<double>(1.0, 0.0) : w[k][j];
            const zd t = conj(wki) * wkj;
            sum.re += t.re * dinv[k];
            sum.im += t.im * dinv[k];
          }
        if (i == j) P[i] = sum.re;
        else {
          P[6 + 2 * (i * (i - 1) / 2 + j)] = sum.re;
          P[6 + 2 * (i * (i - 1) / 2 + j) + 1] = sum.im;
        }
      }
  }
  float Pf[36];
#pragma unroll
  for (int i = 0; i < 36; i++) Pf[i] = (float)P[i];
  store_reals<36>(inv64 + (int64_t)b * 18 * g.Vh, g.Vh, cb, P);
  store_reals<36>(inv32 + (int64_t)b * 9 * g.Vh, g.Vh, cb, Pf);
}

cudaError_t launch_clover_invert(const Geom& g, const void* c64, double tw2, void* inv64, void* inv32, int* flag, cudaStream_t s) {
  const int n = 2 * g.Vh;
  clover_invert_kernel<<<(n + 63) / 64, 64, 0, s>>>(g, (const double2*)c64, tw2, (double2*)inv64, (float4*)inv32, flag);
  return cudaGetLastError();
}
cudaError_t launch_clover_invert_pivot(const Geom& g, const void* c64, double tw2, void* inv64, void* inv32, int* singular, cudaStream_t s) {
  const int n = 2 * g.Vh;
  clover_invert_pivot_kernel<<<(n + 63) / 64, 64, 0, s>>>(g, (const double2*)c64, tw2, (double2*)inv64, (float4*)inv32, singular);
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
