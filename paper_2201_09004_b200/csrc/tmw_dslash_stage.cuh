// tmw_dslash_stage.cuh — the fp32 Dslash stencil with the neighbour spinors of a site tile staged through shared
// memory (BASELINE.json north_star subsystem (2): "neighbour tiles staged through TMA/shared memory"; SURVEY §8(a) A3/A4,
// §8(f1); the hopping part of PAPER.md:62 Eq. (2) for the "12 columns" of PAPER.md:78).
//
// Why: with the links amortised over several right-hand-side columns, the plain kernel (tmw_dslash_impl.cuh) pulls
// 8 neighbour spinors per site and column through L1 — ~700 B per site and column from L2 for 192 B of compulsory spinor
// traffic — and stalls on those loads with 12 warps/SM (profiles/r1_dslash_full.md: DRAM 44-64 %, long scoreboard).
// Here a CTA owns a tile of one time slice, TXH (in x/2) x TY x TZ output sites of parity par, and first copies the input
// sites of that slice the tile needs — the tile's own sites of the other parity plus one row of halo on each side in
// y, z (and one site in x/2 when the tile does not span the whole x extent) — into shared memory with 16-byte
// asynchronous copies (cp.async.cg = LDGSTS, no registers, deep queue), planes of float4 exactly as in global memory.
// The six spatial hops then read their spinors from shared memory (every staged spinor serves ~3 hops); the two
// t hops and the links still come from global memory, and the t hops are computed BEFORE the wait on the
// copies so that their latency overlaps the fill. Periodic wrap is applied per staged row by the index arithmetic of
// the fill (a TMA box would zero-fill instead of wrapping; with cp.async the wrap costs nothing).
#pragma once
#include "tmw_dslash_impl.cuh"

namespace tmw {

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit_wait() {
  asm volatile("cp.async.commit_group;" ::: "memory");
  asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// 24 reals of a staged spinor: plane k at st[k * nslots + slot]
__device__ __forceinline__ void lds_spinor(const float4* st, int nslots, int slot, float* v) {
#pragma unroll
  for (int k = 0; k < 6; k++) {
    const float4 q = st[k * nslots + slot];
    v[4 * k] = q.x;
    v[4 * k + 1] = q.y;
    v[4 * k + 2] = q.z;
    v[4 * k + 3] = q.w;
  }
}

// the two hops of a spatial direction with the neighbour spinors in shared memory (slots sf, sb) and the links from
// global memory (forward: U_mu(x) of this parity at cb; backward: U_mu(x-mu) of the other parity at n.bwd[MU])
template <int NG, int MU, int NR, bool STREAM>
__device__ __forceinline__ void hop_pair_staged(const DslashArgs<float>& a, const Nbr& n, int cb, const float4* st, int nslots, int sf, int sb,
                                                float (&acc)[NR][24]) {
  const int NPG = Planes<float, NG>::N;
  const int64_t Vh = a.g.Vh;
  {
    cx<float> U[9];
    load_link<float, NG, STREAM>((const float4*)a.U[a.par] + (int64_t)MU * NPG * Vh, Vh, cb, U);
#pragma unroll
    for (int j = 0; j < NR; j++) {
      float psi[24];
      lds_spinor(st + j * 6 * nslots, nslots, sf, psi);
      hop<float, MU, true>(psi, U, a.sig, 1.f, acc[j]);
    }
  }
  {
    cx<float> U[9];
    load_link<float, NG, STREAM>((const float4*)a.U[1 - a.par] + (int64_t)MU * NPG * Vh, Vh, n.bwd[MU], U);
#pragma unroll
    for (int j = 0; j < NR; j++) {
      float psi[24];
      lds_spinor(st + j * 6 * nslots, nslots, sb, psi);
      hop<float, MU, false>(psi, U, -a.sig, 1.f, acc[j]);
    }
  }
}

// blockIdx.x = group + ngroups * tile, tile = bx + ntx * (by + nty * (bz + ntz * t)): the CTAs of the column groups of one
// tile are adjacent, so the groups after the first find the links in L2. Dynamic shared memory: NR * 6 * nslots float4.
template <int NG, int EPI, int CLOVER, int NR, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) dslash_stage_kernel(const DslashArgs<float> a, const StageGeom sg) {
  extern __shared__ float4 stage_smem[];
  if (a.skip && *a.skip) return;
  const Geom& g = a.g;
  int tile = blockIdx.x, grp = 0;
  if (a.ngroups > 1) {
    tile = blockIdx.x / a.ngroups;
    grp = blockIdx.x - tile * a.ngroups;
  }
  const int bx = tile % sg.ntx;
  int q = tile / sg.ntx;
  const int by = q % sg.nty;
  q /= sg.nty;
  const int bz = q % sg.ntz;
  const int t = q / sg.ntz;
  const int x0 = bx * sg.txh, y0 = by * sg.ty, z0 = bz * sg.tz;
  int colj[NR], cofs[NR];
  bool valid[NR];
#pragma unroll
  for (int j = 0; j < NR; j++) {
    const int slot = grp * NR + j;
    valid[j] = slot < a.ncol;
    colj[j] = a.col[valid[j] ? slot : a.ncol - 1];
    cofs[j] = colj[j] * a.cstride;
  }
  const int nint = sg.ty * sg.tz;
  // ---- fill: staged slot (row, xs) <- input site (xh, y, z, t) of parity 1 - par, rows wrapped periodically ----
  for (int sl = threadIdx.x; sl < sg.nslots; sl += blockDim.x) {
    const int row = sl / sg.rw, xs = sl - row * sg.rw;
    int y, z;
    if (row < nint) {
      const int zz = row / sg.ty;
      y = y0 + row - zz * sg.ty;
      z = z0 + zz;
    } else if (row < nint + 2 * sg.tz) {  // y halos: below (y0 - 1), then above (y0 + ty)
      const int r = row - nint, hi = r >= sg.tz;
      z = z0 + r - hi * sg.tz;
      y = hi ? (y0 + sg.ty == g.L ? 0 : y0 + sg.ty) : (y0 == 0 ? g.L - 1 : y0 - 1);
    } else {  // z halos
      const int r = row - nint - 2 * sg.tz, hi = r >= sg.ty;
      y = y0 + r - hi * sg.ty;
      z = hi ? (z0 + sg.tz == g.Lz ? 0 : z0 + sg.tz) : (z0 == 0 ? g.Lz - 1 : z0 - 1);
    }
    int xh = xs;
    if (!sg.fullx) {
      xh = x0 - 1 + xs;
      xh = xh < 0 ? g.Lh - 1 : (xh >= g.Lh ? xh - g.Lh : xh);
    }
    const int cbs = xh + g.Lh * (y + g.L * (z + g.Lz * t));
#pragma unroll
    for (int j = 0; j < NR; j++)
#pragma unroll
      for (int k = 0; k < 6; k++) cp_async16(stage_smem + (j * 6 + k) * sg.nslots + sl, (const float4*)a.in + (int64_t)k * g.Vh + cbs + cofs[j]);
  }
  // ---- this thread's output site ----
  const bool active = (int)threadIdx.x < sg.nthr;
  Site s;
  int xl = 0, yy = 0, zz = 0;
  if (active) {
    const int r = threadIdx.x / sg.txh;
    xl = threadIdx.x - r * sg.txh;
    zz = r / sg.ty;
    yy = r - zz * sg.ty;
  }
  s.xh = x0 + xl;
  s.y = y0 + yy;
  s.z = z0 + zz;
  s.t = t;
  s.cb = s.xh + g.Lh * (s.y + g.L * (s.z + g.Lz * s.t));
  const Nbr n = neighbours(g, a.par, s);
  float o[NR][24], r2[NR][3];
#pragma unroll
  for (int j = 0; j < NR; j++)
#pragma unroll
    for (int i = 0; i < 24; i++) o[j][i] = 0.f;
  // the t hops from global memory while the copies are in flight
  if (active) hop_pair<float, NG, 3, NR, NR == 1, 0>(a, n, s.cb, cofs, o);
  cp_async_commit_wait();
  __syncthreads();
  if (active) {
    const int par_x = (s.y + s.z + s.t + a.par) & 1;  // x = 2 xh + par_x: the +x neighbour has x/2 = xh + par_x, the -x one xh + par_x - 1
    const int rowc = yy + sg.ty * zz;
    int xf, xb;
    if (sg.fullx) {
      xf = s.xh + par_x;
      xf = xf == g.Lh ? 0 : xf;
      xb = s.xh + par_x - 1;
      xb = xb < 0 ? g.Lh - 1 : xb;
    } else {
      xf = xl + 1 + par_x;
      xb = xl + par_x;
    }
    const int xc = (sg.fullx) ? s.xh : xl + 1;  // staged x index of the sites with this thread's x/2
    const int base = rowc * sg.rw;
    hop_pair_staged<NG, 0, NR, NR == 1>(a, n, s.cb, stage_smem, sg.nslots, base + xf, base + xb, o);
    const int ryf = (yy + 1 < sg.ty) ? rowc + 1 : nint + sg.tz + zz;
    const int ryb = (yy > 0) ? rowc - 1 : nint + zz;
    hop_pair_staged<NG, 1, NR, NR == 1>(a, n, s.cb, stage_smem, sg.nslots, ryf * sg.rw + xc, ryb * sg.rw + xc, o);
    const int rzf = (zz + 1 < sg.tz) ? rowc + sg.ty : nint + 2 * sg.tz + sg.ty + yy;
    const int rzb = (zz > 0) ? rowc - sg.ty : nint + 2 * sg.tz + yy;
    hop_pair_staged<NG, 2, NR, NR == 1>(a, n, s.cb, stage_smem, sg.nslots, rzf * sg.rw + xc, rzb * sg.rw + xc, o);
    dslash_epilogue<float, NG, EPI, CLOVER, NR, NR == 1>(a, s.cb, cofs, valid, o, r2);
    if (!stored_in_site<EPI, CLOVER>()) {
      if (a.g5) {
#pragma unroll
        for (int j = 0; j < NR; j++)
#pragma unroll
          for (int i = 12; i < 24; i++) o[j][i] = -o[j][i];
      }
#pragma unroll
      for (int j = 0; j < NR; j++)
        if (valid[j] && a.out) store_reals_s<24>(a.out, g.Vh, s.cb + cofs[j], o[j]);
    }
  }
  if (a.red_mode != 0) site_reductions<float, NR, 0>(a, s, active, cofs, colj, valid, o, r2);
}

// launch shapes: the staging buffers allow two CTAs per SM, so 128 registers at 256 threads, 168 at 192
template <int NR> struct StageTune;
template <> struct StageTune<1> { enum { MAXT = 256, MINB = 2 }; };
template <> struct StageTune<2> { enum { MAXT = 256, MINB = 2 }; };
template <> struct StageTune<3> { enum { MAXT = 192, MINB = 2 }; };

template <int NG, int EPI, int CLOVER, int NR> static cudaError_t launch_stage_one(DslashArgs<float> a, const StageGeom& sg, cudaStream_t s) {
  typedef StageTune<NR> TN;
  const int block = (sg.nthr + 31) / 32 * 32;
  if (block > TN::MAXT) return cudaErrorInvalidConfiguration;
  const size_t smem = (size_t)NR * 6 * sg.nslots * sizeof(float4);
  auto kern = dslash_stage_kernel<NG, EPI, CLOVER, NR, TN::MAXT, TN::MINB>;
  // the attribute belongs to (function, device): set it on every launch rather than cache it across devices
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  a.ngroups = (a.ncol + NR - 1) / NR;
  const unsigned grid = (unsigned)((int64_t)sg.ntx * sg.nty * sg.ntz * a.g.T * a.ngroups);
  kern<<<grid, block, smem, s>>>(a, sg);
  return cudaGetLastError();
}

// the kernels the Krylov iteration spends its time in: hop, K1 (all kinds of diagonal part), K2
template <int NG, int NR> static cudaError_t launch_stage_epi(const DslashArgs<float>& a, int epi, int clover, const StageGeom& sg, cudaStream_t s) {
  switch (epi) {
    case EPI_HOP: return launch_stage_one<NG, EPI_HOP, CL_NONE, NR>(a, sg, s);
    case EPI_AINV_HOP:
      if (clover == CL_TWISTED) return launch_stage_one<NG, EPI_AINV_HOP, CL_TWISTED, NR>(a, sg, s);
      return clover ? launch_stage_one<NG, EPI_AINV_HOP, CL_CLOVER, NR>(a, sg, s) : launch_stage_one<NG, EPI_AINV_HOP, CL_NONE, NR>(a, sg, s);
    case EPI_A_XPAY: return clover ? launch_stage_one<NG, EPI_A_XPAY, CL_CLOVER, NR>(a, sg, s) : launch_stage_one<NG, EPI_A_XPAY, CL_NONE, NR>(a, sg, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace tmw
