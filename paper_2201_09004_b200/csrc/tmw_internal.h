// tmw_internal.h — launcher declarations shared by the .cu files of libtmw.so (private to csrc/).
#pragma once
#include "tmw_core.cuh"

namespace tmw {

// ---- stencil (tmw_dslash_f32.cu / tmw_dslash_f64.cu) ----
// ng = stored reals per link (12 | 18), epi = EPI_*, clover = CL_NONE | CL_CLOVER | CL_TWISTED (kind of diagonal part),
// nr = right-hand-side columns per thread (fp32: 1..4; fp64: always 1)
cudaError_t launch_dslash(const DslashArgs<float>& a, int ng, int epi, int clover, int nr, cudaStream_t s);
cudaError_t launch_dslash(const DslashArgs<double>& a, int ng, int epi, int clover, int nr, cudaStream_t s);
// Shared-memory staged fp32 stencil (tmw_dslash_stage.cuh; north_star subsystem (2)): a CTA covers a tile of one time slice and
// stages the input sites the tile's spatial hops need.
struct StageGeom {
  int txh, ty, tz;     // output sites per tile along x/2, y, z (one time slice)
  int ntx, nty, ntz;   // tiles along x/2, y, z
  int fullx;           // the tile spans the whole x extent (txh = Lh): no x halo, the x wrap happens inside the row
  int rw;              // staged sites per row: Lh if fullx, else txh + 2 (one halo site per side)
  int nrows;           // ty*tz interior rows + 2*tz (y halos) + 2*ty (z halos)
  int nslots;          // nrows * rw = float4 per staged plane and column
  int nthr;            // txh * ty * tz active threads (blockDim.x = nthr rounded up to a warp)
};
// epi: EPI_HOP | EPI_AINV_HOP | EPI_A_XPAY; nr = 1..3 columns per thread; the whole lattice, no domain decomposition
cudaError_t launch_dslash_stage(const DslashArgs<float>& a, int ng, int epi, int clover, int nr, const StageGeom& sg, cudaStream_t s);
int stage_max_threads(int nr);  // largest CTA of the staged kernel with nr columns per thread
// loads and stores of the fp32 hopping kernel without its arithmetic (measurement: tmw_time_kernel)
cudaError_t launch_hop_loadonly(const DslashArgs<float>& a, int ng, cudaStream_t s);

// register-only fp32 FMA loop (packed = 0: scalar FFMA, 1: FFMA2 pairs), (SM count) x 8 CTAs of 256 threads, fmas_per_thread FMAs each;
// sink: >= sms * 8 * 256 floats (sms = the device's SM count)
cudaError_t launch_ffma_probe(int packed, int fmas_per_thread, int sms, float* sink, cudaStream_t s);

// ---- domain decomposition (tmw_dd_f32.cu / tmw_dd_f64.cu) ----
// a describes ONE domain (local geometry and fields, a.dd its cuts and receive buffers). pass 0: interior (all sites, the
// hops through a cut skipped, sites on a cut left raw in a.out); pass 1: exterior (the sites on a cut: + ghost terms,
// epilogue, reductions). One column per thread, a.ncol columns per launch.
cudaError_t launch_dslash_dd(const DslashArgs<float>& a, int ng, int epi, int clover, int pass, cudaStream_t s);
cudaError_t launch_dslash_dd(const DslashArgs<double>& a, int ng, int epi, int clover, int pass, cudaStream_t s);
// half spinors for the neighbours of the domain from a.in: send[direction z,t][0: to the neighbour behind, 1: ahead]
cudaError_t launch_face_pack(const DslashArgs<float>& a, int ng, void* const (&send)[2][2], cudaStream_t s);
cudaError_t launch_face_pack(const DslashArgs<double>& a, int ng, void* const (&send)[2][2], cudaStream_t s);
// dst (packed field of domain g, nplanes planes of 16-byte vectors) <- src (the same field of the whole lattice, gVh sites per parity)
cudaError_t launch_extract_planes(const Geom& g, int nplanes, int64_t gVh, const void* src, void* dst, cudaStream_t s);

// out = A in (inverse = 0) or A^{-1} in (inverse = 1) on parity par, site-local
cudaError_t launch_diag(const Diag<float>& d, const Geom& g, int par, bool clover, int inverse, const void* in, void* out, cudaStream_t s);
cudaError_t launch_diag(const Diag<double>& d, const Geom& g, int par, bool clover, int inverse, const void* in, void* out, cudaStream_t s);

// ---- layout (tmw_pack.cu) ----
// canonical gauge [mu][lex][3][3][2] fp64 -> packed per parity: g64 [par][mu][9 planes][Vh] double2,
// g32 [par][mu][NP planes][Vh] float4 with ng32 reals (12 | 18)
cudaError_t launch_pack_gauge(const Geom& g, const double* canon, void* g64_even, void* g64_odd, void* g32_even, void* g32_odd, int ng32, cudaStream_t s);
// canonical spinor fp64 <-> packed parity spinor (prec 0: float4 planes, 1: double2 planes)
cudaError_t launch_pack_spinor(const Geom& g, int par, int prec, const double* canon, void* packed, cudaStream_t s);
cudaError_t launch_unpack_spinor(const Geom& g, int par, int prec, const void* packed, double* canon, cudaStream_t s);
// both parities in one launch (coalesced on the canonical side); [lex0, lex1) = the (local) lexicographic sites to convert
// (lex1 < 0: all), e.g. one t-slab
cudaError_t launch_pack_spinor_both(const Geom& g, int prec, const double* canon, void* packed_even, void* packed_odd, cudaStream_t s, int64_t lex0 = 0, int64_t lex1 = -1);
cudaError_t launch_unpack_spinor_both(const Geom& g, int prec, const void* packed_even, const void* packed_odd, double* canon, cudaStream_t s, int64_t lex0 = 0, int64_t lex1 = -1);

// ---- clover (tmw_clover.cu) ----
// From the packed fp64 gauge (launch_pack_gauge's g64): packed Hermitian blocks C = (c_sw/2) sum sigma F + diag, both
// parities, fp64 [36 planes][Vh] double2 and fp32 [18 planes][Vh] float4.
// su3: the links are SU(3) (the context stores 12-real fp32 links, which requires it): the third row of every plaquette
// product is rebuilt from the first two instead of multiplied out
cudaError_t launch_clover_build(const Geom& g, const void* g64_even, const void* g64_odd, double c_sw, double diag, void* c64_even, void* c64_odd, void* c32_even, void* c32_odd, bool su3, cudaStream_t s);
// inverse blocks of one parity: (C^2 + tw2)^{-1} if tw2 != 0 else C^{-1}. launch_clover_invert: unpivoted LDL^dag in
// registers; *flag (device int) is set if any block met a tiny pivot (its output is then not written) and the caller
// reruns the field with launch_clover_invert_pivot (Gauss-Jordan with pivoting), whose *singular is set on failure.
cudaError_t launch_clover_invert(const Geom& g, const void* c64, double tw2, void* inv64, void* inv32, int* flag, cudaStream_t s);
cudaError_t launch_clover_invert_pivot(const Geom& g, const void* c64, double tw2, void* inv64, void* inv32, int* singular, cudaStream_t s);
// packed [planes][Vh] double2 blocks -> [cb][2][36] doubles
cudaError_t launch_clover_export(const Geom& g, const void* c64, double* dst, cudaStream_t s);

// ---- BLAS-1 with fused reductions (tmw_blas.cu) ----
// Device scalar block of the BiCGStab recurrences (all complex as re,im doubles).
struct Scalars {
  double rho[2];      // <rhat, r>           (sc_omega: <rhat,s> - omega <rhat,t>; resid_convert after a reliable update)
  double rho_old[2];
  double alpha[2];
  double omega[2];
  double beta[2];
  double rhat_v[2];   // <rhat, v>           (accumulated by the first K2)
  double ts[2];       // <t, s>              (accumulated by the second K2, red_mode 4: the next 7 doubles in this order)
  double tt;          // <t, t>
  double rhat_t[2];   // <rhat, t>
  double rhat_s[2];   // <rhat, s>
  double rr;          // <r, r>              (accumulated by update_xrp / resid_convert)
  double nrm;         // generic norm^2 accumulator
  // what the device needs to decide, at the start of an iteration, whether the host must look at this column first
  // (sc_begin_iter with check != 0; the host sets these three whenever it (re)starts the recurrence):
  double stop2;       // (tol |b|)^2: converged when rr <= stop2
  double maxr2;       // largest rr since the last reliable update (0: not set yet, the next rr is taken)
  double brk2;        // (eps_break |rhat|)^2: breakdown when |rho|^2 <= brk2 * rr
  long long trip;     // TRIP_* bits of the last check
};
enum { TRIP_BROKEN = 1, TRIP_CONV = 2, TRIP_RELIABLE = 4, TRIP_BREAKDOWN = 8 };
// GCR(k) scalars (device): see the gcr_* kernels of tmw_blas.cu
enum { GCR_KMAX = 16 };
struct GcrScalars {
  double dots[2 * GCR_KMAX];  // <q_j, w>
  double coef[2 * GCR_KMAX];  // dots_j / nq_j
  double nq[GCR_KMAX];        // <q_j, q_j>
  double nw;                  // <w, w> after orthogonalisation
  double g[2];                // <w, r>
  double a[2];                // g / nw
  double rr;                  // <r, r> after the update
  double pad[2];
};
// One GCR step for the columns of cm after q_i = Mhat r has been stored as vector i of Q: orthogonalise it against
// q_0..q_{i-1} (classical Gram-Schmidt, one pass for the dot products and one for the updates), build p_i alongside, then
// x += a p_i, r -= a q_i with a = <q_i, r>/<q_i, q_i>; gs[c].rr = |r|^2. n16 = 16-byte vectors per spinor; vector j of
// column c of Q / P starts (j*ncw + c) spinors after the base pointer; 5 launches (4 for i = 0).
struct ColMap;
template <typename R> cudaError_t launch_gcr_step(int64_t n16, int i, int ncw, void* Q, void* P, void* x, void* r, GcrScalars* gs, const ColMap& cm, cudaStream_t s);

// The right-hand-side columns a batched launch works on: slot j -> column col[j].
struct ColMap {
  int n;
  unsigned char col[MAXCOL];
};
// Every launcher below is batched: column c of a vector starts c * (column length) after the base pointer and
// uses the scalar block sc[c]; reductions into a plain double* go to out + 4*c.
// sc phase kernels (one thread per column): see tmw_blas.cu
// `attn` (device int[2]) lets the host run one iteration ahead of the device without a round trip per iteration (SURVEY §3b
// "read back only a convergence flag"): attn[0] != 0 = some column needs the host (converged, reliable update due,
// breakdown, non-finite scalar); every kernel of the iteration (`skip` = attn) then returns at once, so that the vectors and
// scalars stay as the last finished iteration left them. attn[1] counts the iterations really done.
// sc_begin_iter: if check != 0, first test every column of cm against its stop2 / maxr2 (delta2 = delta^2) / brk2, record
// Scalars::trip and raise attn[0]; unless attn[0] is raised: zero the accumulators of the two K2 launches, attn[1]++.
cudaError_t launch_sc_begin_iter(Scalars* sc, const ColMap& cm, int* attn, int check, double delta2, cudaStream_t s);
cudaError_t launch_sc_alpha(Scalars* sc, const ColMap& cm, const int* skip, cudaStream_t s);       // alpha = rho / rhat_v
// omega = ts/tt; rho_old = rho; rho = <rhat,s> - omega <rhat,t> (= <rhat, s - omega t>, the new <rhat,r>);
// beta = (rho/rho_old)(alpha/omega); zero rr
cudaError_t launch_sc_omega(Scalars* sc, const ColMap& cm, const int* skip, cudaStream_t s);
// n = number of 16-byte vectors in one column of each array
template <typename R> cudaError_t launch_update_s(int64_t n, void* sv, const void* r, const void* v, const Scalars* sc, const ColMap& cm, const int* skip, cudaStream_t s);     // s = r - alpha v
// x += alpha p + omega s; r = s - omega t; p = r + beta (p - omega v); rr += <r,r>  (the end of one BiCGStab iteration and
// the search direction of the next in one pass: 5 reads + 3 writes instead of 8 + 3 in two kernels)
template <typename R> cudaError_t launch_update_xrp(int64_t n, void* x, void* r, void* p, const void* sv, const void* t, const void* v, Scalars* sc, const ColMap& cm, const int* skip, cudaStream_t s);
// out[4c+0..1] += <a,b>, out[4c+2] += <b,b> (a may be null: only the norm)
template <typename R> cudaError_t launch_dot_norm(int64_t n, const void* a, const void* b, double* out, const ColMap& cm, cudaStream_t s);
// fp64 helpers for the reliable update
// vh = sites per parity of one domain (the fp32 <-> fp64 plane correspondence works per domain block of 24 reals x vh)
template <typename R> cudaError_t launch_acc_y(int64_t n64, int64_t vh, void* y64, void* x, const ColMap& cm, cudaStream_t s);  // y += x; x = 0   (n64 = number of double2 vectors per column)
// r64 = b64 - w64 (w64 may be null: zero); r = (R) r64; rho += <rhat, r>; rr += <r64, r64>. If p is not null (reliable update in the middle of
// the recurrence): p += r_new - r_old, i.e. the search direction already built from the iterated residual is moved to
// the true one.
template <typename R> cudaError_t launch_resid_convert(int64_t n64, int64_t vh, const void* b64, const void* w64, void* r64, void* r, const void* rhat, void* p, Scalars* sc, const ColMap& cm, cudaStream_t s);
// dst(R) = src(double), n64 double2 vectors per column
template <typename R> cudaError_t launch_convert(int64_t n64, int64_t vh, const void* src64, void* dst, const ColMap& cm, cudaStream_t s);
// d = a - b (fp64, n64 double2 vectors per column), out[4c+2] += <d,d>
cudaError_t launch_sub_norm(int64_t n64, const void* a, const void* b, void* d, double* out, const ColMap& cm, cudaStream_t s);

// a += b (fp64, n64 double2 vectors per column)
cudaError_t launch_add64(int64_t n64, void* a, const void* b, const ColMap& cm, cudaStream_t s);

// Clenshaw step (fp64, one column, n64 double2 vectors): out = c*psi + f*(scale*hb + shift*b1) - b2; out may alias b2
cudaError_t launch_clenshaw(int64_t n64, void* out, const void* psi, const void* hb, const void* b1, const void* b2, double c, double f, double scale,
                            double shift, cudaStream_t s);
cudaError_t launch_scale(int64_t n64, void* dst, const void* src, double c, cudaStream_t s);  // dst = c * src

}  // namespace tmw
