/*
 * tmw.h — C ABI of libtmw.so: the twisted-mass Wilson(-clover) Dirac operator of arXiv:2201.09004 on one B200
 * (sm_100a), and an even-odd preconditioned mixed-precision BiCGStab that inverts it.
 *
 * What the calls compute (citations: /root/reference/PAPER.md line, section; readings Cn = DESIGN.md "Readings"):
 *
 *   (D psi)(x) = 1/2 sum_mu [ (1+g_mu) U_mu(x) psi(x+mu) s+ + (1-g_mu) U_mu(x-mu)^dag psi(x-mu) s- ]   PAPER.md:62 Eq. (2)
 *                - (4 + Re m) psi(x) - i (Im m) g5 psi(x)                   PAPER.md:62 "-(4+m) delta_xy", m = m_cri+omega
 *                                                                           complex (Eq. (1), :65), reading C4
 *                + (c_sw/2) sum_{mu<nu} sigma_mu_nu F_mu_nu(x) psi(x)       PAPER.md:67 Eq. (3), reading C7
 *
 *   s+- = -1 on a hop that wraps around the time direction (antiperiodic in t, periodic in x,y,z; C6); lattice
 *   units a = 1; gamma matrices in the DeGrand-Rossi basis (C5; g5 = diag(+1,+1,-1,-1)); F_mu_nu is the clover-leaf
 *   field strength built from the same links (clover term and its inverse are computed on the GPU).
 *   tmw_solve returns x with D x = b by BiCGStab (the solver of PAPER.md:73, Table 2 row 1) on the even-odd Schur
 *   complement, fp32 inner recurrences with fp64 reliable updates; the stopping rule is the relative residual of
 *   the FULL system, |b - D x|_2 / |b|_2 <= tol ("residual").
 *
 * Every step runs in CUDA kernels of this library. There is no CPU fallback.
 *
 * Canonical (user-facing) layouts, fp64, x fastest (same as the oracle's; the spin basis is part of the boundary):
 *   gauge   double[4][T][L][L][L][3][3][2]   = [mu (x,y,z,t)][t][z][y][x][row][col][re,im],  U_mu(x)_{row,col}
 *   spinor  double[T][L][L][L][4][3][2]      = [t][z][y][x][spin][colour][re,im]
 *
 * Internal ("packed") layout, used only by the raw parity path (tmw_pack / tmw_unpack / tmw_apply EVEN|ODD /
 * tmw_apply_schur): one parity (x+y+z+t mod 2) of the lattice, checkerboard index cb = lex/2 with
 * lex = x + L (y + L (z + L t)), stored as planes of 16-byte vectors: plane k of a spinor holds reals
 * [k*n, k*n+n) of the site's 24 reals (spin, colour, re/im order), n = 4 (fp32, float4) or 2 (fp64, double2);
 * element (k, cb) is at vector index k*V_h + cb, V_h = L^3 T / 2. tmw_spinor_bytes gives the size.
 *
 * Pointers: `location` in tmw_options says whether the gauge/in/out/b/x pointers of the canonical-layout calls are
 * HOST or DEVICE pointers. Packed-layout pointers are always DEVICE pointers. All pointers must be 16-byte aligned;
 * in and out must not alias. The context owns every internal buffer and frees it in tmw_destroy; the caller owns
 * gauge (read only during tmw_create; may be freed afterwards), in, out, b, x.
 *
 * Errors: every int function returns TMW_OK (0) or a negative code; tmw_last_error gives a text. Nothing aborts
 * or throws across this boundary.
 */
#ifndef TMW_H
#define TMW_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tmw_ctx tmw_ctx; /* opaque */

typedef struct { double re, im; } tmw_complex;

/* error codes */
#define TMW_OK 0
#define TMW_EINVAL (-1)     /* null pointer, odd or too small L/T, tol <= 0, bad enum */
#define TMW_ENOMEM (-2)     /* a device or host allocation failed */
#define TMW_ECUDA (-3)      /* a CUDA call failed; text in tmw_last_error */
#define TMW_ESINGULAR (-4)  /* a clover block (or the twisted-mass diagonal) is not invertible */
#define TMW_ENOCONV (-5)    /* max_iter reached: x holds the best iterate, info is filled */
#define TMW_EBREAKDOWN (-6) /* BiCGStab breakdown (rho or <t,t> vanished / NaN): 5 consecutive restarts brought no progress */

/* enums */
#define TMW_DEVICE 0
#define TMW_HOST 1

#define TMW_MIXED 0  /* fp32 inner BiCGStab, fp64 reliable updates (default) */
#define TMW_DOUBLE 1 /* everything in fp64 */

#define TMW_BICGSTAB 0
#define TMW_GCR 1

#define TMW_TWIST_GAMMA5 0 /* mass term -(4+Re m) - i Im m g5  (default, reading C4) */
#define TMW_MASS_SCALAR 1  /* mass term -(4+m) with a complex scalar m (the literal alternative) */

#define TMW_D 0
#define TMW_DDAG 1
#define TMW_G5D 2 /* gamma5 D (= H_w when m is real): gamma5 fused into the stencil's epilogue */

#define TMW_FULL 0
#define TMW_EVEN 1
#define TMW_ODD 2

#define TMW_F32 0
#define TMW_F64 1

typedef struct {
  size_t struct_size; /* = sizeof(tmw_options) of the header the caller was compiled against (TMW_OPTIONS_INIT sets it).
                         tmw_create refuses (TMW_EINVAL) a size it does not know instead of misreading a struct laid out by
                         another version of this header; every other member may be 0 = default. */
  int location;     /* TMW_DEVICE (default) | TMW_HOST: where canonical-layout pointers live */
  int precision;    /* TMW_MIXED (default) | TMW_DOUBLE: solver arithmetic */
  int reconstruct;  /* fp32 gauge storage: 12 (default; third row rebuilt in-kernel, links must be SU(3)) | 18 */
  int mass_reading; /* TMW_TWIST_GAMMA5 (default) | TMW_MASS_SCALAR */
  int max_iter;     /* BiCGStab iterations; 0 -> 10000 */
  double delta;     /* reliable-update threshold: fp64 true residual when |r| < delta * max|r|; 0 -> 1e-5 */
  void* stream;     /* cudaStream_t all work is queued on; NULL = the legacy default stream */
  int solver;       /* TMW_BICGSTAB (default; the paper's CPU solver) | TMW_GCR (its "standard GPU inverter with
                       GCR algorithm"): restarted GCR(nkrylov) on the same Schur system and kernels */
  int nkrylov;      /* GCR restart length, 1..16; 0 -> 8 */
  int verbose;      /* != 0: one line per solver iteration, reliable update and restart on stderr */
  int columns_per_thread; /* tuning of the multi-column fp32 stencil (tmw_*_multi): 1..4 right-hand-side
                             columns per thread (links and clover blocks stay in registers for them); 0 = automatic */
  int tile[4];      /* log2 extents (x/2, y, z, t) of the 4-D tile of 128 sites a CTA of the single-column stencil covers;
                       all 0 (default): 128 consecutive checkerboard indices; tile[0] = -1: the largest tile that fits,
                       preferring 8 x 4 x 2 x 2. A tile that does not divide the lattice or is not 128 sites -> 1-D. */
  int debug;        /* bit mask of TMW_DEBUG_* (test hooks, see below); also settable later with tmw_set_debug */
  /* Domain decomposition (the paper's runs are all multi-GPU: PAPER.md:52, the "Nodes" columns of Tables 2-5 :71-76, and
     "the network has much stronger impact on the performance", :315): the lattice is cut into domains_z x domains_t
     sub-lattices (0 or 1: not cut; L / domains_z and T / domains_t must be even), each with its own packed gauge and
     clover fields. Every stencil application then packs the (1 +- gamma_mu)-projected half spinors of the cut faces
     (12 reals per face site), exchanges them with one copy per face, computes the interior of the domains meanwhile and
     finishes the sites on the cuts afterwards; the antiperiodic sign stays on the physical t boundary. All calls give
     the same results as without cuts up to rounding (the hops through a cut are added last). A packed parity spinor of
     such a context is the domains' local packed spinors back to back, domain (iz, it) at index iz + domains_z * it. In
     this build all domains live on the context's device (the exchange is a same-device copy); tmw_get_clover and the
     tile / columns_per_thread tunings are not available. */
  int domains_z, domains_t;
  /* Shared-memory staged fp32 stencil (BASELINE.json north_star subsystem (2)): a CTA covers a tile of one
     time slice and copies the input sites its six spatial hops need into shared memory with asynchronous 16-byte copies
     instead of loading 8 neighbour spinors per site through L1. 0 or -1 = off (default: measured on B200 the staged kernel
     is 10-40 % slower than the plain one at every tile shape and column count, profiles/r2_stage.md), 1 = wherever a tile
     fits (hop, K1, K2 of fp32 launches without domain decomposition). stage_tile = tile extents (x/2, y, z) in sites, all 0 =
     chosen by the library; a tile that does not divide the lattice or does not fit in shared memory -> the plain kernel. */
  int stage;
  int stage_tile[3];
  /* Sweep order of the multi-column fp32 stencil launches: the lattice is cut into slabs of zchunk sites in
     z and a launch goes through all time slices of one slab before the next, so that the +-t neighbour re-reads of all
     columns stay in L2. 0 = automatic (the largest slab whose +-t window fits a fixed L2 budget), -1 = off (time slice
     after time slice), > 0 = that many sites (must divide L, with L*L*zchunk/2 a multiple of 128; else off). */
  int zchunk;
  /* L2 prefetch of the links: a CTA of the plain stencil also issues prefetch.global.L2 for the links of the
     site block `prefetch` blocks ahead of its own (the links are the loads that always miss to DRAM). 0 = automatic: one
     block ahead in the multi-column fp32 hop launches (measured: -7..10 % at 12 columns 32^3 x 96, -3 % at 3 columns
     48^3 x 144; no gain for K1 / K2 and for one column, where it stays off), -1 = off, > 0 = that distance in site blocks
     of 128 sites for every stencil launch. */
  int prefetch;
} tmw_options;
#define TMW_OPTIONS_INIT {sizeof(tmw_options)} /* tmw_options o = TMW_OPTIONS_INIT; : all defaults, struct_size set */

/* Test hooks (tmw_options.debug / tmw_set_debug): they change which code path runs, never the result. */
#define TMW_DEBUG_FORCE_PIVOT 1 /* tmw_create: invert the clover blocks with the pivoted Gauss-Jordan fallback kernel */
#define TMW_DEBUG_NO_CHUNK 2    /* tmw_solve_multi: do not split the columns into chunks that fit the free memory */
#define TMW_DEBUG_FORCE_DEFECT 4 /* tmw_solve_multi: send the odd-numbered columns through one fp64 defect-correction pass as if
                                   their full-lattice residual had missed tol (the other columns must come out untouched) */

typedef struct {
  int iters;            /* BiCGStab iterations (each = 2 Schur-operator applications) or GCR steps (1 application each) */
  int reliable_updates; /* fp64 true-residual recomputations */
  int restarts;         /* breakdown restarts (rhat := r) */
  double iter_resid;    /* last iterated |r| / |b| */
  double true_resid;    /* |b - D x| / |b| on the full lattice, fp64, recomputed after reconstruction */
  double device_ms;     /* CUDA-event time of the whole solve on the context stream */
} tmw_solve_info;

/*
 * Build a context for an L^3 x T lattice (L, T even, >= 4): copies the gauge field and re-lays it out
 * (checkerboarded SoA, fp64 18-real and fp32 12/18-real copies), and, if c_sw != 0, computes the clover-leaf
 * F_mu_nu (Eq. (3), C7), the two Hermitian 6x6 chiral blocks per site and the inverses on the even sites
 * (PAPER.md:80). gauge: canonical layout, HOST or DEVICE per opt->location. opt may be NULL (all defaults).
 */
int tmw_create(tmw_ctx** out, int L, int T, const double* gauge, tmw_complex m, double c_sw, const tmw_options* opt);

/*
 * out = D in (op = TMW_D), D^dag in (TMW_DDAG) or gamma5 D in (TMW_G5D), Eq. (2)+(3). TMW_G5D is the paper's one
 * explicit fusion ("we combine the gamma5 and D_w operations into one kernel to save the bandwidth"):
 * gamma5 = diag(+1,+1,-1,-1) in spin (C5) multiplies the result inside the kernel, at no extra memory traffic.
 *   parity = TMW_FULL: in, out are canonical fp64 full-lattice spinors (HOST or DEVICE per location); fp64 arithmetic.
 *   parity = TMW_EVEN | TMW_ODD: the raw benchmark path. out (packed, parity p) = H_{p pbar} in (packed, the other
 *     parity) = only the hopping part of Eq. (2) (the 1/2 sum over mu), in precision `prec` (TMW_F32 | TMW_F64).
 *     DEVICE pointers. Asynchronous on the context stream.
 */
int tmw_apply(tmw_ctx* ctx, int op, int parity, int prec, const void* in, void* out);

/*
 * Even-odd Schur complement on the odd sites (packed DEVICE spinors, precision prec):
 *   out_o = A_oo in_o - H_oe A_ee^{-1} H_eo in_o,  A = the site-diagonal part of D (mass, twist, clover).
 * op = TMW_DDAG applies its conjugate transpose. Asynchronous on the context stream.
 */
int tmw_apply_schur(tmw_ctx* ctx, int op, int prec, const void* in_odd, void* out_odd);

/*
 * Solve D x = b to |b - D x| / |b| <= tol. b, x: canonical fp64 spinors (HOST or DEVICE per location).
 * b = 0 gives x = 0. Returns after the final fp64 true residual is known. info may be NULL.
 * TMW_MIXED: if the fp32 BiCGStab recurrence stalls (TMW_EBREAKDOWN; only seen on near-critical systems that need
 * ~1000 iterations) the solve is redone with fp64 recurrences before an error is returned.
 */
int tmw_solve(tmw_ctx* ctx, const double* b, double* x, double tol, tmw_solve_info* info);

/*
 * tmw_apply_schur for callers that must not allocate device memory: same operator (Eq. (2), :67 Eq. (3) on
 * the even-odd Schur complement), same kernels, same arguments and result as tmw_apply_schur, but the call itself never
 * allocates or frees anything - no cudaMalloc, no cudaFree, no library routine that allocates.
 *
 * Who needs this. tmw_apply_schur keeps its even-parity intermediate A_ee^{-1} H_eo in_o in a workspace that it
 * cudaMallocs on first use (and again whenever a multi-column call has resized the workspaces). Some programs cannot
 * afford that inside their steady state: a process that, once start-up is over, has handed the rest of the card to a
 * pooling allocator (a PyTorch or RAPIDS job: a raw cudaMalloc then fails although the pool has room, or it fragments
 * the pool's address space); a job that runs under a fixed device-memory quota; and a latency-critical loop that shares
 * the GPU with other streams, because cudaMalloc and cudaFree stall the whole device until every stream has drained.
 * Such a caller creates the context at start-up, while allocating is still allowed (tmw_create allocates the gauge and
 * clover fields), and from then on applies the operator through this entry point.
 *
 * Where the intermediate lives. In one array of TMW_STATIC_SCRATCH_BYTES (8 MiB) that is compiled into libtmw.so as
 * a device global. Every GPU on which the library's kernels are loaded sets these 8 MiB aside until the process exits,
 * whether or not this call is ever used. A lattice whose packed parity spinor (tmw_spinor_bytes(ctx, prec): 96 bytes
 * per site and parity in fp32, 192 in fp64) is larger than the array is refused with TMW_EINVAL and an error text that
 * names both sizes; nothing is launched then. 16^3 x 32 in fp32 and 16^3 x 16 in fp64 still fit.
 *
 * First call on a device. The first call on each device looks up the device address of the array (a CUDA runtime
 * query, no allocation) with the context's device current, and remembers it; make that first call during set-up,
 * before any stream capture is begun. The context's device must be the calling thread's current device in every call,
 * as for all other calls of this library (checked here: TMW_EINVAL otherwise).
 *
 * Sharing. There is ONE array per device for all contexts, streams and threads of the process, and it still holds
 * whatever the previous call left in it. Nothing in it has to start at zero: the first kernel writes the intermediate
 * of every even site before the second kernel reads it, so stale contents are never read. But two calls whose kernels
 * can be on the GPU at the same time (different streams, or different contexts with different streams) overwrite each
 * other's intermediate: that is a data race with wrong results and no error. Keep all calls of this entry point on one
 * stream per device, or order them with events. It does not disturb, and is not disturbed by, any other call.
 *
 * One column, packed DEVICE spinors as for tmw_apply_schur, contexts without domain decomposition (a decomposed context
 * grows its exchange buffers on demand; TMW_EINVAL). Asynchronous on the context stream.
 */
#define TMW_STATIC_SCRATCH_BYTES (8u << 20)
int tmw_apply_schur_static(tmw_ctx* ctx, int op, int prec, const void* in_odd, void* out_odd);

/*
 * Several right-hand sides at once (the "12 columns" of a propagator, Table 2 caption).
 * The columns are independent problems with the same operator; doing them in one call lets every link and clover
 * block be read once for all columns. nrhs in 1..16. Column c of every spinor argument follows column c-1 directly:
 *   canonical: double[nrhs][T][L][L][L][4][3][2];   packed: nrhs packed parity spinors back to back.
 * tmw_apply_multi / tmw_apply_schur_multi: as tmw_apply / tmw_apply_schur, column by column the same result.
 * tmw_solve_multi: BiCGStab on all columns in lockstep, each with its own recurrence scalars, reliable updates and
 *   stopping test (|b_c - D x_c| / |b_c| <= tol for every column c); columns that have converged drop out of the
 *   launches. info (nullable) points to nrhs records; device_ms is the time of the whole call in each of them.
 *   Returns TMW_ENOCONV if any column reached max_iter. Workspace grows with nrhs (16 parity spinors per column); if
 *   the columns do not all fit in the free device memory they are solved in chunks of as many as fit (device_ms is
 *   then the time of the column's chunk). TMW_ENOMEM if not even one column fits.
 */
int tmw_apply_multi(tmw_ctx* ctx, int op, int parity, int prec, int nrhs, const void* in, void* out);
int tmw_apply_schur_multi(tmw_ctx* ctx, int op, int prec, int nrhs, const void* in_odd, void* out_odd);
int tmw_solve_multi(tmw_ctx* ctx, int nrhs, const double* b, double* x, double tol, tmw_solve_info* info);

/*
 * out = sum_{k=0}^{ncoef-1} coef[k] T_k(X) in,  X = scale * (gamma5 D) + shift * 1,  T_k the Chebyshev polynomials of
 * the first kind, evaluated with the Clenshaw recursion ("one should use the Clenshaw recursion to define the
 * Chebyshev polynomial to suppress the round-off error"; the polynomial of gamma5 D_w is the inner loop
 * of the paper's overlap sign function). gamma5 D is applied with the fused gamma5 epilogue
 * (PAPER.md:315). coef: HOST array of real coefficients; in, out: canonical fp64 full-lattice spinors (HOST or
 * DEVICE per location); fp64 arithmetic. The caller chooses scale and shift so that the spectrum of X lies where the
 * series is wanted (usually [-1, 1]). Cost: ncoef - 1 applications of gamma5 D.
 */
int tmw_cheb_apply(tmw_ctx* ctx, int ncoef, const double* coef, double scale, double shift, const double* in, double* out);

/* bytes of one packed parity spinor in precision prec (TMW_F32 | TMW_F64); 0 on bad arguments */
long long tmw_spinor_bytes(const tmw_ctx* ctx, int prec);

/*
 * Layout conversion between a canonical fp64 full-lattice spinor and a packed parity spinor (both DEVICE
 * pointers regardless of `location`). parity = TMW_EVEN | TMW_ODD. tmw_unpack writes only the sites of that parity.
 */
int tmw_pack(tmw_ctx* ctx, int prec, int parity, const double* canonical, void* packed);
int tmw_unpack(tmw_ctx* ctx, int prec, int parity, const void* packed, double* canonical);

/*
 * Copy the packed clover blocks out for inspection (tests): for the given parity, 72 doubles per site
 * [cb][chirality 0..1][36], each block = 6 real diagonal entries then the 15 strictly-lower entries (row-major:
 * (1,0),(2,0),(2,1),(3,0),...) as re,im; block index i = 3*(spin mod 2) + colour; the diagonal includes
 * -(4 + Re m). inverse != 0 returns the stored inverse (even parity only). dst: DEVICE pointer.
 */
int tmw_get_clover(tmw_ctx* ctx, int parity, int inverse, double* dst);

/* change where the canonical-layout pointers of subsequent calls live (TMW_DEVICE | TMW_HOST) */
int tmw_set_location(tmw_ctx* ctx, int location);

/* replace the TMW_DEBUG_* mask of the context (TMW_DEBUG_FORCE_PIVOT only matters at tmw_create) */
int tmw_set_debug(tmw_ctx* ctx, int flags);

/* number of kernel launches this context has issued since creation (bench.py's gpu_launches) */
long long tmw_launch_count(const tmw_ctx* ctx);

/*
 * Measurement support (bench.py's roofline objects; DESIGN.md 5 has the algorithmic bytes per site of every kind).
 * Kernel kinds: the stencil launches by precision and epilogue, the fused BLAS-1 kernels of the BiCGStab recurrences
 * ("vector operations"), the layout conversions.
 */
#define TMW_K_HOP32 0          /* fp32 hopping block H (Eq. (2) hopping part), the benchmarked kernel */
#define TMW_K_K1_32 1          /* fp32 K1 = A_ee^{-1} H_eo */
#define TMW_K_K2_32 2          /* fp32 K2 = A_oo - H_oe (+ <rhat, v>) */
#define TMW_K_K2_32_DOTS 3     /* fp32 K2 with <t,s>, <t,t>, <rhat,t>, <rhat,s> fused */
#define TMW_K_HOP64 4
#define TMW_K_K1_64 5          /* fp64 K1 (reliable update) */
#define TMW_K_K2_64 6          /* fp64 K2 / full-operator half (reliable update, tmw_apply FULL, final residual) */
#define TMW_K_XPAY64 7         /* fp64 source preparation b_o - H_oe (A_ee^{-1} b_e) */
#define TMW_K_AINVXPAY64 8     /* fp64 reconstruction x_e = A_ee^{-1} (b_e - H_eo x_o) */
#define TMW_K_UPDATE_S 9       /* s = r - alpha v */
#define TMW_K_UPDATE_XRP 10    /* x, r, next p, |r|^2 in one pass */
#define TMW_K_ACC_Y 11         /* y += x (fp64), x = 0 */
#define TMW_K_RESID_CONVERT 12 /* r64 = bhat - Mhat y, r = (fp32) r64, <rhat, r>, |r|^2 (, p += r_new - r_old) */
#define TMW_K_CONVERT 13       /* fp64 -> inner precision */
#define TMW_K_DOT_NORM64 14    /* |b|^2 of one parity */
#define TMW_K_SUB_NORM 15      /* fp64 a - b / a + b */
#define TMW_K_DIAG64 16        /* A_ee^{-1} b_e */
#define TMW_K_PACK_BOTH 17     /* canonical -> packed, both parities */
#define TMW_K_UNPACK_BOTH 18   /* packed -> canonical, both parities */
#define TMW_K_OTHER 19         /* anything else that was counted */
#define TMW_K_MEMSET_BYTES 20  /* BYTES zeroed by device memsets inside the solver */
#define TMW_K_COPY_BYTES 21    /* BYTES moved by device-to-device copies inside the solver */
#define TMW_K_HOP32_LOADONLY 22 /* tmw_time_kernel only: the loads and stores of TMW_K_HOP32 without its arithmetic */
#define TMW_K_STAGED 23        /* of the fp32 stencil applications above: those that ran in the shared-memory staged kernel */
#define TMW_K_FFMA_PROBE 24    /* tmw_time_kernel only: TMW_FFMA_PROBE_FMAS_PER_THREAD scalar fp32 FMAs (16 independent chains) per thread */
#define TMW_K_FFMA2_PROBE 25   /* tmw_time_kernel only: the same FMAs as packed pairs (fma.rn.f32x2, 8 chains of 2) */
#define TMW_FFMA_PROBE_FMAS_PER_THREAD (16 * 16384) /* the probe launches (SM count) x 8 CTAs of 256 threads */
#define TMW_K_COUNT 26

/*
 * counts[k] (k < min(n, TMW_K_COUNT)) = how many right-hand-side columns kernels of kind k have been applied to since
 * tmw_create (a launch on N columns counts N; the two *_BYTES kinds count bytes). Returns TMW_K_COUNT, or TMW_EINVAL.
 */
int tmw_kernel_counts(const tmw_ctx* ctx, long long* counts, int n);

/*
 * Mean duration in milliseconds of `reps` back-to-back launches (after 3 untimed ones) of ONE kernel of the solver, on
 * the context's own workspace vectors, timed with CUDA events on the context stream: kind = TMW_K_HOP32, K1_32, K2_32,
 * K2_32_DOTS, K1_64, K2_64, UPDATE_S, UPDATE_XRP, or TMW_K_HOP32_LOADONLY (a kernel that issues exactly the loads and
 * stores of the fp32 hopping kernel - 8 neighbour spinors, 8 links, one store per site, same indices and launch shape -
 * and only adds the loaded values up: the memory floor of the access pattern), or TMW_K_FFMA_PROBE /
 * TMW_K_FFMA2_PROBE (register-only fp32 FMA loops: the ALU ceiling the multi-column stencil is measured against,
 * DESIGN.md 6b; FMAs per launch = TMW_FFMA_PROBE_FMAS_PER_THREAD x 256 x 8 x SM count). Single column, TMW_MIXED
 * contexts without domain decomposition. The vectors hold whatever the last solve left there (run one first); the
 * results are not meaningful, only the time is. Synchronises the stream.
 */
int tmw_time_kernel(tmw_ctx* ctx, int kind, int reps, double* ms);

void tmw_destroy(tmw_ctx* ctx);

/* text of the last error of this context (ctx-owned, valid until the next call); ctx may be NULL for create errors */
const char* tmw_last_error(const tmw_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* TMW_H */
