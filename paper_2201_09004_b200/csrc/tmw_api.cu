// tmw_api.cu — the C ABI of include/tmw.h: context, layout conversion, operator application, and the even-odd
// mixed-precision BiCGStab driver (the solver named at PAPER.md:73). Host code only
// sequences kernel launches and reads a few reduction scalars per iteration; all arithmetic on fields runs in
// the CUDA kernels of this directory.
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>  // header-only: ranges around the phases of create / apply / solve for nsys and ncu --nvtx

#include "../../include/tmw.h"
#include "tmw_internal.h"

namespace {
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};
}  // namespace

using namespace tmw;

enum { NW64 = 14 };
// automatic z-slab of the multi-column sweep (tmw_options.zchunk = 0): the +-t window may take this share of the L2 the
// device reports (3/16 of B200's 126 MB = the 24 MB found best by the sweep of DESIGN.md 5a)
enum { ZCHUNK_L2_SHARE_NUM = 3, ZCHUNK_L2_SHARE_DEN = 16, ZCHUNK_L2_FALLBACK_MB = 126 };
enum { NSLAB = 24 };  // most t-slabs of the pipelined host-pointer tmw_apply

// One domain of a domain-decomposed context: a sub-lattice L x L x (L/Pz) x (T/Pt) with its own packed
// gauge and clover fields and the send / receive buffers of its cuts. Domain (iz, it) has index iz + Pz * it; every
// packed spinor of the context is the domains' local packed spinors back to back in that order.
struct Domain {
  Geom g;
  int iz, it;
  int device;        // CUDA device that holds the domain (all domains of a context share one device in this build)
  void* g64[2];
  void* g32[2];
  void* c64[2];
  void* c32[2];
  void* ci64;
  void* ci32;
  void* send[2][2];  // [direction z, t][0: to the neighbour behind, 1: ahead]
  void* recv[2][2];  // [direction][0: lo ghost (from behind), 1: hi ghost (from ahead)]
};

struct tmw_ctx {
  Geom g;
  int64_t V;
  double m_re, m_im, c_sw;
  tmw_options opt;
  cudaStream_t stream;
  bool clover;
  int ng32;
  void* g64[2];
  void* g32[2];
  void* c64[2];
  void* c32[2];
  void* ci64;  // inverse blocks, even parity
  void* ci32;
  std::vector<void*> owned;  // every device allocation
  // domain decomposition: pz * pt > 1 domains (then g64 ... ci32 above are null and the fields live in dom[])
  int pz, pt;
  std::vector<Domain> dom;
  int vh_loc;        // sites per parity of one domain (= g.Vh without decomposition)
  int ghost_cols;    // columns the send / receive buffers hold
  void* dd_tmp;      // scratch output spinors for stencil launches that keep only a reduction
  size_t dd_tmp_bytes; // its size: grows with the highest column a reduction-only launch has used
  cudaStream_t h2d, d2h;             // copy streams of the pipelined host-pointer tmw_apply (lazily created)
  cudaEvent_t ev_in[NSLAB], ev_out[NSLAB]; // per t-slab: input arrived / output ready
  cudaStream_t comm; // the halo exchange runs here, beside the interior pass on `stream`
  cudaEvent_t ev_pack, ev_comm;
  // lazily allocated workspaces, each sized for ws_cols right-hand-side columns (column c at c * spinor bytes)
  int ws_cols;
  void* w64[NW64];  // packed fp64 parity spinors (0..7 the solver's, 8..13 only for the rare defect-correction pass)
  void* w32[8];   // packed inner-precision parity spinors (fp32 for TMW_MIXED, fp64 for TMW_DOUBLE)
  void* canon[2]; // canonical fp64 full-lattice staging (HOST location only)
  void* gcr_q;       // GCR Krylov vectors q_j, p_j: nkrylov inner-precision parity spinors each (lazily allocated)
  void* gcr_p;
  GcrScalars* gs;       // device
  GcrScalars* gs_host;  // pinned
  int nr32;          // forced columns per thread of the fp32 stencil (1..4), 0 = automatic
  StageGeom stage[4];  // tile of the shared-memory staged fp32 stencil for nr = 1..3 columns per thread (index nr)
  bool stage_ok[4];    // such a tile exists (tmw_options.stage / stage_tile, choose_stage)
  bool verbose;
  int* attn;         // device int[2]: [0] a column needs the host (the queued iteration kernels return at once), [1] iterations done
  int* attn_host;    // pinned int[6]: two lagged copies of attn (one per queued iteration) and the copy of a sync point
  cudaEvent_t ev_lag[2];
  const int* cur_skip;  // what make_args puts into DslashArgs::skip: attn while BiCGStab iterations are being queued, else null
  Scalars* sc;       // MAXCOL scalar blocks
  Scalars* sc_host;  // pinned
  double* red;       // 4 * MAXCOL device doubles
  double* red_host;  // pinned
  cudaEvent_t ev0, ev1;
  int sms;           // SM count and L2 size of the context's device (asked once in tmw_create)
  int64_t l2_bytes;
  long long launches;
  long long kcount[TMW_K_COUNT];  // per kernel kind: column applications (or bytes), see include/tmw.h TMW_K_*
  std::string err;
};

// Sets tmw_ctx::cur_skip for the lifetime of the guard: the LAUNCH / CK macros return from the middle of a block, and a
// skip pointer left behind would make every later stencil launch of the context return without writing.
struct SkipGuard {
  tmw_ctx* c;
  SkipGuard(tmw_ctx* ctx, const int* skip) : c(ctx) { c->cur_skip = skip; }
  ~SkipGuard() { c->cur_skip = nullptr; }
  SkipGuard(const SkipGuard&) = delete;
  SkipGuard& operator=(const SkipGuard&) = delete;
};

static thread_local std::string g_create_err;

static int fail(tmw_ctx* c, int code, const char* msg) {
  if (c) c->err = msg; else g_create_err = msg;
  return code;
}
static int fail_cuda(tmw_ctx* c, cudaError_t e, const char* where) {
  char buf[512];
  snprintf(buf, sizeof(buf), "CUDA error in %s: %s", where, cudaGetErrorString(e));
  cudaGetLastError();
  return fail(c, e == cudaErrorMemoryAllocation ? TMW_ENOMEM : TMW_ECUDA, buf);
}
#define CK(call)                                               \
  do {                                                         \
    cudaError_t e_ = (call);                                   \
    if (e_ != cudaSuccess) return fail_cuda(ctx, e_, #call);   \
  } while (0)
#define LAUNCH(call)                                           \
  do {                                                         \
    cudaError_t e_ = (call);                                   \
    ctx->launches++;                                           \
    if (e_ != cudaSuccess) return fail_cuda(ctx, e_, #call);   \
  } while (0)
// a launch of kernel kind K (TMW_K_*) that works on N right-hand-side columns
#define LAUNCHK(K, N, call)                                    \
  do {                                                         \
    ctx->kcount[K] += (N);                                     \
    LAUNCH(call);                                              \
  } while (0)
// a device memset / device-to-device copy inside the solver (counted in bytes)
#define MEMSETK(ptr, val, bytes)                               \
  do {                                                         \
    ctx->kcount[TMW_K_MEMSET_BYTES] += (long long)(bytes);     \
    CK(cudaMemsetAsync((ptr), (val), (bytes), ctx->stream));   \
  } while (0)
#define COPYK(dst, src, bytes)                                 \
  do {                                                         \
    ctx->kcount[TMW_K_COPY_BYTES] += (long long)(bytes);       \
    CK(cudaMemcpyAsync((dst), (src), (bytes), cudaMemcpyDeviceToDevice, ctx->stream)); \
  } while (0)

static int dev_alloc(tmw_ctx* ctx, void** p, size_t bytes) {
  cudaError_t e = cudaMalloc(p, bytes);
  if (e != cudaSuccess) { *p = nullptr; return fail_cuda(ctx, e, "cudaMalloc"); }
  ctx->owned.push_back(*p);
  return TMW_OK;
}
static void dev_free(tmw_ctx* ctx, void* p) {
  for (size_t i = 0; i < ctx->owned.size(); i++)
    if (ctx->owned[i] == p) { ctx->owned.erase(ctx->owned.begin() + i); break; }
  cudaFree(p);
}

static size_t spinor_bytes(const tmw_ctx* c, int prec) { return (size_t)c->g.Vh * 24 * (prec == TMW_F32 ? 4 : 8); }

// ---- the diagonal part for D (dagger = 0) or D^dagger ----
template <typename R> static Diag<R> make_diag(const tmw_ctx* c, int dagger, const Domain* dm = nullptr) {
  Diag<R> d;
  const double dg = -(4.0 + c->m_re);
  double tu, tl;
  if (c->opt.mass_reading == TMW_TWIST_GAMMA5) { tu = -c->m_im; tl = c->m_im; }
  else { tu = -c->m_im; tl = -c->m_im; }
  if (dagger) { tu = -tu; tl = -tl; }
  d.diag = (R)dg;
  d.tw_up = (R)tu;
  d.tw_lo = (R)tl;
  const double den = dg * dg + tu * tu;
  d.inv_re = (R)(dg / den);
  d.inv_im_up = (R)(-tu / den);
  d.inv_im_lo = (R)(-tl / den);
  d.twisted_clover = (c->clover && c->m_im != 0.0) ? 1 : 0;
  const bool f = sizeof(R) == 4;
  if (dm) {
    d.c[0] = f ? dm->c32[0] : dm->c64[0];
    d.c[1] = f ? dm->c32[1] : dm->c64[1];
    d.cinv[0] = f ? dm->ci32 : dm->ci64;
  } else {
    d.c[0] = f ? c->c32[0] : c->c64[0];
    d.c[1] = f ? c->c32[1] : c->c64[1];
    d.cinv[0] = f ? c->ci32 : c->ci64;
  }
  d.cinv[1] = nullptr;
  return d;
}

static ColMap cols_first(int n) {
  ColMap cm;
  cm.n = n;
  for (int i = 0; i < MAXCOL; i++) cm.col[i] = (unsigned char)(i < n ? i : 0);
  return cm;
}
static void cols_add(ColMap& cm, int c) { cm.col[cm.n++] = (unsigned char)c; }

template <typename R>
static DslashArgs<R> make_args(const tmw_ctx* c, int par, int dagger, const void* in, void* out, const void* aux, double sgn, const ColMap& cm,
                               const Domain* dm = nullptr) {
  DslashArgs<R> a;
  memset(&a, 0, sizeof(a));
  a.in = in;
  a.out = out;
  a.aux = aux;
  const bool f = sizeof(R) == 4;
  if (dm) {
    a.U[0] = f ? dm->g32[0] : dm->g64[0];
    a.U[1] = f ? dm->g32[1] : dm->g64[1];
    a.g = dm->g;
  } else {
    a.U[0] = f ? c->g32[0] : c->g64[0];
    a.U[1] = f ? c->g32[1] : c->g64[1];
    a.g = c->g;
  }
  a.par = par;
  a.sig = dagger ? (R)-1 : (R)1;
  a.coef = (R)(0.5 * sgn);
  a.g5 = 0;
  a.d = make_diag<R>(c, dagger, dm);
  a.red_mode = 0;
  a.dotv = nullptr;
  a.red = nullptr;
  a.ncol = cm.n;
  a.ngroups = 1;
  a.sb0 = 0;
  a.cb_end = a.g.Vh;
  a.cstride = (int)((int64_t)c->g.Vh * 24 * (int64_t)sizeof(R) / 16);
  a.red_stride = 0;
  a.skip = c->cur_skip;
  a.pf_blocks = c->opt.prefetch > 0 ? c->opt.prefetch : 0;  // automatic (0): set per launch in dslash<R>()
  for (int i = 0; i < MAXCOL; i++) a.col[i] = cm.col[i];
  return a;
}
template <typename R> static int ng_of(const tmw_ctx* c) { return sizeof(R) == 4 ? c->ng32 : 18; }

// out(par) = epilogue(H in) for the columns of cm (vectors of column c start c spinors after the base pointers);
// red (if any) is the reduction target of column 0, column c's is red_stride doubles further per column.
// kernel kind (TMW_K_*) of a stencil launch
template <typename R> static int stencil_kind(int epi, int red_mode) {
  const bool f = sizeof(R) == 4;
  switch (epi) {
    case EPI_HOP: return f ? TMW_K_HOP32 : TMW_K_HOP64;
    case EPI_AINV_HOP: return f ? TMW_K_K1_32 : TMW_K_K1_64;
    case EPI_A_XPAY: return f ? (red_mode == 4 ? TMW_K_K2_32_DOTS : TMW_K_K2_32) : TMW_K_K2_64;
    case EPI_XPAY: return f ? TMW_K_OTHER : TMW_K_XPAY64;
    default: return f ? TMW_K_OTHER : TMW_K_AINVXPAY64;
  }
}

static inline int dom_behind(const tmw_ctx* c, const Domain& d, int dir) {
  return dir == 0 ? ((d.iz + c->pz - 1) % c->pz) + c->pz * d.it : d.iz + c->pz * ((d.it + c->pt - 1) % c->pt);
}
static inline int dom_ahead(const tmw_ctx* c, const Domain& d, int dir) {
  return dir == 0 ? ((d.iz + 1) % c->pz) + c->pz * d.it : d.iz + c->pz * ((d.it + 1) % c->pt);
}

// The stencil on a domain-decomposed context. Per application, for every domain:
//   (a) face pack: the half spinors its neighbours need, (1 +- g_mu) projected (and U^dag-multiplied for the backward
//       hops) BEFORE they travel: 12 reals per face site instead of 24;
//   (b) exchange on the stream `comm`: one cudaMemcpyPeerAsync per domain, cut and side (a same-device copy when both
//       domains share a GPU, a peer copy over NVLink otherwise);
//   (c) interior pass on `stream`, concurrent with (b): every hop that stays inside the domain;
//   (d) exterior pass after (b): the sites on a cut get the ghost terms, the epilogue and their share of the fused
//       reductions. The antiperiodic sign sits on the physical t boundary only (DDArgs::bc), never on an internal cut.
// Reductions of all domains accumulate into the same device scalars (one device; several devices would add one small
// all-reduce per reduction here).
template <typename R>
static int dslash_dd(tmw_ctx* ctx, int epi, int par, int dagger, const void* in, void* out, const void* aux, double sgn, const ColMap& cm, int red_mode,
                     const void* dotv, double* red, int red_stride, int g5) {
  const int nd = (int)ctx->dom.size();
  const size_t lb = (size_t)ctx->vh_loc * 24 * sizeof(R);  // bytes of one domain's packed parity spinor
  int cmin = MAXCOL, cmax = 0;
  for (int i = 0; i < cm.n; i++) { cmin = cm.col[i] < cmin ? cm.col[i] : cmin; cmax = cm.col[i] > cmax ? cm.col[i] : cmax; }
  if (cmax + 1 > ctx->ghost_cols) {  // (re)size the send / receive buffers: fp64 half spinors for cmax + 1 columns
    CK(cudaStreamSynchronize(ctx->stream));
    CK(cudaStreamSynchronize(ctx->comm));
    for (Domain& d : ctx->dom)
      for (int dir = 0; dir < 2; dir++)
        for (int k = 0; k < 2; k++) {
          if (d.send[dir][k]) { dev_free(ctx, d.send[dir][k]); d.send[dir][k] = nullptr; }
          if (d.recv[dir][k]) { dev_free(ctx, d.recv[dir][k]); d.recv[dir][k] = nullptr; }
        }
    ctx->ghost_cols = 0;
    for (Domain& d : ctx->dom)
      for (int dir = 0; dir < 2; dir++) {
        if (!(dir == 0 ? ctx->pz > 1 : ctx->pt > 1)) continue;
        const size_t nface = (size_t)d.g.Lh * d.g.L * (dir == 0 ? d.g.T : d.g.Lz);
        for (int k = 0; k < 2; k++) {
          int rc = dev_alloc(ctx, &d.send[dir][k], nface * 12 * 8 * (cmax + 1));
          if (!rc) rc = dev_alloc(ctx, &d.recv[dir][k], nface * 12 * 8 * (cmax + 1));
          if (rc) return rc;
        }
      }
    ctx->ghost_cols = cmax + 1;
  }
  if (!out) {  // only a reduction is wanted, but the interior pass needs somewhere to leave the raw sums of the cut sites
    // column c is written at c whole-lattice packed spinors of precision R: room for columns 0..cmax, no more
    const size_t need = (size_t)ctx->g.Vh * 24 * sizeof(R) * (cmax + 1);
    if (need > ctx->dd_tmp_bytes) {
      CK(cudaStreamSynchronize(ctx->stream));
      if (ctx->dd_tmp) { dev_free(ctx, ctx->dd_tmp); ctx->dd_tmp = nullptr; ctx->dd_tmp_bytes = 0; }
      int rc = dev_alloc(ctx, &ctx->dd_tmp, need);
      if (rc) return rc;
      ctx->dd_tmp_bytes = need;
    }
    out = ctx->dd_tmp;
  }
  std::vector<DslashArgs<R>> A(nd);
  for (int k = 0; k < nd; k++) {
    const Domain& d = ctx->dom[k];
    DslashArgs<R>& a = A[k];
    a = make_args<R>(ctx, par, dagger, (const char*)in + k * lb, (char*)out + k * lb, aux ? (const char*)aux + k * lb : nullptr, sgn, cm, &d);
    a.cstride = (int)((int64_t)ctx->g.Vh * 24 * (int64_t)sizeof(R) / 16);  // a column = the packed spinor of the WHOLE lattice
    a.g5 = g5;
    a.red_mode = red_mode;
    a.dotv = dotv ? (const char*)dotv + k * lb : nullptr;
    a.red = red;
    a.red_stride = red_stride;
    a.dd.part[0] = ctx->pz > 1;
    a.dd.part[1] = ctx->pt > 1;
    for (int dir = 0; dir < 2; dir++) {
      a.dd.nface[dir] = d.g.Lh * d.g.L * (dir == 0 ? d.g.T : d.g.Lz);
      a.dd.gstride[dir] = a.dd.nface[dir] * (int)(12 * sizeof(R) / 16);
      a.dd.ghost[dir][0] = d.recv[dir][0];
      a.dd.ghost[dir][1] = d.recv[dir][1];
      a.dd.bc[dir][0] = a.dd.bc[dir][1] = (R)1;
    }
    if (d.it == 0) a.dd.bc[1][0] = (R)-1;            // the backward t hop of the first time slice wraps around the lattice
    if (d.it == ctx->pt - 1) a.dd.bc[1][1] = (R)-1;  // the forward t hop of the last one
  }
  const int ng = ng_of<R>(ctx);
  const int clv = !ctx->clover ? CL_NONE : (ctx->m_im != 0.0 ? CL_TWISTED : CL_CLOVER);
  ctx->kcount[stencil_kind<R>(epi, red_mode)] += cm.n;
  for (int k = 0; k < nd; k++) LAUNCH(launch_face_pack(A[k], ng, ctx->dom[k].send, ctx->stream));
  CK(cudaEventRecord(ctx->ev_pack, ctx->stream));
  CK(cudaStreamWaitEvent(ctx->comm, ctx->ev_pack, 0));
  for (int k = 0; k < nd; k++) {
    const Domain& d = ctx->dom[k];
    for (int dir = 0; dir < 2; dir++) {
      if (!A[k].dd.part[dir]) continue;
      const size_t colb = (size_t)A[k].dd.gstride[dir] * 16, off = colb * cmin, bytes = colb * (cmax - cmin + 1);
      const Domain& nb = ctx->dom[dom_behind(ctx, d, dir)];
      const Domain& na = ctx->dom[dom_ahead(ctx, d, dir)];
      CK(cudaMemcpyPeerAsync((char*)nb.recv[dir][1] + off, nb.device, (const char*)d.send[dir][0] + off, d.device, bytes, ctx->comm));
      CK(cudaMemcpyPeerAsync((char*)na.recv[dir][0] + off, na.device, (const char*)d.send[dir][1] + off, d.device, bytes, ctx->comm));
    }
  }
  CK(cudaEventRecord(ctx->ev_comm, ctx->comm));
  for (int k = 0; k < nd; k++) LAUNCH(launch_dslash_dd(A[k], ng, epi, clv, 0, ctx->stream));
  CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_comm, 0));
  for (int k = 0; k < nd; k++) LAUNCH(launch_dslash_dd(A[k], ng, epi, clv, 1, ctx->stream));
  return TMW_OK;
}

// Does this launch go through the shared-memory staged kernel (fp32 hop / K1 / K2 on the whole lattice)? nr may be lowered
// to the most columns per thread the staged kernel has a tile for. Opt-in only (tmw_options.stage = 1): measured on B200 it
// loses to the plain kernel at every tile shape and column count (profiles/r2_stage.md).
template <typename R> static bool use_stage(tmw_ctx* ctx, int epi, int ncol, int cb1, int& nr) {
  if (sizeof(R) != 4 || ctx->opt.stage <= 0 || cb1 >= 0 || !ctx->dom.empty()) return false;
  if (epi != EPI_HOP && epi != EPI_AINV_HOP && epi != EPI_A_XPAY) return false;
  int n = nr > 3 ? 3 : nr;
  while (n >= 1 && !ctx->stage_ok[n]) n--;
  if (n < 1) return false;
  if (n != nr) {  // regroup the columns evenly
    const int groups = (ncol + n - 1) / n;
    n = (ncol + groups - 1) / groups;
    if (!ctx->stage_ok[n]) return false;
  }
  nr = n;
  return true;
}
static cudaError_t launch_stage(const DslashArgs<float>& a, int ng, int epi, int clv, int nr, const StageGeom& sg, cudaStream_t s) {
  return launch_dslash_stage(a, ng, epi, clv, nr, sg, s);
}
static cudaError_t launch_stage(const DslashArgs<double>&, int, int, int, int, const StageGeom&, cudaStream_t) { return cudaErrorInvalidValue; }

// cb0, cb1 (optional): restrict the launch to the output sites with checkerboard index in [cb0, cb1), cb0 a multiple of 128
template <typename R>
static int dslash(tmw_ctx* ctx, int epi, int par, int dagger, const void* in, void* out, const void* aux, double sgn, const ColMap& cm,
                  int red_mode = 0, const void* dotv = nullptr, double* red = nullptr, int red_stride = 0, int g5 = 0, int cb0 = 0, int cb1 = -1) {
  for (int i = 0; i < cm.n; i++)  // the kernels add column * cstride to a 32-bit site index
    if (((int64_t)cm.col[i] + 1) * ((int64_t)ctx->g.Vh * 24 * (int64_t)sizeof(R) / 16) >= ((int64_t)1 << 31))
      return fail(ctx, TMW_EINVAL, "lattice too large for this many right-hand-side columns in one call");
  if (!ctx->dom.empty()) return dslash_dd<R>(ctx, epi, par, dagger, in, out, aux, sgn, cm, red_mode, dotv, red, red_stride, g5);
  DslashArgs<R> a = make_args<R>(ctx, par, dagger, in, out, aux, sgn, cm);
  a.g5 = g5;
  a.red_mode = red_mode;
  a.dotv = dotv;
  a.red = red;
  a.red_stride = red_stride;
  // automatic link prefetch: one site block ahead in the multi-column hop launches, the one case where it was measured to pay
  if (ctx->opt.prefetch == 0 && sizeof(R) == 4 && epi == EPI_HOP && cm.n >= 2) a.pf_blocks = 1;
  if (cb1 >= 0) { a.sb0 = cb0 / 128; a.cb_end = cb1; }
  else if (sizeof(R) == 4 && cm.n >= 2 && !a.g.tiled) {
    // multi-column launch: z-slab sweep order (Geom::zc) so that the +-t window of all columns fits in L2
    int zc = 0;
    const int64_t row = (int64_t)a.g.Lh * a.g.L;  // sites of one z of a time slice
    if (ctx->opt.zchunk > 0) {
      zc = ctx->opt.zchunk;
    } else if (ctx->opt.zchunk == 0) {
      const int64_t budget = ctx->l2_bytes / ZCHUNK_L2_SHARE_DEN * ZCHUNK_L2_SHARE_NUM;  // in + out spinors of all columns over the 2-slice window
      for (int d = a.g.Lz; d >= 1; d--)
        if (a.g.Lz % d == 0 && (row * d) % 128 == 0 && 2 * row * d * 96 * 2 * cm.n <= budget) { zc = d; break; }
      if (zc == a.g.Lz) zc = 0;  // everything fits: keep the plain order
    }
    if (zc > 0 && zc < a.g.Lz && a.g.Lz % zc == 0 && (row * zc) % 128 == 0) { a.g.zc = zc; a.g.nbzt = (int)(row * zc / 128); }
  }
  // columns per thread: as even a split of the columns into groups of at most nr32 as possible
  int nr = 1;
  if (sizeof(R) == 4 && cm.n > 1) {
    if (ctx->nr32 > 0) {  // tmw_options.columns_per_thread
      const int groups = (cm.n + ctx->nr32 - 1) / ctx->nr32;
      nr = (cm.n + groups - 1) / groups;
    } else {  // 2 columns per thread (the fastest) unless 3 wastes fewer slots of a ragged last group
      nr = ((cm.n + 2) / 3 * 3 < (cm.n + 1) / 2 * 2) ? 3 : 2;
    }
  }
  const int clv = !ctx->clover ? CL_NONE : (ctx->m_im != 0.0 ? CL_TWISTED : CL_CLOVER);
  if (use_stage<R>(ctx, epi, cm.n, cb1, nr)) {
    ctx->kcount[TMW_K_STAGED] += cm.n;
    LAUNCHK(stencil_kind<R>(epi, red_mode), cm.n, launch_stage(a, ng_of<R>(ctx), epi, clv, nr, ctx->stage[nr], ctx->stream));
    return TMW_OK;
  }
  LAUNCHK(stencil_kind<R>(epi, red_mode), cm.n, launch_dslash(a, ng_of<R>(ctx), epi, clv, nr, ctx->stream));
  return TMW_OK;
}
// out = A^{-1} in (inverse) or A in on parity par, one column, fp64 (every domain of a decomposed context)
static int diag64(tmw_ctx* ctx, int par, int inverse, const void* in, void* out) {
  ctx->kcount[TMW_K_DIAG64]++;
  if (ctx->dom.empty()) {
    LAUNCH(launch_diag(make_diag<double>(ctx, 0), ctx->g, par, ctx->clover, inverse, in, out, ctx->stream));
    return TMW_OK;
  }
  const size_t lb = (size_t)ctx->vh_loc * 24 * 8;
  for (size_t k = 0; k < ctx->dom.size(); k++)
    LAUNCH(launch_diag(make_diag<double>(ctx, 0, &ctx->dom[k]), ctx->dom[k].g, par, ctx->clover, inverse, (const char*)in + k * lb, (char*)out + k * lb, ctx->stream));
  return TMW_OK;
}
// canonical fp64 spinor <-> the packed parity spinors of the context (every domain)
static int pack_both(tmw_ctx* ctx, int prec, const double* canon, void* pe, void* po) {
  ctx->kcount[TMW_K_PACK_BOTH]++;
  if (ctx->dom.empty()) { LAUNCH(launch_pack_spinor_both(ctx->g, prec, canon, pe, po, ctx->stream)); return TMW_OK; }
  const size_t lb = (size_t)ctx->vh_loc * 24 * (prec == TMW_F32 ? 4 : 8);
  for (size_t k = 0; k < ctx->dom.size(); k++) LAUNCH(launch_pack_spinor_both(ctx->dom[k].g, prec, canon, (char*)pe + k * lb, (char*)po + k * lb, ctx->stream));
  return TMW_OK;
}
static int unpack_both(tmw_ctx* ctx, int prec, const void* pe, const void* po, double* canon) {
  ctx->kcount[TMW_K_UNPACK_BOTH]++;
  if (ctx->dom.empty()) { LAUNCH(launch_unpack_spinor_both(ctx->g, prec, pe, po, canon, ctx->stream)); return TMW_OK; }
  const size_t lb = (size_t)ctx->vh_loc * 24 * (prec == TMW_F32 ? 4 : 8);
  for (size_t k = 0; k < ctx->dom.size(); k++) LAUNCH(launch_unpack_spinor_both(ctx->dom[k].g, prec, (const char*)pe + k * lb, (const char*)po + k * lb, canon, ctx->stream));
  return TMW_OK;
}

// Schur operator on the odd sites: out = A_oo in - H_oe A_ee^{-1} H_eo in  (tmp: even-parity scratch)
// The conjugate transpose is A_oo^dag in - H_eo^dag (A_ee^dag)^{-1} H_oe^dag in: the same two kernels with the
// daggered projectors / twist, because (H_oe)^dag = the daggered hopping block from odd to even.
template <typename R>
static int schur(tmw_ctx* ctx, int dagger, const void* in, void* out, void* tmp, const ColMap& cm, int red_mode = 0, const void* dotv = nullptr,
                 double* red = nullptr, int red_stride = 0) {
  int rc = dslash<R>(ctx, EPI_AINV_HOP, 0, dagger, in, tmp, nullptr, 1.0, cm);
  if (rc) return rc;
  return dslash<R>(ctx, EPI_A_XPAY, 1, dagger, tmp, out, in, -1.0, cm, red_mode, dotv, red, red_stride);
}

// Thread -> site mapping of the single-column stencil kernels (Geom::tiled), from tmw_options.tile: all 0 -> 1-D (CTA b =
// 128 consecutive cb); tile[0] = -1 -> the largest power-of-two 4-D tile of 128 sites that divides the lattice,
// preferring 8 (xh) x 4 (y) x 2 (z) x 2 (t); else those log2 extents. Measured on B200: the tiled mapping
// changes neither the time nor the DRAM traffic of the stencil, so it stays an opt-in tuning knob.
static void choose_tile(Geom& g, const int* tile) {
  g.tiled = 0;
  g.lx = g.ly = g.lz = g.lt = 0;
  g.ntx = g.nty = 1;
  int l[4] = {tile[0], tile[1], tile[2], tile[3]};
  if (l[0] == 0 && l[1] == 0 && l[2] == 0 && l[3] == 0) return;
  const int ext[4] = {g.Lh, g.L, g.Lz, g.T};
  if (l[0] < 0) {
    const int want[4] = {3, 2, 1, 1};
    int left = 7;
    for (int d = 0; d < 4; d++) {
      l[d] = 0;
      while (l[d] < want[d] && ext[d] % (2 << l[d]) == 0) l[d]++;
      left -= l[d];
    }
    for (int d = 3; d >= 1 && left > 0; d--)  // fill up from t, z, y if x (or another extent) fell short
      while (left > 0 && ext[d] % (2 << l[d]) == 0) { l[d]++; left--; }
    if (left != 0) return;
  }
  int sum = 0;
  for (int d = 0; d < 4; d++) {
    if (l[d] < 0 || l[d] > 7 || ext[d] % (1 << l[d]) != 0) return;
    sum += l[d];
  }
  if (sum != 7) return;
  g.tiled = 1;
  g.lx = l[0]; g.ly = l[1]; g.lz = l[2]; g.lt = l[3];
  g.ntx = g.Lh >> g.lx;
  g.nty = g.L >> g.ly;
}

// Tile of the staged stencil (tmw_dslash_stage.cuh) for nr columns per thread: txh | Lh, ty | L, tz | L with at most
// stage_max_threads(nr) threads and nr * 6 * nslots float4 of shared memory. Automatic choice: the tile with the fewest
// staged sites per output site among those that are whole warps, at least 96 threads, and leave room for two CTAs per SM
// (<= 112 KB each); a forced tile (tmw_options.stage_tile) or stage = 1 only has to fit at all (<= 226 KB).
static bool make_stage(const Geom& g, int nr, int txh, int ty, int tz, size_t budget, StageGeom& sg) {
  if (txh < 1 || ty < 2 || tz < 2 || g.Lh % txh || g.L % ty || g.Lz % tz) return false;
  sg.txh = txh; sg.ty = ty; sg.tz = tz;
  sg.ntx = g.Lh / txh; sg.nty = g.L / ty; sg.ntz = g.Lz / tz;
  sg.fullx = (txh == g.Lh);
  sg.rw = sg.fullx ? g.Lh : txh + 2;
  sg.nrows = ty * tz + 2 * tz + 2 * ty;
  sg.nslots = sg.nrows * sg.rw;
  sg.nthr = txh * ty * tz;
  if ((sg.nthr + 31) / 32 * 32 > stage_max_threads(nr)) return false;
  return (size_t)nr * 6 * sg.nslots * 16 <= budget;
}
static bool choose_stage(const Geom& g, int nr, const tmw_options& o, StageGeom& best) {
  if (o.stage <= 0 || g.tiled) return false;
  if (o.stage_tile[0] || o.stage_tile[1] || o.stage_tile[2]) return make_stage(g, nr, o.stage_tile[0], o.stage_tile[1], o.stage_tile[2], 226 * 1024, best);
  bool found = false;
  double best_ratio = 0;
  for (int pass = 0; pass < 2 && !found; pass++) {  // pass 1 (stage = 1 only): any tile that fits
    if (pass == 1 && o.stage != 1) break;
    for (int txh = g.Lh; txh >= 1; txh--) {
      if (g.Lh % txh) continue;
      for (int ty = 8; ty >= 2; ty >>= 1)
        for (int tz = 8; tz >= 2; tz >>= 1) {
          StageGeom sg;
          if (!make_stage(g, nr, txh, ty, tz, pass == 0 ? 112 * 1024 : 226 * 1024, sg)) continue;
          if (pass == 0 && (sg.nthr % 32 || sg.nthr < 96)) continue;
          const double ratio = (double)sg.nslots / sg.nthr;
          if (!found || ratio < best_ratio - 1e-9 || (ratio < best_ratio + 1e-9 && sg.nthr > best.nthr)) { best = sg; best_ratio = ratio; found = true; }
        }
    }
  }
  return found;
}

extern "C" {

const char* tmw_last_error(const tmw_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

void tmw_destroy(tmw_ctx* ctx) {
  if (!ctx) return;
  cudaStreamSynchronize(ctx->stream);
  for (void* p : ctx->owned) cudaFree(p);
  if (ctx->sc_host) cudaFreeHost(ctx->sc_host);
  if (ctx->red_host) cudaFreeHost(ctx->red_host);
  if (ctx->gs_host) cudaFreeHost(ctx->gs_host);
  if (ctx->attn_host) cudaFreeHost(ctx->attn_host);
  for (int i = 0; i < 2; i++) if (ctx->ev_lag[i]) cudaEventDestroy(ctx->ev_lag[i]);
  if (ctx->comm) { cudaStreamSynchronize(ctx->comm); cudaStreamDestroy(ctx->comm); }
  if (ctx->h2d) { cudaStreamSynchronize(ctx->h2d); cudaStreamDestroy(ctx->h2d); }
  if (ctx->d2h) { cudaStreamSynchronize(ctx->d2h); cudaStreamDestroy(ctx->d2h); }
  for (int i = 0; i < NSLAB; i++) {
    if (ctx->ev_in[i]) cudaEventDestroy(ctx->ev_in[i]);
    if (ctx->ev_out[i]) cudaEventDestroy(ctx->ev_out[i]);
  }
  if (ctx->ev_pack) cudaEventDestroy(ctx->ev_pack);
  if (ctx->ev_comm) cudaEventDestroy(ctx->ev_comm);
  if (ctx->ev0) cudaEventDestroy(ctx->ev0);
  if (ctx->ev1) cudaEventDestroy(ctx->ev1);
  delete ctx;
}

int tmw_create(tmw_ctx** out, int L, int T, const double* gauge, tmw_complex m, double c_sw, const tmw_options* opt) {
  NvtxRange nvtx("tmw_create");
  if (!out) return fail(nullptr, TMW_EINVAL, "tmw_create: out is null");
  *out = nullptr;
  if (!gauge) return fail(nullptr, TMW_EINVAL, "tmw_create: gauge is null");
  if (L < 4 || T < 4 || (L & 1) || (T & 1)) return fail(nullptr, TMW_EINVAL, "tmw_create: L and T must be even and >= 4");
  const int64_t V = (int64_t)L * L * L * T;
  if (V / 2 >= (int64_t)1 << 31) return fail(nullptr, TMW_EINVAL, "tmw_create: lattice too large");
  tmw_options o;
  memset(&o, 0, sizeof(o));
  if (opt) {
    if (opt->struct_size != sizeof(tmw_options))
      return fail(nullptr, TMW_EINVAL, "tmw_create: tmw_options.struct_size is not sizeof(tmw_options) of this library (set it, e.g. with TMW_OPTIONS_INIT; a header of another version?)");
    o = *opt;
  }
  if (o.reconstruct == 0) o.reconstruct = 12;
  if (o.max_iter == 0) o.max_iter = 10000;
  if (o.nkrylov == 0) o.nkrylov = 8;  // GCR(8) beats GCR(16) on every config (orthogonalisation traffic)
  if (o.delta == 0.0) o.delta = 1e-5;  // the fewest fp64 passes without costing iterations
  if ((o.location != TMW_DEVICE && o.location != TMW_HOST) || (o.precision != TMW_MIXED && o.precision != TMW_DOUBLE) ||
      (o.reconstruct != 12 && o.reconstruct != 18) || (o.mass_reading != TMW_TWIST_GAMMA5 && o.mass_reading != TMW_MASS_SCALAR) ||
      o.max_iter < 0 || !(o.delta > 0.0) || !(o.delta < 1.0) || (o.solver != TMW_BICGSTAB && o.solver != TMW_GCR) || o.nkrylov < 1 ||
      o.nkrylov > GCR_KMAX || o.columns_per_thread < 0 || o.columns_per_thread > 4 ||
      (o.debug & ~(TMW_DEBUG_FORCE_PIVOT | TMW_DEBUG_NO_CHUNK | TMW_DEBUG_FORCE_DEFECT)) || o.stage < -1 || o.stage > 1 || o.stage_tile[0] < 0 ||
      o.stage_tile[1] < 0 || o.stage_tile[2] < 0 || o.zchunk < -1 || o.prefetch < -1)
    return fail(nullptr, TMW_EINVAL, "tmw_create: bad option value");
  if (!isfinite(m.re) || !isfinite(m.im) || !isfinite(c_sw)) return fail(nullptr, TMW_EINVAL, "tmw_create: non-finite parameter");
  const int pz = o.domains_z > 1 ? o.domains_z : 1, pt = o.domains_t > 1 ? o.domains_t : 1;
  if (o.domains_z < 0 || o.domains_t < 0 || L % (2 * pz) != 0 || T % (2 * pt) != 0)
    return fail(nullptr, TMW_EINVAL, "tmw_create: domains_z / domains_t must divide L / T into even local extents");
  tmw_ctx* ctx = new (std::nothrow) tmw_ctx();
  if (!ctx) return fail(nullptr, TMW_ENOMEM, "tmw_create: host allocation failed");
  ctx->g.L = L; ctx->g.T = T; ctx->g.Lh = L / 2; ctx->g.Vh = (int)(V / 2);
  ctx->g.Lz = L; ctx->g.oz = 0; ctx->g.ot = 0; ctx->g.GT = T;
  ctx->g.sy = L / 2; ctx->g.sz = (L / 2) * L; ctx->g.st = (L / 2) * L * L;
  choose_tile(ctx->g, o.tile);
  ctx->ws_cols = 1;
  ctx->pz = pz; ctx->pt = pt;
  ctx->vh_loc = ctx->g.Vh / (pz * pt);
  ctx->nr32 = o.columns_per_thread;
  for (int nr = 0; nr < 4; nr++) ctx->stage_ok[nr] = (nr >= 1 && nr <= 3 && pz * pt == 1) ? choose_stage(ctx->g, nr, o, ctx->stage[nr]) : false;
  ctx->verbose = o.verbose != 0;
  {
    int dev = 0, sms = 0, l2 = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev);
    if (e != cudaSuccess) {
      const int rc = fail_cuda(nullptr, e, "tmw_create: device attributes");
      delete ctx;
      return rc;
    }
    ctx->sms = sms > 0 ? sms : 148;
    ctx->l2_bytes = l2 > 0 ? (int64_t)l2 : (int64_t)ZCHUNK_L2_FALLBACK_MB << 20;
  }
  ctx->V = V;
  ctx->m_re = m.re; ctx->m_im = m.im; ctx->c_sw = c_sw;
  ctx->opt = o;
  ctx->stream = (cudaStream_t)o.stream;
  ctx->clover = (c_sw != 0.0);
  ctx->ng32 = o.reconstruct;
  ctx->launches = 0;
  memset(ctx->kcount, 0, sizeof(ctx->kcount));
  int rc = TMW_OK;
  // from here on errors must free ctx
#define CKC(call)                                                       \
  do {                                                                  \
    cudaError_t e_ = (call);                                            \
    if (e_ != cudaSuccess) {                                            \
      rc = fail_cuda(nullptr, e_, #call);                               \
      tmw_destroy(ctx);                                                 \
      return rc;                                                        \
    }                                                                   \
  } while (0)
#define CKA(p, bytes)                                                   \
  do {                                                                  \
    rc = dev_alloc(ctx, (void**)(p), (bytes));                          \
    if (rc) { g_create_err = ctx->err; tmw_destroy(ctx); return rc; }   \
  } while (0)
  if (!ctx->clover) {
    const double dg = -(4.0 + m.re);
    if (dg * dg + m.im * m.im == 0.0) { tmw_destroy(ctx); return fail(nullptr, TMW_ESINGULAR, "tmw_create: 4 + m = 0, the diagonal part is singular"); }
  }
  CKC(cudaMallocHost((void**)&ctx->sc_host, MAXCOL * sizeof(Scalars)));
  CKC(cudaMallocHost((void**)&ctx->red_host, 4 * MAXCOL * sizeof(double)));
  CKC(cudaEventCreate(&ctx->ev0));
  CKC(cudaEventCreate(&ctx->ev1));
  CKA(&ctx->sc, MAXCOL * sizeof(Scalars));
  CKA(&ctx->red, 4 * MAXCOL * sizeof(double));
  CKC(cudaMallocHost((void**)&ctx->attn_host, 6 * sizeof(int)));
  CKA(&ctx->attn, 2 * sizeof(int));
  for (int i = 0; i < 2; i++) CKC(cudaEventCreateWithFlags(&ctx->ev_lag[i], cudaEventDisableTiming));
  CKC(cudaMallocHost((void**)&ctx->gs_host, MAXCOL * sizeof(GcrScalars)));
  CKA(&ctx->gs, MAXCOL * sizeof(GcrScalars));
  const size_t Vh = (size_t)ctx->g.Vh;
  const int np32 = (ctx->ng32 == 12) ? 3 : 5;
  for (int p = 0; p < 2; p++) {
    CKA(&ctx->g64[p], Vh * 4 * 9 * 16);
    CKA(&ctx->g32[p], Vh * 4 * np32 * 16);
  }
  const double* gdev = gauge;
  void* staging = nullptr;
  if (o.location == TMW_HOST) {
    CKA(&staging, (size_t)V * 4 * 18 * 8);
    CKC(cudaMemcpyAsync(staging, gauge, (size_t)V * 4 * 18 * 8, cudaMemcpyHostToDevice, ctx->stream));
    gdev = (const double*)staging;
  }
  CKC(launch_pack_gauge(ctx->g, gdev, ctx->g64[0], ctx->g64[1], ctx->g32[0], ctx->g32[1], ctx->ng32, ctx->stream));
  ctx->launches++;
  if (ctx->clover) {
    for (int p = 0; p < 2; p++) {
      CKA(&ctx->c64[p], Vh * 36 * 16);
      CKA(&ctx->c32[p], Vh * 18 * 16);
    }
    CKA(&ctx->ci64, Vh * 36 * 16);
    CKA(&ctx->ci32, Vh * 18 * 16);
    CKC(launch_clover_build(ctx->g, ctx->g64[0], ctx->g64[1], c_sw, -(4.0 + m.re), ctx->c64[0], ctx->c64[1], ctx->c32[0], ctx->c32[1], ctx->ng32 == 12, ctx->stream));
    ctx->launches++;
    int* flag = (int*)ctx->red;
    CKC(cudaMemsetAsync(flag, 0, sizeof(int), ctx->stream));
    const double tw2 = m.im * m.im;
    CKC(launch_clover_invert(ctx->g, ctx->c64[0], tw2, ctx->ci64, ctx->ci32, flag, ctx->stream));
    ctx->launches++;
    int hflag = 0;
    CKC(cudaMemcpyAsync(&hflag, flag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CKC(cudaStreamSynchronize(ctx->stream));
    if (o.debug & TMW_DEBUG_FORCE_PIVOT) hflag = 1;  // tests: force the fallback
    if (hflag) {  // a tiny pivot without pivoting: redo the field with the pivoted kernel, which decides singularity
      CKC(cudaMemsetAsync(flag, 0, sizeof(int), ctx->stream));
      CKC(launch_clover_invert_pivot(ctx->g, ctx->c64[0], tw2, ctx->ci64, ctx->ci32, flag, ctx->stream));
      ctx->launches++;
      CKC(cudaMemcpyAsync(&hflag, flag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
      CKC(cudaStreamSynchronize(ctx->stream));
    }
    if (hflag) { tmw_destroy(ctx); return fail(nullptr, TMW_ESINGULAR, "tmw_create: a clover block on an even site is singular"); }
  }
  CKC(cudaStreamSynchronize(ctx->stream));
  if (staging) dev_free(ctx, staging);
  if (pz * pt > 1) {
    // Domain decomposition: every domain gets its own packed gauge and clover fields, cut out of the
    // whole-lattice ones built above (the clover leaves reach across the cuts, so F is computed before the split); the
    // whole-lattice copies are then released. Split in t first, then z (tmw_options.domains_t / domains_z).
    CKC(cudaStreamCreateWithFlags(&ctx->comm, cudaStreamNonBlocking));
    CKC(cudaEventCreateWithFlags(&ctx->ev_pack, cudaEventDisableTiming));
    CKC(cudaEventCreateWithFlags(&ctx->ev_comm, cudaEventDisableTiming));
    int device = 0;
    CKC(cudaGetDevice(&device));
    const int64_t gVh = ctx->g.Vh;
    for (int it = 0; it < pt; it++)
      for (int iz = 0; iz < pz; iz++) {
        Domain d;
        memset(&d, 0, sizeof(d));
        d.g = ctx->g;
        d.g.tiled = 0;
        d.g.Lz = L / pz; d.g.T = T / pt;
        d.g.oz = iz * d.g.Lz; d.g.ot = it * d.g.T;
        d.g.Vh = ctx->vh_loc;
        d.g.st = d.g.sz * d.g.Lz;
        d.iz = iz; d.it = it; d.device = device;
        const size_t lv = (size_t)d.g.Vh;
        for (int p = 0; p < 2; p++) {
          CKA(&d.g64[p], lv * 36 * 16);
          CKA(&d.g32[p], lv * 4 * np32 * 16);
          CKC(launch_extract_planes(d.g, 36, gVh, ctx->g64[p], d.g64[p], ctx->stream));
          CKC(launch_extract_planes(d.g, 4 * np32, gVh, ctx->g32[p], d.g32[p], ctx->stream));
          if (ctx->clover) {
            CKA(&d.c64[p], lv * 36 * 16);
            CKA(&d.c32[p], lv * 18 * 16);
            CKC(launch_extract_planes(d.g, 36, gVh, ctx->c64[p], d.c64[p], ctx->stream));
            CKC(launch_extract_planes(d.g, 18, gVh, ctx->c32[p], d.c32[p], ctx->stream));
          }
        }
        if (ctx->clover) {
          CKA(&d.ci64, lv * 36 * 16);
          CKA(&d.ci32, lv * 18 * 16);
          CKC(launch_extract_planes(d.g, 36, gVh, ctx->ci64, d.ci64, ctx->stream));
          CKC(launch_extract_planes(d.g, 18, gVh, ctx->ci32, d.ci32, ctx->stream));
        }
        ctx->launches += ctx->clover ? 10 : 4;
        ctx->dom.push_back(d);
      }
    CKC(cudaStreamSynchronize(ctx->stream));
    for (int p = 0; p < 2; p++) {
      dev_free(ctx, ctx->g64[p]); dev_free(ctx, ctx->g32[p]); ctx->g64[p] = ctx->g32[p] = nullptr;
      if (ctx->clover) { dev_free(ctx, ctx->c64[p]); dev_free(ctx, ctx->c32[p]); ctx->c64[p] = ctx->c32[p] = nullptr; }
    }
    if (ctx->clover) { dev_free(ctx, ctx->ci64); dev_free(ctx, ctx->ci32); ctx->ci64 = ctx->ci32 = nullptr; }
  }
  *out = ctx;
  return TMW_OK;
#undef CKC
#undef CKA
}

long long tmw_spinor_bytes(const tmw_ctx* ctx, int prec) {
  if (!ctx || (prec != TMW_F32 && prec != TMW_F64)) return 0;
  return (long long)spinor_bytes(ctx, prec);
}
long long tmw_launch_count(const tmw_ctx* ctx) { return ctx ? ctx->launches : 0; }
int tmw_kernel_counts(const tmw_ctx* ctx, long long* counts, int n) {
  if (!ctx || !counts || n < 0) return TMW_EINVAL;
  for (int i = 0; i < n && i < TMW_K_COUNT; i++) counts[i] = ctx->kcount[i];
  return TMW_K_COUNT;
}
int tmw_set_location(tmw_ctx* ctx, int location) {
  if (!ctx) return TMW_EINVAL;
  if (location != TMW_DEVICE && location != TMW_HOST) return fail(ctx, TMW_EINVAL, "tmw_set_location: bad location");
  ctx->opt.location = location;
  return TMW_OK;
}

int tmw_set_debug(tmw_ctx* ctx, int flags) {
  if (!ctx) return TMW_EINVAL;
  if (flags & ~(TMW_DEBUG_FORCE_PIVOT | TMW_DEBUG_NO_CHUNK | TMW_DEBUG_FORCE_DEFECT)) return fail(ctx, TMW_EINVAL, "tmw_set_debug: unknown flag");
  ctx->opt.debug = flags;
  return TMW_OK;
}

int tmw_pack(tmw_ctx* ctx, int prec, int parity, const double* canonical, void* packed) {
  if (!ctx) return TMW_EINVAL;
  if (!canonical || !packed || (prec != TMW_F32 && prec != TMW_F64) || (parity != TMW_EVEN && parity != TMW_ODD)) return fail(ctx, TMW_EINVAL, "tmw_pack: bad argument");
  if (!ctx->dom.empty()) {  // the domains' local packed spinors back to back
    const size_t lb = (size_t)ctx->vh_loc * 24 * (prec == TMW_F32 ? 4 : 8);
    for (size_t k = 0; k < ctx->dom.size(); k++) LAUNCH(launch_pack_spinor(ctx->dom[k].g, parity == TMW_ODD, prec, canonical, (char*)packed + k * lb, ctx->stream));
    return TMW_OK;
  }
  LAUNCH(launch_pack_spinor(ctx->g, parity == TMW_ODD, prec, canonical, packed, ctx->stream));
  return TMW_OK;
}
int tmw_unpack(tmw_ctx* ctx, int prec, int parity, const void* packed, double* canonical) {
  if (!ctx) return TMW_EINVAL;
  if (!canonical || !packed || (prec != TMW_F32 && prec != TMW_F64) || (parity != TMW_EVEN && parity != TMW_ODD)) return fail(ctx, TMW_EINVAL, "tmw_unpack: bad argument");
  if (!ctx->dom.empty()) {
    const size_t lb = (size_t)ctx->vh_loc * 24 * (prec == TMW_F32 ? 4 : 8);
    for (size_t k = 0; k < ctx->dom.size(); k++) LAUNCH(launch_unpack_spinor(ctx->dom[k].g, parity == TMW_ODD, prec, (const char*)packed + k * lb, canonical, ctx->stream));
    return TMW_OK;
  }
  LAUNCH(launch_unpack_spinor(ctx->g, parity == TMW_ODD, prec, packed, canonical, ctx->stream));
  return TMW_OK;
}

int tmw_get_clover(tmw_ctx* ctx, int parity, int inverse, double* dst) {
  if (!ctx) return TMW_EINVAL;
  if (!dst || (parity != TMW_EVEN && parity != TMW_ODD)) return fail(ctx, TMW_EINVAL, "tmw_get_clover: bad argument");
  if (!ctx->clover) return fail(ctx, TMW_EINVAL, "tmw_get_clover: context has no clover term (c_sw = 0)");
  if (inverse && parity != TMW_EVEN) return fail(ctx, TMW_EINVAL, "tmw_get_clover: the inverse is stored on the even parity only");
  if (!ctx->dom.empty()) return fail(ctx, TMW_EINVAL, "tmw_get_clover: not available on a domain-decomposed context (the blocks live per domain)");
  const void* src = inverse ? ctx->ci64 : ctx->c64[parity == TMW_ODD];
  LAUNCH(launch_clover_export(ctx->g, src, dst, ctx->stream));
  return TMW_OK;
}

}  // extern "C"

// ---- workspaces ----
static void release_ws(tmw_ctx* ctx) {
  for (int i = 0; i < NW64; i++) if (ctx->w64[i]) { dev_free(ctx, ctx->w64[i]); ctx->w64[i] = nullptr; }
  for (int i = 0; i < 8; i++) if (ctx->w32[i]) { dev_free(ctx, ctx->w32[i]); ctx->w32[i] = nullptr; }
  for (int i = 0; i < 2; i++) if (ctx->canon[i]) { dev_free(ctx, ctx->canon[i]); ctx->canon[i] = nullptr; }
  if (ctx->gcr_q) { dev_free(ctx, ctx->gcr_q); ctx->gcr_q = nullptr; }
  if (ctx->gcr_p) { dev_free(ctx, ctx->gcr_p); ctx->gcr_p = nullptr; }
}
// make the workspaces hold `cols` columns (existing smaller ones are released and re-made on demand)
static int need_cols(tmw_ctx* ctx, int cols) {
  if (cols <= ctx->ws_cols) return TMW_OK;
  cudaError_t e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaStreamSynchronize");
  release_ws(ctx);
  ctx->ws_cols = cols;
  return TMW_OK;
}
// A failed workspace allocation (TMW_ENOMEM: too many columns for this lattice) releases every workspace and goes back
// to one column, so that the context stays usable for smaller calls.
static int ws_alloc(tmw_ctx* ctx, void** p, size_t bytes) {
  const int rc = dev_alloc(ctx, p, bytes);
  if (rc) {
    cudaStreamSynchronize(ctx->stream);
    release_ws(ctx);
    ctx->ws_cols = 1;
  }
  return rc;
}
static int need_w64(tmw_ctx* ctx, int n) {
  for (int i = 0; i < n; i++)
    if (!ctx->w64[i]) { int rc = ws_alloc(ctx, &ctx->w64[i], spinor_bytes(ctx, TMW_F64) * ctx->ws_cols); if (rc) return rc; }
  return TMW_OK;
}
static int need_w32(tmw_ctx* ctx, int n, int prec) {
  for (int i = 0; i < n; i++)
    if (!ctx->w32[i]) { int rc = ws_alloc(ctx, &ctx->w32[i], spinor_bytes(ctx, prec) * ctx->ws_cols); if (rc) return rc; }
  return TMW_OK;
}
static int need_canon(tmw_ctx* ctx) {
  for (int i = 0; i < 2; i++)
    if (!ctx->canon[i]) { int rc = ws_alloc(ctx, &ctx->canon[i], (size_t)ctx->V * 24 * 8 * ctx->ws_cols); if (rc) return rc; }
  return TMW_OK;
}
static inline void* colp(void* base, int c, size_t bytes) { return (char*)base + (size_t)c * bytes; }
static inline const void* colp(const void* base, int c, size_t bytes) { return (const char*)base + (size_t)c * bytes; }

// out_p = A in_p + H in_pbar for both parities, fp64 packed
static int full_apply64(tmw_ctx* ctx, int dagger, const void* in_e, const void* in_o, void* out_e, void* out_o, const ColMap& cm, int g5 = 0) {
  int rc = dslash<double>(ctx, EPI_A_XPAY, 0, dagger, in_o, out_e, in_e, 1.0, cm, 0, nullptr, nullptr, 0, g5);
  if (rc) return rc;
  return dslash<double>(ctx, EPI_A_XPAY, 1, dagger, in_e, out_o, in_o, 1.0, cm, 0, nullptr, nullptr, 0, g5);
}

// tmw_apply FULL with HOST pointers, one column: the canonical spinor is cut into S t-slabs (contiguous both in the
// canonical array and in checkerboard order) and three streams work on them at once, so that both PCIe directions are
// busy: h2d uploads slab after slab (the LAST slab first: the periodic t-neighbour of slab 0); the context stream packs
// every slab as it arrives and applies the operator to slab k as soon as slabs k-1, k, k+1 are there, then unpacks it;
// d2h downloads every finished slab. Only the last two slabs cannot overlap their upload.
static int apply_full_host_pipelined(tmw_ctx* ctx, int dagger, int g5, const double* in, double* out) {
  const int T = ctx->g.T;
  int S = 1;
  for (int d = 2; d <= NSLAB && d <= T; d++) if (T % d == 0) S = d;  // as many slabs as there are events: a short tail
  if (S < 3) S = 1;
  const int dt = T / S;
  if (!ctx->h2d) {
    CK(cudaStreamCreateWithFlags(&ctx->h2d, cudaStreamNonBlocking));
    CK(cudaStreamCreateWithFlags(&ctx->d2h, cudaStreamNonBlocking));
    for (int i = 0; i < NSLAB; i++) {
      CK(cudaEventCreateWithFlags(&ctx->ev_in[i], cudaEventDisableTiming));
      CK(cudaEventCreateWithFlags(&ctx->ev_out[i], cudaEventDisableTiming));
    }
  }
  int rc;
  void** W = ctx->w64;
  const ColMap one = cols_first(1);
  const int64_t slice = (int64_t)ctx->g.L * ctx->g.L * ctx->g.L;  // lexicographic sites per time slice
  const size_t slab_bytes = (size_t)slice * dt * 24 * 8;
  const int slab_cb = ctx->g.st * dt;                            // checkerboard sites per parity and slab
  double* cin = (double*)ctx->canon[0];
  double* cout = (double*)ctx->canon[1];
  // the copy streams start after whatever the context stream still has queued on the staging buffers
  CK(cudaEventRecord(ctx->ev0, ctx->stream));
  CK(cudaStreamWaitEvent(ctx->h2d, ctx->ev0, 0));
  CK(cudaStreamWaitEvent(ctx->d2h, ctx->ev0, 0));
  for (int j = 0; j < S; j++) {  // upload order: S-1, 0, 1, ..., S-2
    const int k = (j + S - 1) % S;
    CK(cudaMemcpyAsync((char*)cin + k * slab_bytes, (const char*)in + k * slab_bytes, slab_bytes, cudaMemcpyHostToDevice, ctx->h2d));
    CK(cudaEventRecord(ctx->ev_in[k], ctx->h2d));
  }
  auto pack_slab = [&](int k) -> int {
    CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_in[k], 0));
    ctx->kcount[TMW_K_PACK_BOTH]++;
    LAUNCH(launch_pack_spinor_both(ctx->g, 1, cin, W[0], W[1], ctx->stream, k * slice * dt, (k + 1) * slice * dt));
    return TMW_OK;
  };
  auto do_slab = [&](int k) -> int {
    const int c0 = k * slab_cb, c1 = (k + 1) * slab_cb;
    int r = dslash<double>(ctx, EPI_A_XPAY, 0, dagger, W[1], W[2], W[0], 1.0, one, 0, nullptr, nullptr, 0, g5, c0, c1);
    if (!r) r = dslash<double>(ctx, EPI_A_XPAY, 1, dagger, W[0], W[3], W[1], 1.0, one, 0, nullptr, nullptr, 0, g5, c0, c1);
    if (r) return r;
    ctx->kcount[TMW_K_UNPACK_BOTH]++;
    LAUNCH(launch_unpack_spinor_both(ctx->g, 1, W[2], W[3], cout, ctx->stream, k * slice * dt, (k + 1) * slice * dt));
    CK(cudaEventRecord(ctx->ev_out[k], ctx->stream));
    CK(cudaStreamWaitEvent(ctx->d2h, ctx->ev_out[k], 0));
    CK(cudaMemcpyAsync((char*)out + k * slab_bytes, (const char*)cout + k * slab_bytes, slab_bytes, cudaMemcpyDeviceToHost, ctx->d2h));
    return TMW_OK;
  };
  if ((rc = pack_slab(S - 1))) return rc;
  if (S > 1 && (rc = pack_slab(0))) return rc;
  for (int k = 0; k < S; k++) {
    if (k + 1 < S - 1 && (rc = pack_slab(k + 1))) return rc;  // slab S-1 is already packed
    if ((rc = do_slab(k))) return rc;
  }
  CK(cudaStreamSynchronize(ctx->d2h));
  CK(cudaStreamSynchronize(ctx->stream));
  return TMW_OK;
}

extern "C" int tmw_apply_multi(tmw_ctx* ctx, int op, int parity, int prec, int nrhs, const void* in, void* out) {
  NvtxRange nvtx("tmw_apply");
  if (!ctx) return TMW_EINVAL;
  if (!in || !out || in == out) return fail(ctx, TMW_EINVAL, "tmw_apply: null or aliased pointers");
  if ((op != TMW_D && op != TMW_DDAG && op != TMW_G5D) || (parity != TMW_FULL && parity != TMW_EVEN && parity != TMW_ODD)) return fail(ctx, TMW_EINVAL, "tmw_apply: bad op or parity");
  if (nrhs < 1 || nrhs > MAXCOL) return fail(ctx, TMW_EINVAL, "tmw_apply: nrhs must be in 1..16");
  const int dagger = (op == TMW_DDAG), g5 = (op == TMW_G5D);
  const ColMap cm = cols_first(nrhs);
  if (parity != TMW_FULL) {
    if (prec != TMW_F32 && prec != TMW_F64) return fail(ctx, TMW_EINVAL, "tmw_apply: bad precision");
    const int par = (parity == TMW_ODD);
    if (prec == TMW_F32) return dslash<float>(ctx, EPI_HOP, par, dagger, in, out, nullptr, 1.0, cm, 0, nullptr, nullptr, 0, g5);
    return dslash<double>(ctx, EPI_HOP, par, dagger, in, out, nullptr, 1.0, cm, 0, nullptr, nullptr, 0, g5);
  }
  int rc = need_cols(ctx, nrhs);
  if (rc) return rc;
  if ((rc = need_w64(ctx, 4))) return rc;
  const double* cin = (const double*)in;
  double* cout = (double*)out;
  const size_t cbytes = (size_t)ctx->V * 24 * 8, b64 = spinor_bytes(ctx, TMW_F64);
  if (ctx->opt.location == TMW_HOST) {
    rc = need_canon(ctx);
    if (rc) return rc;
    if (nrhs == 1 && ctx->dom.empty() && !ctx->g.tiled && ctx->g.st % 128 == 0) return apply_full_host_pipelined(ctx, dagger, g5, (const double*)in, (double*)out);
    CK(cudaMemcpyAsync(ctx->canon[0], in, cbytes * nrhs, cudaMemcpyHostToDevice, ctx->stream));
    cin = (const double*)ctx->canon[0];
    cout = (double*)ctx->canon[1];
  }
  for (int c = 0; c < nrhs; c++) {
    if ((rc = pack_both(ctx, 1, (const double*)colp(cin, c, cbytes), colp(ctx->w64[0], c, b64), colp(ctx->w64[1], c, b64)))) return rc;
  }
  rc = full_apply64(ctx, dagger, ctx->w64[0], ctx->w64[1], ctx->w64[2], ctx->w64[3], cm, g5);
  if (rc) return rc;
  for (int c = 0; c < nrhs; c++) {
    if ((rc = unpack_both(ctx, 1, colp(ctx->w64[2], c, b64), colp(ctx->w64[3], c, b64), (double*)colp(cout, c, cbytes)))) return rc;
  }
  if (ctx->opt.location == TMW_HOST) {
    CK(cudaMemcpyAsync(out, cout, cbytes * nrhs, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
  }
  return TMW_OK;
}
extern "C" int tmw_apply(tmw_ctx* ctx, int op, int parity, int prec, const void* in, void* out) {
  return tmw_apply_multi(ctx, op, parity, prec, 1, in, out);
}

// Chebyshev series of X = scale * gamma5 D + shift by the Clenshaw recursion, fp64, full lattice:
//   b_{n} = b_{n+1} = 0;  b_k = c_k psi + 2 X b_{k+1} - b_{k+2} (k = n-1 .. 1);  out = c_0 psi + X b_1 - b_2.
// Each step = gamma5 D fused in the two stencil launches + one fused vector kernel per parity.
//   w64: 0,1 psi (e,o); 2,3 and 4,5 the two recursion vectors; 6,7 H b_1
extern "C" int tmw_cheb_apply(tmw_ctx* ctx, int ncoef, const double* coef, double scale, double shift, const double* in, double* out) {
  if (!ctx) return TMW_EINVAL;
  if (!coef || !in || !out || in == out) return fail(ctx, TMW_EINVAL, "tmw_cheb_apply: null or aliased pointers");
  if (ncoef < 1 || !isfinite(scale) || !isfinite(shift)) return fail(ctx, TMW_EINVAL, "tmw_cheb_apply: ncoef must be >= 1, scale and shift finite");
  for (int k = 0; k < ncoef; k++) if (!isfinite(coef[k])) return fail(ctx, TMW_EINVAL, "tmw_cheb_apply: non-finite coefficient");
  int rc;
  if ((rc = need_w64(ctx, 8))) return rc;
  cudaStream_t s = ctx->stream;
  const double* cin = in;
  double* cout = out;
  const size_t cbytes = (size_t)ctx->V * 24 * 8;
  if (ctx->opt.location == TMW_HOST) {
    if ((rc = need_canon(ctx))) return rc;
    CK(cudaMemcpyAsync(ctx->canon[0], in, cbytes, cudaMemcpyHostToDevice, s));
    cin = (const double*)ctx->canon[0];
    cout = (double*)ctx->canon[1];
  }
  void** W = ctx->w64;
  const int64_t n64 = (int64_t)ctx->g.Vh * 12;
  const ColMap one = cols_first(1);
  if ((rc = pack_both(ctx, 1, cin, W[0], W[1]))) return rc;
  int b1 = 2, b2 = 4;  // indices of the (even) buffers of b_{k+1}, b_{k+2}
  if (ncoef == 1) {
    for (int p = 0; p < 2; p++) LAUNCH(launch_scale(n64, W[b1 + p], W[p], coef[0], s));
  } else {
    for (int p = 0; p < 2; p++) {
      LAUNCH(launch_scale(n64, W[b1 + p], W[p], coef[ncoef - 1], s));  // b_{n-1} = c_{n-1} psi
      CK(cudaMemsetAsync(W[b2 + p], 0, (size_t)n64 * 16, s));
    }
    for (int k = ncoef - 2; k >= 0; k--) {
      if ((rc = full_apply64(ctx, 0, W[b1], W[b1 + 1], W[6], W[7], one, 1))) return rc;
      const double f = (k == 0) ? 1.0 : 2.0;
      for (int p = 0; p < 2; p++) LAUNCH(launch_clenshaw(n64, W[b2 + p], W[p], W[6 + p], W[b1 + p], W[b2 + p], coef[k], f, scale, shift, s));
      const int t = b1; b1 = b2; b2 = t;  // the new vector was written over b_{k+2}
    }
  }
  if ((rc = unpack_both(ctx, 1, W[b1], W[b1 + 1], cout))) return rc;
  if (ctx->opt.location == TMW_HOST) {
    CK(cudaMemcpyAsync(out, cout, cbytes, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
  }
  return TMW_OK;
}

extern "C" int tmw_apply_schur_multi(tmw_ctx* ctx, int op, int prec, int nrhs, const void* in_odd, void* out_odd) {
  if (!ctx) return TMW_EINVAL;
  if (!in_odd || !out_odd || in_odd == out_odd) return fail(ctx, TMW_EINVAL, "tmw_apply_schur: null or aliased pointers");
  if ((op != TMW_D && op != TMW_DDAG) || (prec != TMW_F32 && prec != TMW_F64)) return fail(ctx, TMW_EINVAL, "tmw_apply_schur: bad op or precision");
  if (nrhs < 1 || nrhs > MAXCOL) return fail(ctx, TMW_EINVAL, "tmw_apply_schur: nrhs must be in 1..16");
  const int dagger = (op == TMW_DDAG);
  int rc;
  if ((rc = need_cols(ctx, nrhs))) return rc;
  if ((rc = need_w64(ctx, 1))) return rc;  // even-parity scratch for nrhs columns
  const ColMap cm = cols_first(nrhs);
  if (prec == TMW_F64) return schur<double>(ctx, dagger, in_odd, out_odd, ctx->w64[0], cm);
  // fp32: the scratch columns are fp32 spinors back to back at the start of the (twice as large) fp64 workspace
  return schur<float>(ctx, dagger, in_odd, out_odd, ctx->w64[0], cm);
}
extern "C" int tmw_apply_schur(tmw_ctx* ctx, int op, int prec, const void* in_odd, void* out_odd) {
  return tmw_apply_schur_multi(ctx, op, prec, 1, in_odd, out_odd);
}

// ---- tmw_apply_schur_static (include/tmw.h): the Schur operator for callers that must not allocate ----
// The even-parity intermediate of K1 -> K2 lives in this array instead of the cudaMalloc'ed workspace w64[0]. It is part of
// the library image: every device that loads libtmw.so's kernels holds these bytes until the process ends.
// In HOST code the name g_static_scratch is only a handle for the runtime, not a device address (a kernel given
// `g_static_scratch` itself would fault, or scribble over host memory where the GPU can reach it): the device address
// comes from cudaGetSymbolAddress, asked in this translation unit, once per device, with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[TMW_STATIC_SCRATCH_BYTES];

namespace {
enum { STATIC_MAX_DEVICES = 64 };
void* g_static_ptr[STATIC_MAX_DEVICES];  // device address of g_static_scratch on device d, null until first asked
std::mutex g_static_mutex;
}  // namespace

// Device address of the static scratch array on the current device (which must be the context's). No allocation.
static int static_scratch_ptr(tmw_ctx* ctx, void** out) {
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(ctx, TMW_EINVAL, "tmw_apply_schur_static: device ordinal out of range");
  cudaPointerAttributes attr;
  CK(cudaPointerGetAttributes(&attr, ctx->g64[1]));  // the context's own gauge field tells which device it lives on
  if (attr.type != cudaMemoryTypeDevice || attr.device != dev)
    return fail(ctx, TMW_EINVAL, "tmw_apply_schur_static: the context's device is not the calling thread's current device");
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[dev]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaGetSymbolAddress(g_static_scratch)");
    if (!p || ((uintptr_t)p & 255)) return fail(ctx, TMW_ECUDA, "tmw_apply_schur_static: bad address for the static scratch array");
    g_static_ptr[dev] = p;
  }
  *out = g_static_ptr[dev];
  return TMW_OK;
}

extern "C" int tmw_apply_schur_static(tmw_ctx* ctx, int op, int prec, const void* in_odd, void* out_odd) {
  if (!ctx) return TMW_EINVAL;
  if (!in_odd || !out_odd || in_odd == out_odd) return fail(ctx, TMW_EINVAL, "tmw_apply_schur_static: null or aliased pointers");
  if ((op != TMW_D && op != TMW_DDAG) || (prec != TMW_F32 && prec != TMW_F64)) return fail(ctx, TMW_EINVAL, "tmw_apply_schur_static: bad op or precision");
  if (!ctx->dom.empty())
    return fail(ctx, TMW_EINVAL, "tmw_apply_schur_static: not available on a domain-decomposed context (its exchange buffers are allocated on demand)");
  const size_t need = spinor_bytes(ctx, prec);
  if (need > (size_t)TMW_STATIC_SCRATCH_BYTES) {
    char buf[256];
    snprintf(buf, sizeof(buf), "tmw_apply_schur_static: a packed parity spinor of this lattice takes %zu bytes, the static scratch array holds %zu (TMW_STATIC_SCRATCH_BYTES); use tmw_apply_schur",
             need, (size_t)TMW_STATIC_SCRATCH_BYTES);
    return fail(ctx, TMW_EINVAL, buf);
  }
  void* tmp = nullptr;
  int rc = static_scratch_ptr(ctx, &tmp);
  if (rc) return rc;
  // K1 writes the intermediate of every even site, K2 reads only those: nothing in the array has to be cleared first
  const int dagger = (op == TMW_DDAG);
  const ColMap cm = cols_first(1);
  if (prec == TMW_F64) return schur<double>(ctx, dagger, in_odd, out_odd, tmp, cm);
  return schur<float>(ctx, dagger, in_odd, out_odd, tmp, cm);
}

// ---- the solver ----
namespace {

struct ColState {
  double bnorm, rnorm, maxr, rhat_norm;
  bool done;    // converged (or b = 0)
  int iters, updates, restarts;
  double r_upd;  // true residual at the last reliable update / restart (what y stands for)
  double best;   // smallest true residual seen at a restart
  int stalled;   // consecutive restarts that did not improve on it
  double iter_resid, true_resid;
};

// download the scalar blocks and wait
int fetch_scalars(tmw_ctx* ctx) {
  CK(cudaMemcpyAsync(ctx->sc_host, ctx->sc, MAXCOL * sizeof(Scalars), cudaMemcpyDeviceToHost, ctx->stream));
  CK(cudaStreamSynchronize(ctx->stream));
  return TMW_OK;
}
int push_scalars(tmw_ctx* ctx) {
  CK(cudaMemcpyAsync(ctx->sc, ctx->sc_host, MAXCOL * sizeof(Scalars), cudaMemcpyHostToDevice, ctx->stream));
  // the pinned block is rewritten by the host right after some pushes: wait for the copy
  CK(cudaStreamSynchronize(ctx->stream));
  return TMW_OK;
}
int fetch_red(tmw_ctx* ctx) {
  CK(cudaMemcpyAsync(ctx->red_host, ctx->red, 4 * MAXCOL * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
  CK(cudaStreamSynchronize(ctx->stream));
  return TMW_OK;
}
void reset_recurrence(Scalars* h) {
  h->rho_old[0] = h->alpha[0] = h->omega[0] = 1.0;
  h->rho_old[1] = h->alpha[1] = h->omega[1] = 0.0;
}

// BiCGStab (van der Vorst) on the odd-site Schur systems Mhat y_c = bhat_c of the columns c with !cs[c].done, inner
// precision R, fp64 reliable updates. The columns run in lockstep, each with its own scalars; every launch covers the
// columns that still iterate (ColMap), so links and clover blocks are read once for all of them.
//   w64: 0 b_e, 1 b_o, 2 bhat_o, 3 y, 4 r64, 5 tmp_e64, 6 w (Mhat y), 7 x_e
//   w32: 0 r, 1 rhat, 2 p, 3 v, 4 s, 5 t, 6 x, 7 tmp_e
template <typename R>
int solve_schur(tmw_ctx* ctx, int ncols, double tol, ColState* cs) {
  cudaStream_t s = ctx->stream;
  const int64_t n64 = (int64_t)ctx->g.Vh * 12;                           // double2 vectors per fp64 parity spinor
  const int64_t nR = (int64_t)ctx->g.Vh * 24 * (int64_t)sizeof(R) / 16;  // 16-byte vectors per inner spinor
  const size_t bytesR = (size_t)nR * 16, bytes64 = (size_t)n64 * 16;
  void** W = ctx->w64;
  void** X = ctx->w32;
  void *r = X[0], *rhat = X[1], *p = X[2], *v = X[3], *sv = X[4], *t = X[5], *x = X[6], *tmp = X[7];
  Scalars* h = ctx->sc_host;
  const int SCD = (int)(sizeof(Scalars) / sizeof(double));
  double* red_rhat_v = (double*)((char*)ctx->sc + offsetof(Scalars, rhat_v));
  double* red_ts = (double*)((char*)ctx->sc + offsetof(Scalars, ts));
  // restart when |rho| = |<rhat,r>| has decayed to the noise of the vectors relative to |rhat||r|: the dot products are
  // accumulated in fp64, so for fp32 vectors that floor is ~1e-9 (rounding of r, ~6e-8/sqrt(N) per step), not 1e-6
  const double eps_break = sizeof(R) == 4 ? 1e-8 : 1e-12;
  const bool verbose = ctx->verbose;  // per-iteration residual log on stderr
  int rc;
  ColMap act;
  act.n = 0;
  for (int c = 0; c < ncols; c++) if (!cs[c].done) cols_add(act, c);
  if (act.n == 0) return TMW_OK;
  // y = 0, r64 = bhat, r = (R) r64, rhat = r, x = p = v = 0
  // only the columns that are iterated: W[3] of the others holds their finished solution (defect-correction pass)
  for (int i = 0; i < act.n; i++) {
    MEMSETK(colp(W[3], act.col[i], bytes64), 0, bytes64);
    MEMSETK(colp(x, act.col[i], bytesR), 0, bytesR);
  }
  LAUNCHK(TMW_K_CONVERT, act.n, launch_convert<R>(n64, ctx->vh_loc, W[2], rhat, act, s));
  memset(h, 0, MAXCOL * sizeof(Scalars));
  if ((rc = push_scalars(ctx))) return rc;
  LAUNCHK(TMW_K_RESID_CONVERT, act.n, launch_resid_convert<R>(n64, ctx->vh_loc, W[2], nullptr, W[4], r, rhat, nullptr, ctx->sc, act, s));  // r64 = bhat - 0; rho = <rhat,r>; rr = |r64|^2
  if ((rc = fetch_scalars(ctx))) return rc;
  // what the device compares against at the start of an iteration (Scalars::stop2 / maxr2 / brk2)
  auto arm = [&](int c) {
    h[c].stop2 = (tol * cs[c].bnorm) * (tol * cs[c].bnorm);
    h[c].maxr2 = cs[c].maxr * cs[c].maxr;
    h[c].brk2 = (eps_break * cs[c].rhat_norm) * (eps_break * cs[c].rhat_norm);
    h[c].trip = 0;
  };
  for (int i = 0; i < act.n; i++) {
    const int c = act.col[i];
    reset_recurrence(&h[c]);
    cs[c].rnorm = cs[c].maxr = cs[c].rhat_norm = cs[c].r_upd = cs[c].best = sqrt(h[c].rr);
    cs[c].iter_resid = cs[c].rnorm / cs[c].bnorm;
    if (cs[c].rnorm <= tol * cs[c].bnorm) cs[c].done = true;
    arm(c);
  }
  if ((rc = push_scalars(ctx))) return rc;
  // p = r for the first iteration; later p comes out of update_xrp (v is written by the first K2 before it is read)
  for (int i = 0; i < act.n; i++) COPYK(colp(p, act.col[i], bytesR), colp(r, act.col[i], bytesR), bytesR);
  const int max_iter = ctx->opt.max_iter;
  // The host queues iterations ahead of the device and looks at the scalars only at SYNC POINTS: when the device has raised
  // attn[0] (it tests every column at the start of each iteration, sc_begin_iter; all kernels of the queued iterations then
  // return at once, so nothing moves past the iteration that tripped), when max_iter is near, or every iteration if verbose.
  // Between sync points the host only waits for the 8-byte copy of attn of the iteration BEFORE the one it has just queued,
  // so the device always has an iteration in its queue ("read back only a convergence flag").
  const double delta2 = ctx->opt.delta * ctx->opt.delta;
  int* const lag = ctx->attn_host;       // lag[2 * (e & 1)]: attn after queued iteration e
  int* const attn_now = ctx->attn_host + 4;
  CK(cudaMemsetAsync(ctx->attn, 0, 2 * sizeof(int), s));
  int k = 0;    // iterations done, as of the last sync point
  int enq = 0;  // iterations queued since then
  for (;;) {
    act.n = 0;
    for (int c = 0; c < ncols; c++) if (!cs[c].done) cols_add(act, c);
    if (act.n == 0) return TMW_OK;
    long long per_iter[TMW_K_COUNT];  // what one iteration adds to the kernel counts
    memcpy(per_iter, ctx->kcount, sizeof(per_iter));
    {
      SkipGuard skip_guard(ctx, ctx->attn);  // cur_skip = attn until the end of this block, on every way out of it
      LAUNCH(launch_sc_begin_iter(ctx->sc, act, ctx->attn, enq > 0, delta2, s));
      rc = schur<R>(ctx, 0, p, v, tmp, act, 1, rhat, red_rhat_v, SCD);
      if (!rc) {
        LAUNCH(launch_sc_alpha(ctx->sc, act, ctx->attn, s));
        LAUNCHK(TMW_K_UPDATE_S, act.n, launch_update_s<R>(nR, sv, r, v, ctx->sc, act, ctx->attn, s));
        rc = schur<R>(ctx, 0, sv, t, tmp, act, 4, rhat, red_ts, SCD);  // <t,s>, <t,t>, <rhat,t>, <rhat,s>
      }
      if (!rc) {
        LAUNCH(launch_sc_omega(ctx->sc, act, ctx->attn, s));                                        // omega, rho' = <rhat, s - omega t>, beta
        LAUNCHK(TMW_K_UPDATE_XRP, act.n, launch_update_xrp<R>(nR, x, r, p, sv, t, v, ctx->sc, act, ctx->attn, s));  // x, r, and p of the next iteration
      }
    }
    if (rc) return rc;
    for (int i = 0; i < TMW_K_COUNT; i++) per_iter[i] = ctx->kcount[i] - per_iter[i];
    enq++;
    bool sync_now = verbose || k + enq >= max_iter;
    if (!sync_now) {
      CK(cudaMemcpyAsync(lag + 2 * (enq & 1), ctx->attn, 2 * sizeof(int), cudaMemcpyDeviceToHost, s));
      CK(cudaEventRecord(ctx->ev_lag[enq & 1], s));
      if (enq >= 2) {
        CK(cudaEventSynchronize(ctx->ev_lag[(enq - 1) & 1]));
        sync_now = lag[2 * ((enq - 1) & 1)] != 0;
      }
    }
    if (!sync_now) continue;
    // ---- sync point: the state is the one after iteration attn[1]; iterations queued beyond it did nothing ----
    CK(cudaMemcpyAsync(attn_now, ctx->attn, 2 * sizeof(int), cudaMemcpyDeviceToHost, s));
    if ((rc = fetch_scalars(ctx))) return rc;
    {
      const int skipped = k + enq - attn_now[1];  // their launches returned at once: not work of the path (tmw_kernel_counts)
      for (int i = 0; i < TMW_K_COUNT; i++) ctx->kcount[i] -= skipped * per_iter[i];
    }
    k = attn_now[1];
    enq = 0;
    const bool tripped = attn_now[0] != 0;
    if (tripped) CK(cudaMemsetAsync(ctx->attn, 0, sizeof(int), s));
    ColMap upd, brk;  // columns that take a reliable update now / whose iterate is corrupted
    upd.n = brk.n = 0;
    bool broken[MAXCOL];
    for (int i = 0; i < act.n; i++) {
      const int c = act.col[i];
      ColState& q = cs[c];
      q.iters = k;
      broken[c] = !isfinite(h[c].rr) || !isfinite(h[c].rho[0]) || !isfinite(h[c].rho[1]);
      const long long trip = tripped ? h[c].trip : 0;
      if (h[c].maxr2 > q.maxr * q.maxr) q.maxr = sqrt(h[c].maxr2);  // the device tracked it over the iterations the host did not see
      q.rnorm = broken[c] ? q.maxr : sqrt(h[c].rr);
      if (verbose)
        fprintf(stderr, "[tmw] col %d it %d |r|/|b| %.3e rho (%.3e,%.3e) alpha (%.3e,%.3e) omega (%.3e,%.3e) <rhat,v> (%.3e,%.3e) tt %.3e\n", c, k,
                sqrt(h[c].rr) / q.bnorm, h[c].rho[0], h[c].rho[1], h[c].alpha[0], h[c].alpha[1], h[c].omega[0], h[c].omega[1], h[c].rhat_v[0],
                h[c].rhat_v[1], h[c].tt);
      if (!broken[c]) q.iter_resid = q.rnorm / q.bnorm;
      const bool conv = !broken[c] && q.rnorm <= tol * q.bnorm;
      if (broken[c] || conv || (trip & ~(long long)TRIP_BREAKDOWN) || q.rnorm < ctx->opt.delta * q.maxr || k >= max_iter) {
        cols_add(upd, c);
        if (broken[c]) cols_add(brk, c);
      } else if (q.rnorm > q.maxr) {
        q.maxr = q.rnorm;
      }
    }
    if (upd.n > 0) {
      // reliable update: y += x (skipped if the iterate is corrupted), true residual in fp64
      ColMap good;
      good.n = 0;
      for (int i = 0; i < upd.n; i++) if (!broken[upd.col[i]]) cols_add(good, upd.col[i]);
      if (good.n > 0) LAUNCHK(TMW_K_ACC_Y, good.n, launch_acc_y<R>(n64, ctx->vh_loc, W[3], x, good, s));
      for (int i = 0; i < brk.n; i++) MEMSETK(colp(x, brk.col[i], bytesR), 0, bytesR);
      if ((rc = schur<double>(ctx, 0, W[3], W[6], W[5], upd))) return rc;
      for (int i = 0; i < upd.n; i++) {
        const int c = upd.col[i];
        h[c].rho[0] = h[c].rho[1] = 0.0;
        h[c].rr = 0.0;
        if (broken[c]) reset_recurrence(&h[c]);
      }
      if ((rc = push_scalars(ctx))) return rc;
      // r := true residual; the search direction update_xrp already built from the iterated r moves with it
      LAUNCHK(TMW_K_RESID_CONVERT, upd.n, launch_resid_convert<R>(n64, ctx->vh_loc, W[2], W[6], W[4], r, rhat, p, ctx->sc, upd, s));
      if ((rc = fetch_scalars(ctx))) return rc;
      for (int i = 0; i < upd.n; i++) {
        const int c = upd.col[i];
        ColState& q = cs[c];
        q.updates++;
        q.rnorm = q.maxr = q.r_upd = sqrt(h[c].rr);
        q.iter_resid = q.rnorm / q.bnorm;
        if (verbose) fprintf(stderr, "[tmw]   col %d reliable update %d: true |r|/|b| %.3e rho (%.3e,%.3e)\n", c, q.updates, q.rnorm / q.bnorm, h[c].rho[0], h[c].rho[1]);
        if (!isfinite(q.rnorm)) return fail(ctx, TMW_EBREAKDOWN, "tmw_solve: non-finite true residual");
        if (q.rnorm <= tol * q.bnorm) q.done = true;
        arm(c);
      }
      if ((rc = push_scalars(ctx))) return rc;
    }
    if (k >= max_iter) break;
    ColMap rst;  // breakdown: restart the recurrence with rhat = r (C11)
    rst.n = 0;
    for (int i = 0; i < act.n; i++) {
      const int c = act.col[i];
      if (cs[c].done) continue;
      const double rho_abs = hypot(h[c].rho[0], h[c].rho[1]);
      if (broken[c] || !(rho_abs > eps_break * cs[c].rhat_norm * cs[c].rnorm)) {  // (the device's TRIP_BREAKDOWN is this test on its own copy)
        if (verbose) fprintf(stderr, "[tmw]   col %d breakdown: |rho| %.3e vs %.3e * %.3e * %.3e -> restart\n", c, rho_abs, eps_break, cs[c].rhat_norm, cs[c].rnorm);
        cs[c].restarts++;
        cols_add(rst, c);
      }
    }
    if (rst.n > 0) {
      // fold the current iterate into y first so that r is the residual of y - unless the recurrence has wandered off
      // (corrupted, or its residual is above the one y already has): then the iterate is dropped
      ColMap keep;
      keep.n = 0;
      for (int i = 0; i < rst.n; i++) {
        const int c = rst.col[i];
        if (!broken[c] && cs[c].rnorm <= cs[c].r_upd) cols_add(keep, c);
        else MEMSETK(colp(x, c, bytesR), 0, bytesR);
      }
      if (keep.n > 0) LAUNCHK(TMW_K_ACC_Y, keep.n, launch_acc_y<R>(n64, ctx->vh_loc, W[3], x, keep, s));
      if ((rc = schur<double>(ctx, 0, W[3], W[6], W[5], rst))) return rc;
      for (int i = 0; i < rst.n; i++) {
        const int c = rst.col[i];
        memset(&h[c], 0, sizeof(Scalars));
        reset_recurrence(&h[c]);
      }
      if ((rc = push_scalars(ctx))) return rc;
      LAUNCHK(TMW_K_SUB_NORM, rst.n, launch_sub_norm(n64, W[2], W[6], W[4], ctx->red, rst, s));  // r64 = bhat - Mhat y (norm discarded)
      LAUNCHK(TMW_K_CONVERT, rst.n, launch_convert<R>(n64, ctx->vh_loc, W[4], rhat, rst, s));
      LAUNCHK(TMW_K_RESID_CONVERT, rst.n, launch_resid_convert<R>(n64, ctx->vh_loc, W[2], W[6], W[4], r, rhat, nullptr, ctx->sc, rst, s));
      for (int i = 0; i < rst.n; i++)  // p = r
        COPYK(colp(p, rst.col[i], bytesR), colp(r, rst.col[i], bytesR), bytesR);
      if ((rc = fetch_scalars(ctx))) return rc;
      for (int i = 0; i < rst.n; i++) {
        const int c = rst.col[i];
        ColState& q = cs[c];
        q.rnorm = q.maxr = q.rhat_norm = q.r_upd = sqrt(h[c].rr);
        q.iter_resid = q.rnorm / q.bnorm;
        q.updates++;
        if (verbose) fprintf(stderr, "[tmw]   col %d restart %d: true |r|/|b| %.3e\n", c, q.restarts, q.iter_resid);
        arm(c);
        if (q.rnorm <= tol * q.bnorm) { q.done = true; continue; }
        // restarts are cheap and a long solve may need many; give up only when they stop paying
        if (q.rnorm < 0.9 * q.best) { q.best = q.rnorm; q.stalled = 0; }
        else if (++q.stalled > 5) return fail(ctx, TMW_EBREAKDOWN, "tmw_solve: BiCGStab breakdown: no progress over 5 consecutive restarts");
      }
      if ((rc = push_scalars(ctx))) return rc;
    }
  }
  for (int c = 0; c < ncols; c++)
    if (!cs[c].done) return fail(ctx, TMW_ENOCONV, "tmw_solve: max_iter reached");
  return TMW_OK;
}


// Restarted GCR(k) (the paper's GPU solver) on the Schur systems of the columns c with
// !cs[c].done, inner precision R, restarted from the fp64 true residual (the same reliable update as in solve_schur). The
// columns run in lockstep like BiCGStab's: per step one Mhat application (K1, K2) over the columns still stepping, so that
// links and clover blocks are read once for all of them, and the five launches of launch_gcr_step; a column leaves the
// steps of a cycle when it has converged or its residual has dropped by delta, and all columns of the cycle restart together.
//   w64 as in solve_schur; w32: 0 r, 1 zero (the rhat slot of resid_convert), 6 x, 7 tmp_e
//   gcr_q, gcr_p: nkrylov x ws_cols inner-precision spinors, vector j of column c at (j * ws_cols + c)
template <typename R>
int solve_gcr(tmw_ctx* ctx, int ncols, double tol, ColState* cs) {
  cudaStream_t s = ctx->stream;
  const int64_t n64 = (int64_t)ctx->g.Vh * 12;
  const int64_t nR = (int64_t)ctx->g.Vh * 24 * (int64_t)sizeof(R) / 16;
  const size_t bytesR = (size_t)nR * 16, bytes64 = (size_t)n64 * 16;
  const int k = ctx->opt.nkrylov, ncw = ctx->ws_cols;
  void** W = ctx->w64;
  void** X = ctx->w32;
  int rc;
  if (!ctx->gcr_q) { if ((rc = ws_alloc(ctx, &ctx->gcr_q, bytesR * k * ncw))) return rc; }
  if (!ctx->gcr_p) { if ((rc = ws_alloc(ctx, &ctx->gcr_p, bytesR * k * ncw))) return rc; }
  void *r = X[0], *x = X[6], *tmp = X[7];
  Scalars* h = ctx->sc_host;
  GcrScalars* gh = ctx->gs_host;
  const bool verbose = ctx->verbose;
  const int max_iter = ctx->opt.max_iter;
  bool given_up[MAXCOL] = {false};  // max_iter reached
  for (int c = 0; c < ncols; c++) {
    if (cs[c].done) continue;
    CK(cudaMemsetAsync(colp(W[3], c, bytes64), 0, bytes64, s));
    CK(cudaMemsetAsync(colp(W[6], c, bytes64), 0, bytes64, s));
    CK(cudaMemsetAsync(colp(X[1], c, bytesR), 0, bytesR, s));
  }
  for (;;) {
    ColMap cyc;  // the columns of this cycle
    cyc.n = 0;
    for (int c = 0; c < ncols; c++) if (!cs[c].done && !given_up[c]) cols_add(cyc, c);
    if (cyc.n == 0) break;
    // true residuals r64 = bhat - Mhat y (W[6] holds Mhat y), r = (R) r64, |r64|^2
    memset(h, 0, MAXCOL * sizeof(Scalars));
    if ((rc = push_scalars(ctx))) return rc;
    LAUNCHK(TMW_K_RESID_CONVERT, cyc.n, launch_resid_convert<R>(n64, ctx->vh_loc, W[2], W[6], W[4], r, X[1], nullptr, ctx->sc, cyc, s));
    if ((rc = fetch_scalars(ctx))) return rc;
    ColMap step;  // the columns still stepping
    step.n = 0;
    for (int i = 0; i < cyc.n; i++) {
      const int c = cyc.col[i];
      ColState& q = cs[c];
      q.rnorm = q.maxr = sqrt(h[c].rr);
      q.iter_resid = q.rnorm / q.bnorm;
      if (verbose) fprintf(stderr, "[tmw] gcr col %d cycle %d it %d true |r|/|b| %.3e\n", c, q.updates, q.iters, q.iter_resid);
      if (!isfinite(q.rnorm)) return fail(ctx, TMW_EBREAKDOWN, "tmw_solve: non-finite true residual");
      if (q.rnorm <= tol * q.bnorm) q.done = true;
      else if (q.iters >= max_iter) given_up[c] = true;
      else cols_add(step, c);
    }
    if (step.n == 0) continue;
    cyc = step;
    for (int i = 0; i < cyc.n; i++) CK(cudaMemsetAsync(colp(x, cyc.col[i], bytesR), 0, bytesR, s));
    CK(cudaMemsetAsync(ctx->gs, 0, MAXCOL * sizeof(GcrScalars), s));
    for (int i = 0; i < k && step.n > 0; i++) {
      // q_i = Mhat r (orthogonalised in launch_gcr_step), p_i = r - ...
      if ((rc = schur<R>(ctx, 0, r, (char*)ctx->gcr_q + (size_t)i * ncw * bytesR, tmp, step))) return rc;
      LAUNCH(launch_gcr_step<R>(nR, i, ncw, ctx->gcr_q, ctx->gcr_p, x, r, ctx->gs, step, s));
      ctx->launches += (i > 0) ? 4 : 3;  // launch_gcr_step is 5 launches (4 for the first vector)
      CK(cudaMemcpyAsync(gh, ctx->gs, MAXCOL * sizeof(GcrScalars), cudaMemcpyDeviceToHost, s));
      CK(cudaStreamSynchronize(s));
      ColMap next;
      next.n = 0;
      for (int j = 0; j < step.n; j++) {
        const int c = step.col[j];
        ColState& q = cs[c];
        q.iters++;
        if (!isfinite(gh[c].rr) || !(gh[c].nw > 0.0)) return fail(ctx, TMW_EBREAKDOWN, "tmw_solve: GCR breakdown (Mhat p vanished or non-finite)");
        const double rn = sqrt(gh[c].rr);
        q.iter_resid = rn / q.bnorm;
        if (verbose) fprintf(stderr, "[tmw] gcr col %d it %d |r|/|b| %.3e\n", c, q.iters, q.iter_resid);
        if (!(rn <= tol * q.bnorm || rn < ctx->opt.delta * q.maxr || q.iters >= max_iter)) cols_add(next, c);
      }
      step = next;
    }
    // restart: y += x, Mhat y in fp64
    LAUNCHK(TMW_K_ACC_Y, cyc.n, launch_acc_y<R>(n64, ctx->vh_loc, W[3], x, cyc, s));
    if ((rc = schur<double>(ctx, 0, W[3], W[6], W[5], cyc))) return rc;
    for (int i = 0; i < cyc.n; i++) cs[cyc.col[i]].updates++;
  }
  for (int c = 0; c < ncols; c++)
    if (given_up[c]) return fail(ctx, TMW_ENOCONV, "tmw_solve: max_iter reached");
  return TMW_OK;
}

}  // namespace

// The columns of cm: from the packed fp64 source W[0] (even), W[1] (odd) to the packed solution W[7] (even), W[3] (odd).
//   A7: bhat_o = b_o - H_oe A_ee^{-1} b_e;  Krylov iterations on Mhat y = bhat_o;  x_o = y, x_e = A_ee^{-1} (b_e - H_eo x_o)
// cs[c].done marks the columns that are NOT to be iterated (already solved, or b = 0). Returns TMW_OK or TMW_ENOCONV.
static int solve_packed(tmw_ctx* ctx, int nrhs, const ColMap& cm, double tol, ColState* cs) {
  const bool dbl = ctx->opt.precision == TMW_DOUBLE;
  cudaStream_t s = ctx->stream;
  void** W = ctx->w64;
  const size_t b64 = spinor_bytes(ctx, TMW_F64);
  int rc, status = TMW_OK;
  for (int i = 0; i < cm.n; i++)
    if ((rc = diag64(ctx, 0, 1, colp(W[0], cm.col[i], b64), colp(W[5], cm.col[i], b64)))) return rc;
  if ((rc = dslash<double>(ctx, EPI_XPAY, 1, 0, W[5], W[2], W[1], -1.0, cm))) return rc;
  {
    NvtxRange nvtx_it("tmw_solve: Krylov iterations");
    if (ctx->opt.solver == TMW_GCR) {
      status = dbl ? solve_gcr<double>(ctx, nrhs, tol, cs) : solve_gcr<float>(ctx, nrhs, tol, cs);
    } else {
      status = dbl ? solve_schur<double>(ctx, nrhs, tol, cs) : solve_schur<float>(ctx, nrhs, tol, cs);
    }
  }
  if (status != TMW_OK && status != TMW_ENOCONV) return status;
  if ((rc = dslash<double>(ctx, EPI_AINV_XPAY, 0, 0, W[3], W[7], W[0], -1.0, cm))) return rc;
  return status;
}

// |b - D x| / |b| of the full system in fp64 for the columns of cm (b in W[0], W[1]; x in W[7], W[3]): the difference and
// its norm are fused into the two launches of the full operator. With store_e/store_o the products D x themselves are
// written there (both parities) instead.
static int full_residual(tmw_ctx* ctx, const ColMap& cm, ColState* cs) {
  void** W = ctx->w64;
  int rc;
  CK(cudaMemsetAsync(ctx->red, 0, 4 * MAXCOL * sizeof(double), ctx->stream));
  if ((rc = dslash<double>(ctx, EPI_A_XPAY, 0, 0, W[3], nullptr, W[7], 1.0, cm, 3, W[0], ctx->red, 4))) return rc;
  if ((rc = dslash<double>(ctx, EPI_A_XPAY, 1, 0, W[7], nullptr, W[3], 1.0, cm, 3, W[1], ctx->red, 4))) return rc;
  if ((rc = fetch_red(ctx))) return rc;
  for (int i = 0; i < cm.n; i++) cs[cm.col[i]].true_resid = sqrt(ctx->red_host[4 * cm.col[i] + 2]) / cs[cm.col[i]].bnorm;
  return TMW_OK;
}

// nrhs columns that are known to fit in the workspaces (tmw_solve_multi below splits a call into such chunks)
static int solve_chunk(tmw_ctx* ctx, int nrhs, const double* b, double* x, double tol, tmw_solve_info* info) {
  const bool dbl = ctx->opt.precision == TMW_DOUBLE;
  int rc;
  if ((rc = need_cols(ctx, nrhs))) return rc;
  if ((rc = need_w64(ctx, 8))) return rc;
  if ((rc = need_w32(ctx, 8, dbl ? TMW_F64 : TMW_F32))) return rc;
  cudaStream_t s = ctx->stream;
  const size_t cbytes = (size_t)ctx->V * 24 * 8, b64 = spinor_bytes(ctx, TMW_F64);
  const double* cb = b;
  double* cx_ = x;
  if (ctx->opt.location == TMW_HOST) {
    if ((rc = need_canon(ctx))) return rc;
    cb = (const double*)ctx->canon[0];
    cx_ = (double*)ctx->canon[1];
  }
  CK(cudaEventRecord(ctx->ev0, s));
  if (ctx->opt.location == TMW_HOST) CK(cudaMemcpyAsync(ctx->canon[0], b, cbytes * nrhs, cudaMemcpyHostToDevice, s));
  void** W = ctx->w64;
  const int64_t n64 = (int64_t)ctx->g.Vh * 12;
  ColState cs[MAXCOL];
  memset(cs, 0, sizeof(cs));
  const ColMap all = cols_first(nrhs);
  // A0: split b into parities, |b|
  for (int c = 0; c < nrhs; c++) {
    if ((rc = pack_both(ctx, 1, (const double*)colp(cb, c, cbytes), colp(W[0], c, b64), colp(W[1], c, b64)))) return rc;
  }
  CK(cudaMemsetAsync(ctx->red, 0, 4 * MAXCOL * sizeof(double), s));
  LAUNCHK(TMW_K_DOT_NORM64, all.n, launch_dot_norm<double>(n64, nullptr, W[0], ctx->red, all, s));
  LAUNCHK(TMW_K_DOT_NORM64, all.n, launch_dot_norm<double>(n64, nullptr, W[1], ctx->red, all, s));
  if ((rc = fetch_red(ctx))) return rc;
  ColMap nz;  // columns with b != 0
  nz.n = 0;
  for (int c = 0; c < nrhs; c++) {
    cs[c].bnorm = sqrt(ctx->red_host[4 * c + 2]);
    if (!isfinite(cs[c].bnorm)) return fail(ctx, TMW_EINVAL, "tmw_solve: b has non-finite entries");
    if (cs[c].bnorm == 0.0) {
      cs[c].done = true;
      CK(cudaMemsetAsync(colp(cx_, c, cbytes), 0, cbytes, s));
    } else {
      cols_add(nz, c);
    }
  }
  int status = TMW_OK;
  if (nz.n > 0) {
    status = solve_packed(ctx, nrhs, nz, tol, cs);
    if (status != TMW_OK && status != TMW_ENOCONV) return status;
    if ((rc = full_residual(ctx, nz, cs))) return rc;
    // The stopping rule of include/tmw.h is the residual of the FULL system, but the iteration is stopped on the odd-site
    // Schur residual; the two agree only as far as the fp64 A_ee^{-1} is well conditioned (with near-singular clover
    // blocks the even-site defect grows as cond(A_ee) * eps). Columns that converged on the Schur system but whose full
    // residual is above tol get fp64 defect correction: solve D e = b - D x the same way, x += e (at most twice).
    for (int round = 0; round < 2 && status == TMW_OK; round++) {
      ColMap bad;
      bad.n = 0;
      for (int i = 0; i < nz.n; i++) {
        const int c = nz.col[i];
        const bool forced = round == 0 && (ctx->opt.debug & TMW_DEBUG_FORCE_DEFECT) && (c & 1);  // test hook: a strict subset
        if (!(cs[c].true_resid <= tol) || forced) cols_add(bad, c);
      }
      if (bad.n == 0) break;
      if (ctx->verbose) fprintf(stderr, "[tmw] defect correction %d for %d column(s): full residual %.3e > tol\n", round + 1, bad.n, cs[bad.col[0]].true_resid);
      if ((rc = need_w64(ctx, NW64))) return rc;
      int it0[MAXCOL], up0[MAXCOL];
      for (int i = 0; i < bad.n; i++) {
        const int c = bad.col[i];
        CK(cudaMemcpyAsync(colp(W[10], c, b64), colp(W[0], c, b64), b64, cudaMemcpyDeviceToDevice, s));  // b
        CK(cudaMemcpyAsync(colp(W[11], c, b64), colp(W[1], c, b64), b64, cudaMemcpyDeviceToDevice, s));
        CK(cudaMemcpyAsync(colp(W[12], c, b64), colp(W[7], c, b64), b64, cudaMemcpyDeviceToDevice, s));  // x
        CK(cudaMemcpyAsync(colp(W[13], c, b64), colp(W[3], c, b64), b64, cudaMemcpyDeviceToDevice, s));
        it0[c] = cs[c].iters;
        up0[c] = cs[c].updates;
      }
      if ((rc = full_apply64(ctx, 0, W[7], W[3], W[8], W[9], bad))) return rc;        // D x
      LAUNCHK(TMW_K_SUB_NORM, bad.n, launch_sub_norm(n64, W[10], W[8], W[0], ctx->red, bad, s));              // b := b - D x (norm discarded)
      LAUNCHK(TMW_K_SUB_NORM, bad.n, launch_sub_norm(n64, W[11], W[9], W[1], ctx->red, bad, s));
      for (int c = 0; c < nrhs; c++) cs[c].done = true;
      for (int i = 0; i < bad.n; i++) cs[bad.col[i]].done = false;
      status = solve_packed(ctx, nrhs, bad, tol, cs);                                 // e, to the same absolute target tol |b|
      if (status != TMW_OK && status != TMW_ENOCONV) return status;
      LAUNCHK(TMW_K_SUB_NORM, bad.n, launch_add64(n64, W[7], W[12], bad, s));                                 // x = x + e
      LAUNCHK(TMW_K_SUB_NORM, bad.n, launch_add64(n64, W[3], W[13], bad, s));
      for (int i = 0; i < bad.n; i++) {
        const int c = bad.col[i];
        CK(cudaMemcpyAsync(colp(W[0], c, b64), colp(W[10], c, b64), b64, cudaMemcpyDeviceToDevice, s));
        CK(cudaMemcpyAsync(colp(W[1], c, b64), colp(W[11], c, b64), b64, cudaMemcpyDeviceToDevice, s));
        cs[c].iters += it0[c];
        cs[c].updates += up0[c];
      }
      if ((rc = full_residual(ctx, bad, cs))) return rc;
    }
    for (int i = 0; i < nz.n; i++) {
      const int c = nz.col[i];
      if ((rc = unpack_both(ctx, 1, colp(W[7], c, b64), colp(W[3], c, b64), (double*)colp(cx_, c, cbytes)))) return rc;
      if (status == TMW_OK && !(cs[c].true_resid <= tol)) {
        status = TMW_ENOCONV;
        fail(ctx, TMW_ENOCONV, "tmw_solve: the Schur system converged but the full-lattice residual stays above tol (ill-conditioned A_ee)");
      }
    }
  }
  if (ctx->opt.location == TMW_HOST) CK(cudaMemcpyAsync(x, cx_, cbytes * nrhs, cudaMemcpyDeviceToHost, s));
  CK(cudaEventRecord(ctx->ev1, s));
  CK(cudaStreamSynchronize(s));
  float ms = 0;
  CK(cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
  if (info) {
    for (int c = 0; c < nrhs; c++) {
      info[c].iters = cs[c].iters;
      info[c].reliable_updates = cs[c].updates;
      info[c].restarts = cs[c].restarts;
      info[c].iter_resid = cs[c].iter_resid;
      info[c].true_resid = cs[c].true_resid;
      info[c].device_ms = ms;
    }
  }
  return status;
}

extern "C" int tmw_solve_multi(tmw_ctx* ctx, int nrhs, const double* b, double* x, double tol, tmw_solve_info* info) {
  NvtxRange nvtx("tmw_solve");
  if (!ctx) return TMW_EINVAL;
  if (!b || !x || b == x) return fail(ctx, TMW_EINVAL, "tmw_solve: null or aliased pointers");
  if (!(tol > 0.0) || !isfinite(tol)) return fail(ctx, TMW_EINVAL, "tmw_solve: tol must be > 0");
  if (nrhs < 1 || nrhs > MAXCOL) return fail(ctx, TMW_EINVAL, "tmw_solve: nrhs must be in 1..16");
  if (info) memset(info, 0, sizeof(*info) * nrhs);
  // How many columns fit at once: 8 fp64 + 8 inner-precision parity spinors per column (+ 2 canonical staging spinors
  // for HOST pointers) out of the free device memory plus what the workspaces already hold. More columns than that are
  // solved chunk after chunk (as even as possible); TMW_DEBUG_NO_CHUNK disables the split (the call then fails with
  // TMW_ENOMEM if the columns do not fit).
  int chunk = nrhs;
  if (nrhs > 1 && !(ctx->opt.debug & TMW_DEBUG_NO_CHUNK)) {
    const size_t b64 = spinor_bytes(ctx, TMW_F64), bin = spinor_bytes(ctx, ctx->opt.precision == TMW_DOUBLE ? TMW_F64 : TMW_F32);
    const size_t cbytes = (size_t)ctx->V * 24 * 8;
    // GCR: 2 nkrylov Krylov vectors per column on top (the columns step together)
    const size_t gcr = ctx->opt.solver == TMW_GCR ? 2 * (size_t)ctx->opt.nkrylov * bin : 0;
    // decomposed contexts: one more fp64 parity spinor per column for the reduction-only launches of the final residual (dd_tmp)
    const size_t per_col = 8 * b64 + 8 * bin + gcr + (ctx->opt.location == TMW_HOST ? 2 * cbytes : 0) + (ctx->dom.empty() ? 0 : b64);
    size_t held = 0;
    for (int i = 0; i < NW64; i++) if (ctx->w64[i]) held += b64 * ctx->ws_cols;
    for (int i = 0; i < 8; i++) if (ctx->w32[i]) held += bin * ctx->ws_cols;
    for (int i = 0; i < 2; i++) if (ctx->canon[i]) held += cbytes * ctx->ws_cols;
    size_t free_b = 0, total_b = 0;
    CK(cudaMemGetInfo(&free_b, &total_b));
    if (ctx->gcr_q) held += gcr * ctx->ws_cols;
    const double avail = 0.92 * (double)(free_b + held);
    const size_t fit = avail > 0 ? (size_t)avail / per_col : 0;
    if (fit < (size_t)nrhs && ctx->ws_cols < nrhs) {
      chunk = fit < 1 ? 1 : (int)fit;
      if (chunk < ctx->ws_cols) chunk = ctx->ws_cols;  // what is already allocated fits by construction
      const int nchunks = (nrhs + chunk - 1) / chunk;
      chunk = (nrhs + nchunks - 1) / nchunks;
    }
  }
  int status = TMW_OK;
  const size_t cdoubles = (size_t)ctx->V * 24;
  for (int c0 = 0; c0 < nrhs; c0 += chunk) {
    const int n = nrhs - c0 < chunk ? nrhs - c0 : chunk;
    int rc = solve_chunk(ctx, n, b + c0 * cdoubles, x + c0 * cdoubles, tol, info ? info + c0 : nullptr);
    if (rc == TMW_EBREAKDOWN && ctx->opt.precision == TMW_MIXED && ctx->opt.solver == TMW_BICGSTAB) {
      // the fp32 recurrence stalled (near-critical system): redo the chunk with fp64 recurrences, which hold out longer
      CK(cudaStreamSynchronize(ctx->stream));
      for (int i = 0; i < 8; i++) if (ctx->w32[i]) { dev_free(ctx, ctx->w32[i]); ctx->w32[i] = nullptr; }
      ctx->opt.precision = TMW_DOUBLE;
      rc = solve_chunk(ctx, n, b + c0 * cdoubles, x + c0 * cdoubles, tol, info ? info + c0 : nullptr);
      ctx->opt.precision = TMW_MIXED;
      cudaStreamSynchronize(ctx->stream);
      for (int i = 0; i < 8; i++) if (ctx->w32[i]) { dev_free(ctx, ctx->w32[i]); ctx->w32[i] = nullptr; }
    }
    if (rc != TMW_OK && rc != TMW_ENOCONV) return rc;
    if (rc == TMW_ENOCONV) status = rc;
  }
  return status;
}

extern "C" int tmw_solve(tmw_ctx* ctx, const double* b, double* x, double tol, tmw_solve_info* info) {
  return tmw_solve_multi(ctx, 1, b, x, tol, info);
}

extern "C" int tmw_time_kernel(tmw_ctx* ctx, int kind, int reps, double* ms) {
  if (!ctx) return TMW_EINVAL;
  if (!ms || reps < 1) return fail(ctx, TMW_EINVAL, "tmw_time_kernel: bad argument");
  if (ctx->opt.precision != TMW_MIXED || !ctx->dom.empty()) return fail(ctx, TMW_EINVAL, "tmw_time_kernel: needs a TMW_MIXED context without domain decomposition");
  if ((kind == TMW_K_FFMA_PROBE || kind == TMW_K_FFMA2_PROBE) && spinor_bytes(ctx, TMW_F32) < (size_t)ctx->sms * 8 * 256 * 4)
    return fail(ctx, TMW_EINVAL, "tmw_time_kernel: the lattice is too small to hold the probe's output");
  int rc;
  if ((rc = need_w64(ctx, 8))) return rc;
  if ((rc = need_w32(ctx, 8, TMW_F32))) return rc;
  void** W = ctx->w64;
  void** X = ctx->w32;
  const ColMap one = cols_first(1);
  const int64_t nR = (int64_t)ctx->g.Vh * 24 * 4 / 16;
  const int SCD = (int)(sizeof(Scalars) / sizeof(double));
  double* red_rhat_v = (double*)((char*)ctx->sc + offsetof(Scalars, rhat_v));
  double* red_ts = (double*)((char*)ctx->sc + offsetof(Scalars, ts));
  long long saved[TMW_K_COUNT];
  memcpy(saved, ctx->kcount, sizeof(saved));
  const long long launches0 = ctx->launches;
  auto run = [&]() -> int {
    switch (kind) {
      case TMW_K_HOP32: return dslash<float>(ctx, EPI_HOP, 1, 0, X[7], X[3], nullptr, 1.0, one);
      case TMW_K_K1_32: return dslash<float>(ctx, EPI_AINV_HOP, 0, 0, X[2], X[7], nullptr, 1.0, one);
      case TMW_K_K2_32: return dslash<float>(ctx, EPI_A_XPAY, 1, 0, X[7], X[3], X[2], -1.0, one, 1, X[1], red_rhat_v, SCD);
      case TMW_K_K2_32_DOTS: return dslash<float>(ctx, EPI_A_XPAY, 1, 0, X[7], X[5], X[4], -1.0, one, 4, X[1], red_ts, SCD);
      case TMW_K_K1_64: return dslash<double>(ctx, EPI_AINV_HOP, 0, 0, W[3], W[5], nullptr, 1.0, one);
      case TMW_K_K2_64: return dslash<double>(ctx, EPI_A_XPAY, 1, 0, W[5], W[6], W[3], -1.0, one);
      case TMW_K_UPDATE_S: LAUNCH(launch_update_s<float>(nR, X[4], X[0], X[3], ctx->sc, one, nullptr, ctx->stream)); return TMW_OK;
      case TMW_K_UPDATE_XRP: LAUNCH(launch_update_xrp<float>(nR, X[6], X[0], X[2], X[4], X[5], X[3], ctx->sc, one, nullptr, ctx->stream)); return TMW_OK;
      case TMW_K_FFMA_PROBE:
      case TMW_K_FFMA2_PROBE: LAUNCH(launch_ffma_probe(kind == TMW_K_FFMA2_PROBE, TMW_FFMA_PROBE_FMAS_PER_THREAD, ctx->sms, (float*)X[7], ctx->stream)); return TMW_OK;
      case TMW_K_HOP32_LOADONLY: {
        DslashArgs<float> a = make_args<float>(ctx, 1, 0, X[7], X[3], nullptr, 1.0, one);
        LAUNCH(launch_hop_loadonly(a, ctx->ng32, ctx->stream));
        return TMW_OK;
      }
    }
    return fail(ctx, TMW_EINVAL, "tmw_time_kernel: this kind cannot be timed alone");
  };
  for (int i = 0; i < 3; i++) if ((rc = run())) return rc;
  CK(cudaEventRecord(ctx->ev0, ctx->stream));
  for (int i = 0; i < reps; i++) if ((rc = run())) return rc;
  CK(cudaEventRecord(ctx->ev1, ctx->stream));
  CK(cudaStreamSynchronize(ctx->stream));
  float t = 0;
  CK(cudaEventElapsedTime(&t, ctx->ev0, ctx->ev1));
  *ms = (double)t / reps;
  memcpy(ctx->kcount, saved, sizeof(saved));  // probing does not count as work of the path
  ctx->launches = launches0;
  return TMW_OK;
}
