/*
 * tmw_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct fp64 CPU implementation of what the hot path computes: the twisted-mass
 * Wilson(-clover) Dirac operator of arXiv:2201.09004 Eqs. (1)-(3) and a full-lattice
 * BiCGStab (the solver named in PAPER.md:73, Table 2 row 1). Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this. It shares no code, header, table or helper with
 * the CUDA library under paper_2201_09004_b200/csrc/, and never includes or links it.
 *
 * Written naively on purpose: lexicographic array-of-structures, explicit 4x4 gamma matrices applied to full
 * 4-spinors (no spin-projection trick), full 3x3 links (no 12-real reconstruction), no even-odd checkerboarding,
 * no blocking or fusion. OpenMP only splits the outermost site loop.
 *
 * Definition implemented (readings C1-C8; lattice units a = 1, C18):
 *
 *   (D psi)(x) = 1/2 sum_mu [ (1+g_mu) U_mu(x)        psi(x+mu) s+_mu(x)
 *                           + (1-g_mu) U_mu(x-mu)^dag psi(x-mu) s-_mu(x) ]        PAPER.md:62 Eq. 2, hopping part (C1, C3)
 *                - (4 + Re m) psi(x) - i (Im m) g5 psi(x)                          PAPER.md:62 "-(4+m) delta_xy", reading C4
 *                + (c_sw/2) sum_{mu<nu} sigma_mu_nu F_mu_nu(x) psi(x)              PAPER.md:67 Eq. 3, reading C7
 *
 *   s+-_mu(x) = -1 when mu = t and the hop wraps around the lattice (antiperiodic in time, C6), else +1;
 *   x, y, z periodic. m = m_cri + omega is complex. mass_reading = 1 selects the literal
 *   alternative -(4+m)*1 with a complex scalar (C4, TMW_MASS_SCALAR).
 *   gamma matrices: DeGrand-Rossi basis (C5; the only basis the paper mentions).
 *   sigma_mu_nu = (i/2)[g_mu, g_nu];  F_mu_nu = (Q_mu_nu - Q_mu_nu^dag)/(8i) with Q the sum of the four plaquette
 *   leaves around x in the (mu,nu) plane, no trace subtraction, gauge links periodic in all four directions (C7).
 *   D^dag is the conjugate transpose, written out from the definition (see site_apply).
 *
 * PINS (tests/test_oracle_*.py, run with -m "not gpu"): free-field and constant-abelian-background closed-form
 * spectra; gamma5-hermiticity; adjoint dot test and dense conjugate transpose on 2^4; twisted-mass identity
 * |D(m)psi|^2 = |D(Re m)psi|^2 + (Im m)^2|psi|^2; gauge covariance incl. clover; F = 0 on unit / pure-gauge
 * fields; uniform abelian flux F_xy = sin(B) T3; dense LU solve on 2^4 and 4^4; free propagator by Fourier sum.
 * The sign and prefactor of the clover term of Eq. 3 relative to the hopping term of Eq. 2 (the paper prints no number
 * and Eq. 3 is schematic) are pinned by what the term is for, "O(a) improvement": in a uniform abelian
 * field the Wilson term lifts the would-be zero modes to B/2 and the clover term at c_sw = 1 must cancel that lift
 * (test_clover_sign_is_the_improving_one: sigma_min = B/2 at c_sw = 0, O(B^2) at +1, B at -1), on a fully periodic
 * lattice (antiperiodic_t = 0). No function of this file is "parity unpinned".
 *
 * Layouts (canonical, fp64, x fastest; same as include/tmw.h):
 *   gauge  [mu=0..3 (x,y,z,t)][t][z][y][x][row][col] complex   U_mu(x)_{row,col}
 *   spinor [t][z][y][x][spin][colour] complex
 *   F      [site][plane 0..5 = (xy,xz,xt,yz,yt,zt)][row][col] complex
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

/* ---- gamma matrices, DeGrand-Rossi basis, GAMMA[mu][row][col], mu = x,y,z,t ---- */
static const cplx GAMMA[4][4][4] = {
    /* g_x */ {{0, 0, 0, I}, {0, 0, I, 0}, {0, -I, 0, 0}, {-I, 0, 0, 0}},
    /* g_y */ {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    /* g_z */ {{0, 0, I, 0}, {0, 0, 0, -I}, {-I, 0, 0, 0}, {0, I, 0, 0}},
    /* g_t */ {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}},
};

static void mat4_mul(const cplx a[4][4], const cplx b[4][4], cplx c[4][4]) {
  for (int i = 0; i < 4; i++)
    for (int j = 0; j < 4; j++) {
      cplx s = 0;
      for (int k = 0; k < 4; k++) s += a[i][k] * b[k][j];
      c[i][j] = s;
    }
}

/* g5 = g_x g_y g_z g_t */
static void gamma5(cplx g5[4][4]) {
  cplx a[4][4], b[4][4];
  mat4_mul(GAMMA[0], GAMMA[1], a);
  mat4_mul(a, GAMMA[2], b);
  mat4_mul(b, GAMMA[3], g5);
}

/* sigma_mu_nu = (i/2) (g_mu g_nu - g_nu g_mu) */
static void sigma_munu(int mu, int nu, cplx s[4][4]) {
  cplx a[4][4], b[4][4];
  mat4_mul(GAMMA[mu], GAMMA[nu], a);
  mat4_mul(GAMMA[nu], GAMMA[mu], b);
  for (int i = 0; i < 4; i++)
    for (int j = 0; j < 4; j++) s[i][j] = 0.5 * I * (a[i][j] - b[i][j]);
}

/* exported for the tests: mu = 0..3 -> g_mu, mu = 4 -> g5; out[4][4] complex */
void orc_gamma(int mu, double* out) {
  cplx g[4][4];
  if (mu == 4) gamma5(g);
  else memcpy(g, GAMMA[mu], sizeof(g));
  memcpy(out, g, sizeof(g));
}
void orc_sigma(int mu, int nu, double* out) {
  cplx s[4][4];
  sigma_munu(mu, nu, s);
  memcpy(out, s, sizeof(s));
}

/* ---- lattice geometry ---- */
typedef struct {
  int L, T;
  int64_t V;
} lat_t;

static inline int64_t site_index(const lat_t* g, const int c[4]) {
  return c[0] + (int64_t)g->L * (c[1] + (int64_t)g->L * (c[2] + (int64_t)g->L * c[3]));
}
static inline void site_coords(const lat_t* g, int64_t s, int c[4]) {
  c[0] = (int)(s % g->L); s /= g->L;
  c[1] = (int)(s % g->L); s /= g->L;
  c[2] = (int)(s % g->L); s /= g->L;
  c[3] = (int)s;
}
static inline int extent(const lat_t* g, int mu) { return mu == 3 ? g->T : g->L; }

/* neighbour of c in direction mu by step d (+1/-1), periodic; *wrapped = 1 if the hop crossed the boundary */
static inline int64_t neighbour(const lat_t* g, const int c[4], int mu, int d, int* wrapped) {
  int n[4] = {c[0], c[1], c[2], c[3]};
  int e = extent(g, mu);
  n[mu] += d;
  *wrapped = 0;
  if (n[mu] >= e) { n[mu] -= e; *wrapped = 1; }
  if (n[mu] < 0) { n[mu] += e; *wrapped = 1; }
  return site_index(g, n);
}

static inline const cplx* link(const lat_t* g, const cplx* U, int mu, int64_t s) { return U + 9 * ((int64_t)mu * g->V + s); }

/* ---- 3x3 helpers ---- */
static void m3_mul(const cplx* a, const cplx* b, cplx* c) { /* c = a b */
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      cplx s = 0;
      for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
      c[3 * i + j] = s;
    }
}
static void m3_dag(const cplx* a, cplx* c) {
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) c[3 * i + j] = conj(a[3 * j + i]);
}
/* out = a b c d for four 3x3 matrices */
static void m3_mul4(const cplx* a, const cplx* b, const cplx* c, const cplx* d, cplx* out) {
  cplx t1[9], t2[9];
  m3_mul(a, b, t1);
  m3_mul(t1, c, t2);
  m3_mul(t2, d, out);
}

/* ---- clover field strength, SURVEY.md §8(c) C7 ----
 * Q_mu_nu(x) =  U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
 *             + U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
 *             + U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
 *             + U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
 * F_mu_nu = (Q - Q^dag) / (8i).  Gauge-link geometry is periodic in all directions.
 */
static void field_strength_site(const lat_t* g, const cplx* U, int64_t s, cplx F[6][9]) {
  int c[4], w;
  site_coords(g, s, c);
  int plane = 0;
  for (int mu = 0; mu < 4; mu++)
    for (int nu = mu + 1; nu < 4; nu++, plane++) {
      int cp[4], cm[4];
      int64_t x = s;
      int64_t xpm = neighbour(g, c, mu, +1, &w);  /* x+mu */
      int64_t xpn = neighbour(g, c, nu, +1, &w);  /* x+nu */
      int64_t xmm = neighbour(g, c, mu, -1, &w);  /* x-mu */
      int64_t xmn = neighbour(g, c, nu, -1, &w);  /* x-nu */
      site_coords(g, xmm, cm);
      site_coords(g, xpm, cp);
      int64_t xmm_pn = neighbour(g, cm, nu, +1, &w); /* x-mu+nu */
      int64_t xmm_mn = neighbour(g, cm, nu, -1, &w); /* x-mu-nu */
      int64_t xpm_mn = neighbour(g, cp, nu, -1, &w); /* x+mu-nu */
      cplx d1[9], d2[9], leaf[9], Q[9];
      memset(Q, 0, sizeof(Q));
      /* leaf 1 */
      m3_dag(link(g, U, mu, xpn), d1);
      m3_dag(link(g, U, nu, x), d2);
      m3_mul4(link(g, U, mu, x), link(g, U, nu, xpm), d1, d2, leaf);
      for (int i = 0; i < 9; i++) Q[i] += leaf[i];
      /* leaf 2 */
      m3_dag(link(g, U, mu, xmm_pn), d1);
      m3_dag(link(g, U, nu, xmm), d2);
      m3_mul4(link(g, U, nu, x), d1, d2, link(g, U, mu, xmm), leaf);
      for (int i = 0; i < 9; i++) Q[i] += leaf[i];
      /* leaf 3 */
      m3_dag(link(g, U, mu, xmm), d1);
      m3_dag(link(g, U, nu, xmm_mn), d2);
      m3_mul4(d1, d2, link(g, U, mu, xmm_mn), link(g, U, nu, xmn), leaf);
      for (int i = 0; i < 9; i++) Q[i] += leaf[i];
      /* leaf 4 */
      m3_dag(link(g, U, nu, xmn), d1);
      m3_dag(link(g, U, mu, x), d2);
      m3_mul4(d1, link(g, U, mu, xmn), link(g, U, nu, xpm_mn), d2, leaf);
      for (int i = 0; i < 9; i++) Q[i] += leaf[i];
      for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) F[plane][3 * i + j] = (Q[3 * i + j] - conj(Q[3 * j + i])) / (8.0 * I);
    }
}

/* F for all sites: out[V][6][3][3] complex */
void orc_field_strength(int L, int T, const double* gauge, double* out) {
  lat_t g = {L, T, (int64_t)L * L * L * T};
  const cplx* U = (const cplx*)gauge;
  cplx* F = (cplx*)out;
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < g.V; s++) field_strength_site(&g, U, s, (cplx(*)[9])(F + 54 * s));
}

/* ---- the operator at one site ---- */
typedef struct {
  double m_re, m_im, c_sw;
  int dagger;       /* 0: D, 1: D^dag */
  int mass_reading; /* 0: gamma5 twist (C4), 1: complex scalar mass */
  int antiperiodic_t; /* 1: C6 (default); 0: fully periodic, used only by oracle self-tests */
} op_t;

/* r[s][c] += coef * sum_{s'} M[s][s'] w[s'][c] */
static void spin_acc(const cplx M[4][4], cplx coef, const cplx w[4][3], cplx r[4][3]) {
  for (int s = 0; s < 4; s++)
    for (int sp = 0; sp < 4; sp++)
      for (int c = 0; c < 3; c++) r[s][c] += coef * M[s][sp] * w[sp][c];
}

/*
 * D:      row x of the matrix D(x,y).
 * D^dag:  (D^dag psi)(x) = sum_y [D(y,x)]^dag psi(y). The block D(y,x) with x = y + eta*mu is
 *         1/2 (1 + eta g_mu) (x) U_mu(y, y+eta mu) s; its conjugate transpose is 1/2 (1 + eta g_mu) (x) U_mu(y,y+eta mu)^dag s
 *         (g_mu Hermitian). For eta = +1, y = x - mu:  1/2 (1+g_mu) U_mu(x-mu)^dag psi(x-mu);
 *         for eta = -1, y = x + mu, U_mu(y, y-mu) = U_mu(x)^dag so the dagger gives 1/2 (1-g_mu) U_mu(x) psi(x+mu).
 *         The site-diagonal part is conjugate-transposed: -(4+Re m) + i Im m g5 (g5 Hermitian), clover Hermitian.
 */
static void site_apply(const lat_t* g, const cplx* U, const cplx (*Fsite)[9], const op_t* op, const cplx* in, int64_t s,
                       cplx out[4][3]) {
  int c[4];
  site_coords(g, s, c);
  cplx r[4][3];
  memset(r, 0, sizeof(r));
  cplx one_pm[4][4];
  for (int mu = 0; mu < 4; mu++) {
    for (int dir = +1; dir >= -1; dir -= 2) {
      int wrapped;
      int64_t y = neighbour(g, c, mu, dir, &wrapped);
      double sgn = (mu == 3 && wrapped && op->antiperiodic_t) ? -1.0 : 1.0;
      /* colour part: forward hop uses U_mu(x), backward hop uses U_mu(x-mu)^dag */
      cplx Umat[9];
      if (dir > 0) memcpy(Umat, link(g, U, mu, s), sizeof(Umat));
      else m3_dag(link(g, U, mu, y), Umat);
      const cplx* psi = in + 12 * y;
      cplx w[4][3];
      for (int sp = 0; sp < 4; sp++)
        for (int a = 0; a < 3; a++) {
          cplx t = 0;
          for (int b = 0; b < 3; b++) t += Umat[3 * a + b] * psi[3 * sp + b];
          w[sp][a] = t;
        }
      /* spin part: D uses (1 + dir*g_mu); D^dag uses (1 - dir*g_mu) */
      double eta = op->dagger ? -(double)dir : (double)dir;
      for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) one_pm[i][j] = (i == j ? 1.0 : 0.0) + eta * GAMMA[mu][i][j];
      spin_acc(one_pm, 0.5 * sgn, w, r);
    }
  }
  const cplx* psi = in + 12 * s;
  /* mass term */
  if (op->mass_reading == 0) {
    cplx g5[4][4];
    gamma5(g5);
    double mim = op->dagger ? -op->m_im : op->m_im;
    for (int sp = 0; sp < 4; sp++)
      for (int a = 0; a < 3; a++) {
        r[sp][a] -= (4.0 + op->m_re) * psi[3 * sp + a];
        for (int sq = 0; sq < 4; sq++) r[sp][a] -= I * mim * g5[sp][sq] * psi[3 * sq + a];
      }
  } else {
    cplx m = op->m_re + I * (op->dagger ? -op->m_im : op->m_im);
    for (int sp = 0; sp < 4; sp++)
      for (int a = 0; a < 3; a++) r[sp][a] -= (4.0 + m) * psi[3 * sp + a];
  }
  /* clover term */
  if (op->c_sw != 0.0) {
    cplx Floc[6][9];
    if (!Fsite) { field_strength_site(g, U, s, Floc); Fsite = Floc; }
    int plane = 0;
    for (int mu = 0; mu < 4; mu++)
      for (int nu = mu + 1; nu < 4; nu++, plane++) {
        cplx sig[4][4], w[4][3];
        sigma_munu(mu, nu, sig);
        for (int sp = 0; sp < 4; sp++)
          for (int a = 0; a < 3; a++) {
            cplx t = 0;
            for (int b = 0; b < 3; b++) t += Fsite[plane][3 * a + b] * psi[3 * sp + b];
            w[sp][a] = t;
          }
        spin_acc(sig, 0.5 * op->c_sw, w, r);
      }
  }
  memcpy(out, r, sizeof(r));
}

/* out = D in (or D^dag in) on the full lattice. F may be NULL: then F is recomputed at every site when c_sw != 0. */
void orc_apply(int L, int T, const double* gauge, const double* F, double m_re, double m_im, double c_sw, int dagger,
               int mass_reading, int antiperiodic_t, const double* in, double* out) {
  lat_t g = {L, T, (int64_t)L * L * L * T};
  op_t op = {m_re, m_im, c_sw, dagger, mass_reading, antiperiodic_t};
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < g.V; s++) {
    const cplx(*Fs)[9] = F ? (const cplx(*)[9])((const cplx*)F + 54 * s) : NULL;
    site_apply(&g, (const cplx*)gauge, Fs, &op, (const cplx*)in, s, (cplx(*)[3])((cplx*)out + 12 * s));
  }
}

/* the same, but only at the n listed lexicographic sites: out[n][4][3]. F is recomputed on the fly. */
void orc_apply_sites(int L, int T, const double* gauge, double m_re, double m_im, double c_sw, int dagger,
                     int mass_reading, int antiperiodic_t, const double* in, int64_t n, const int64_t* sites, double* out) {
  lat_t g = {L, T, (int64_t)L * L * L * T};
  op_t op = {m_re, m_im, c_sw, dagger, mass_reading, antiperiodic_t};
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < n; k++)
    site_apply(&g, (const cplx*)gauge, NULL, &op, (const cplx*)in, sites[k], (cplx(*)[3])((cplx*)out + 12 * k));
}

/* ---- BiCGStab (van der Vorst), full lattice, fp64; SURVEY.md §8(c) C11 ----
 * x0 = 0, r0 = b, rhat = r0, rho = alpha = omega = 1, v = p = 0; loop:
 *   rho' = <rhat,r>; beta = (rho'/rho)(alpha/omega); p = r + beta (p - omega v); v = A p; alpha = rho'/<rhat,v>;
 *   s = r - alpha v; t = A s; omega = <t,s>/<t,t>; x += alpha p + omega s; r = s - omega t
 * with <a,b> = sum conj(a_i) b_i. Stop when |r| <= tol |b|. Returns 0 on convergence, 1 if max_iter was reached,
 * 2 on breakdown. *true_resid = |b - D x| / |b| recomputed at the end.
 * Breakdown rule (C11): when |rho'| <= 1e-12 |rhat| |r| (rhat and r numerically orthogonal) the recurrence is
 * restarted with rhat = r, rho = alpha = omega = 1, p = v = 0 (at most 5 times). This is not a corner case here: for
 * a point source rhat = b is a single component, s vanishes at the source site after the first half step and the
 * there-and-back hop (1 -+ g_mu)(1 +- g_mu) = 0 makes <rhat, D s> = 0 exactly, so rho' = 0 at the second iteration.
 */
static cplx vdot(int64_t n, const cplx* a, const cplx* b) {
  double re = 0, im = 0;
#pragma omp parallel for reduction(+ : re, im) schedule(static)
  for (int64_t i = 0; i < n; i++) {
    cplx t = conj(a[i]) * b[i];
    re += creal(t);
    im += cimag(t);
  }
  return re + I * im;
}

int orc_bicgstab(int L, int T, const double* gauge, const double* F, double m_re, double m_im, double c_sw, int dagger,
                 int mass_reading, int antiperiodic_t, const double* b_, double* x_, double tol, int max_iter, int* iters,
                 double* true_resid) {
  int64_t n = 12 * (int64_t)L * L * L * T;
  const cplx* b = (const cplx*)b_;
  cplx* x = (cplx*)x_;
  cplx *r = malloc(n * sizeof(cplx)), *rhat = malloc(n * sizeof(cplx)), *p = calloc(n, sizeof(cplx)),
       *v = calloc(n, sizeof(cplx)), *s = malloc(n * sizeof(cplx)), *t = malloc(n * sizeof(cplx));
  int status = 1;
  memset(x, 0, n * sizeof(cplx));
  memcpy(r, b, n * sizeof(cplx));
  memcpy(rhat, b, n * sizeof(cplx));
  double bnorm = sqrt(creal(vdot(n, b, b)));
  cplx rho = 1, alpha = 1, omega = 1;
  double rhat_norm = bnorm, rnorm = bnorm;
  int k = 0, restarts = 0;
  if (bnorm == 0.0) { status = 0; goto done; }
  for (k = 1; k <= max_iter; k++) {
    cplx rho1 = vdot(n, rhat, r);
    if (!(cabs(rho1) > 1e-12 * rhat_norm * rnorm)) { /* breakdown (or NaN): restart with rhat = r */
      if (rho1 != rho1 || restarts >= 5) { status = 2; break; }
      restarts++;
      memcpy(rhat, r, n * sizeof(cplx));
      memset(p, 0, n * sizeof(cplx));
      memset(v, 0, n * sizeof(cplx));
      rhat_norm = rnorm;
      rho = alpha = omega = 1;
      rho1 = rnorm * rnorm;
    }
    cplx beta = (rho1 / rho) * (alpha / omega);
    for (int64_t i = 0; i < n; i++) p[i] = r[i] + beta * (p[i] - omega * v[i]);
    orc_apply(L, T, gauge, F, m_re, m_im, c_sw, dagger, mass_reading, antiperiodic_t, (double*)p, (double*)v);
    alpha = rho1 / vdot(n, rhat, v);
    for (int64_t i = 0; i < n; i++) s[i] = r[i] - alpha * v[i];
    orc_apply(L, T, gauge, F, m_re, m_im, c_sw, dagger, mass_reading, antiperiodic_t, (double*)s, (double*)t);
    double tt = creal(vdot(n, t, t));
    if (tt == 0.0 || tt != tt) { /* s = 0: x + alpha p is exact */
      for (int64_t i = 0; i < n; i++) x[i] += alpha * p[i];
      status = (tt == 0.0) ? 0 : 2;
      break;
    }
    omega = vdot(n, t, s) / tt;
    for (int64_t i = 0; i < n; i++) {
      x[i] += alpha * p[i] + omega * s[i];
      r[i] = s[i] - omega * t[i];
    }
    rho = rho1;
    rnorm = sqrt(creal(vdot(n, r, r)));
    if (rnorm <= tol * bnorm) { status = 0; break; }
  }
done:
  if (iters) *iters = k > max_iter ? max_iter : k;
  if (true_resid) {
    if (bnorm == 0.0) *true_resid = 0.0;
    else {
      orc_apply(L, T, gauge, F, m_re, m_im, c_sw, dagger, mass_reading, antiperiodic_t, (double*)x, (double*)t);
      for (int64_t i = 0; i < n; i++) t[i] = b[i] - t[i];
      *true_resid = sqrt(creal(vdot(n, t, t))) / bnorm;
    }
  }
  free(r); free(rhat); free(p); free(v); free(s); free(t);
  return status;
}

int orc_num_threads(void) {
#ifdef _OPENMP
  extern int omp_get_max_threads(void);
  return omp_get_max_threads();
#else
  return 1;
#endif
}
