/*
 * synth.c — seeded synthetic input generators (harness side).
 *
 * This file holds NONE of the method's arithmetic (no Dirac operator, no clover, no solver). It only
 * manufactures inputs: random SU(3) gauge links, Z2 / Gaussian spinors. Both the CPU oracle and the CUDA
 * library receive the arrays produced here; neither of them includes or links this file.
 *
 * Recipe (BASELINE.json configs[0]):
 *   link  U = exp(i * eps * H),  H = sum_{a=1..8} c_a lambda_a  (standard Gell-Mann matrices, tr(l_a l_b) = 2 d_ab,
 *   no factor 1/2),  c_a i.i.d. N(0,1);  then re-unitarised: Gram-Schmidt on rows 0,1 and row 2 = conj(row0 x row1).
 *   RNG: counter based (order- and thread-independent): splitmix64 finaliser of (seed, stream, index) -> uniforms
 *   -> Box-Muller.
 *
 * Layout of a link array of n matrices: [n][row 3][col 3][re,im] doubles (row-major 3x3 complex).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <string.h>

typedef double complex cplx;

static inline uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

/* one 64-bit word for the counter (seed, stream, idx, k) */
static inline uint64_t rnd_u64(uint64_t seed, uint64_t stream, uint64_t idx, uint64_t k) {
  uint64_t h = mix64(seed ^ 0xD1B54A32D192ED03ULL);
  h = mix64(h ^ (stream * 0xA24BAED4963EE407ULL));
  h = mix64(h ^ idx);
  h = mix64(h ^ (k * 0x9FB21C651E98DF25ULL));
  return h;
}

/* uniform in (0,1): 53 random bits, never 0 */
static inline double rnd_unif(uint64_t seed, uint64_t stream, uint64_t idx, uint64_t k) {
  return ((double)(rnd_u64(seed, stream, idx, k) >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

/* standard normal number j of counter idx (Box-Muller; pairs share two uniforms) */
static inline double rnd_normal(uint64_t seed, uint64_t stream, uint64_t idx, uint64_t j) {
  double u1 = rnd_unif(seed, stream, idx, 2 * (j >> 1));
  double u2 = rnd_unif(seed, stream, idx, 2 * (j >> 1) + 1);
  double r = sqrt(-2.0 * log(u1));
  double a = 6.283185307179586476925286766559 * u2;
  return (j & 1) ? r * sin(a) : r * cos(a);
}

static void mat_mul(const cplx a[9], const cplx b[9], cplx c[9]) {
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      cplx s = 0;
      for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
      c[3 * i + j] = s;
    }
}

/* H = sum c_a lambda_a, Gell-Mann */
static void gellmann_sum(const double c[8], cplx h[9]) {
  const double s3 = 0.57735026918962576450914878050196; /* 1/sqrt(3) */
  h[0] = c[2] + c[7] * s3;
  h[4] = -c[2] + c[7] * s3;
  h[8] = -2.0 * c[7] * s3;
  h[1] = c[0] - I * c[1];
  h[3] = c[0] + I * c[1];
  h[2] = c[3] - I * c[4];
  h[6] = c[3] + I * c[4];
  h[5] = c[5] - I * c[6];
  h[7] = c[5] + I * c[6];
}

/* u = exp(i*eps*h): scaling and squaring with a degree-18 Taylor polynomial */
static void su3_exp(const cplx h[9], double eps, cplx u[9]) {
  double nrm = 0;
  for (int i = 0; i < 9; i++) nrm += creal(h[i]) * creal(h[i]) + cimag(h[i]) * cimag(h[i]);
  nrm = sqrt(nrm) * fabs(eps);
  int sq = 0;
  while (nrm > 0.25) { nrm *= 0.5; sq++; }
  double sc = eps / (double)(1ULL << sq);
  cplx x[9], term[9], tmp[9];
  for (int i = 0; i < 9; i++) x[i] = I * sc * h[i];
  for (int i = 0; i < 9; i++) { u[i] = (i % 4 == 0) ? 1.0 : 0.0; term[i] = u[i]; }
  for (int k = 1; k <= 18; k++) {
    mat_mul(term, x, tmp);
    for (int i = 0; i < 9; i++) { term[i] = tmp[i] / (double)k; u[i] += term[i]; }
  }
  for (int s = 0; s < sq; s++) {
    mat_mul(u, u, tmp);
    memcpy(u, tmp, sizeof(tmp));
  }
}

static void reunitarise(cplx u[9]) {
  double n0 = 0;
  for (int j = 0; j < 3; j++) n0 += creal(u[j] * conj(u[j]));
  n0 = 1.0 / sqrt(n0);
  for (int j = 0; j < 3; j++) u[j] *= n0;
  cplx d = 0;
  for (int j = 0; j < 3; j++) d += conj(u[j]) * u[3 + j];
  for (int j = 0; j < 3; j++) u[3 + j] -= d * u[j];
  double n1 = 0;
  for (int j = 0; j < 3; j++) n1 += creal(u[3 + j] * conj(u[3 + j]));
  n1 = 1.0 / sqrt(n1);
  for (int j = 0; j < 3; j++) u[3 + j] *= n1;
  u[6] = conj(u[1] * u[5] - u[2] * u[4]);
  u[7] = conj(u[2] * u[3] - u[0] * u[5]);
  u[8] = conj(u[0] * u[4] - u[1] * u[3]);
}

/* n random SU(3) matrices, counter index = first + i */
void synth_su3(int64_t n, double eps, uint64_t seed, uint64_t stream, int64_t first, double* out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; i++) {
    double c[8];
    for (int a = 0; a < 8; a++) c[a] = rnd_normal(seed, stream, (uint64_t)(first + i), (uint64_t)a);
    cplx h[9], u[9];
    gellmann_sum(c, h);
    su3_exp(h, eps, u);
    reunitarise(u);
    memcpy(out + 18 * i, u, sizeof(u));
  }
}

/* gauge field in the canonical layout [mu][t][z][y][x][3][3][2]; counter = mu*V + site; stream 1 */
void synth_gauge(int L, int T, double eps, uint64_t seed, double* out) {
  int64_t V = (int64_t)L * L * L * T;
  synth_su3(4 * V, eps, seed, 1, 0, out);
}

/* n complex numbers, each +-1 + 0i with equal probability (stream 2) */
void synth_z2(int64_t n, uint64_t seed, double* out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; i++) {
    out[2 * i] = (rnd_u64(seed, 2, (uint64_t)i, 0) >> 63) ? 1.0 : -1.0;
    out[2 * i + 1] = 0.0;
  }
}

/* n complex Gaussians, re and im i.i.d. N(0,1) (stream 3) */
void synth_gauss(int64_t n, uint64_t seed, double* out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; i++) {
    out[2 * i] = rnd_normal(seed, 3, (uint64_t)i, 0);
    out[2 * i + 1] = rnd_normal(seed, 3, (uint64_t)i, 1);
  }
}
