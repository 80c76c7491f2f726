/* su3gen.c -- seeded synthetic lattice fields (input generator ONLY).
 *
 * This module holds none of the method's arithmetic (no 3x3 matrix product, no
 * layout index map).  It only draws the inputs of the SU(3)xSU(3) streaming
 * test of PAPER.md section 4 (Listing 3), which the paper itself
 * never specifies ("x", "y" are just lattice fields); the recipe is the
 * reading S10-S14 of SURVEY.md section 8(c), restated in DESIGN.md:
 *
 *   counter-based RNG keyed by (seed, field id, logical matrix index m, draw)
 *   -> 53-bit uniforms in (0,1) -> Box-Muller -> complex Gaussian 3x3
 *   -> modified Gram-Schmidt on the rows, applied twice
 *   -> multiply by exp(-i*arg(det)/3)  (principal branch) so that det = 1.
 *
 * Output is always the LOGICAL order  out[m][i][j][re,im]  in fp64, m =
 * site*n_lorentz + mu, which makes a field independent of layout, thread count
 * and generation order.  Both the oracle and the CUDA path consume the arrays
 * produced here; neither shares code with this file.
 */
#include <math.h>
#include <stdint.h>

static inline uint64_t mix64(uint64_t z) { /* splitmix64 finaliser */
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
  z ^= z >> 27; z *= 0x94D049BB133111EBULL;
  z ^= z >> 31; return z;
}

static inline uint64_t field_key(uint64_t seed, uint64_t field_id) {
  return mix64(mix64(seed) ^ (0xD1B54A32D192ED03ULL * (field_id + 1)));
}

/* uniform in (0,1): 53 random bits * 2^-53 + 2^-54, never 0 and never 1 */
static inline double u01(uint64_t key, uint64_t ctr) {
  uint64_t r = mix64(key + 0x9E3779B97F4A7C15ULL * (ctr + 1));
  return (double)(r >> 11) * 0x1.0p-53 + 0x1.0p-54;
}

/* 9 Box-Muller pairs: pair e gives (re, im) of element e, each ~ N(0, sigma^2) */
static void gauss9(uint64_t key, uint64_t m, double sigma, double a[18]) {
  for (int e = 0; e < 9; e++) {
    double u1 = u01(key, m * 18 + 2 * (uint64_t)e);
    double u2 = u01(key, m * 18 + 2 * (uint64_t)e + 1);
    double r = sigma * sqrt(-2.0 * log(u1));
    double t = 6.283185307179586476925286766559 * u2;
    a[2 * e] = r * cos(t);
    a[2 * e + 1] = r * sin(t);
  }
}

/* raw 64-bit draws, exposed so that tests can pin the counter scheme */
void su3gen_raw(uint64_t seed, uint64_t field_id, uint64_t ctr0, int64_t n, uint64_t *out) {
  uint64_t key = field_key(seed, field_id);
  for (int64_t i = 0; i < n; i++)
    out[i] = mix64(key + 0x9E3779B97F4A7C15ULL * (ctr0 + (uint64_t)i + 1));
}

void su3gen_uniform(uint64_t seed, uint64_t field_id, uint64_t ctr0, int64_t n, double *out) {
  uint64_t key = field_key(seed, field_id);
  for (int64_t i = 0; i < n; i++) out[i] = u01(key, ctr0 + (uint64_t)i);
}

/* complex Gaussian 3x3 field, E|a_ij|^2 = variance (re, im ~ N(0, variance/2)) */
void su3gen_gaussian(uint64_t seed, uint64_t field_id, int64_t m0, int64_t count,
                     double variance, double *out) {
  uint64_t key = field_key(seed, field_id);
  double sigma = sqrt(0.5 * variance);
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < count; q++) gauss9(key, (uint64_t)(m0 + q), sigma, out + 18 * q);
}

/* rows of a: a[3*r + j] complex as (re,im) pairs */
static void mgs_rows(double a[18]) {
  for (int r = 0; r < 3; r++) {
    double *v = a + 6 * r;
    for (int p = 0; p < r; p++) {
      const double *u = a + 6 * p;
      double cr = 0.0, ci = 0.0; /* c = <u, v> = sum_j conj(u_j) v_j */
      for (int j = 0; j < 3; j++) {
        cr += u[2 * j] * v[2 * j] + u[2 * j + 1] * v[2 * j + 1];
        ci += u[2 * j] * v[2 * j + 1] - u[2 * j + 1] * v[2 * j];
      }
      for (int j = 0; j < 3; j++) { /* v -= c u */
        double ur = u[2 * j], ui = u[2 * j + 1];
        v[2 * j] -= cr * ur - ci * ui;
        v[2 * j + 1] -= cr * ui + ci * ur;
      }
    }
    double n2 = 0.0;
    for (int j = 0; j < 6; j++) n2 += v[j] * v[j];
    double s = 1.0 / sqrt(n2);
    for (int j = 0; j < 6; j++) v[j] *= s;
  }
}

static void det3(const double a[18], double *dr, double *di) {
#define RE(e) a[2 * (e)]
#define IM(e) a[2 * (e) + 1]
#define CMUL(xr, xi, yr, yi, zr, zi) do { zr = (xr) * (yr) - (xi) * (yi); zi = (xr) * (yi) + (xi) * (yr); } while (0)
  double m0r, m0i, m1r, m1i, tr, ti, sr = 0.0, si = 0.0;
  /* cofactor expansion along row 0 */
  const int c[3][4] = {{4, 8, 5, 7}, {5, 6, 3, 8}, {3, 7, 4, 6}};
  for (int j = 0; j < 3; j++) {
    CMUL(RE(c[j][0]), IM(c[j][0]), RE(c[j][1]), IM(c[j][1]), m0r, m0i);
    CMUL(RE(c[j][2]), IM(c[j][2]), RE(c[j][3]), IM(c[j][3]), m1r, m1i);
    CMUL(RE(j), IM(j), m0r - m1r, m0i - m1i, tr, ti);
    sr += tr; si += ti;
  }
  *dr = sr; *di = si;
#undef RE
#undef IM
#undef CMUL
}

/* random SU(3) field */
void su3gen_su3(uint64_t seed, uint64_t field_id, int64_t m0, int64_t count, double *out) {
  uint64_t key = field_key(seed, field_id);
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < count; q++) {
    double *a = out + 18 * q;
    gauss9(key, (uint64_t)(m0 + q), 1.0, a);
    mgs_rows(a);
    mgs_rows(a); /* twice: one pass leaves ~3e-13 on ill-conditioned draws (S11) */
    double dr, di;
    det3(a, &dr, &di);
    double th = atan2(di, dr) / 3.0; /* principal branch (S12) */
    double pr = cos(th), pi = -sin(th);
    for (int e = 0; e < 9; e++) {
      double xr = a[2 * e], xi = a[2 * e + 1];
      a[2 * e] = xr * pr - xi * pi;
      a[2 * e + 1] = xr * pi + xi * pr;
    }
  }
}
