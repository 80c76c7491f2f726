/* su3_oracle.c -- the ORACLE: a plain, slow, obviously correct CPU statement of
 * what the SU(3)xSU(3) streaming hot path computes.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product (the CUDA library, its
 * Python binding) may import, link or call this file; only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs do.
 * It shares no source, header, table or helper with the CUDA path.
 *
 * What it follows (P:N = /root/reference/PAPER.md line N):
 *   - the site loop `for(ss<_osites) _odata[ss] = eval(ss,expr)`      P:76-89, Listing 1
 *   - `z = x*y` on Lattice<Su3f>, complex 3x3 per site                P:113-126, section 4, Listing 3
 *   - composite expressions evaluated inside that one site loop       P:91-109, Listing 2
 *     (z = x*y*w parsed left-to-right as (x*y)*w; z = x*y + v)
 *   - vector layout: the lattice is split into N_sub "virtual nodes",
 *     the split lives at the level of the basic complex type
 *   - extract/merge: lane l of every matrix element <-> one scalar
 *     3x3 matrix
 * The method reaches exactly the plain definition (no approximation), so the
 * oracle IS the definition: z_ij = sum_k x_ik y_kj, k ascending, complex
 * multiply as 4 real multiplies + 2 adds, in fp64, no FMA contraction
 * (compile with -ffp-contract=off).  Where the paper is silent the readings
 * S1-S7 of DESIGN.md apply (element order, site order, the vector layout map,
 * the default split of W, the Lorentz index position).
 *
 * fp32 fields: the oracle reads the fp32 storage, promotes exactly to double,
 * computes and KEEPS the result in double (reading S16).
 *
 * Every function below is pinned by tests/test_oracle_pins.py (hand-computed
 * integer products, identity/zero, closed-form SU(3) elements, unitarity/det
 * closure, associativity, numpy.matmul cross-check, brute force on 2^4 / 4^4,
 * index spot values, layout agreement).  Nothing here is "parity unpinned".
 */
#include <stdint.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int32_t L[4];    /* lattice extents                                         */
  int32_t nl;      /* matrices per site: 1 (colour matrix) or 4 (gauge field) */
  int32_t layout;  /* 0 = scalar site-major, 1 = vector (virtual nodes)       */
  int32_t W;       /* sites interleaved lane-wise; 1 for the scalar layout    */
  int32_t simd[4]; /* virtual-node grid, product = W                          */
} orc_geom;

/* Reading S4: hand out factors of two starting at d=3 and moving down, wrapping. */
void orc_default_simd(int W, int32_t simd[4]) {
  for (int d = 0; d < 4; d++) simd[d] = 1;
  int d = 3;
  while (W > 1) {
    simd[d] *= 2;
    W /= 2;
    d = (d + 3) % 4; /* 3,2,1,0,3,... */
  }
}

/* returns 0 on success, nonzero if the geometry is not admissible */
int orc_geom_init(orc_geom *g, const int32_t L[4], int nl, int layout, int W, const int32_t simd[4]) {
  if (!g || !L) return 1;
  if (nl != 1 && nl != 4) return 2;
  if (layout != 0 && layout != 1) return 2;
  if (W < 1 || W > 32 || (W & (W - 1))) return 2;
  if (layout == 0 && W != 1) return 2;
  for (int d = 0; d < 4; d++) {
    if (L[d] <= 0) return 2;
    g->L[d] = L[d];
  }
  g->nl = nl; g->layout = layout; g->W = W;
  int any = 0;
  if (simd) for (int d = 0; d < 4; d++) any |= simd[d];
  if (any) {
    int p = 1;
    for (int d = 0; d < 4; d++) {
      if (simd[d] <= 0) return 2;
      g->simd[d] = simd[d];
      p *= simd[d];
    }
    if (p != W) return 2;
  } else {
    orc_default_simd(W, g->simd);
  }
  for (int d = 0; d < 4; d++) if (g->L[d] % g->simd[d]) return 2;
  return 0;
}

int64_t orc_volume(const orc_geom *g) {
  return (int64_t)g->L[0] * g->L[1] * g->L[2] * g->L[3];
}
int64_t orc_nreals(const orc_geom *g) { return orc_volume(g) * g->nl * 18; }

/* Virtual-node map (reading S3): site -> (outer site o, lane l).
 * x[d] from site with x0 fastest (S2); r[d] = L[d]/simd[d];
 * oc[d] = x[d] mod r[d] (position inside the sub-lattice), ic[d] = x[d] div r[d]
 * (which sub-lattice); o = lexicographic index of oc over r, l = lexicographic
 * index of ic over simd, both d=0 fastest. */
void orc_site_to_outer(const orc_geom *g, int64_t site, int64_t *o, int32_t *l) {
  int64_t oo = 0, ostride = 1;
  int32_t ll = 0, lstride = 1;
  for (int d = 0; d < 4; d++) {
    int32_t xd = (int32_t)(site % g->L[d]);
    site /= g->L[d];
    int32_t r = g->L[d] / g->simd[d];
    oo += (int64_t)(xd % r) * ostride;  ostride *= r;
    ll += (xd / r) * lstride;           lstride *= g->simd[d];
  }
  *o = oo; *l = ll;
}

/* Offset, in units of REALS, of (site, mu, row i, col j, reim).
 * scalar (S1,S2,S6): (((site*nl + mu)*9 + 3i+j)*2 + reim
 * vector (S3):       ((((o*nl + mu)*9 + 3i+j)*W + l)*2 + reim                   */
int64_t orc_index(const orc_geom *g, int64_t site, int mu, int i, int j, int reim) {
  int e = 3 * i + j;
  if (g->layout == 0) return ((site * g->nl + mu) * 9 + e) * 2 + reim;
  int64_t o; int32_t l;
  orc_site_to_outer(g, site, &o, &l);
  return (((o * g->nl + mu) * 9 + e) * g->W + l) * 2 + reim;
}

static inline double rd(const void *p, int prec, int64_t idx) {
  return prec == 8 ? ((const double *)p)[idx] : (double)((const float *)p)[idx];
}

/* load the 3x3 complex matrix (site,mu) into a[i][j][reim], promoted to double */
static void load33(const orc_geom *g, int prec, const void *f, int64_t site, int mu, double a[3][3][2]) {
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++)
      for (int c = 0; c < 2; c++) a[i][j][c] = rd(f, prec, orc_index(g, site, mu, i, j, c));
}

static void store33(const orc_geom *g, double *f, int64_t site, int mu, double a[3][3][2]) {
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++)
      for (int c = 0; c < 2; c++) f[orc_index(g, site, mu, i, j, c)] = a[i][j][c];
}

/* c = a.b : c_ij = sum_k a_ik b_kj, k ascending; 4 real mul + 2 add per term (S7) */
static void mat33(double a[3][3][2], double b[3][3][2], double c[3][3][2]) {
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      double re = 0.0, im = 0.0;
      for (int k = 0; k < 3; k++) {
        double ar = a[i][k][0], ai = a[i][k][1], br = b[k][j][0], bi = b[k][j][1];
        re += ar * br - ai * bi;
        im += ar * bi + ai * br;
      }
      c[i][j][0] = re; c[i][j][1] = im;
    }
}

/* z = x*y.  x,y in storage precision `prec` (4 or 8 bytes per real), z double. */
void orc_mul(const orc_geom *g, int prec, const void *x, const void *y, double *z) {
  int64_t V = orc_volume(g);
#pragma omp parallel for schedule(static)
  for (int64_t site = 0; site < V; site++)
    for (int mu = 0; mu < g->nl; mu++) {
      double a[3][3][2], b[3][3][2], c[3][3][2];
      load33(g, prec, x, site, mu, a);
      load33(g, prec, y, site, mu, b);
      mat33(a, b, c);
      store33(g, z, site, mu, c);
    }
}

/* z = (x*y)*w, left-associative as C++ parses x*y*w; T in fp64, one site. */
void orc_mul3(const orc_geom *g, int prec, const void *x, const void *y, const void *w, double *z) {
  int64_t V = orc_volume(g);
#pragma omp parallel for schedule(static)
  for (int64_t site = 0; site < V; site++)
    for (int mu = 0; mu < g->nl; mu++) {
      double a[3][3][2], b[3][3][2], d[3][3][2], t[3][3][2], c[3][3][2];
      load33(g, prec, x, site, mu, a);
      load33(g, prec, y, site, mu, b);
      load33(g, prec, w, site, mu, d);
      mat33(a, b, t);
      mat33(t, d, c);
      store33(g, z, site, mu, c);
    }
}

/* z = x*y + v (the `v1+v2+v1*v2` pattern of P:104-106 on matrices) */
void orc_mul_add(const orc_geom *g, int prec, const void *x, const void *y, const void *v, double *z) {
  int64_t V = orc_volume(g);
#pragma omp parallel for schedule(static)
  for (int64_t site = 0; site < V; site++)
    for (int mu = 0; mu < g->nl; mu++) {
      double a[3][3][2], b[3][3][2], d[3][3][2], c[3][3][2];
      load33(g, prec, x, site, mu, a);
      load33(g, prec, y, site, mu, b);
      load33(g, prec, v, site, mu, d);
      mat33(a, b, c);
      for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++)
          for (int q = 0; q < 2; q++) c[i][j][q] = c[i][j][q] + d[i][j][q];
      store33(g, z, site, mu, c);
    }
}

/* z = value of a postfix expression over matrix fields, evaluated per site inside the one site loop
 * (Listing 1: `eval(ss, expr)` walks the expression tree at every site; Listing 2:
 * `v3 = v1+v2+v1*v2` is one pass, no temporaries in memory).  The tree is given in postfix order as a
 * string: a digit '0'..'7' pushes operand field ops[digit] at this site, '+', '-', '*' pop b then a and push
 * a+b, a-b, a.b (matrix product, mat33 above).  Every intermediate lives in fp64 for the one site.
 * Returns 0, or nonzero if the program is malformed (bad token, operand index >= nops, stack under-/
 * overflow (depth > 8), or not exactly one value left). */
int orc_expr(const orc_geom *g, int prec, int nops, const void *const *ops, const char *prog, double *z) {
  int depth = 0, n = 0;
  for (const char *t = prog; *t; t++, n++) {
    if (*t >= '0' && *t <= '7') { if (*t - '0' >= nops) return 2; if (++depth > 8) return 3; }
    else if (*t == '+' || *t == '-' || *t == '*') { if (depth < 2) return 4; depth--; }
    else return 1;
  }
  if (depth != 1) return 5;
  int64_t V = orc_volume(g);
#pragma omp parallel for schedule(static)
  for (int64_t site = 0; site < V; site++)
    for (int mu = 0; mu < g->nl; mu++) {
      double st[8][3][3][2];
      int sp = 0;
      for (const char *t = prog; *t; t++) {
        if (*t >= '0' && *t <= '7') {
          load33(g, prec, ops[*t - '0'], site, mu, st[sp++]);
        } else {
          double (*a)[3][2] = st[sp - 2], (*b)[3][2] = st[sp - 1], c[3][3][2];
          if (*t == '*') mat33(a, b, c);
          else
            for (int i = 0; i < 3; i++)
              for (int j = 0; j < 3; j++)
                for (int q = 0; q < 2; q++) c[i][j][q] = (*t == '+') ? a[i][j][q] + b[i][j][q] : a[i][j][q] - b[i][j][q];
          memcpy(a, c, sizeof c);
          sp--;
        }
      }
      store33(g, z, site, mu, st[0]);
    }
  return 0;
}

/* layout conversion = pure permutation of reals, bit copy (lane l of
 * each of the 9 vector elements <-> one scalar matrix).  `prec` bytes per real. */
int orc_convert(const orc_geom *gd, const orc_geom *gs, int prec, void *dst, const void *src) {
  for (int d = 0; d < 4; d++) if (gd->L[d] != gs->L[d]) return 3;
  if (gd->nl != gs->nl) return 3;
  int64_t V = orc_volume(gs);
#pragma omp parallel for schedule(static)
  for (int64_t site = 0; site < V; site++)
    for (int mu = 0; mu < gs->nl; mu++)
      for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++)
          for (int c = 0; c < 2; c++)
            memcpy((char *)dst + prec * orc_index(gd, site, mu, i, j, c),
                   (const char *)src + prec * orc_index(gs, site, mu, i, j, c), (size_t)prec);
  return 0;
}

/* Neighbour of `site` at displacement `disp` (any integer) along dimension `dim`, periodic:
 * x[dim] -> (x[dim] + disp) mod L[dim], site order S2 (x0 fastest). */
int64_t orc_neighbour(const orc_geom *g, int64_t site, int dim, int disp) {
  int64_t stride = 1;
  for (int d = 0; d < dim; d++) stride *= g->L[d];
  int64_t xd = (site / stride) % g->L[dim];
  int64_t nd = ((xd + disp) % g->L[dim] + g->L[dim]) % g->L[dim];
  return site + (nd - xd) * stride;
}

/* Circular shift, Grid's `Cshift(x, dim, disp)` (named by the paper as the next obstacle):
 * z[s] = x[s + disp*dim_hat] for every site s and every mu; a pure permutation of matrices, bit copy,
 * `prec` bytes per real, any layout (in the vector layout a shift across a sub-lattice boundary moves
 * a matrix to another lane -- here that is simply what the index function says). */
int orc_cshift(const orc_geom *g, int prec, void *z, const void *x, int dim, int disp) {
  if (dim < 0 || dim > 3) return 1;
  int64_t V = orc_volume(g);
#pragma omp parallel for schedule(static)
  for (int64_t site = 0; site < V; site++) {
    int64_t from = orc_neighbour(g, site, dim, disp);
    for (int mu = 0; mu < g->nl; mu++)
      for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++)
          for (int c = 0; c < 2; c++)
            memcpy((char *)z + prec * orc_index(g, site, mu, i, j, c),
                   (const char *)x + prec * orc_index(g, from, mu, i, j, c), (size_t)prec);
  }
  return 0;
}

/* z[s] = x[s] . y[s + disp*dim_hat]: the site-local product with a shifted second operand, the building
 * block of covariant shifts / plaquettes ("Cshift ... stencil operators").  fp64 result. */
int orc_mul_shift(const orc_geom *g, int prec, const void *x, const void *y, int dim, int disp, double *z) {
  if (dim < 0 || dim > 3) return 1;
  int64_t V = orc_volume(g);
#pragma omp parallel for schedule(static)
  for (int64_t site = 0; site < V; site++) {
    int64_t from = orc_neighbour(g, site, dim, disp);
    for (int mu = 0; mu < g->nl; mu++) {
      double a[3][3][2], b[3][3][2], c[3][3][2];
      load33(g, prec, x, site, mu, a);
      load33(g, prec, y, from, mu, b);
      mat33(a, b, c);
      store33(g, z, site, mu, c);
    }
  }
  return 0;
}

/* ---- colour-vector fields (3 complex per (site, mu)) and y = U.psi (f4; the building block
 * of the Dslash-type stencil operators the paper says it is porting).  Layout by the same readings as the
 * matrix field with 3 components instead of 9:
 *   scalar: ((site*nl + mu)*3 + i)*2 + reim        vector: (((o*nl + mu)*3 + i)*W + l)*2 + reim          */
int64_t orc_index_vec(const orc_geom *g, int64_t site, int mu, int i, int reim) {
  if (g->layout == 0) return ((site * g->nl + mu) * 3 + i) * 2 + reim;
  int64_t o; int32_t l;
  orc_site_to_outer(g, site, &o, &l);
  return (((o * g->nl + mu) * 3 + i) * g->W + l) * 2 + reim;
}

/* y_i = sum_j U_ij psi_j, j ascending, 4 real mul + 2 add per term (S7); fp64 result. */
void orc_matvec(const orc_geom *g, int prec, const void *U, const void *psi, double *y) {
  int64_t V = orc_volume(g);
#pragma omp parallel for schedule(static)
  for (int64_t site = 0; site < V; site++)
    for (int mu = 0; mu < g->nl; mu++) {
      double a[3][3][2];
      load33(g, prec, U, site, mu, a);
      for (int i = 0; i < 3; i++) {
        double re = 0.0, im = 0.0;
        for (int j = 0; j < 3; j++) {
          double br = rd(psi, prec, orc_index_vec(g, site, mu, j, 0)), bi = rd(psi, prec, orc_index_vec(g, site, mu, j, 1));
          re += a[i][j][0] * br - a[i][j][1] * bi;
          im += a[i][j][0] * bi + a[i][j][1] * br;
        }
        y[orc_index_vec(g, site, mu, i, 0)] = re;
        y[orc_index_vec(g, site, mu, i, 1)] = im;
      }
    }
}

/* layout permutation of a colour-vector field, bit copy */
int orc_convert_vec(const orc_geom *gd, const orc_geom *gs, int prec, void *dst, const void *src) {
  for (int d = 0; d < 4; d++) if (gd->L[d] != gs->L[d]) return 3;
  if (gd->nl != gs->nl) return 3;
  int64_t V = orc_volume(gs);
#pragma omp parallel for schedule(static)
  for (int64_t site = 0; site < V; site++)
    for (int mu = 0; mu < gs->nl; mu++)
      for (int i = 0; i < 3; i++)
        for (int c = 0; c < 2; c++)
          memcpy((char *)dst + prec * orc_index_vec(gd, site, mu, i, c),
                 (const char *)src + prec * orc_index_vec(gs, site, mu, i, c), (size_t)prec);
  return 0;
}

/* ---- real scalar fields, the paper's own example of the expression engine (Listing 2):
 *   Lattice<double> v1, v2, v3;  v1 = 1.0;  v2 = 2.0;  v3 = v1+v2;  v3 = v1+v2+v1*v2;
 * One real per (site, mu); '+', '-', '*' act element-wise, so no layout map is involved: the field is just n
 * reals.  Same postfix convention and the same validity rules as orc_expr; fp64 result. */
int orc_expr_real(int64_t n, int prec, int nops, const void *const *ops, const char *prog, double *z) {
  int depth = 0;
  for (const char *t = prog; *t; t++) {
    if (*t >= '0' && *t <= '7') { if (*t - '0' >= nops) return 2; if (++depth > 8) return 3; }
    else if (*t == '+' || *t == '-' || *t == '*') { if (depth < 2) return 4; depth--; }
    else return 1;
  }
  if (depth != 1) return 5;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; i++) {
    double st[8];
    int sp = 0;
    for (const char *t = prog; *t; t++) {
      if (*t >= '0' && *t <= '7') st[sp++] = rd(ops[*t - '0'], prec, i);
      else {
        double b = st[--sp], a = st[--sp];
        st[sp++] = *t == '+' ? a + b : (*t == '-' ? a - b : a * b);
      }
    }
    z[i] = st[0];
  }
  return 0;
}

/* Host STREAM triad a[i] = b[i] + s*c[i] (the line the paper draws next to its curves), best of `reps`
 * passes over n doubles, returned in GB/s counting 24 bytes per element.  A measurement aid of bench.py's
 * cpu_baseline leg: it is NOT part of the method and nothing above uses it. */
#include <stdlib.h>
#include <time.h>
double orc_stream_triad(int64_t n, int reps) {
  double *a = malloc(sizeof(double) * (size_t)n), *b = malloc(sizeof(double) * (size_t)n), *c = malloc(sizeof(double) * (size_t)n);
  double best = 0.0;
  if (a && b && c && n > 0) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; i++) { a[i] = 0.0; b[i] = 1.0; c[i] = 2.0; } /* first touch */
    for (int r = 0; r < reps; r++) {
      struct timespec t0, t1;
      clock_gettime(CLOCK_MONOTONIC, &t0);
#pragma omp parallel for schedule(static)
      for (int64_t i = 0; i < n; i++) a[i] = b[i] + 3.0 * c[i];
      clock_gettime(CLOCK_MONOTONIC, &t1);
      const double s = (double)(t1.tv_sec - t0.tv_sec) + 1e-9 * (double)(t1.tv_nsec - t0.tv_nsec);
      const double gbs = 24.0 * (double)n / s / 1e9;
      if (gbs > best) best = gbs;
    }
    if (a[n / 2] != 7.0) best = -1.0;
  }
  free(a); free(b); free(c);
  return best;
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}
