/*
 * sws_oracle.c -- TEST INFRASTRUCTURE.  Plain, slow, obviously-correct CPU
 * implementation of the nonlinear residual E(u) of
 *   Pethiyagoda, McCue, Moroney & Back, "Jacobian-free Newton-Krylov methods
 *   with GPU acceleration for computing nonlinear ship wave patterns"
 *   (arXiv 1403.5044; /root/reference/PAPER.md, cited below as L<line>).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares NO code with
 * the CUDA path (paper_1403_5044_b200/csrc) and never includes its headers.
 *
 * It is the paper's algorithm written out step by step, in the paper's order
 * and notation (1-based k = 1..N along x, l = 1..M along y in comments; arrays
 * are 0-based with node (k,l) at [(l-1)*N + (k-1)]).  No blocking, fusion or
 * reordering.  The only parallelism is an OpenMP `for` over the independent
 * integral-equation rows E2_{k,l}.
 *
 * Compiled three times: -DREAL=double -DSUF=f64 (the timed baseline),
 * -DREAL="long double" -DSUF=f80 (x86 80-bit accuracy reference), and
 * -DCSTEP -DSUF=c80 (REAL = long double _Complex): the SAME residual code run
 * on u + i h v, whose imaginary part / h is the exact directional derivative
 * J(u) v = d/d sigma E(u + sigma v) at sigma = 0 (complex-step differentiation:
 * no subtraction, truncation error O(h^2) with h = 1e-40).  That is the oracle
 * of the analytic Jacobian action (the limit of eq. (25) L219 as sigma -> 0);
 * it contains no hand-derived derivative formula.  Every function of u the
 * residual uses is analytic (sqrt and asinh of arguments with positive real
 * part, rational expressions); |.| is applied to mesh geometry only.
 *
 * Readings of the paper where it is silent/garbled are DESIGN.md "Readings"
 * Q1..Q12; each is flagged at the line that uses it.
 *
 * Pins (tests/test_oracle_pins.py): P1 full-plane identity, P2 Gauss flux,
 * P3 spline == scipy CubicSpline, P4 sum of weights, P5 closed-form I vs
 * adaptive quadrature, P6 uniform stream, P7 tilted plane, P8 O(h^2)
 * convergence, P9 linear-Jacobian closed forms B.5/B.6 and B.2, layout tests;
 * for the complex-step Jacobian action: PJ1 the same closed forms B.5/B.6/B.2
 * to round-off, PJ2 Richardson-extrapolated central differences of the f80
 * residual at a nonlinear state, PJ3 the linear radiation rows applied to v.
 * PW (tests/test_oracle_jfnk.py): the ROOT of this residual, found by the oracle's
 * own Newton driver, is the steady wave pattern of linear theory (centre-line
 * wavelength 2 pi F^2 under refinement, F^2 scaling, nothing upstream).
 * PG (tests/test_oracle_green.py): for a manufactured harmonic psi on a curved
 * surface, the K1 sum (PG1) and the whole row E2 the residual returns (PG2)
 * converge at O(h^2) to the two sides of Green's third identity, evaluated by
 * adaptive quadrature of continuous integrands that contain none of K1, K2, S2,
 * I.  P1b: the returned row against eq. (12) assembled from full-plane direct
 * sums with the printed signs.  tests/test_oracle_mutations.py compiles ~30
 * single-line mutations of THIS file and requires the named pin to fail on each.
 * The paper prints no numeric value of E for any worked example, so what pins
 * the residual at an arbitrary u is PG2 (to the O(h^2) discretisation error)
 * and P1b/P7 (to round-off).  The nonlinear terms of the Bernoulli row E1 are pinned
 * by PB (an exact potential flow a x + b y + c z under a doubly tilted plane: the first
 * term of (13) must return (a^2 + b^2 + c^2)/2 with all four slopes and the cross term
 * live) and A, B, C of L177 by PS (S2 is the singular part of K2: h (K2 - S2) -> 0 at
 * the nodes next to a target under refinement, only for these A, B, C); (zeta* + 1)^2
 * in the source term by PH (the term is harmonic in (x*, y*, zeta*) and symmetric
 * about z = -1).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <tgmath.h>

#ifdef CSTEP
#include <complex.h>
#undef REAL
#define REAL long double _Complex
#define RREAL long double             /* quantities that never depend on u */
#define RE(z) creall(z)
#else
#ifndef REAL
#define REAL double
#endif
#define RREAL REAL
#define RE(z) (z)
#endif
#ifndef SUF
#define SUF f64
#endif
#define CAT_(a, b) a##_##b
#define CAT(a, b) CAT_(a, b)
#define FN(name) CAT(name, SUF)

typedef struct {
  int N, M;           /* mesh nodes in x and y                       (L145) */
  double x1, y1;      /* first node; x1 = upstream truncation        (L162) */
  double dx, dy;      /* spacings Delta x, Delta y                   (L145) */
  double froude, eps; /* F eq.(9); epsilon eq.(6)                   */
  double n_rad;       /* n in x f_x + n f = 0, paper value 0.05      (L189) */
  int dy_scheme;      /* 0 cubic spline (L160); 1 finite differences (Q3)   */
} sws_oracle_params;

typedef struct {
  int N, M;
  REAL *x, *y;                 /* x_k, y_l */
  REAL *zeta, *phi;            /* nodal values */
  REAL *zeta_x, *phi_x;        /* unknown slopes, from u */
  REAL *zeta_y, *phi_y;        /* y-derivatives (spline or FD) */
} fields_t;

#define AT(k, l) ((size_t)(l) * (size_t)N + (size_t)(k)) /* 0-based k,l */

static const REAL PI_R = (REAL)3.14159265358979323846264338327950288L;

/* ---------------------------------------------------------------------- */
/* Dense LU with partial pivoting; the spline's linear system is solved by */
/* the plainest possible method.                                           */
static int lu_factor(int n, RREAL *A, int *piv) {
  for (int c = 0; c < n; ++c) {
    int p = c;
    RREAL best = fabs(A[(size_t)c * n + c]);
    for (int r = c + 1; r < n; ++r) {
      RREAL v = fabs(A[(size_t)r * n + c]);
      if (v > best) { best = v; p = r; }
    }
    if (best == 0) return -1;
    piv[c] = p;
    if (p != c)
      for (int j = 0; j < n; ++j) {
        RREAL t = A[(size_t)c * n + j];
        A[(size_t)c * n + j] = A[(size_t)p * n + j];
        A[(size_t)p * n + j] = t;
      }
    for (int r = c + 1; r < n; ++r) {
      RREAL f = A[(size_t)r * n + c] / A[(size_t)c * n + c];
      A[(size_t)r * n + c] = f;
      for (int j = c + 1; j < n; ++j) A[(size_t)r * n + j] -= f * A[(size_t)c * n + j];
    }
  }
  return 0;
}

static void lu_solve(int n, const RREAL *A, const int *piv, REAL *b) {
  for (int c = 0; c < n; ++c) {
    int p = piv[c];
    if (p != c) { REAL t = b[c]; b[c] = b[p]; b[p] = t; }
    for (int r = c + 1; r < n; ++r) b[r] -= A[(size_t)r * n + c] * b[c];
  }
  for (int r = n - 1; r >= 0; --r) {
    REAL s = b[r];
    for (int j = r + 1; j < n; ++j) s -= A[(size_t)r * n + j] * b[j];
    b[r] = s / A[(size_t)r * n + r];
  }
}

/* ---------------------------------------------------------------------- */
/* y-derivative of the M values f_1..f_M of one x-line (spacing h).        */
/* L160: "zeta_y [is] computed by fitting a cubic spline through the points */
/* zeta_{k,1..M}".  End conditions are not printed; reading Q3: clamped     */
/* zero slope at y_1 when y_1 = 0 (the y -> -y images of L107-109 assume an  */
/* even extension), otherwise not-a-knot; not-a-knot at y_M.  The unknowns   */
/* are the knot slopes m_l = S'(y_l).  With d_l = (f_{l+1}-f_l)/h:           */
/*   C2 continuity at interior knots:  m_{l-1} + 4 m_l + m_{l+1} = 3(d_{l-1}+d_l) */
/*   not-a-knot (S''' continuous) at y_2:     m_1 - m_3 = 2(d_1 - d_2)       */
/*   not-a-knot at y_{M-1}:          m_{M-2} - m_M = 2(d_{M-2} - d_{M-1})    */
/* The matrix does not depend on f: it is factorised once per call.          */
typedef struct { int M; int clamped_first; RREAL *LU; int *piv; } spline_t;

static int spline_setup(spline_t *s, int M, int clamped_first) {
  s->M = M; s->clamped_first = clamped_first;
  s->LU = (RREAL *)calloc((size_t)M * M, sizeof(RREAL));
  s->piv = (int *)calloc((size_t)M, sizeof(int));
  if (!s->LU || !s->piv) return -1;
  RREAL *A = s->LU;
  if (clamped_first) {
    A[0] = 1;                                   /* m_1 = 0 */
  } else {
    A[0] = 1; A[2] = -1;                        /* m_1 - m_3 = 2(d_1 - d_2) */
  }
  for (int l = 1; l < M - 1; ++l) {
    A[(size_t)l * M + l - 1] = 1; A[(size_t)l * M + l] = 4; A[(size_t)l * M + l + 1] = 1;
  }
  A[(size_t)(M - 1) * M + M - 3] = 1; A[(size_t)(M - 1) * M + M - 1] = -1;
  return lu_factor(M, A, s->piv);
}

static void spline_free(spline_t *s) { free(s->LU); free(s->piv); }

/* f, m: strided by `stride` (one x-line of a node array). rhs: scratch [M]. */
static void spline_slopes(const spline_t *s, REAL h, const REAL *f, size_t stride, REAL *m,
                          REAL *rhs) {
  int M = s->M;
#define F_(l) f[(size_t)(l) * stride]
#define D_(l) ((F_((l) + 1) - F_(l)) / h)
  rhs[0] = s->clamped_first ? (REAL)0 : 2 * (D_(0) - D_(1));
  for (int l = 1; l < M - 1; ++l) rhs[l] = 3 * (D_(l - 1) + D_(l));
  rhs[M - 1] = 2 * (D_(M - 3) - D_(M - 2));
  lu_solve(M, s->LU, s->piv, rhs);
  for (int l = 0; l < M; ++l) m[(size_t)l * stride] = rhs[l];
#undef D_
}

/* Reading Q3, dy_scheme = 1 ("finite differences", BASELINE.json north_star): */
/* central differences inside; at y_1: 0 if y_1 = 0 (symmetry) else 3-point    */
/* one-sided; at y_M: 3-point one-sided.                                        */
static void fd_slopes(int M, int sym_first, REAL h, const REAL *f, size_t stride, REAL *m) {
  m[0] = sym_first ? (REAL)0 : (-3 * F_(0) + 4 * F_(1) - F_(2)) / (2 * h);
  for (int l = 1; l < M - 1; ++l) m[(size_t)l * stride] = (F_(l + 1) - F_(l - 1)) / (2 * h);
  m[(size_t)(M - 1) * stride] = (3 * F_(M - 1) - 4 * F_(M - 2) + F_(M - 3)) / (2 * h);
#undef F_
}

/* ---------------------------------------------------------------------- */
static void fields_free(fields_t *f) {
  free(f->x); free(f->y); free(f->zeta); free(f->phi);
  free(f->zeta_x); free(f->phi_x); free(f->zeta_y); free(f->phi_y);
  memset(f, 0, sizeof *f);
}

/* Entry idx of the state: u[idx], or u[idx] + i h v[idx] in the complex-step build. */
#ifdef CSTEP
#define UVAL(arr_u, arr_v, idx) ((REAL)(arr_u)[idx] + _Complex_I * (cs_h * (RREAL)(arr_v)[idx]))
#else
#define UVAL(arr_u, arr_v, idx) ((REAL)(arr_u)[idx])
#endif

/* Steps 1-3 of the residual: unpack u, x-trapezoid, y-derivatives.  (v, cs_h): the
 * complex-step direction and step; used by the CSTEP build only. */
static int fields_build(const sws_oracle_params *p, const double *u, const double *v, RREAL cs_h,
                        fields_t *f) {
  (void)v; (void)cs_h;
  int N = p->N, M = p->M;
  size_t S = (size_t)N * M;
  memset(f, 0, sizeof *f);
  f->N = N; f->M = M;
  f->x = (REAL *)malloc(N * sizeof(REAL)); f->y = (REAL *)malloc(M * sizeof(REAL));
  f->zeta = (REAL *)malloc(S * sizeof(REAL)); f->phi = (REAL *)malloc(S * sizeof(REAL));
  f->zeta_x = (REAL *)malloc(S * sizeof(REAL)); f->phi_x = (REAL *)malloc(S * sizeof(REAL));
  f->zeta_y = (REAL *)malloc(S * sizeof(REAL)); f->phi_y = (REAL *)malloc(S * sizeof(REAL));
  if (!f->x || !f->y || !f->zeta || !f->phi || !f->zeta_x || !f->phi_x || !f->zeta_y || !f->phi_y) {
    fields_free(f); return -2;
  }
  REAL dx = (REAL)p->dx, dy = (REAL)p->dy;
  /* L145: regular mesh.  x_k = x_1 + (k-1) dx evaluated in double (the mesh  */
  /* is an FP64 input of the problem), then widened.                          */
  for (int k = 0; k < N; ++k) f->x[k] = (REAL)(p->x1 + (double)k * p->dx);
  for (int l = 0; l < M; ++l) f->y[l] = (REAL)(p->y1 + (double)l * p->dy);

  /* eq. (18): u = [phi_{1,l}, (phi_x)_{1..N,l}]_{l=1..M}, then the same for zeta. */
  const size_t off_zeta = (size_t)(N + 1) * M;
  for (int l = 0; l < M; ++l) {
    const size_t lp = (size_t)l * (N + 1), lz = off_zeta + (size_t)l * (N + 1);
    for (int k = 0; k < N; ++k) {
      f->phi_x[AT(k, l)] = UVAL(u, v, lp + 1 + k);
      f->zeta_x[AT(k, l)] = UVAL(u, v, lz + 1 + k);
    }
    /* eq. (19): zeta_{k+1,l} = zeta_{k,l} + (dx/2)((zeta_x)_{k,l} + (zeta_x)_{k+1,l}); */
    /* L160: "Values of phi ... similarly computed using phi_x".                             */
    f->phi[AT(0, l)] = UVAL(u, v, lp);
    f->zeta[AT(0, l)] = UVAL(u, v, lz);
    for (int k = 0; k + 1 < N; ++k) {
      f->zeta[AT(k + 1, l)] = f->zeta[AT(k, l)] + (dx / 2) * (f->zeta_x[AT(k, l)] + f->zeta_x[AT(k + 1, l)]);
      f->phi[AT(k + 1, l)] = f->phi[AT(k, l)] + (dx / 2) * (f->phi_x[AT(k, l)] + f->phi_x[AT(k + 1, l)]);
    }
  }
  /* L160: y-derivatives along each x-line k. */
  int sym = (p->y1 == 0.0);
  if (p->dy_scheme == 0) {
    spline_t sp;
    if (spline_setup(&sp, M, sym) != 0) { spline_free(&sp); fields_free(f); return -3; }
    REAL *rhs = (REAL *)malloc(M * sizeof(REAL));
    for (int k = 0; k < N; ++k) {
      spline_slopes(&sp, dy, f->zeta + k, (size_t)N, f->zeta_y + k, rhs);
      spline_slopes(&sp, dy, f->phi + k, (size_t)N, f->phi_y + k, rhs);
    }
    free(rhs); spline_free(&sp);
  } else {
    for (int k = 0; k < N; ++k) {
      fd_slopes(M, sym, dy, f->zeta + k, (size_t)N, f->zeta_y + k);
      fd_slopes(M, sym, dy, f->phi + k, (size_t)N, f->phi_y + k);
    }
  }
  return 0;
}

/* ---------------------------------------------------------------------- */
/* Kernels at one source node (x,y) for one target (x*,y*)  (L107, L109, L169-172).
 * K1 is garbled in PAPER.md L107 (both denominators printed with (y-y*)^2);
 * reading Q1: the second (image) term has (y+y*)^2 in the denominator, as in
 * K2 (L109), S2 (L172) and K3 (L139).  Reading Q2: zeta_x, zeta_y in K1 are
 * taken at the source node (x,y). */
static void pair_kernels(REAL x, REAL y, REAL zeta, REAL zeta_x, REAL zeta_y,
                         REAL xs, REAL ys, REAL zetas, REAL A, REAL B, REAL C,
                         REAL *K1, REAL *K2, REAL *S2) {
  REAL ddx = x - xs, dm = y - ys, dp = y + ys, dz = zeta - zetas;
  REAL Rm2 = ddx * ddx + dm * dm + dz * dz;   /* direct */
  REAL Rp2 = ddx * ddx + dp * dp + dz * dz;   /* image y* -> -y* */
  REAL Rm = sqrt(Rm2), Rp = sqrt(Rp2);
  *K1 = (dz - ddx * zeta_x - dm * zeta_y) / (Rm2 * Rm) + (dz - ddx * zeta_x - dp * zeta_y) / (Rp2 * Rp);
  *K2 = 1 / Rm + 1 / Rp;
  *S2 = 1 / sqrt(A * ddx * ddx + B * ddx * dm + C * dm * dm)      /* (21) L169 */
      + 1 / sqrt(A * ddx * ddx - B * ddx * dp + C * dp * dp);     /* (22) L172 */
}

/* Antiderivative G(s,t) with d^2G/ds dt = 1/sqrt(A s^2 + B s t + C t^2)
 * (reading Q5; the paper only says "exactly in terms of logarithms", L187).
 * D = 4AC - B^2 > 0.  A term whose prefactor (t or s) is 0 is 0. */
static REAL G_antiderivative(REAL A, REAL B, REAL C, REAL s, REAL t) {
  REAL D = 4 * A * C - B * B, g = 0;
  if (t != 0) g += (t / sqrt(A)) * asinh((2 * A * s + B * t) / (fabs(t) * sqrt(D)));
  if (s != 0) g += (s / sqrt(C)) * asinh((2 * C * t + B * s) / (fabs(s) * sqrt(D)));
  return g;
}

static REAL box_integral(REAL A, REAL B, REAL C, REAL s1, REAL s2, REAL t1, REAL t2) {
  return G_antiderivative(A, B, C, s2, t2) - G_antiderivative(A, B, C, s1, t2)
       - G_antiderivative(A, B, C, s2, t1) + G_antiderivative(A, B, C, s1, t1);
}

/* eq. (23): I = int_{y_1}^{y_M} int_{x_1}^{x_N} S2 dx dy, both terms of S2.
 * Direct term: s = x - x*, t = y - y*.  Image term: t' = -(y + y*), which maps
 * A s^2 - B s (y+y*) + C (y+y*)^2 onto A s^2 + B s t' + C t'^2. */
static REAL S2_integral(REAL A, REAL B, REAL C, REAL xs, REAL ys, REAL xa, REAL xb, REAL ya, REAL yb) {
  return box_integral(A, B, C, xa - xs, xb - xs, ya - ys, yb - ys)
       + box_integral(A, B, C, xa - xs, xb - xs, -(yb + ys), -(ya + ys));
}

/* Starred (half-mesh) value by two-point interpolation, L162 / L454. */
#define STAR(arr, k, l) (((arr)[AT(k, l)] + (arr)[AT((k) + 1, l)]) / 2)

/* Trapezoid weight w(i,j) = dx dy c_i c_j, c = 1/2 on the first/last index (L189, reading Q4). */
static REAL weight(const sws_oracle_params *p, int i, int j) {
  REAL ci = (i == 0 || i == p->N - 1) ? (REAL)0.5 : (REAL)1;
  REAL cj = (j == 0 || j == p->M - 1) ? (REAL)0.5 : (REAL)1;
  return (REAL)p->dx * (REAL)p->dy * ci * cj;
}

/* A, B, C of L177 at the half-mesh point (k, l): the coefficients of the quadratic form
 *   A (x - x*)^2 + B (x - x*)(y - y*) + C (y - y*)^2
 * under the square root of S2 (L169-172), from the starred slopes.  The ONE place they are
 * formed: E2_row, E2_terms and sws_oracle_row_abc all call this.
 * Pin (test_PS_S2_is_the_singular_part_of_K2): S2 exists to cancel the 1/R singularity of K2
 * at the target, so R^2 = Q + O(h^3) at the nodes next to it, i.e. h (K2 - S2) -> 0 under
 * mesh refinement - which holds only for these A, B, C. */
static void star_ABC(const fields_t *f, int k, int l, REAL *A, REAL *B, REAL *C) {
  int N = f->N;
  REAL zxs = STAR(f->zeta_x, k, l), zys = STAR(f->zeta_y, k, l);
  *A = 1 + zxs * zxs; *B = 2 * zxs * zys; *C = 1 + zys * zys; /* L177 */
}

/* The six pieces of E2_{k,l} (0-based k = 0..N-2, l = 0..M-1):
 * out[0] = 2 pi (phi* - x*)
 * out[1] = eps / sqrt(x*^2 + y*^2 + (zeta* + 1)^2)
 * out[2] = sum w (phi_ij - phi* - x_i + x*) K1
 * out[3] = sum w (zeta_x)_ij K2
 * out[4] = sum w S2
 * out[5] = I
 * E2 = out0 + out1 - out2 - (out3 - zeta_x* out4) - zeta_x* out5
 * (eq. (12) L101 moved to one side with the sign convention of B.1 L431). */
static void E2_terms(const sws_oracle_params *p, const fields_t *f, int k, int l, REAL out[6], REAL *zxs_out) {
  int N = f->N, M = f->M;
  REAL xs = (f->x[k] + f->x[k + 1]) / 2, ys = f->y[l];        /* L162 */
  REAL zs = STAR(f->zeta, k, l), ps = STAR(f->phi, k, l);
  REAL zxs = STAR(f->zeta_x, k, l);
  REAL A, B, C;
  star_ABC(f, k, l, &A, &B, &C);
  REAL s1 = 0, s2 = 0, s3 = 0;
  for (int j = 0; j < M; ++j)
    for (int i = 0; i < N; ++i) {
      REAL K1, K2, S2, w = weight(p, i, j);
      pair_kernels(f->x[i], f->y[j], f->zeta[AT(i, j)], f->zeta_x[AT(i, j)], f->zeta_y[AT(i, j)],
                   xs, ys, zs, A, B, C, &K1, &K2, &S2);
      s1 += w * (f->phi[AT(i, j)] - ps - f->x[i] + xs) * K1;
      s2 += w * f->zeta_x[AT(i, j)] * K2;
      s3 += w * S2;
    }
  out[0] = 2 * PI_R * (ps - xs);
  out[1] = (REAL)p->eps / sqrt(xs * xs + ys * ys + (zs + 1) * (zs + 1));
  out[2] = s1; out[3] = s2; out[4] = s3;
  out[5] = S2_integral(A, B, C, xs, ys, f->x[0], f->x[N - 1], f->y[0], f->y[M - 1]);
  *zxs_out = zxs;
}

/* E2_{k,l}: the integral equation (12) L101 with the singularity subtraction of
 * L181: sum w [ (phi - phi* - x + x*) K1 + zeta_x K2 - zeta_x* S2 ] + zeta_x* I. */
static REAL E2_row(const sws_oracle_params *p, const fields_t *f, int k, int l) {
  int N = f->N, M = f->M;
  REAL xs = (f->x[k] + f->x[k + 1]) / 2, ys = f->y[l];
  REAL zs = STAR(f->zeta, k, l), ps = STAR(f->phi, k, l);
  REAL zxs = STAR(f->zeta_x, k, l);
  REAL A, B, C;
  star_ABC(f, k, l, &A, &B, &C);
  REAL sum = 0;
  for (int j = 0; j < M; ++j)
    for (int i = 0; i < N; ++i) {
      REAL K1, K2, S2;
      pair_kernels(f->x[i], f->y[j], f->zeta[AT(i, j)], f->zeta_x[AT(i, j)], f->zeta_y[AT(i, j)],
                   xs, ys, zs, A, B, C, &K1, &K2, &S2);
      sum += weight(p, i, j) * ((f->phi[AT(i, j)] - ps - f->x[i] + xs) * K1
                                + f->zeta_x[AT(i, j)] * K2 - zxs * S2);
    }
  /* I of eq. (23); named I_S2 because <tgmath.h> defines the macro I. */
  REAL I_S2 = S2_integral(A, B, C, xs, ys, f->x[0], f->x[N - 1], f->y[0], f->y[M - 1]);
  return 2 * PI_R * (ps - xs) + (REAL)p->eps / sqrt(xs * xs + ys * ys + (zs + 1) * (zs + 1))
       - sum - zxs * I_S2;
}

/* E1_{k,l}: Bernoulli, eq. (13), at the starred values (reading Q6: average
 * nodal values first, then evaluate). */
static REAL E1_row(const sws_oracle_params *p, const fields_t *f, int k, int l) {
  int N = f->N;
  REAL zs = STAR(f->zeta, k, l);
  REAL zx = STAR(f->zeta_x, k, l), zy = STAR(f->zeta_y, k, l);
  REAL px = STAR(f->phi_x, k, l), py = STAR(f->phi_y, k, l);
  REAL F2 = (REAL)p->froude * (REAL)p->froude;
  return ((1 + zx * zx) * py * py + (1 + zy * zy) * px * px - 2 * zx * zy * px * py)
             / (1 + zx * zx + zy * zy) / 2
       + zs / F2 - (REAL)0.5;
}

/* Residual in App. A order (L421):
 *   first half, per l:  [E3_l, E4_l, E1_{1..N-1,l}];  second half: [E5_l, E6_l, E2_{1..N-1,l}].
 * rows (optional): flat target indices t = l*(N-1) + k whose E2 is wanted;
 * every other E2 entry is NaN.  rows == NULL: all.  Output widened REAL. */
static int residual_cs(const sws_oracle_params *p, const double *u, const double *v, RREAL cs_h,
                       const int *rows, int nrows, REAL *E) {
  int N = p->N, M = p->M;
  if (N < 3 || M < 4 || !(p->dx > 0) || !(p->dy > 0)) return -1;
  fields_t f;
  int rc = fields_build(p, u, v, cs_h, &f);
  if (rc) return rc;
  size_t half = (size_t)(N + 1) * M;
  REAL x1 = f.x[0], n = (REAL)p->n_rad, dx = (REAL)p->dx;
  for (int l = 0; l < M; ++l) {
    REAL *e = E + (size_t)l * (N + 1), *e2 = E + half + (size_t)l * (N + 1);
    /* eq. (24) L191-197 / App. A; second derivatives by forward difference */
    /* of the first derivative (L201, printed explicitly in B.1 L431).           */
    e[0] = x1 * (f.phi_x[AT(0, l)] - 1) + n * (f.phi[AT(0, l)] - x1);                     /* E3 */
    e[1] = x1 * ((f.phi_x[AT(1, l)] - f.phi_x[AT(0, l)]) / dx) + n * (f.phi_x[AT(0, l)] - 1); /* E4 */
    e2[0] = x1 * f.zeta_x[AT(0, l)] + n * f.zeta[AT(0, l)];                               /* E5 */
    e2[1] = x1 * ((f.zeta_x[AT(1, l)] - f.zeta_x[AT(0, l)]) / dx) + n * f.zeta_x[AT(0, l)]; /* E6 */
    for (int k = 0; k + 1 < N; ++k) {
      e[2 + k] = E1_row(p, &f, k, l);
      e2[2 + k] = (REAL)NAN;
    }
  }
  int T = (N - 1) * M, cnt = rows ? nrows : T;
#pragma omp parallel for schedule(dynamic, 8)
  for (int r = 0; r < cnt; ++r) {
    int t = rows ? rows[r] : r;
    if (t < 0 || t >= T) continue;
    int l = t / (N - 1), k = t % (N - 1);
    E[half + (size_t)l * (N + 1) + 2 + k] = E2_row(p, &f, k, l);
  }
  fields_free(&f);
  return 0;
}

static int residual_real(const sws_oracle_params *p, const double *u, const int *rows, int nrows, REAL *E) {
  return residual_cs(p, u, u, 0, rows, nrows, E);   /* zero step: the plain residual */
}

/* ============================ exported C-ABI ============================ */

int FN(sws_oracle_residual)(const sws_oracle_params *p, const double *u, const int *rows, int nrows, double *E) {
  size_t n = (size_t)2 * (p->N + 1) * p->M;
  REAL *Er = (REAL *)malloc(n * sizeof(REAL));
  if (!Er) return -2;
  int rc = residual_real(p, u, rows, nrows, Er);
  if (!rc) for (size_t i = 0; i < n; ++i) E[i] = (double)RE(Er[i]);
  free(Er);
  return rc;
}

/* Finite-difference Jacobian action, literally eq. (25):
 *   JV = (E(u_b) - E(u)) / sigma,   u_b = fl64(fma(sigma, v, u))  (reading Q9:
 * the perturbed state is an FP64 vector, formed with ONE rounding per entry).
 * The difference and the division are done in REAL before rounding to double.
 * Epert (optional) receives E(u_b). */
int FN(sws_oracle_jv)(const sws_oracle_params *p, const double *u, const double *v, double sigma,
                      const int *rows, int nrows, double *JV, double *Epert) {
  size_t n = (size_t)2 * (p->N + 1) * p->M;
  double *ub = (double *)malloc(n * sizeof(double));
  REAL *E0 = (REAL *)malloc(n * sizeof(REAL)), *E1 = (REAL *)malloc(n * sizeof(REAL));
  int rc = -2;
  if (ub && E0 && E1) {
    for (size_t i = 0; i < n; ++i) ub[i] = fma(sigma, v[i], u[i]);
    rc = residual_real(p, u, rows, nrows, E0);
    if (!rc) rc = residual_real(p, ub, rows, nrows, E1);
    if (!rc) for (size_t i = 0; i < n; ++i) {
      JV[i] = (double)RE((E1[i] - E0[i]) / (REAL)sigma);
      if (Epert) Epert[i] = (double)RE(E1[i]);
    }
  }
  free(ub); free(E0); free(E1);
  return rc;
}

/* sigma = 1e-7 (1 + ||u||_2) / ||v||_2  (BASELINE.json configs; the paper only says
 * "a suitably-chosen shift [1]", L221). */
double FN(sws_oracle_sigma)(int n, const double *u, const double *v) {
  REAL su = 0, sv = 0;
  for (int i = 0; i < n; ++i) { su += (REAL)u[i] * (REAL)u[i]; sv += (REAL)v[i] * (REAL)v[i]; }
  return (double)RE((REAL)1e-7 * (1 + sqrt(su)) / sqrt(sv));
}

/* --- pieces exposed so that the pins can reach every term separately --- */

/* Nodal fields after steps 1-3; each out array [M*N], index l*N + k. */
int FN(sws_oracle_fields)(const sws_oracle_params *p, const double *u, double *zeta, double *phi,
                          double *zeta_y, double *phi_y) {
  fields_t f;
  int rc = fields_build(p, u, u, 0, &f);
  if (rc) return rc;
  size_t S = (size_t)p->N * p->M;
  for (size_t i = 0; i < S; ++i) {
    zeta[i] = (double)RE(f.zeta[i]); phi[i] = (double)RE(f.phi[i]);
    zeta_y[i] = (double)RE(f.zeta_y[i]); phi_y[i] = (double)RE(f.phi_y[i]);
  }
  fields_free(&f);
  return 0;
}

/* out[0..5] as documented at E2_terms; out[6] = zeta_x*. */
int FN(sws_oracle_e2_terms)(const sws_oracle_params *p, const double *u, int k, int l, double *out) {
  if (k < 0 || k >= p->N - 1 || l < 0 || l >= p->M) return -1;
  fields_t f;
  int rc = fields_build(p, u, u, 0, &f);
  if (rc) return rc;
  REAL o[6], zxs;
  E2_terms(p, &f, k, l, o, &zxs);
  for (int i = 0; i < 6; ++i) out[i] = (double)RE(o[i]);
  out[6] = (double)RE(zxs);
  fields_free(&f);
  return 0;
}

/* out3 = {A, B, C} the rows E2_{k,l} use (0-based k, l), and *zs_out = zeta* (optional). */
int FN(sws_oracle_row_abc)(const sws_oracle_params *p, const double *u, int k, int l, double *out3, double *zs_out) {
  if (k < 0 || k >= p->N - 1 || l < 0 || l >= p->M) return -1;
  fields_t f;
  int rc = fields_build(p, u, u, 0, &f);
  if (rc) return rc;
  int N = f.N;
  REAL A, B, C;
  star_ABC(&f, k, l, &A, &B, &C);
  out3[0] = (double)RE(A); out3[1] = (double)RE(B); out3[2] = (double)RE(C);
  if (zs_out) *zs_out = (double)RE(STAR(f.zeta, k, l));
  fields_free(&f);
  return 0;
}

void FN(sws_oracle_pair_kernels)(double x, double y, double zeta, double zeta_x, double zeta_y,
                                 double xs, double ys, double zetas, double A, double B, double C,
                                 double *out3) {
  REAL K1, K2, S2;
  pair_kernels(x, y, zeta, zeta_x, zeta_y, xs, ys, zetas, A, B, C, &K1, &K2, &S2);
  out3[0] = (double)RE(K1); out3[1] = (double)RE(K2); out3[2] = (double)RE(S2);
}

double FN(sws_oracle_s2_integral)(double A, double B, double C, double xs, double ys,
                                  double xa, double xb, double ya, double yb) {
  return (double)RE(S2_integral(A, B, C, xs, ys, xa, xb, ya, yb));
}

double FN(sws_oracle_box_integral)(double A, double B, double C, double s1, double s2, double t1, double t2) {
  return (double)RE(box_integral(A, B, C, s1, s2, t1, t2));
}

double FN(sws_oracle_weight)(const sws_oracle_params *p, int i, int j) { return (double)RE(weight(p, i, j)); }

/* y-derivative of one line of M samples (spacing h), same routine the residual uses. */
int FN(sws_oracle_dy_line)(int M, double h, int scheme, int first_is_symmetric, const double *f, double *m) {
  REAL *fr = (REAL *)malloc(M * sizeof(REAL)), *mr = (REAL *)malloc(M * sizeof(REAL));
  REAL *rhs = (REAL *)malloc(M * sizeof(REAL));
  int rc = 0;
  for (int l = 0; l < M; ++l) fr[l] = (REAL)f[l];
  if (scheme == 0) {
    spline_t sp;
    rc = spline_setup(&sp, M, first_is_symmetric);
    if (!rc) spline_slopes(&sp, (REAL)h, fr, 1, mr, rhs);
    spline_free(&sp);
  } else {
    fd_slopes(M, first_is_symmetric, (REAL)h, fr, 1, mr);
  }
  for (int l = 0; l < M; ++l) m[l] = (double)RE(mr[l]);
  free(fr); free(mr); free(rhs);
  return rc;
}

int FN(sws_oracle_sizeof_real)(void) { return (int)sizeof(REAL); }


#ifdef CSTEP
/* Exact Jacobian action J(u) v = d/d sigma E(u + sigma v)|_{sigma=0} (the limit of eq. (25)
 * L219), by complex-step differentiation of the residual above:
 *   JV = Im E(u + i h v) / h,   h = 1e-40  (no cancellation; truncation O(h^2)).
 * rows as in sws_oracle_residual (E2 rows not asked for are NaN).  E0 (optional) receives
 * Re E(u + i h v) = E(u) + O(h^2). */
int FN(sws_oracle_jv_exact)(const sws_oracle_params *p, const double *u, const double *v,
                            const int *rows, int nrows, double *JV, double *E0) {
  size_t n = (size_t)2 * (p->N + 1) * p->M;
  const RREAL h = 1e-40L;
  REAL *Ec = (REAL *)malloc(n * sizeof(REAL));
  if (!Ec) return -2;
  int rc = residual_cs(p, u, v, h, rows, nrows, Ec);
  if (!rc) for (size_t i = 0; i < n; ++i) {
    RREAL re = creall(Ec[i]);
    JV[i] = (re != re) ? (double)NAN : (double)(cimagl(Ec[i]) / h);
    if (E0) E0[i] = (double)re;
  }
  free(Ec);
  return rc;
}
#endif
