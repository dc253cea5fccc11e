// Device primitives shared by the all-pairs kernels (sws_allpairs.cu, sws_allpairs_f32.cu): the FP64
// reciprocal square root and the far-field (Euler-Maclaurin) form of the S2 column sums.
// Citations "L<n>" are lines of /root/reference/PAPER.md; "Qn" are DESIGN.md readings.
#pragma once
#include <cuda_runtime.h>

#include "sws_internal.cuh"

namespace sws {

// 1/sqrt(x) for normal positive x, full double precision.
// Seed: MUFU.RSQ64H (PTX rsqrt.approx.ftz.f64: works on the upper 32 bits of x, so the seed
// carries a relative error d with |d| < ~2^-20).  With e = 1 - x y0^2 (= -2d - d^2) the
// exact result is y0 (1 - e)^(-1/2) = y0 (1 + e/2 + 3e^2/8 + 5e^3/16 + ...); the two-term
// correction below leaves 5/16 |e|^3 < 2^-59, i.e. below the rounding of the final FMA.
// 5 FP64 instructions (DMUL, DFMA, DFMA, DMUL, DFMA) + 1 MUFU.
//
// Operand shapes matter on B200: a DFMA with three DISTINCT register sources issues every
// 3 cycles per SM sub-partition, one with <= 2 distinct registers (a repeated operand, an
// immediate) every 2 (measured).  Every step
// here is written with at most two distinct registers: the last one is
// y0 + y0 * (e p) = fma(y0, e p, y0), not fma(y0 e, p, y0).
__device__ __forceinline__ double rsqrt_seed(double x) {
#ifdef SWS_RSQRT_F32SEED
  // Experiment of round 2: FP32 seed, cvt + MUFU.RSQ + cvt instead of MUFU.RSQ64H + the
  // move that zeroes its low word.  Measured slower at 721x241: 59.9 against 54.5 ms per launch (the two F2F
  // conversions cost more issue than the move they save); kept behind this build flag for the record, off.
  float xf, yf;
  asm("cvt.rn.f32.f64 %0, %1;" : "=f"(xf) : "d"(x));
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(yf) : "f"(xf));
  double y;
  asm("cvt.f64.f32 %0, %1;" : "=d"(y) : "f"(yf));
  return y;
#else
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
#endif
}

// The same with the seed's low word taken from `lo` instead of being zeroed (any value does: the seed carries 20
// bits anyway).  When `lo` is the low word of a value that dies where x is formed, ptxas writes the MUFU result
// into that value's register pair and the move that zeroes the low word disappears.
__device__ __forceinline__ double rsqrt_fp64_lo(double x, int lo) {
  const double y0 = __hiloint2double(__double2hiint(rsqrt_seed(x)), lo);
  const double t = x * y0;
  const double e = fma(-t, y0, 1.0);
  const double p = fma(0.375, e, 0.5);
  const double w = e * p;
  return fma(y0, w, y0);
}

__device__ __forceinline__ double rsqrt_fp64(double x) {
  const double y0 = rsqrt_seed(x);
  const double t = x * y0;
  const double e = fma(-t, y0, 1.0);
  const double p = fma(0.375, e, 0.5);
  const double w = e * p;
  return fma(y0, w, y0);
}

// ---------------------------------------------------------------------------------------
// Far-field form of the S2 column sums.
//
// For one target and one source column the S2 terms of the quadrature are, up to 1/sqrt(C),
//     sum_j c_j [ f(y_j; c) + f(y_j; -c) ],   f(y; c) = ((y - c)^2 + g)^(-1/2),
// a composite trapezoid sum (step dy, c_j = 1/2 at both ends, reading Q4) of a function that
// does NOT depend on the source data: c and g depend on the target's A, B, C and on x_i - x*
// only.  f is analytic with its nearest singularities at y = c +- i sqrt(g), sqrt(g) ~ |x_i - x*|,
// so once sqrt(g) >= r dy the sum equals its Euler-Maclaurin expansion to round-off:
//     dy sum_j c_j f(y_j) = int_a^b f dy + sum_{k=1..K} B_2k dy^2k / (2k)! (f^(2k-1)(b) - f^(2k-1)(a)) + R_K,
//     int f dy = asinh((y - c) / sqrt(g)),
//     f^(n)(y) = (-1)^n n! P_n(mu) / rho^(n+1),  rho = sqrt((y-c)^2 + g), mu = (y - c) / rho
// (P_n = Legendre polynomial: 1/rho is the generating function of P_n), i.e. the k-th term is
//     -(B_2k / 2k) (dy / rho)^2k P_{2k-1}(mu)  at b minus the same at a.
// With K = 7 and r = 8 the remainder is < 1e-16 / sqrt(g) (measured against 50-digit sums over
// the whole range of c), below the rounding of the direct sum itself.
// The same quantity, evaluated another way: the result still matches the oracle's plain sum.
// Cost: 216 FP64 instructions per (target, column) in SASS (y1 = 0 form: 100 DFMA + 93 DMUL + 23 DADD = 2 x 59 for
// the end-point tails, the rest one log1p and two divisions; counted with cuobjdump) instead of 16 per pair
// x M pairs: 0.9 per pair at M = 241.
// (default r = kEmRadius of sws_internal.cuh; sws_set_farfield changes it, r <= 0 sums directly)

// sum_{k=1..K} (B_2k / 2k) s^k P_{2k-1}(mu) at the end point u = y_e - c, s = (dy / rho)^2;  *rho = sqrt(u^2 + g).
// K = 7 in general (s <= 1/64 at the far-field radius).  Most end points are much farther from the target than the
// radius, and the series is cut where its next term is below 1e-18: K = 3 when s <= 1e-4 (rho >= 100 dy; next term
// s^4 / 240 <= 4e-19), K = 5 when s <= 1.5e-3 (rho >= 26 dy; next term 0.021 s^6 <= 3e-19).  The choice depends on
// the lane's own s only (lanes of a warp are neighbouring targets and mostly agree).
__device__ __forceinline__ double em_tail(const double u, const double g, const double h2, double* rho) {
  const double r2 = fma(u, u, g);
  const double ri = rsqrt_fp64(r2);
  *rho = r2 * ri;
  const double mu = u * ri;
  const double s = h2 * (ri * ri);
  double P[14];
  P[0] = 1.0;
  P[1] = mu;
#pragma unroll
  for (int n = 1; n <= 4; ++n)  // (n+1) P_{n+1} = (2n+1) mu P_n - n P_{n-1}
    P[n + 1] = ((2.0 * n + 1.0) / (n + 1.0)) * (mu * P[n]) - (n / (n + 1.0)) * P[n - 1];
#ifndef SWS_EM_FULL_SERIES
  if (s <= 1e-4) {
    double t = (1.0 / 252.0) * P[5];            // B_6 / 6
    t = fma(s, t, (-1.0 / 120.0) * P[3]);       // B_4 / 4
    t = fma(s, t, (1.0 / 12.0) * P[1]);         // B_2 / 2
    return s * t;
  }
#endif
#pragma unroll
  for (int n = 5; n <= 8; ++n)
    P[n + 1] = ((2.0 * n + 1.0) / (n + 1.0)) * (mu * P[n]) - (n / (n + 1.0)) * P[n - 1];
#ifndef SWS_EM_FULL_SERIES
  if (s <= 1.5e-3) {
    double t = (1.0 / 132.0) * P[9];            // B_10 / 10
    t = fma(s, t, (-1.0 / 240.0) * P[7]);       // B_8 / 8
    t = fma(s, t, (1.0 / 252.0) * P[5]);
    t = fma(s, t, (-1.0 / 120.0) * P[3]);
    t = fma(s, t, (1.0 / 12.0) * P[1]);
    return s * t;
  }
#endif
#pragma unroll
  for (int n = 9; n <= 12; ++n)
    P[n + 1] = ((2.0 * n + 1.0) / (n + 1.0)) * (mu * P[n]) - (n / (n + 1.0)) * P[n - 1];
  double t = (1.0 / 12.0) * P[13];              // B_14 / 14
  t = fma(s, t, (-691.0 / 32760.0) * P[11]);    // B_12 / 12
  t = fma(s, t, (1.0 / 132.0) * P[9]);          // B_10 / 10
  t = fma(s, t, (-1.0 / 240.0) * P[7]);         // B_8 / 8
  t = fma(s, t, (1.0 / 252.0) * P[5]);          // B_6 / 6
  t = fma(s, t, (-1.0 / 120.0) * P[3]);         // B_4 / 4
  t = fma(s, t, (1.0 / 12.0) * P[1]);           // B_2 / 2
  return s * t;
}

// dy * (trapezoid sum of f(.; c) over the nodes a, a + dy, ..., b), by the expansion above
__device__ __forceinline__ double em_interval(const double a, const double b, const double c, const double g,
                                              const double h2) {
  const double ua = a - c, ub = b - c;
  double rhoa, rhob;
  const double ta = em_tail(ua, g, h2, &rhoa);
  const double tb = em_tail(ub, g, h2, &rhob);
  // asinh(ub / sqrt g) - asinh(ua / sqrt g) = log(q),  q = L(ub) / L(ua),  L(u) = u + rho = g / (rho - u),
  // each L taken in the form without cancellation.  q - 1 = (L(ub) - L(ua)) / L(ua) with
  // L(ub) - L(ua) = (b - a) (L(ua) + L(ub)) / (rho_a + rho_b), so log(q) = log1p((b - a)(1 + q) / (rho_a + rho_b))
  // keeps full relative accuracy when the interval is short against sqrt(g) (q -> 1).
  const double nb = ub >= 0.0 ? ub + rhob : g, db = ub >= 0.0 ? 1.0 : rhob - ub;
  const double na = ua >= 0.0 ? ua + rhoa : g, da = ua >= 0.0 ? 1.0 : rhoa - ua;
  // (b - a)(1 + q) / (rho_a + rho_b) with q = (nb da) / (db na), as ONE quotient of sums of positive products
  const double den = db * na;
  return log1p((b - a) * fma(nb, da, den) / ((rhoa + rhob) * den)) - (tb - ta);
}

struct EmGeom {
  double y1, yM;   // first and last node of a column
  double h2, inv_h;  // dy^2, 1 / dy
  double gmin;     // (r dy)^2; a column is "far" for a target when g >= gmin  (inf: never)
  int sym;         // y1 == 0: direct + image = one trapezoid sum over [-yM, yM]
};

// sum_j c_j [ f(y_j; c) + f(y_j; -c) ]  (unit node weights, as the direct loop accumulates it)
__device__ __forceinline__ double s2_column_em(const EmGeom& e, const double c, const double g) {
  const double v = e.sym ? em_interval(-e.yM, e.yM, c, g, e.h2)
                         : em_interval(e.y1, e.yM, c, g, e.h2) + em_interval(e.y1, e.yM, -c, g, e.h2);
  return v * e.inv_h;
}

// ---------------------------------------------------------------------------------------
// The same for the sums the analytic Jacobian action needs (sws_jv_exact.cu): with u = f(y; c),
// s = y - c,
//     F0 = sum c_j u,   F3 = sum c_j u^3,   F3s = sum c_j s u^3        (data independent as well).
// Integrals: int u = asinh(s / sqrt g), int u^3 = s / (g rho) = mu / g, int s u^3 = -1 / rho.
// End corrections, from f^(n) above and from u^3 = -2 du/dg, s u^3 = -du/ds:
//     u     : -(B_2k / 2k) (dy/rho)^2k P_{2k-1}(mu)
//     u^3   : -(B_2k / 2k) (dy/rho)^2k P'_{2k}(mu) / rho^2        (mu P'_n + (n+1) P_n = P'_{n+1})
//     s u^3 : - B_2k       (dy/rho)^2k P_{2k}(mu)  / rho
// K = 7, same radius: remainders < 2e-17, 2e-16, 4e-15 of the respective sums at r = 8 (50-digit check).
struct Em3 {
  double f0, f3, f3s;
};

__device__ __forceinline__ Em3 em_tail3(const double u, const double g, const double h2, double* rho, double* ri_o,
                                        double* mu_o) {
  const double r2 = fma(u, u, g);
  const double ri = rsqrt_fp64(r2);
  *rho = r2 * ri;
  *ri_o = ri;
  const double mu = u * ri;
  *mu_o = mu;
  const double s = h2 * (ri * ri);
  double P[15], D[15];  // P_n(mu), P'_n(mu)
  P[0] = 1.0; P[1] = mu;
  D[0] = 0.0; D[1] = 1.0;
#pragma unroll
  for (int n = 1; n <= 13; ++n) {
    P[n + 1] = ((2.0 * n + 1.0) / (n + 1.0)) * (mu * P[n]) - (n / (n + 1.0)) * P[n - 1];
    D[n + 1] = fma(mu, D[n], (n + 1.0) * P[n]);
  }
  constexpr double c1 = 1.0 / 12.0, c2 = -1.0 / 120.0, c3 = 1.0 / 252.0, c4 = -1.0 / 240.0, c5 = 1.0 / 132.0,
                   c6 = -691.0 / 32760.0, c7 = 1.0 / 12.0;  // B_2k / 2k
  Em3 t;
  double a = c7 * P[13];
  a = fma(s, a, c6 * P[11]); a = fma(s, a, c5 * P[9]); a = fma(s, a, c4 * P[7]);
  a = fma(s, a, c3 * P[5]); a = fma(s, a, c2 * P[3]); a = fma(s, a, c1 * P[1]);
  t.f0 = s * a;
  a = c7 * D[14];
  a = fma(s, a, c6 * D[12]); a = fma(s, a, c5 * D[10]); a = fma(s, a, c4 * D[8]);
  a = fma(s, a, c3 * D[6]); a = fma(s, a, c2 * D[4]); a = fma(s, a, c1 * D[2]);
  t.f3 = (s * a) * (ri * ri);
  a = (14.0 * c7) * P[14];  // B_2k = 2k (B_2k / 2k)
  a = fma(s, a, (12.0 * c6) * P[12]); a = fma(s, a, (10.0 * c5) * P[10]); a = fma(s, a, (8.0 * c4) * P[8]);
  a = fma(s, a, (6.0 * c3) * P[6]); a = fma(s, a, (4.0 * c2) * P[4]); a = fma(s, a, (2.0 * c1) * P[2]);
  t.f3s = (s * a) * ri;
  return t;
}

// dy * (trapezoid sums of u, u^3, s u^3 over the nodes a, a + dy, ..., b) for the centre c
__device__ __forceinline__ Em3 em_interval3(const double a, const double b, const double c, const double g,
                                            const double h2) {
  const double ua = a - c, ub = b - c;
  double rhoa, rhob, ria, rib, mua, mub;
  const Em3 ta = em_tail3(ua, g, h2, &rhoa, &ria, &mua);
  const Em3 tb = em_tail3(ub, g, h2, &rhob, &rib, &mub);
  const double nb = ub >= 0.0 ? ub + rhob : g, db = ub >= 0.0 ? 1.0 : rhob - ub;
  const double na = ua >= 0.0 ? ua + rhoa : g, da = ua >= 0.0 ? 1.0 : rhoa - ua;
  const double q = (nb * da) / (db * na);
  Em3 r;
  r.f0 = log1p((b - a) * (1.0 + q) / (rhoa + rhob)) - (tb.f0 - ta.f0);
  r.f3 = (mub - mua) / g - (tb.f3 - ta.f3);
  r.f3s = (ria - rib) - (tb.f3s - ta.f3s);
  return r;
}

// Unit-node-weight column sums, direct + image:
//   f0 = sum c_j (u- + u+),  f3 = sum c_j (u-^3 + u+^3),  f3s = sum c_j (s- u-^3 - s+ u+^3),  s-+ = y_j -+ c
__device__ __forceinline__ Em3 s2_column_em3(const EmGeom& e, const double c, const double g) {
  Em3 r;
  if (e.sym) {  // one trapezoid sum over [-yM, yM]; the image half contributes -s+ u+^3
    r = em_interval3(-e.yM, e.yM, c, g, e.h2);
  } else {
    const Em3 d = em_interval3(e.y1, e.yM, c, g, e.h2), m = em_interval3(e.y1, e.yM, -c, g, e.h2);
    r.f0 = d.f0 + m.f0; r.f3 = d.f3 + m.f3; r.f3s = d.f3s - m.f3s;
  }
  r.f0 *= e.inv_h; r.f3 *= e.inv_h; r.f3s *= e.inv_h;
  return r;
}

// The far/near decision is taken per WARP (all 32 targets of the warp must be far), so the j loop
// has no divergence.  Used by k_allpairs and by the counting kernel of sws_farfield_stats.
__device__ __forceinline__ bool column_is_far(const double g, const double gmin) {
  return __all_sync(0xffffffffu, g >= gmin) != 0;
}

// The all-pairs kernels hand the targets to their threads in TRANSPOSED order, slot = k M + l (k = x index
// of the midpoint, l = y-line), so that the 32 targets of a warp share one x* (two at most): the columns that
// are near for the warp are then the 2 r columns around one target instead of 32 + 2 r.  t = l (N-1) + k is
// the index everything is stored by.
__device__ __forceinline__ int target_of_slot(const int slot, const int N, const int M) {
  const int k = slot / M, l = slot - k * M;
  return l * (N - 1) + k;
}

// Host: the far-field geometry of a context's mesh and its current radius.
inline EmGeom em_geometry(const sws_ctx* c) {
  const Mesh& m = c->mesh;
  EmGeom e;
  e.y1 = m.y1;
  e.yM = m.y1 + (m.M - 1) * m.dy;
  e.h2 = m.dy * m.dy;
  e.inv_h = 1.0 / m.dy;
  const double r = c->em_radius;
  e.gmin = r > 0.0 ? (r * m.dy) * (r * m.dy) : __builtin_inf();
  e.sym = m.sym_first;
  return e;
}

}  // namespace sws
