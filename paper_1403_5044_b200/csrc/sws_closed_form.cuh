// Closed form of I = int int S2 dx dy over the truncated rectangle (eq. (23), reading Q5) and the
// local part of the integral-equation row, shared by sws_fields.cu (FP32 variant, analytic Jacobian action) and
// sws_allpairs.cu (FP64 path: evaluated by an extra CTA row of the all-pairs launch, concurrently with the pair
// loops - 8 asinh per target are ~10 us of dependent latency that a small mesh would otherwise wait for).
#pragma once
#include <math_constants.h>

#include "sws_internal.cuh"

namespace sws {

// a5.  Antiderivative G with d2G/ds dt = 1/sqrt(A s^2 + B s t + C t^2) (reading Q5; the paper
// says only "exactly in terms of logarithms", L187).  D = 4AC - B^2 > 0.  A term whose
// prefactor is 0 is 0 (the limit of t asinh(c/|t|) as t -> 0).
__device__ __forceinline__ double G_anti(double A, double B, double C, double sqA, double sqC, double sqD, double s,
                         double t) {
  double g = 0.0;
  if (t != 0.0) g += (t / sqA) * asinh((2 * A * s + B * t) / (fabs(t) * sqD));
  if (s != 0.0) g += (s / sqC) * asinh((2 * C * t + B * s) / (fabs(s) * sqD));
  return g;
}

__device__ __forceinline__ double box_int(double A, double B, double C, double sqA, double sqC, double sqD,
                          double s1, double s2, double t1, double t2) {
  return G_anti(A, B, C, sqA, sqC, sqD, s2, t2) - G_anti(A, B, C, sqA, sqC, sqD, s1, t2) -
         G_anti(A, B, C, sqA, sqC, sqD, s2, t1) + G_anti(A, B, C, sqA, sqC, sqD, s1, t1);
}

// a5 + a6 (local part) of one target: 2 pi (phi* - x*) + eps / sqrt(x*^2 + y*^2 + (zeta* + 1)^2) - zeta_x* I, with
// I over [xa, xb] x [ya, yb], direct + image term (image: t' = -(y + y*) maps A s^2 - B s (y+y*) + C (y+y*)^2 onto
// the direct form); when ya = 0 the two boxes share the edge t = -y* and are one box over [-(yb + y*), yb - y*].
__device__ __forceinline__ double e2_local(const TgtRec& tr, const double eps, const double xa, const double xb,
                                           const double ya, const double yb) {
  const double A = tr.A, B = tr.B, C = tr.C, xs = tr.xs, ys = tr.ys, zs = tr.zs;
  const double sqA = sqrt(A), sqC = sqrt(C), sqD = sqrt(4 * A * C - B * B);
  const double s1 = xa - xs, s2 = xb - xs;
  double I;
  if (ya == 0.0) {
    I = box_int(A, B, C, sqA, sqC, sqD, s1, s2, -(yb + ys), yb - ys);
  } else {
    I = box_int(A, B, C, sqA, sqC, sqD, s1, s2, ya - ys, yb - ys) +
        box_int(A, B, C, sqA, sqC, sqD, s1, s2, -(yb + ys), -(ya + ys));
  }
  const double rho2 = xs * xs + ys * ys + (zs + 1.0) * (zs + 1.0);
  return 2.0 * CUDART_PI * tr.psis + eps / sqrt(rho2) - tr.zxs * I;
}

}  // namespace sws
