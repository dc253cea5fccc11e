// The pair term of the all-pairs quadrature (step a4, eq. (12) PAPER.md L101 with K1 L107, K2 L109, S2 L169-172)
// and the per-thread constants it works with: shared by the staged kernel (sws_allpairs.cu) and the
// uniform-operand kernel (sws_allpairs_const.cuh).  Citations "L<n>" are lines of /root/reference/PAPER.md.
#pragma once
#include "sws_farfield.cuh"
#include "sws_internal.cuh"

namespace sws {

// Per-thread constants of one target and of the current source column, split into what is GEOMETRY (the same
// for every state of a batch: the mesh does not move) and what depends on the state.
// The S2 quadratic forms are used with the square completed (C > 0):
//   A dx^2 + B dx (y-y*) + C (y-y*)^2 = C [ (y - c)^2 + g ],
//   A dx^2 - B dx (y+y*) + C (y+y*)^2 = C [ (y + c)^2 + g ],
//   c = y* - (B / 2C) dx,   g = (A/C - (B/2C)^2) dx^2 = (4AC - B^2) dx^2 / (4 C^2) > 0,
// so that each form costs one add and one two-register FMA per pair, c and g are per
// (target, column), and the common factor 1/sqrt(C) is applied once per target at the end.
struct TgtG {
  double ys, ys2, ys4;  // y*, 2 y*, 4 y*: the image terms follow from the direct ones (below)
};
struct TgtS {
  double zs, psis;  // zeta*, phi* - x*
};
struct ColG {
  double dx, dx2;  // x_i - x*, its square
};
struct ColS {
  double c, g;  // the S2 constants above (A, B, C belong to the state)
};

// One source node against one target: adds (phi-phi*-x+x*) K1 + zeta_x K2 to a1 and, if S2T,
// sqrt(C) S2 to aS (unit weight).  S2T = false is the far-field form: the S2 terms of the
// whole column come from s2_column_em() below, 27 FP64 instructions + 2 MUFU.RSQ64H remain.
// dm = y_j - y* is passed in: it is geometry, formed once per (target, node) for all states of the CTA.
template <bool S2T>
__device__ __forceinline__ void pair_term(const double2 zp, const double2 sl, const double yj, const double dm,
                                          const TgtG& tg, const TgtS& ts, const ColG& cg, const ColS& cs,
                                          double& a1, double& aS) {
  const double z = zp.x, psi = zp.y, zx = sl.x, zy = sl.y;
  // Image terms from the direct ones (all y >= 0, sws_setup): (y + y*)^2 = (y - y*)^2 + 4 y y* and
  // y + y* = (y - y*) + 2 y*, so y + y* itself is never formed: one DADD less per pair.  R+^2 >= R-^2, so
  // the rounding of R-^2 it inherits is below its own.
  const double dz = z - ts.zs;
  const double q = fma(dz, dz, cg.dx2);
  const double Rm2 = fma(dm, dm, q);
  const double Rp2 = fma(tg.ys4, yj, Rm2);
#ifdef SWS_SEED_ZERO
  const double rm = rsqrt_fp64(Rm2);
#else
  // q dies in Rm2, so the seed of 1/R- is built in q's register pair and the move that zeroes the seed's low
  // word disappears (721x241, constant-bank kernel: 50.2 -> 49.4 ms per state; -DSWS_SEED_ZERO: the plain seed)
  const double rm = rsqrt_fp64_lo(Rm2, __double2loint(q));
#endif
  const double rp = rsqrt_fp64(Rp2);
  // K1 numerators: zeta - zeta* - (x-x*) zeta_x - (y -+ y*) zeta_y, slopes at the source (Q2)
  const double n0 = fma(-cg.dx, zx, dz);
  const double nm = fma(-dm, zy, n0);
  const double np = fma(-tg.ys2, zy, nm);
  const double dpsi = psi - ts.psis;
#ifdef SWS_TAIL_CUBES
  // rounds 1-2: K1 with explicit cubes, then K2; 10 FP64 instructions (-DSWS_TAIL_CUBES, kept for the record)
  const double rm3 = (rm * rm) * rm;
  const double rp3 = (rp * rp) * rp;
  const double k1 = fma(np, rp3, nm * rm3);
  a1 = fma(dpsi, k1, a1);
  a1 = fma(zx, rm + rp, a1);  // K2 = 1/R- + 1/R+
#else
  // dpsi K1 + zeta_x K2 = (1/R-) [zeta_x + dpsi n- / R-^2] + (1/R+) [zeta_x + dpsi n+ / R+^2]: the third factor of
  // each cube and the K2 sum ride the two accumulating FMAs - 9 FP64 instructions instead of 10 (cfg5: 54.5 -> 53.2 ms)
  const double bm = dpsi * nm, bp = dpsi * np;
  const double cm = fma(bm, rm * rm, zx);
  const double cp = fma(bp, rp * rp, zx);
  a1 = fma(rm, cm, a1);
  a1 = fma(rp, cp, a1);
#endif
  if (S2T) {
    // S2 (eqs. (21), (22)) up to the factor 1/sqrt(C)
    const double sm = yj - cs.c;
    const double sp = yj + cs.c;
    const double Qm = fma(sm, sm, cs.g);
    const double Qp = fma(sp, sp, cs.g);
    aS += rsqrt_fp64(Qm) + rsqrt_fp64(Qp);
  }
}

}  // namespace sws
