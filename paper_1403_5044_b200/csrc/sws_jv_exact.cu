// The analytic Jacobian action  JV_d = J(u) v_d = d/d sigma E(u + sigma v_d) at sigma = 0,
// d = 1..b: the limit of eq. (25) that JFNK approximates by a finite
// difference, formed here by differentiating every step a0-a9 of E by hand.
// No shift sigma, no subtraction of two residuals, hence none of the eps_mach / sigma
// rounding floor of the quotient (Q9).
//
// Linearisation of the all-pairs term (a4).  For one pair (source ij, target *), unit weight,
//   T = dpsi K1 + zeta_x K2 - zeta_x* S2,   dpsi = (phi - x)_ij - (phi* - x*),
//   K1 = n- r-^3 + n+ r+^3,  n-+ = dz - dx zeta_x - d-+ zeta_y,  r-+ = (dx^2 + d-+^2 + dz^2)^(-1/2),
//   K2 = r- + r+                                                   (L107-109, readings Q1, Q2)
// the mesh geometry dx = x_i - x*, d-+ = y_j -+ y* is fixed, so with dz = zeta_ij - zeta*
//   d(r)    = -r^3 dz d(dz),        d(r^3) = -3 r^5 dz d(dz),
//   dT = K1                                  d(psi_ij)  - K1 (...) d(psi*)
//      + [R3 (dpsi - zeta_x dz) - 3 dpsi dz N5] (d(zeta_ij) - d(zeta*))
//      + [K2 - dpsi dx R3]                      d(zeta_x)_ij
//      - [dpsi D3]                              d(zeta_y)_ij          - d(zeta_x* S2),
//   R3 = r-^3 + r+^3,  N5 = n- r-^5 + n+ r+^5,  D3 = d- r-^3 + d+ r+^3.
// The four bracketed coefficients depend on the base state only: they are computed ONCE per
// pair and applied to all b directions (4 DFMA per pair per direction), which is what makes a
// batch of b products cost (71 + 4 b) FP64 instructions per pair instead of 45 (b + 1).
// S2 = (C Q-)^(-1/2) + (C Q+)^(-1/2) (completed squares, see sws_allpairs.cu) depends on the
// direction only through A, B, C of the target:
//   d(sum w S2) = -1/2 C^(-3/2) [ dA sum w dx^2 (u-^3 + u+^3) + dB sum w dx (d- u-^3 - d+ u+^3)
//                                 + dC sum w (d-^2 u-^3 + d+^2 u+^3) ],   u-+ = Q-+^(-1/2),
// three more sums shared by all directions.  The per-target pieces d(psi*), d(zeta*), d(zeta_x*),
// dA, dB, dC multiply sums over the sources and are applied after the pair loop
// (k_assemble_lin).  Everything O(NM) (reconstruction, spline, midpoints, Bernoulli, the closed
// form I) is linearised in k_reconstruct (lin mode), k_dy (linear as it stands), k_targets_lin.
#include <math_constants.h>

#include <type_traits>

#include "sws_farfield.cuh"
#include "sws_internal.cuh"
#include "sws_stage.cuh"

namespace sws {

#ifndef SWS_LIN_ORDER
#define SWS_LIN_ORDER 1  // 1: coefficient-major accumulation, 0: direction-major
#endif
#ifndef SWS_LIN_UNROLL
#define SWS_LIN_UNROLL 1
#endif
#ifndef SWS_LIN_MINB16
#define SWS_LIN_MINB16 3
#endif
#ifndef SWS_LIN_THREADS
#define SWS_LIN_THREADS 128  // threads (= targets) per CTA of k_allpairs_lin
#endif

// ---------------------------------------------------------------------------------------
// Per node / per target linearisation for direction d (grid.z).  Base fields = state 0 of the
// planes, direction fields = state d + 1 (written by k_reconstruct in lin mode and k_dy).
//   dsrc  [group][i][j][BT] records {d zeta, d phi, d zeta_x, -d zeta_y}  (transposed like src)
//   dtgt  [d][t] {d zeta*, d phi*, d zeta_x*, dA, dB, dC}
//   e2lin [d][t] = 2 pi d phi* - eps (zeta*+1) d zeta* / rho*^3 - d zeta_x* I - zeta_x* dI
//   JV[d] Bernoulli rows: the derivative of eq. (13) L113 at the starred values.
__global__ void __launch_bounds__(128) k_targets_lin(Mesh m, int BT, const double* __restrict__ x,
                                                     const double* __restrict__ y,
                                                     const double* __restrict__ zeta,
                                                     const double* __restrict__ zx,
                                                     const double* __restrict__ px,
                                                     const double* __restrict__ zy,
                                                     const double* __restrict__ py,
                                                     const double* __restrict__ phi,
                                                     const double4* __restrict__ tgtI, double4* dsrc,
                                                     DTgtRec* dtgt, double* e2lin, double* JV) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= m.N) return;
  const int N = m.N, M = m.M, l = blockIdx.y, d = blockIdx.z;
  const size_t nb = (size_t)l * N + k;             // base node (state 0)
  const size_t nd = (size_t)(d + 1) * m.S + nb;    // direction node
  const double dz0 = zeta[nd], dp0 = phi[nd], dzx0 = zx[nd], dpx0 = px[nd], dzy0 = zy[nd], dpy0 = py[nd];

  // direction-interleaved source records: one (i, j) node holds BT consecutive 32 B records
  const int g = d / BT, dd = d - g * BT;
  dsrc[(((size_t)g * N + k) * M + l) * BT + dd] = make_double4(dz0, dp0, dzx0, -dzy0);
  if (k >= N - 1) return;

  // base starred values (L162) and their derivatives (same two-point averages: linear)
  const double xs = (x[k] + x[k + 1]) / 2, ys = y[l];
  const double zs = (zeta[nb] + zeta[nb + 1]) / 2;
  const double zxs = (zx[nb] + zx[nb + 1]) / 2, zys = (zy[nb] + zy[nb + 1]) / 2;
  const double pxs = (px[nb] + px[nb + 1]) / 2, pys = (py[nb] + py[nb + 1]) / 2;
  const double dzs = (dz0 + zeta[nd + 1]) / 2, dps = (dp0 + phi[nd + 1]) / 2;
  const double dzxs = (dzx0 + zx[nd + 1]) / 2, dzys = (dzy0 + zy[nd + 1]) / 2;
  const double dpxs = (dpx0 + px[nd + 1]) / 2, dpys = (dpy0 + py[nd + 1]) / 2;

  // A = 1 + zeta_x*^2, B = 2 zeta_x* zeta_y*, C = 1 + zeta_y*^2  (L177)
  const double dA = 2.0 * zxs * dzxs, dB = 2.0 * (dzxs * zys + zxs * dzys), dC = 2.0 * zys * dzys;

  const size_t t = (size_t)l * (N - 1) + k, td = (size_t)d * m.T + t;
  DTgtRec r;
  r.dzs = dzs; r.dpsis = dps; r.dzxs = dzxs; r.dA = dA; r.dB = dB; r.dC = dC;
  dtgt[td] = r;

  // Bernoulli row: E1 = num / (2 den) + zeta*/F^2 - 1/2,
  //   num = (1+zx^2) py^2 + (1+zy^2) px^2 - 2 zx zy px py,  den = 1 + zx^2 + zy^2
  {
    const double A1 = 1.0 + zxs * zxs, C1 = 1.0 + zys * zys;
    const double num = A1 * pys * pys + C1 * pxs * pxs - 2.0 * zxs * zys * pxs * pys;
    const double den = 1.0 + zxs * zxs + zys * zys;
    const double dnum = dA * pys * pys + 2.0 * A1 * pys * dpys + dC * pxs * pxs + 2.0 * C1 * pxs * dpxs -
                        2.0 * (dzxs * zys * pxs * pys + zxs * dzys * pxs * pys + zxs * zys * dpxs * pys +
                               zxs * zys * pxs * dpys);
    const double dden = dA + dC;
    JV[(size_t)d * m.n + (size_t)l * (N + 1) + 2 + k] =
        0.5 * (dnum - num * dden / den) / den + dzs / (m.froude * m.froude);
  }
  // local part of the integral-equation row
  const double4 I4 = tgtI[t];  // {I, I_A, I_B, I_C}
  const double rho2 = xs * xs + ys * ys + (zs + 1.0) * (zs + 1.0);
  const double rho = sqrt(rho2);
  e2lin[td] = 2.0 * CUDART_PI * dps - m.eps * (zs + 1.0) * dzs / (rho2 * rho) - dzxs * I4.x -
              zxs * (I4.y * dA + I4.z * dB + I4.w * dC);
}

// ---------------------------------------------------------------------------------------
// The all-pairs kernel of the analytic Jacobian action.  Same decomposition as k_allpairs
// (one thread = one target, 128 targets per CTA, a CTA walks a group of source columns staged
// by bulk async copies; every lane reads the same shared-memory record), plus the BT direction
// records of each staged node.  Output per (column group, target): 6 direction-independent
// sums and BT direction sums, [chunk][6 + BT][T] (coalesced in t), reduced in fixed order by
// k_assemble_lin.
__device__ __forceinline__ double rsqrt_seed_l(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}

// identical to rsqrt_fp64 of sws_allpairs.cu (MUFU.RSQ64H seed + one third-order correction)
__device__ __forceinline__ double rsqrt_l(double x) {
  const double y0 = rsqrt_seed_l(x);
  const double t = x * y0;
  const double e = fma(-t, y0, 1.0);
  const double p = fma(0.375, e, 0.5);
  const double w = e * p;
  return fma(y0, w, y0);
}

struct LinT {  // per target
  double ys, zs, psis;
};
struct LinC {  // per (target, column)
  double dx, dx2, c, g;
};
struct LinS {  // direction-independent sums of one thread
  double cpsi, cz;       // sum w K1, sum w [coefficient of d zeta]
  double s0;             // sum w (u- + u+)                       (sqrt(C) S2)
  double u3, u3y, u3yy;  // per column: sum_j w (u-^3 + u+^3), (d- u-^3 - d+ u+^3), (d-^2 u-^3 + d+^2 u+^3)
};

// MODE 0: everything (sws_jv_exact_batch).  MODE 1: the direction-independent sums only
// (sws_linearize: they depend on u alone, so a Newton step forms them once).  MODE 2: the
// direction sums only (sws_jv_apply): no S2, 41 + 4 BT FP64 instructions per pair.
// S2T = false: far column, the S2 sums of the whole column come from s2_column_em3 (sws_farfield.cuh).
template <int BT, bool SCALE, int MODE, bool S2T>
__device__ __forceinline__ void pair_lin(const double2 zp, const double2 sl, const double yj,
                                         const double4* __restrict__ dv, const double wgt,
                                         const LinT& t, const LinC& c, LinS& s, double (&acc)[BT]) {
  const double z = zp.x, psi = zp.y, zx = sl.x, zy = sl.y;
  const double dm = yj - t.ys, dp = yj + t.ys, dz = z - t.zs;
  const double q = fma(dz, dz, c.dx2);
  const double rm = rsqrt_l(fma(dm, dm, q)), rp = rsqrt_l(fma(dp, dp, q));
  const double n0 = fma(-c.dx, zx, dz);
  const double nm = fma(-dm, zy, n0), np = fma(-dp, zy, n0);
  const double rm2 = rm * rm, rp2 = rp * rp;
  const double rm3 = rm2 * rm, rp3 = rp2 * rp;
  const double am = nm * rm3, ap = np * rp3;
  double K1 = am + ap;
  const double N5 = fma(am, rm2, ap * rp2);
  const double R3 = rm3 + rp3;
  const double D3 = fma(dm, rm3, dp * rp3);
  const double K2 = rm + rp;
  const double dpsi = psi - t.psis;
  const double t1 = fma(-zx, dz, dpsi);
  const double t3 = (dpsi * dz) * N5;
  double cz = fma(-3.0, t3, R3 * t1);
  double czx = fma(-c.dx, dpsi * R3, K2);
  double czy = dpsi * D3;  // applied to the stored -d zeta_y
  if (SCALE) {  // trapezoid half weights on the first/last row and column (Q4)
    K1 *= wgt; cz *= wgt; czx *= wgt; czy *= wgt;
  }
  if (MODE != 2) {
    s.cpsi += K1;
    s.cz += cz;
  }
  if (MODE != 2 && S2T) {
    // S2 and its A, B, C sensitivities
    const double sm = yj - c.c, sp = yj + c.c;
    double um = rsqrt_l(fma(sm, sm, c.g)), up = rsqrt_l(fma(sp, sp, c.g));
    double um3 = (um * um) * um, up3 = (up * up) * up;
    if (SCALE) { um *= wgt; up *= wgt; um3 *= wgt; up3 *= wgt; }
    s.s0 += um + up;
    s.u3 += um3 + up3;
    const double vm = dm * um3, vp = dp * up3;
    s.u3y += vm - vp;
    s.u3yy = fma(dm, vm, s.u3yy);
    s.u3yy = fma(dp, vp, s.u3yy);
  }
  if (MODE == 1) return;
  // Coefficient-major order: runs of BT DFMAs that share one coefficient register in the same
  // operand slot (the operand-reuse cache then leaves two fresh 64-bit register reads per DFMA,
  // which is what the FP64 pipe can be fed at full rate).
  const double2* dv2 = reinterpret_cast<const double2*>(dv);
#if SWS_LIN_ORDER == 1
  {
    double2 lo[BT];
#pragma unroll
    for (int d = 0; d < BT; ++d) lo[d] = dv2[2 * d];  // {d zeta, d phi}
#pragma unroll
    for (int d = 0; d < BT; ++d) acc[d] = fma(K1, lo[d].y, acc[d]);
#pragma unroll
    for (int d = 0; d < BT; ++d) acc[d] = fma(cz, lo[d].x, acc[d]);
  }
  {
    double2 hi[BT];
#pragma unroll
    for (int d = 0; d < BT; ++d) hi[d] = dv2[2 * d + 1];  // {d zeta_x, -d zeta_y}
#pragma unroll
    for (int d = 0; d < BT; ++d) acc[d] = fma(czx, hi[d].x, acc[d]);
#pragma unroll
    for (int d = 0; d < BT; ++d) acc[d] = fma(czy, hi[d].y, acc[d]);
  }
#else
#pragma unroll
  for (int d = 0; d < BT; ++d) {
    const double2 lo = dv2[2 * d], hi = dv2[2 * d + 1];
    double a = acc[d];
    a = fma(K1, lo.y, a);
    a = fma(cz, lo.x, a);
    a = fma(czx, hi.x, a);
    a = fma(czy, hi.y, a);
    acc[d] = a;
  }
#endif
}

struct LinArgs {
  const SrcRec* src;    // [N][M] base state
  const double4* dsrc;  // [group][N][M][BT]
  const double* x;
  const double* y;
  const TgtRec* tgt;    // [T] base state
  double* out;          // [group][chunk][6 + BT][T]
  int N, M, T;
  int chunks, cols_per_chunk, seg_len, nseg;
  EmGeom em;
};

constexpr int kLinUnroll = SWS_LIN_UNROLL;
constexpr int kLinThreads = SWS_LIN_THREADS;
constexpr int kLinShared = 6;  // direction-independent sums per (chunk, target)

template <int BT, int MODE>
__global__ void __launch_bounds__(kLinThreads, (BT >= 16 ? SWS_LIN_MINB16 : BT >= 8 ? 3 : 4) * (128 / kLinThreads))
    k_allpairs_lin(const LinArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int DV = MODE == 1 ? 0 : BT;          // direction records staged per node
  constexpr int NSH = MODE == 2 ? 0 : kLinShared; // direction-independent sums written
  const int seg_pad = a.seg_len;  // even
  SrcRec* s_rec = reinterpret_cast<SrcRec*>(smem_raw);                          // [kStages][seg]
  double4* s_dv = reinterpret_cast<double4*>(s_rec + (size_t)kStages * seg_pad);  // [kStages][seg][DV]
  double* s_y = reinterpret_cast<double*>(s_dv + (size_t)kStages * seg_pad * DV);  // [kStages][seg]
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(s_y + (size_t)kStages * seg_pad);

  const int tid = threadIdx.x;
  const int tile = blockIdx.x, chunk = blockIdx.y, group = blockIdx.z;
  const int slot = tile * kLinThreads + tid;  // transposed target order (sws_farfield.cuh)
  const int tc = target_of_slot(slot < a.T ? slot : a.T - 1, a.N, a.M);
  const int t = slot < a.T ? tc : a.T;

  const TgtRec tr = a.tgt[tc];
  const LinT tg = {tr.ys, tr.zs, tr.psis};
  const double xs = tr.xs;
  const double kb = tr.B / (2.0 * tr.C);
  const double kg = tr.A / tr.C - kb * kb;

  const int c0 = chunk * a.cols_per_chunk;
  const int c1 = min(a.N, c0 + a.cols_per_chunk);
  const int nitems = (c1 - c0) * a.nseg;
  const double4* dsrc = a.dsrc + (size_t)group * a.N * a.M * BT;
  (void)dsrc;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&s_bar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  auto issue = [&](int q) {
    const int s = q % kStages;
    const int i = c0 + q / a.nseg, j0 = (q % a.nseg) * a.seg_len;
    const int len = min(a.seg_len, a.M - j0);
    const uint32_t rec_bytes = (uint32_t)len * (uint32_t)sizeof(SrcRec);
    const uint32_t dv_bytes = (uint32_t)len * (uint32_t)(DV * sizeof(double4));
    const uint32_t y_bytes = (uint32_t)((len + 1) & ~1) * 8u;
    mbar_expect_tx(&s_bar[s], rec_bytes + dv_bytes + y_bytes);
    bulk_g2s(s_rec + (size_t)s * seg_pad, a.src + (size_t)i * a.M + j0, rec_bytes, &s_bar[s]);
    if (DV > 0)
      bulk_g2s(s_dv + (size_t)s * seg_pad * DV, dsrc + ((size_t)i * a.M + j0) * DV, dv_bytes, &s_bar[s]);
    bulk_g2s(s_y + (size_t)s * seg_pad, a.y + j0, y_bytes, &s_bar[s]);
  };

  if (tid == 0 && nitems > 0) issue(0);

  double acc[BT];
#pragma unroll
  for (int d = 0; d < BT; ++d) acc[d] = 0.0;
  LinS tot = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};  // u3* here: already scaled by dx^2, dx, 1

  for (int q = 0; q < nitems; ++q) {
    const int s = q % kStages;
    if (tid == 0 && q + 1 < nitems) issue(q + 1);

    const int i = c0 + q / a.nseg, j0 = (q % a.nseg) * a.seg_len;
    const int len = min(a.seg_len, a.M - j0);
    LinC cc;
    cc.dx = __ldg(a.x + i) - xs;
    cc.dx2 = cc.dx * cc.dx;
    cc.c = fma(-kb, cc.dx, tg.ys);
    cc.g = kg * cc.dx2;
    const bool edge_col = (i == 0 || i == a.N - 1);
    const double ci = edge_col ? 0.5 : 1.0;

    mbar_wait(&s_bar[s], (uint32_t)((q / kStages) & 1));

    const double2* rec = reinterpret_cast<const double2*>(s_rec + (size_t)s * seg_pad);
    const double4* dv = s_dv + (size_t)s * seg_pad * DV;
    const double* yy = s_y + (size_t)s * seg_pad;
    LinS col = {tot.cpsi, tot.cz, tot.s0, 0.0, 0.0, 0.0};
    auto walk = [&](auto s2t) {
      constexpr bool S2T = decltype(s2t)::value;
      int jlo = 0, jhi = len;
      if (j0 == 0) {
        pair_lin<BT, true, MODE, S2T>(rec[0], rec[1], yy[0], dv, 0.5 * ci, tg, cc, col, acc);
        jlo = 1;
      }
      const bool last = (j0 + len == a.M);
      if (last) jhi = len - 1;
      if (edge_col) {
        for (int j = jlo; j < jhi; ++j)
          pair_lin<BT, true, MODE, S2T>(rec[2 * j], rec[2 * j + 1], yy[j], dv + (size_t)j * DV, ci, tg, cc, col,
                                        acc);
      } else {
#pragma unroll (MODE == 0 ? kLinUnroll : 2)
        for (int j = jlo; j < jhi; ++j)
          pair_lin<BT, false, MODE, S2T>(rec[2 * j], rec[2 * j + 1], yy[j], dv + (size_t)j * DV, 1.0, tg, cc, col,
                                         acc);
      }
      if (last && jhi >= jlo)
        pair_lin<BT, true, MODE, S2T>(rec[2 * jhi], rec[2 * jhi + 1], yy[jhi], dv + (size_t)jhi * DV, 0.5 * ci, tg,
                                      cc, col, acc);
    };
    if (MODE != 2 && column_is_far(cc.g, a.em.gmin)) {  // warp-uniform
      walk(std::false_type{});
      if (j0 == 0) {  // the column's S2 sums, once: d- = s- - beta, d+ = s+ + beta, beta = y* - c
        const Em3 e3 = s2_column_em3(a.em, cc.c, cc.g);
        const double beta = tg.ys - cc.c;
        col.s0 = fma(ci, e3.f0, col.s0);
        col.u3 = ci * e3.f3;
        col.u3y = ci * fma(-beta, e3.f3, e3.f3s);
        col.u3yy = ci * (fma(-cc.g, e3.f3, e3.f0) + beta * fma(beta, e3.f3, -2.0 * e3.f3s));
      }
    } else {
      walk(std::true_type{});
    }
    tot.cpsi = col.cpsi; tot.cz = col.cz; tot.s0 = col.s0;
    tot.u3 = fma(cc.dx2, col.u3, tot.u3);
    tot.u3y = fma(cc.dx, col.u3y, tot.u3y);
    tot.u3yy += col.u3yy;
    __syncthreads();
  }

  if (t < a.T) {
    double* o = a.out + ((size_t)(group * a.chunks + chunk) * (NSH + DV)) * a.T + t;
    if (MODE != 2) {
      o[0] = tot.cpsi;
      o[(size_t)1 * a.T] = tot.cz;
      o[(size_t)2 * a.T] = tot.s0;
      o[(size_t)3 * a.T] = tot.u3;
      o[(size_t)4 * a.T] = tot.u3y;
      o[(size_t)5 * a.T] = tot.u3yy;
    }
    if (MODE != 1) {
#pragma unroll
      for (int d = 0; d < BT; ++d) o[(size_t)(NSH + d) * a.T] = acc[d];
    }
  }
}

// JV_d[E2 row of t] = e2lin_d - dx dy { sum_chunks acc_d - d psi*_d sum K1 - d zeta*_d sum cz
//                     - d zeta_x*_d / sqrt(C) sum (u-+u+)
//                     + zeta_x* / (2 C^(3/2)) (dA_d U3 + dB_d U3y + dC_d U3yy) }
__global__ void __launch_bounds__(256) k_assemble_lin(Mesh m, int BT, int chunks, int nsh,
                                                      const double* __restrict__ sums,
                                                      const TgtRec* __restrict__ tgt,
                                                      const DTgtRec* __restrict__ dtgt,
                                                      const double* __restrict__ e2lin,
                                                      const double* __restrict__ part, double* JV) {
  // nsh = 6: `part` rows are [group][chunk][6 + BT] (fused kernel); nsh = 0: [group][chunk][BT]
  // and the six direction-independent sums come pre-reduced from `sums` [6][T] (sws_linearize)
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= m.T) return;
  const int d = blockIdx.y, g = d / BT, dd = d - g * BT;
  const size_t T = m.T, stride = (size_t)(nsh + BT) * T;
  const double* p = part + (size_t)g * chunks * stride + t;
  double sh[kLinShared] = {0, 0, 0, 0, 0, 0}, sa = 0.0;
  for (int c = 0; c < chunks; ++c) {
    const double* pc = p + (size_t)c * stride;
    if (nsh) {
#pragma unroll
      for (int q = 0; q < kLinShared; ++q) sh[q] += pc[(size_t)q * T];
    }
    sa += pc[(size_t)(nsh + dd) * T];
  }
  if (!nsh) {
#pragma unroll
    for (int q = 0; q < kLinShared; ++q) sh[q] = sums[(size_t)q * T + t];
  }
  const TgtRec tr = tgt[t];
  const DTgtRec dr = dtgt[(size_t)d * T + t];
  const double rC = 1.0 / sqrt(tr.C);
  const double dsum = sa - dr.dpsis * sh[0] - dr.dzs * sh[1] - dr.dzxs * rC * sh[2] +
                      0.5 * tr.zxs * rC * rC * rC * (dr.dA * sh[3] + dr.dB * sh[4] + dr.dC * sh[5]);
  const int l = t / (m.N - 1), k = t - l * (m.N - 1);
  JV[(size_t)d * m.n + (size_t)(m.N + 1) * m.M + (size_t)l * (m.N + 1) + 2 + k] =
      e2lin[(size_t)d * T + t] - (m.dx * m.dy) * dsum;
}

// sums[q][t] = sum over column groups (fixed order) of the MODE 1 partials [chunk][6][T]
__global__ void __launch_bounds__(256) k_reduce_base(int T, int chunks, const double* __restrict__ part,
                                                     double* __restrict__ sums) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= T) return;
  const int q = blockIdx.y;
  double a = 0.0;
  for (int c = 0; c < chunks; ++c) a += part[((size_t)c * kLinShared + q) * T + t];
  sums[(size_t)q * T + t] = a;
}

// ---------------------------------------------------------------------------------------
// host side

int lin_tile(int b) { return b <= 1 ? 1 : b <= 4 ? 4 : b <= 8 ? 8 : 16; }

static int lin_seg_cap(int DV) {
  // nodes per staged segment: stage = seg (32 + 8 + 32 DV) bytes, two stages <= ~36 KB per CTA
  int seg = (18 * 1024) / (40 + 32 * DV);
  seg &= ~1;
  if (seg > kSegMax) seg = kSegMax;
  if (seg < 8) seg = 8;
  return seg;
}

static size_t lin_smem_bytes(int DV, int seg) {
  return (size_t)kStages * seg * (sizeof(SrcRec) + sizeof(double) + DV * sizeof(double4)) +
         kStages * sizeof(uint64_t);
}

template <int BT, int MODE>
static cudaError_t lin_configure_one(int* occ) {
  const int DV = MODE == 1 ? 0 : BT;
  const size_t smem = lin_smem_bytes(DV, lin_seg_cap(DV));
  cudaError_t e = cudaFuncSetAttribute(k_allpairs_lin<BT, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)smem + 64);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, k_allpairs_lin<BT, MODE>, kLinThreads, smem);
}

cudaError_t lin_configure(sws_ctx* c) {
  cudaError_t e = lin_configure_one<1, 0>(&c->lin_occ[0]);
  if (e == cudaSuccess) e = lin_configure_one<4, 0>(&c->lin_occ[1]);
  if (e == cudaSuccess) e = lin_configure_one<8, 0>(&c->lin_occ[2]);
  if (e == cudaSuccess) e = lin_configure_one<16, 0>(&c->lin_occ[3]);
  if (e == cudaSuccess) e = lin_configure_one<1, 2>(&c->lin_occ2[0]);
  if (e == cudaSuccess) e = lin_configure_one<4, 2>(&c->lin_occ2[1]);
  if (e == cudaSuccess) e = lin_configure_one<8, 2>(&c->lin_occ2[2]);
  if (e == cudaSuccess) e = lin_configure_one<16, 2>(&c->lin_occ2[3]);
  if (e == cudaSuccess) e = lin_configure_one<1, 1>(&c->lin_occ1);
  return e;
}

static int lin_occ_of(const sws_ctx* c, int BT, int mode) {
  const int i = BT == 1 ? 0 : BT == 4 ? 1 : BT == 8 ? 2 : 3;
  const int o = mode == 1 ? c->lin_occ1 : mode == 2 ? c->lin_occ2[i] : c->lin_occ[i];
  return o > 0 ? o : 1;
}

// Launch geometry of the analytic all-pairs kernels: same tiles, a column split chosen from the
// mesh, the SM count and the kernel's occupancy (wave quantisation), and short staged
// segments (the direction records make a node 40 + 32 BT bytes).
// mode 0: fused (6 + BT rows per (group, chunk, target)); 1: base sums (6 rows); 2: directions (BT rows)
PairPlan make_lin_plan(const sws_ctx* c, int BT, int groups, int mode) {
  const Mesh& m = c->mesh;
  const int DV = mode == 1 ? 0 : BT, rows = (mode == 2 ? 0 : kLinShared) + DV;
  PairPlan p;
  p.tiles = (m.T + kLinThreads - 1) / kLinThreads;
  const int cap = lin_seg_cap(DV);
  p.nseg = (m.M + cap - 1) / cap;
  int seg = (m.M + p.nseg - 1) / p.nseg;
  p.seg_len = (seg + 1) & ~1;
  p.nseg = (m.M + p.seg_len - 1) / p.seg_len;
  const long slots = (long)c->sm_count * lin_occ_of(c, BT, mode);
  int min_cols = (256 + m.M - 1) / m.M;
  int cmax = m.N / (min_cols > 0 ? min_cols : 1);
  if (cmax < 1) cmax = 1;
  // the partial-sum buffer holds [group][chunk][rows][T]
  const long cap_chunks = (long)(c->part_rows / ((size_t)groups * rows));
  if (cmax > cap_chunks) cmax = (int)cap_chunks;
  if (cmax > 256) cmax = 256;
  if (cmax < 1) cmax = 1;
  int best = 1;
  double best_cost = 1e300;
  for (int ch = 1; ch <= cmax; ++ch) {
    const int cols = (m.N + ch - 1) / ch;
    if ((m.N + cols - 1) / cols != ch) continue;
    const long ctas = (long)p.tiles * ch * groups;
    const long waves = (ctas + slots - 1) / slots;
    const double cost = (double)waves * (cols + 0.25) + 1e-3 * ch;
    if (cost < best_cost) { best_cost = cost; best = ch; }
  }
  p.cols_per_chunk = (m.N + best - 1) / best;
  p.chunks = (m.N + p.cols_per_chunk - 1) / p.cols_per_chunk;
  return p;
}

cudaError_t launch_targets_lin(sws_ctx* c, int b, int BT, double* JV, cudaStream_t st) {
  const Mesh& m = c->mesh;
  dim3 grid((m.N + 127) / 128, m.M, b);
  k_targets_lin<<<grid, 128, 0, st>>>(m, BT, c->x, c->y, c->zeta, c->zx, c->px, c->zy, c->py, c->phi,
                                      c->tgtI, c->dsrc, c->dtgt, c->e2lin, JV);
  return cudaGetLastError();
}

template <int BT, int MODE>
static cudaError_t launch_lin_t(sws_ctx* c, int groups, const PairPlan& plan, cudaStream_t st) {
  const Mesh& m = c->mesh;
  LinArgs a;
  a.src = c->src; a.dsrc = c->dsrc; a.x = c->x; a.y = c->y; a.tgt = c->tgt; a.out = c->part;
  a.N = m.N; a.M = m.M; a.T = m.T;
  a.chunks = plan.chunks; a.cols_per_chunk = plan.cols_per_chunk;
  a.seg_len = plan.seg_len; a.nseg = plan.nseg;
  a.em = em_geometry(c);
  dim3 grid(plan.tiles, plan.chunks, groups);
  k_allpairs_lin<BT, MODE><<<grid, kLinThreads, lin_smem_bytes(MODE == 1 ? 0 : BT, plan.seg_len), st>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_allpairs_lin(sws_ctx* c, int BT, int groups, int mode, const PairPlan& plan, cudaStream_t st) {
  if (mode == 1) return launch_lin_t<1, 1>(c, 1, plan, st);
  if (mode == 2) {
    switch (BT) {
      case 1: return launch_lin_t<1, 2>(c, groups, plan, st);
      case 4: return launch_lin_t<4, 2>(c, groups, plan, st);
      case 8: return launch_lin_t<8, 2>(c, groups, plan, st);
      default: return launch_lin_t<16, 2>(c, groups, plan, st);
    }
  }
  switch (BT) {
    case 1: return launch_lin_t<1, 0>(c, groups, plan, st);
    case 4: return launch_lin_t<4, 0>(c, groups, plan, st);
    case 8: return launch_lin_t<8, 0>(c, groups, plan, st);
    default: return launch_lin_t<16, 0>(c, groups, plan, st);
  }
}

cudaError_t launch_reduce_base(sws_ctx* c, const PairPlan& plan, cudaStream_t st) {
  dim3 grid((c->mesh.T + 255) / 256, kLinShared);
  k_reduce_base<<<grid, 256, 0, st>>>(c->mesh.T, plan.chunks, c->part, c->lin_sums);
  return cudaGetLastError();
}

// mode 0: partials of the fused kernel; mode 2: direction partials + c->lin_sums
cudaError_t launch_assemble_lin(sws_ctx* c, int b, int BT, int mode, const PairPlan& plan, double* JV,
                                cudaStream_t st) {
  const Mesh& m = c->mesh;
  dim3 grid((m.T + 255) / 256, b);
  k_assemble_lin<<<grid, 256, 0, st>>>(m, BT, plan.chunks, mode == 2 ? 0 : kLinShared, c->lin_sums, c->tgt,
                                       c->dtgt, c->e2lin, c->part, JV);
  return cudaGetLastError();
}

}  // namespace sws
