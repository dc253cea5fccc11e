// Steps a0-a3, a5-a9 of the residual (everything that is O(NM)): unpack + x-trapezoid
// reconstruction + radiation rows, y-derivatives, midpoint values with A/B/C, the closed
// form I, Bernoulli rows, assembly of the integral-equation rows, and the small kernels of
// the batched finite-difference Jv (shift, quotient).  Citations: PAPER.md lines.
//
// These kernels use explicitly rounded __dadd_rn/__dmul_rn where the paper's formula is a
// short expression, so that no FMA contraction changes the rounding of the nodal fields.
#include <cooperative_groups.h>
#include <math_constants.h>

#include "sws_closed_form.cuh"
#include "sws_internal.cuh"

namespace sws {

#define ADD(a, b) __dadd_rn((a), (b))
#define SUB(a, b) __dadd_rn((a), -(b))
#define MUL(a, b) __dmul_rn((a), (b))

__device__ __forceinline__ double* state_out(double* F0, double* Fpert, int state, int n) {
  return state == 0 ? F0 : Fpert + (size_t)(state - 1) * n;
}

// ---------------------------------------------------------------------------------------
// a0 + a1 + a8.  One CTA per (y-line l, state).  eq. (18): the line block of u is
// [phi_{1,l}, (phi_x)_{1..N,l}]; the zeta half follows at offset (N+1)M.  eq. (19):
// zeta_{k+1,l} = zeta_{k,l} + (dx/2)((zeta_x)_{k,l} + (zeta_x)_{k+1,l}), same for phi (L160).
// The increments are formed by all threads; the running sum itself is sequential (one
// thread per field) so that its rounding is that of the recurrence as printed.
// Radiation rows eq. (24) L191-197 / App. A L417 with forward differences (L201, B.1 L431).
// One (y-line l, state) by the whole CTA; sm: 4 N doubles of shared memory.  Ends with the line written to the
// planes; the caller synchronises the CTA before the shared memory is used again.
__device__ __forceinline__ void reconstruct_line(const double* __restrict__ u, const double* __restrict__ V,
                                                 const double* __restrict__ sigma, const Mesh& m, const int lin,
                                                 const int l, const int state, double* sm, double* s_first,
                                                 double* zeta, double* phi, double* zx, double* px, double* F0,
                                                 double* Fpert) {
  const int N = m.N, tid = threadIdx.x;
  double* s_zx = sm;
  double* s_px = sm + N;
  double* s_z = sm + 2 * (size_t)N;
  double* s_p = sm + 3 * (size_t)N;

  const size_t half = (size_t)(N + 1) * m.M;
  const size_t offp = (size_t)l * (N + 1), offz = half + offp;
  const double* v = state > 0 ? V + (size_t)(state - 1) * m.n : nullptr;
  const double sg = state > 0 ? sigma[state - 1] : 0.0;
  // lin != 0 (analytic Jacobian action, sws_jv_exact_batch): state s >= 1 is the DIRECTION v_{s-1}
  // itself - the reconstruction (19) is linear and homogeneous in u, so the same recurrence
  // applied to v gives the directional derivatives of the nodal fields.
  const bool dir = lin && state > 0;
  auto get = [&](size_t idx) -> double {
    if (dir) return v[idx];
    const double a = u[idx];
    return v ? fma(sg, v[idx], a) : a;  // u_b = fl(u + sigma v), one rounding per entry
  };
  for (int k = tid; k < N; k += blockDim.x) {
    s_px[k] = get(offp + 1 + k);
    s_zx[k] = get(offz + 1 + k);
  }
  if (tid == 0) s_first[0] = get(offp);
  if (tid == 32) s_first[1] = get(offz);
  __syncthreads();
  const double hdx = m.dx / 2;
  for (int k = tid; k + 1 < N; k += blockDim.x) {
    s_z[k + 1] = MUL(hdx, ADD(s_zx[k], s_zx[k + 1]));
    s_p[k + 1] = MUL(hdx, ADD(s_px[k], s_px[k + 1]));
  }
  __syncthreads();
  if (tid == 0) {
    double acc = s_first[0];
    s_p[0] = acc;
    for (int k = 1; k < N; ++k) { acc = ADD(acc, s_p[k]); s_p[k] = acc; }
  } else if (tid == 32) {
    double acc = s_first[1];
    s_z[0] = acc;
    for (int k = 1; k < N; ++k) { acc = ADD(acc, s_z[k]); s_z[k] = acc; }
  } else if (tid == 64) {
    // a8: E3..E6 at x_1 (n = n_rad); positions App. A
    double* F = state_out(F0, Fpert, state, m.n);
    const double x1 = m.x1, nr = m.n_rad;
    const double p1 = s_first[0], z1 = s_first[1];
    // derivative rows: the constants (-1, -x_1) of E3, E4 drop out (B.1 L431)
    const double one = dir ? 0.0 : 1.0, xoff = dir ? 0.0 : x1;
    F[offp + 0] = ADD(MUL(x1, SUB(s_px[0], one)), MUL(nr, SUB(p1, xoff)));
    F[offp + 1] = ADD(MUL(x1, SUB(s_px[1], s_px[0]) / m.dx), MUL(nr, SUB(s_px[0], one)));
    F[offz + 0] = ADD(MUL(x1, s_zx[0]), MUL(nr, z1));
    F[offz + 1] = ADD(MUL(x1, SUB(s_zx[1], s_zx[0]) / m.dx), MUL(nr, s_zx[0]));
  }
  __syncthreads();
  const size_t base = ((size_t)state * m.M + l) * N;
  for (int k = tid; k < N; k += blockDim.x) {
    zeta[base + k] = s_z[k];
    phi[base + k] = s_p[k];
    zx[base + k] = s_zx[k];
    px[base + k] = s_px[k];
  }
}

__global__ void __launch_bounds__(256) k_reconstruct(const double* __restrict__ u,
                                                     const double* __restrict__ V,
                                                     const double* __restrict__ sigma, Mesh m,
                                                     int lin, int first, double* zeta, double* phi, double* zx,
                                                     double* px, double* F0, double* Fpert) {
  extern __shared__ double sm[];
  __shared__ double s_first[2];
  reconstruct_line(u, V, sigma, m, lin, blockIdx.x, blockIdx.y + first, sm, s_first, zeta, phi, zx, px, F0, Fpert);
}

// ---------------------------------------------------------------------------------------
// a2.  y-derivatives along each x-line k (L160).  One thread per (k, field, state); the
// planes are [l][k] so a warp's accesses are coalesced at every step of the march.
// dy_scheme 0: cubic spline, unknowns = knot slopes m_l, d_l = (f_{l+1}-f_l)/h:
//   interior  m_{l-1} + 4 m_l + m_{l+1} = 3 (d_{l-1} + d_l)
//   first     m_1 = 0 (y_1 = 0, even extension, Q3)  or not-a-knot, reduced with the first
//             interior row to  m_1 + 2 m_2 = (5 d_1 + d_2)/2
//   last      not-a-knot, reduced with the last interior row to
//             2 m_{M-1} + m_M = (d_{M-2} + 5 d_{M-1})/2
// solved by the Thomas recurrences with the data-independent factors cp[], inv[] made in
// sws_setup.  The output plane is used as the forward-sweep scratch.
// The march along one x-line: F_(l) reads the field at line l, O_(l) names the output at line l (also the
// forward-sweep scratch).  Same operations in the same order whichever memory the accessors name.
template <class FA, class OA>
__device__ __forceinline__ void dy_line(const Mesh& m, const double* __restrict__ cp,
                                        const double* __restrict__ inv, FA F_, OA O_) {
  const int M = m.M;
  const double h = m.dy;
  if (m.dy_scheme == 0) {
    double f0 = F_(0), f1 = F_(1), f2 = F_(2);
    double dprev = SUB(f1, f0) / h, dcur = SUB(f2, f1) / h;  // d_0, d_1
    double r = m.sym_first ? 0.0 : ADD(MUL(5.0, dprev), dcur) / 2;
    double g = MUL(r, inv[0]);
    O_(0) = g;
    for (int l = 1; l < M - 1; ++l) {
      // here dprev = d_{l-1}, dcur = d_l
      r = MUL(3.0, ADD(dprev, dcur));
      g = MUL(SUB(r, g), inv[l]);  // a_l = 1
      O_(l) = g;
      if (l + 2 < M) {
        const double fn = F_(l + 2);
        dprev = dcur;
        dcur = SUB(fn, f2) / h;
        f2 = fn;
      }
    }
    // after the loop dprev = d_{M-3}, dcur = d_{M-2}
    r = ADD(dprev, MUL(5.0, dcur)) / 2;
    g = MUL(SUB(r, MUL(2.0, g)), inv[M - 1]);  // a_{M-1} = 2
    O_(M - 1) = g;
    for (int l = M - 2; l >= 0; --l) {
      g = SUB(O_(l), MUL(cp[l], g));
      O_(l) = g;
    }
  } else {
    // finite differences (BASELINE.json wording; reading Q3)
    const double h2 = 2 * h;
    O_(0) = m.sym_first ? 0.0 : ADD(ADD(MUL(-3.0, F_(0)), MUL(4.0, F_(1))), -F_(2)) / h2;
    for (int l = 1; l < M - 1; ++l) O_(l) = SUB(F_(l + 1), F_(l - 1)) / h2;
    O_(M - 1) = ADD(SUB(MUL(3.0, F_(M - 1)), MUL(4.0, F_(M - 2))), F_(M - 3)) / h2;
  }
}

__global__ void __launch_bounds__(128) k_dy(Mesh m, int first, const double* __restrict__ cp,
                                            const double* __restrict__ inv, const double* zeta,
                                            const double* phi, double* zy, double* py) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= m.N) return;
  const int N = m.N, state = blockIdx.z + first;
  const size_t base = (size_t)state * m.S + k;
  const double* f = (blockIdx.y == 0 ? zeta : phi) + base;
  double* out = (blockIdx.y == 0 ? zy : py) + base;
  dy_line(m, cp, inv, [&](int l) { return f[(size_t)l * N]; }, [&](int l) -> double& { return out[(size_t)l * N]; });
}

// The same with the 32 x-lines of a warp staged in shared memory ([l][lane], coalesced both ways): every step
// of the two dependent sweeps then costs a shared-memory access instead of a global one (the march is pure
// latency: 2 M dependent steps; 220 -> ~25 us at M = 241, which is 1/3 of a residual on the 91x31 mesh).
// One CTA: the 32 x-lines kblock*32 .. +31 of one field of one state; s_dy: (2 M 32 + 2 M) doubles of shared
// memory.  Every thread of the CTA takes part in the loads, the stores and the passes whose elements are
// independent; the two dependent sweeps are marched by warp 0, one x-line per lane.  Called by all threads.
__device__ __forceinline__ void dy_block_staged(const Mesh& m, const double* __restrict__ cp,
                                                const double* __restrict__ inv, const int kblock, const int field,
                                                const int state, double* s_dy, const double* zeta,
                                                const double* phi, double* zy, double* py) {
  const int N = m.N, M = m.M, tid = threadIdx.x, nt = blockDim.x, lane = tid & 31;
  const int k0 = kblock * 32;
  const double* f = (field == 0 ? zeta : phi) + (size_t)state * m.S;
  double* out = (field == 0 ? zy : py) + (size_t)state * m.S;
  double* sa = s_dy;                       // [M][32]
  double* sb = s_dy + (size_t)M * 32;      // [M][32]
  double* s_inv = sb + (size_t)M * 32;     // [M]
  double* s_cp = s_inv + M;                // [M]
  const int tot = M * 32;
#pragma unroll 8
  for (int e = tid; e < tot; e += nt) {    // rows of 32 consecutive doubles: coalesced
    const int k = k0 + (e & 31);
    sa[e] = f[(size_t)(e >> 5) * N + (k < N ? k : N - 1)];
  }
  for (int l = tid; l < M; l += nt) { s_inv[l] = inv[l]; s_cp[l] = cp[l]; }
  __syncthreads();
  if (m.dy_scheme == 0) {
    // The spline march of dy_line() with its operations regrouped, not changed: first every d_l and every
    // right-hand side (independent of one another: the FP64 divisions overlap and spread over the CTA), then the
    // two dependent sweeps, whose chain per step is one subtraction and one multiplication.  Same values.
    const double h = m.dy;
    for (int e = tid; e < tot - 32; e += nt) sb[e] = SUB(sa[e + 32], sa[e]) / h;  // d_l, l = 0 .. M-2
    __syncthreads();
    for (int e = tid; e < tot; e += nt) {  // right-hand sides r_l into sa (f is no longer needed)
      const int l = e >> 5;
      double r;
      if (l == 0) r = m.sym_first ? 0.0 : ADD(MUL(5.0, sb[e]), sb[e + 32]) / 2;
      else if (l == M - 1) r = ADD(sb[e - 64], MUL(5.0, sb[e - 32])) / 2;
      else r = MUL(3.0, ADD(sb[e - 32], sb[e]));
      sa[e] = r;
    }
    __syncthreads();
    if (tid < 32) {
#define SA(l) sa[(l) * 32 + lane]
      double g = MUL(SA(0), s_inv[0]);
      SA(0) = g;
#pragma unroll 4
      for (int l = 1; l < M - 1; ++l) {
        g = MUL(SUB(SA(l), g), s_inv[l]);  // a_l = 1
        SA(l) = g;
      }
      g = MUL(SUB(SA(M - 1), MUL(2.0, g)), s_inv[M - 1]);  // a_{M-1} = 2
      SA(M - 1) = g;
#pragma unroll 4
      for (int l = M - 2; l >= 0; --l) {
        g = SUB(SA(l), MUL(s_cp[l], g));
        SA(l) = g;
      }
#undef SA
    }
  } else if (tid < 32) {
    dy_line(m, cp, inv, [&](int l) { return sa[l * 32 + lane]; }, [&](int l) -> double& { return sb[l * 32 + lane]; });
  }
  __syncthreads();
  const double* res = m.dy_scheme == 0 ? sa : sb;
#pragma unroll 8
  for (int e = tid; e < tot; e += nt) {
    const int k = k0 + (e & 31);
    if (k < N) out[(size_t)(e >> 5) * N + k] = res[e];
  }
  __syncthreads();  // the shared memory may be reused by the caller's next item
}

constexpr int kDyStagedThreads = 256;
__global__ void __launch_bounds__(kDyStagedThreads) k_dy_staged(Mesh m, int first, const double* __restrict__ cp,
                                                               const double* __restrict__ inv, const double* zeta,
                                                               const double* phi, double* zy, double* py) {
  extern __shared__ double s_dy[];
  dy_block_staged(m, cp, inv, blockIdx.x, blockIdx.y, blockIdx.z + first, s_dy, zeta, phi, zy, py);
}

// a5: the closed form of I lives in sws_closed_form.cuh (shared with the all-pairs kernel, whose extra CTA row
// evaluates it concurrently with the pair loops).

// The same antiderivative together with its partial derivatives with respect to A, B, C
// (analytic Jacobian action: dI = I_A dA + I_B dB + I_C dC).  With Q = A s^2 + B s t + C t^2,
// w1, w2 the two asinh arguments above, and 1 + w1^2 = 4 A Q / (t^2 D):
//   dG/dB = 2 sqrt(Q) / D
//   dG/dA = -B sqrt(Q) / (A D) - t asinh(w1) / (2 A^(3/2))
//   dG/dC = -B sqrt(Q) / (C D) - s asinh(w2) / (2 C^(3/2))
// (checked: d^2/ds dt of dG/dB is -s t / (2 Q^(3/2)) = d/dB of the integrand).
struct G4 {
  double g, gA, gB, gC;
};

__device__ G4 G_anti4(double A, double B, double C, double sqA, double sqC, double sqD, double s,
                      double t) {
  const double D = sqD * sqD;
  const double sqQ = sqrt(A * s * s + B * s * t + C * t * t);
  const double a1 = t != 0.0 ? t * asinh((2 * A * s + B * t) / (fabs(t) * sqD)) : 0.0;
  const double a2 = s != 0.0 ? s * asinh((2 * C * t + B * s) / (fabs(s) * sqD)) : 0.0;
  G4 r;
  r.g = a1 / sqA + a2 / sqC;
  r.gB = 2.0 * sqQ / D;
  r.gA = -B * sqQ / (A * D) - a1 / (2.0 * A * sqA);
  r.gC = -B * sqQ / (C * D) - a2 / (2.0 * C * sqC);
  return r;
}

__device__ G4 box_int4(double A, double B, double C, double sqA, double sqC, double sqD, double s1,
                       double s2, double t1, double t2) {
  const G4 a = G_anti4(A, B, C, sqA, sqC, sqD, s2, t2), b = G_anti4(A, B, C, sqA, sqC, sqD, s1, t2),
           c = G_anti4(A, B, C, sqA, sqC, sqD, s2, t1), d = G_anti4(A, B, C, sqA, sqC, sqD, s1, t1);
  G4 r;
  r.g = a.g - b.g - c.g + d.g;
  r.gA = a.gA - b.gA - c.gA + d.gA;
  r.gB = a.gB - b.gB - c.gB + d.gB;
  r.gC = a.gC - b.gC - c.gC + d.gC;
  return r;
}

// a3 + a5 + a6 (local part) + a7 + packing of the transposed source records.
// One thread per node (k, l) of one state; threads with k < N-1 also own target (k, l).
// One node (k, l) of one state.
__device__ __forceinline__ void target_node(const Mesh& m, const int k, const int l, const int state,
                                            const double* __restrict__ x, const double* __restrict__ y,
                                            const double* zeta, const double* phi, const double* zx,
                                            const double* px, const double* zy, const double* py, SrcRec* src,
                                            SrcRecF* srcf, TgtRec* tgt, double* e2loc, double4* tgtI, double* F0,
                                            double* Fpert) {
  const int N = m.N, M = m.M;
  const size_t nd = (size_t)state * m.S + (size_t)l * N + k;
  const double xk = x[k], yl = y[l];
  const double z0 = zeta[nd], p0 = phi[nd], zx0 = zx[nd], px0 = px[nd], zy0 = zy[nd], py0 = py[nd];

  SrcRec r;
  r.z = z0; r.psi = SUB(p0, xk); r.zx = zx0; r.zy = zy0;
  src[(size_t)state * m.S + (size_t)k * M + l] = r;  // transposed [i][j]
  if (srcf) {  // FP32 variant (Q12): zeta as hi + lo, packed-instruction operands duplicated
    SrcRecF f;
    f.z_hi = (float)r.z; f.z_lo = (float)(r.z - (double)f.z_hi);
    f.psi = f.psi_dup = (float)r.psi;
    f.zx = f.zx_dup = (float)r.zx;
    f.nzy = f.nzy_dup = -(float)r.zy;
    srcf[(size_t)state * m.S + (size_t)k * M + l] = f;
  }
  if (k >= N - 1) return;

  // two-point interpolation to the half-mesh point, L162 / L454
  const double xs = ADD(xk, x[k + 1]) / 2, ys = yl;
  const double zs = ADD(z0, zeta[nd + 1]) / 2, ps = ADD(p0, phi[nd + 1]) / 2;
  const double zxs = ADD(zx0, zx[nd + 1]) / 2, zys = ADD(zy0, zy[nd + 1]) / 2;
  const double pxs = ADD(px0, px[nd + 1]) / 2, pys = ADD(py0, py[nd + 1]) / 2;
  const double zx2 = MUL(zxs, zxs), zy2 = MUL(zys, zys);
  const double A = ADD(1.0, zx2), B = MUL(MUL(2.0, zxs), zys), C = ADD(1.0, zy2);  // L177

  const size_t t = (size_t)l * (N - 1) + k, ts = (size_t)state * m.T + t;
  TgtRec tr;
  tr.xs = xs; tr.ys = ys; tr.zs = zs; tr.psis = SUB(ps, xs); tr.zxs = zxs;
  tr.A = A; tr.B = B; tr.C = C;
  tgt[ts] = tr;

  double* F = state_out(F0, Fpert, state, m.n);
  // a7: Bernoulli, eq. (13) L113 at the starred values (Q6)
  {
    const double t1 = MUL(MUL(ADD(1.0, zx2), pys), pys);
    const double t2 = MUL(MUL(ADD(1.0, zy2), pxs), pxs);
    const double t3 = MUL(MUL(MUL(MUL(2.0, zxs), zys), pxs), pys);
    const double num = SUB(ADD(t1, t2), t3);
    const double den = ADD(ADD(1.0, zx2), zy2);
    const double F2 = MUL(m.froude, m.froude);
    F[(size_t)l * (N + 1) + 2 + k] = SUB(ADD(num / den / 2, zs / F2), 0.5);
  }
  // a5: I = int int S2 over [x_1,x_N] x [y_1,y_M], direct + image term, eq. (23) L185.
  // Image: t' = -(y + y*) maps A s^2 - B s (y+y*) + C (y+y*)^2 onto the direct form.
  const double sqA = sqrt(A), sqC = sqrt(C), sqD = sqrt(4 * A * C - B * B);
  const double s1 = x[0] - xs, s2 = x[N - 1] - xs;
  const double ya = y[0], yb = y[M - 1];
  if (tgtI) {
    // analytic Jacobian action: {I, dI/dA, dI/dB, dI/dC} of the base state; the residual rows
    // of this state are not needed (and not formed) in that mode
    G4 r;
    if (ya == 0.0) {
      r = box_int4(A, B, C, sqA, sqC, sqD, s1, s2, -(yb + ys), yb - ys);
    } else {
      const G4 r1 = box_int4(A, B, C, sqA, sqC, sqD, s1, s2, ya - ys, yb - ys);
      const G4 r2 = box_int4(A, B, C, sqA, sqC, sqD, s1, s2, -(yb + ys), -(ya + ys));
      r.g = r1.g + r2.g; r.gA = r1.gA + r2.gA; r.gB = r1.gB + r2.gB; r.gC = r1.gC + r2.gC;
    }
    tgtI[t] = make_double4(r.g, r.gA, r.gB, r.gC);
    return;
  }
  // a5 + a6 local part; e2loc == NULL: the FP64 all-pairs launch forms it itself (its CTA row 0), off this path
  if (e2loc) e2loc[ts] = e2_local(tr, m.eps, x[0], x[N - 1], ya, yb);
}

__global__ void __launch_bounds__(128) k_targets(Mesh m, const double* __restrict__ x,
                                                 const double* __restrict__ y,
                                                 const double* __restrict__ zeta,
                                                 const double* __restrict__ phi,
                                                 const double* __restrict__ zx,
                                                 const double* __restrict__ px,
                                                 const double* __restrict__ zy,
                                                 const double* __restrict__ py, SrcRec* src,
                                                 SrcRecF* srcf, TgtRec* tgt, double* e2loc, double4* tgtI,
                                                 double* F0, double* Fpert) {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // see k_fields_fused
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= m.N) return;
  target_node(m, k, blockIdx.y, blockIdx.z, x, y, zeta, phi, zx, px, zy, py, src, srcf, tgt, e2loc, tgtI, F0, Fpert);
}

// ---------------------------------------------------------------------------------------
// a0-a3, a5, a6 (local), a7, a8 in ONE cooperative launch: the three O(NM) stages above run as phases of one
// grid, separated by grid-wide barriers, instead of three dependent launches.  On the paper's small meshes
// (Table 1: 91x31 ... 361x121) the residual is launch-latency bound outside the all-pairs kernel, and
// this takes two launches and their drain/fill gaps out of every evaluation.  The phases call the very device
// functions of k_reconstruct, k_dy_staged and k_targets: same operations, same order, same roundings.
struct FusedArgs {
  const double* u;
  const double* V;
  const double* sigma;
  Mesh m;
  int states;
  const double* cp;
  const double* inv;
  const double* x;
  const double* y;
  double *zeta, *phi, *zx, *px, *zy, *py;
  SrcRec* src;
  SrcRecF* srcf;
  TgtRec* tgt;
  double* e2loc;
  double *F0, *Fpert;
};

__global__ void __launch_bounds__(256) k_fields_fused(const FusedArgs a) {
  extern __shared__ double sm[];  // max(4 N, 2 M 32 + 2 M) doubles
  __shared__ double s_first[2];
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  const Mesh& m = a.m;
  // phase 1: unpack + x-trapezoid + radiation rows, one (line, state) per CTA pass
  for (int item = blockIdx.x; item < m.M * a.states; item += gridDim.x) {
    reconstruct_line(a.u, a.V, a.sigma, m, 0, item % m.M, item / m.M, sm, s_first, a.zeta, a.phi, a.zx, a.px, a.F0,
                     a.Fpert);
    __syncthreads();
  }
  grid.sync();
  // phase 2: y-derivatives, one (block of 32 x-lines, field, state) per CTA pass
  {
    const int kblocks = (m.N + 31) / 32;
    for (int item = blockIdx.x; item < kblocks * 2 * a.states; item += gridDim.x)
      dy_block_staged(m, a.cp, a.inv, item % kblocks, (item / kblocks) & 1, item / (2 * kblocks), sm, a.zeta, a.phi,
                      a.zy, a.py);
  }
  grid.sync();
  // the all-pairs launch that follows may be scheduled from here on (it waits for this grid to complete before it
  // reads anything: griddepcontrol.wait at its top), which hides its launch latency behind phase 3
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  // phase 3: midpoints, A/B/C, Bernoulli rows, closed-form I, source/target records: one node per thread pass
  const size_t total = (size_t)m.S * a.states;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    const int state = (int)(idx / m.S);
    const int rem = (int)(idx - (size_t)state * m.S);
    const int l = rem / m.N, k = rem - l * m.N;
    target_node(m, k, l, state, a.x, a.y, a.zeta, a.phi, a.zx, a.px, a.zy, a.py, a.src, a.srcf, a.tgt, a.e2loc,
                nullptr, a.F0, a.Fpert);
  }
}

// a6 + a9: E2_{k,l} = local - sum over chunks (fixed order) of the all-pairs partials.
__global__ void __launch_bounds__(256) k_assemble(Mesh m, int chunks, const double* __restrict__ e2loc,
                                                  const double* __restrict__ part, double* F0,
                                                  double* Fpert) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= m.T) return;
  const int state = blockIdx.y;
  const double* p = part + (size_t)state * chunks * m.T + t;
  double s = 0.0;
  for (int c = 0; c < chunks; ++c) s += p[(size_t)c * m.T];
  const int l = t / (m.N - 1), k = t - l * (m.N - 1);
  double* F = state_out(F0, Fpert, state, m.n);
  F[(size_t)(m.N + 1) * m.M + (size_t)l * (m.N + 1) + 2 + k] = e2loc[(size_t)state * m.T + t] - s;
}

// ---------------------------------------------------------------------------------------
// a10 helpers.  sigma_b = 1e-7 (1 + ||u||_2) / ||v_b||_2 (BASELINE.json; the paper says only
// "a suitably-chosen shift", L221).  Two-stage fixed-order reduction: repeatable.
__global__ void __launch_bounds__(256) k_sumsq(const double* __restrict__ u, const double* __restrict__ V,
                                               int n, double* part) {
  const int row = blockIdx.y;  // 0: u, r >= 1: v_{r-1}
  const double* a = row == 0 ? u : V + (size_t)(row - 1) * n;
  double s = 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < (size_t)n;
       i += (size_t)gridDim.x * blockDim.x)
    s = fma(a[i], a[i], s);
  __shared__ double sh[256];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) part[(size_t)row * gridDim.x + blockIdx.x] = sh[0];
}

__global__ void k_sigma(const double* __restrict__ part, int nblk, int b, double* sigma) {
  const int r = threadIdx.x;
  if (r >= b) return;
  double su = 0.0, sv = 0.0;
  for (int i = 0; i < nblk; ++i) su += part[i];
  for (int i = 0; i < nblk; ++i) sv += part[(size_t)(r + 1) * nblk + i];
  // v_b = 0: sigma_b = 0 marks the direction; u_b = u and k_quotient writes the exact row J 0 = 0
  sigma[r] = sv > 0.0 ? 1e-7 * (1.0 + sqrt(su)) / sqrt(sv) : 0.0;
}

// eq. (25): JV_b = (E(u_b) - E(u)) / sigma_b
__global__ void __launch_bounds__(256) k_quotient(const double* __restrict__ F0,
                                                  const double* __restrict__ Fpert,
                                                  const double* __restrict__ sigma, int n, double* JV) {
  const int b = blockIdx.y;
  const double sg = sigma[b];
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < (size_t)n;
       i += (size_t)gridDim.x * blockDim.x)
    JV[(size_t)b * n + i] = sg != 0.0 ? (Fpert[(size_t)b * n + i] - F0[i]) / sg : 0.0;
}

// ---------------------------------------------------------------------------------------
// host launchers

size_t reconstruct_smem_bytes(int N) { return (size_t)4 * N * sizeof(double); }

constexpr size_t kDyStagedMaxSmem = 200 * 1024;
constexpr int kFusedMaxNodes = 1 << 17;  // the fused fields launch is used up to this many mesh nodes
static size_t dy_staged_smem_bytes(int M) { return ((size_t)2 * M * 32 + 2 * M) * sizeof(double); }

cudaError_t fields_configure(const sws_ctx* c) {
  // The attribute belongs to the FUNCTION (per device), not to a context: it is always set to the largest size any
  // context may ask for (sws_setup bounds N; kDyStagedMaxSmem bounds the staged column), so that setting up a small
  // mesh cannot take the limit away from a larger context that is still alive.
  cudaError_t e = cudaFuncSetAttribute(k_reconstruct, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  if (e != cudaSuccess) return e;
  (void)c;
  return cudaFuncSetAttribute(k_dy_staged, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kDyStagedMaxSmem);
}

// The fused launch is used when both the line buffers of phase 1 and the staged block of phase 2 fit the CTA's
// shared memory and the device can co-schedule the grid (cooperative launch); decided once per context.
static size_t fused_smem_bytes(const Mesh& m) {
  const size_t a = reconstruct_smem_bytes(m.N), b = dy_staged_smem_bytes(m.M);
  return a > b ? a : b;
}

cudaError_t fused_configure(sws_ctx* c) {
  c->fused_grid = 0;
  const size_t smem = fused_smem_bytes(c->mesh);
  if (smem > kDyStagedMaxSmem) return cudaSuccess;
  // Larger meshes gain nothing (the all-pairs kernel is > 99 % of the evaluation there) and phase 3 would run
  // at the low occupancy the staged block of phase 2 dictates.
  if (c->mesh.S > kFusedMaxNodes) return cudaSuccess;
  int coop = 0;
  cudaError_t e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device);
  if (e != cudaSuccess || !coop) return e;
  e = cudaFuncSetAttribute(k_fields_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kDyStagedMaxSmem);  // see fields_configure
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_fields_fused, 256, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) return cudaSuccess;
  if (occ > 2) occ = 2;  // a small grid keeps the two grid barriers cheap; the phases are latency bound
  c->fused_grid = occ * c->sm_count;
  return cudaSuccess;
}

cudaError_t launch_fields_fused(sws_ctx* c, const double* u, const double* V, int states, double* F0, double* Fpert,
                                cudaStream_t st) {
  const Mesh& m = c->mesh;
  FusedArgs a;
  a.u = u; a.V = V; a.sigma = c->sigma; a.m = m; a.states = states;
  a.cp = c->sp_cp; a.inv = c->sp_inv; a.x = c->x; a.y = c->y;
  a.zeta = c->zeta; a.phi = c->phi; a.zx = c->zx; a.px = c->px; a.zy = c->zy; a.py = c->py;
  // FP64 path: the all-pairs launch forms e2loc itself (its local CTA row); the FP32 variant keeps it here
  a.src = c->src; a.srcf = c->srcf; a.tgt = c->tgt; a.e2loc = c->params.precision == 0 ? nullptr : c->e2loc;
  a.F0 = F0; a.Fpert = Fpert;
  // no more CTAs than the largest phase has work for
  size_t work = ((size_t)m.S * states + 255) / 256;
  const size_t w1 = (size_t)m.M * states, w2 = (size_t)((m.N + 31) / 32) * 2 * states;
  if (w1 > work) work = w1;
  if (w2 > work) work = w2;
  int grid = c->fused_grid;
  if ((size_t)grid > work) grid = (int)work;
  void* args[] = {(void*)&a};
  return cudaLaunchCooperativeKernel((const void*)k_fields_fused, dim3(grid), dim3(256), args, fused_smem_bytes(m), st);
}

cudaError_t launch_reconstruct(sws_ctx* c, const double* u, const double* V, int states, int lin,
                               double* F0, double* Fpert, cudaStream_t st, int first) {
  const Mesh& m = c->mesh;
  dim3 grid(m.M, states - first);
  k_reconstruct<<<grid, 256, reconstruct_smem_bytes(m.N), st>>>(u, V, c->sigma, m, lin, first, c->zeta, c->phi,
                                                                 c->zx, c->px, F0, Fpert);
  return cudaGetLastError();
}

cudaError_t launch_dy(sws_ctx* c, int states, cudaStream_t st, int first) {
  const Mesh& m = c->mesh;
  const size_t smem = dy_staged_smem_bytes(m.M);
  if (smem <= kDyStagedMaxSmem) {
    dim3 grid((m.N + 31) / 32, 2, states - first);
    k_dy_staged<<<grid, kDyStagedThreads, smem, st>>>(m, first, c->sp_cp, c->sp_inv, c->zeta, c->phi, c->zy, c->py);
  } else {  // very long columns: march in global memory
    dim3 grid((m.N + 127) / 128, 2, states - first);
    k_dy<<<grid, 128, 0, st>>>(m, first, c->sp_cp, c->sp_inv, c->zeta, c->phi, c->zy, c->py);
  }
  return cudaGetLastError();
}

cudaError_t launch_targets(sws_ctx* c, int states, double* F0, double* Fpert, double4* tgtI,
                           cudaStream_t st) {
  const Mesh& m = c->mesh;
  dim3 grid((m.N + 127) / 128, m.M, states);
  // residual path in FP64 (no tgtI): e2loc is formed by the all-pairs launch's local CTA row instead
  double* e2loc = (c->params.precision == 0 && !tgtI) ? nullptr : c->e2loc;
  k_targets<<<grid, 128, 0, st>>>(m, c->x, c->y, c->zeta, c->phi, c->zx, c->px, c->zy, c->py, c->src,
                                  c->srcf, c->tgt, e2loc, tgtI, F0, Fpert);
  return cudaGetLastError();
}

cudaError_t launch_assemble(sws_ctx* c, int states, const PairPlan& plan, double* F0, double* Fpert,
                            cudaStream_t st) {
  const Mesh& m = c->mesh;
  dim3 grid((m.T + 255) / 256, states);
  k_assemble<<<grid, 256, 0, st>>>(m, plan.chunks, c->e2loc, c->part, F0, Fpert);
  return cudaGetLastError();
}

cudaError_t launch_sigma(sws_ctx* c, const double* u, const double* V, int b, cudaStream_t st) {
  dim3 grid(kNormBlocks, b + 1);
  k_sumsq<<<grid, 256, 0, st>>>(u, V, c->mesh.n, c->norm_part);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_sigma<<<1, ((b + 31) / 32) * 32, 0, st>>>(c->norm_part, kNormBlocks, b, c->sigma);
  return cudaGetLastError();
}

cudaError_t launch_jv_quotient(sws_ctx* c, const double* F0, const double* Fpert, int b, double* JV,
                               cudaStream_t st) {
  const int n = c->mesh.n;
  int bx = (n + 255) / 256;
  if (bx > 1024) bx = 1024;
  dim3 grid(bx, b);
  k_quotient<<<grid, 256, 0, st>>>(F0, Fpert, c->sigma, n, JV);
  return cudaGetLastError();
}

}  // namespace sws
