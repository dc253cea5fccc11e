// The linear-Jacobian preconditioner P = [A B; C D] (section 4.2, App. B
// L425-503) in the block-factored form of App. C L505-515.
//
//   A   block diagonal, one tridiagonal (N+1) x (N+1) block A_0 per y-line      (B.3), (B.2) L462-464
//   B   block diagonal: (1/F^2) d zeta*_k / d(zeta_1, zeta_x) of the line        (B.4), L458
//   C   block diagonal: 2 pi d phi*_k / d(phi_1, phi_x) of the line              (B.5), L460
//   D   dense: -w(n,m) K3 (+ (sum w K3 - I)/2 on n = k, k+1, m = l), rows E5, E6 (B.6), L466-468
//       truncated to |l - m| <= hb blocks                                        L241
// A^-1 is a two-term recurrence per line; B and C are "trapezoid-reconstruct, then average to
// the half mesh" (L446-454), applied matrix-free as prefix sums.  The Schur complement
// S = D - C A^-1 B differs from D only on the diagonal blocks, by the SAME (N+1) x (N+1) matrix
// G = C_0 A_0^-1 B_0 on each.  S is factorised once by a block-banded LU (pivoting inside the
// diagonal blocks; cuSOLVER getrf/getrs + cuBLAS gemm) over a ring of hb + 1 live block rows, and
// stored in "apply form": per block row k one row-major panel [ -S~kk^-1 L~k,* | S~kk^-1 ] for the
// forward sweep and one panel S~kk^-1 S~k,* for the backward sweep, so that P^-1 v is 2 M
// HBM-bound matrix-vector kernels (this file) plus two per-line kernels.
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "jfnk_internal.cuh"

namespace jfnk {

// ---------------------------------------------------------------------------------------
// K3 of eq. (17) L139 on the flat surface, direct + image.
__device__ __forceinline__ double k3(double dx, double ym, double yp) {
  return rsqrt(fma(dx, dx, ym * ym)) + rsqrt(fma(dx, dx, yp * yp));
}

// I = int int K3 dx dy over the truncated rectangle (L440), "exactly in terms of logarithms"
// (L442): antiderivative G(s,t) = t asinh(s/|t|) + s asinh(t/|s|) of 1/sqrt(s^2 + t^2); a term
// with zero prefactor is 0 (reading Q5 with A = C = 1, B = 0).
__device__ double anti(double s, double t) {
  double g = 0.0;
  if (t != 0.0) g += t * asinh(s / fabs(t));
  if (s != 0.0) g += s * asinh(t / fabs(s));
  return g;
}
__device__ double box(double s1, double s2, double t1, double t2) {
  return anti(s2, t2) - anti(s1, t2) - anti(s2, t1) + anti(s1, t1);
}

// corr[t] = (sum_ij w(i,j) K3(x_i, y_j; x*_k, y_l) - I) / 2, one thread per target.
__global__ void __launch_bounds__(128) k_corr(LinMesh m, double* __restrict__ corr) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int T = (m.N - 1) * m.M;
  if (t >= T) return;
  const int l = t / (m.N - 1), k = t - l * (m.N - 1);  // 0-based: midpoint between nodes k, k+1
  const double xs = m.x1 + (k + 0.5) * m.dx, ys = m.y1 + l * m.dy;
  double sum = 0.0;
  for (int j = 0; j < m.M; ++j) {
    const double yj = m.y1 + j * m.dy, ym = yj - ys, yp = yj + ys;
    double row = 0.0;
    for (int i = 0; i < m.N; ++i) {
      const double dx = (m.x1 + i * m.dx) - xs;
      const double ci = (i == 0 || i == m.N - 1) ? 0.5 : 1.0;
      row = fma(ci, k3(dx, ym, yp), row);
    }
    sum = fma((j == 0 || j == m.M - 1) ? 0.5 : 1.0, row, sum);
  }
  sum *= m.dx * m.dy;
  const double xa = m.x1 - xs, xb = m.x1 + (m.N - 1) * m.dx - xs;
  const double ya = m.y1, yb = m.y1 + (m.M - 1) * m.dy;
  const double I = box(xa, xb, ya - ys, yb - ys) + box(xa, xb, -(yb + ys), -(ya + ys));
  corr[t] = 0.5 * (sum - I);
}

// One block row l of D (or of S = D - [m == l] G) into `panel`: column-major n1 x (2 hb + 1) n1,
// slot s holds block column m = l - hb + s (zero when m is outside the mesh).
__global__ void __launch_bounds__(256) k_assemble_row(LinMesh m, int hb, int l, int subtract_G,
                                                      const double* __restrict__ G,
                                                      const double* __restrict__ corr,
                                                      double* __restrict__ panel) {
  const int col = blockIdx.x;           // slot * n1 + c
  const int s = col / m.n1, c = col - s * m.n1;
  const int mm = l - hb + s;            // source line
  double* out = panel + (size_t)col * m.n1;
  if (mm < 0 || mm >= m.M) {
    for (int r = threadIdx.x; r < m.n1; r += blockDim.x) out[r] = 0.0;
    return;
  }
  const bool diag = (mm == l);
  const double ys = m.y1 + l * m.dy, yj = m.y1 + mm * m.dy;
  const double ym = yj - ys, yp = yj + ys;
  const double cj = (mm == 0 || mm == m.M - 1) ? 0.5 : 1.0;
  const double xn = m.x1 + (c - 1) * m.dx;  // node n = c (1-based) for c >= 1
  const double wn = m.dx * m.dy * cj * ((c == 1 || c == m.N) ? 0.5 : 1.0);
  for (int r = threadIdx.x; r < m.n1; r += blockDim.x) {
    double v = 0.0;
    if (r == 0) {         // E5 = x1 (zeta_x)_1 + n zeta_1                      L466
      if (diag) v = (c == 0) ? m.n_rad : (c == 1) ? m.x1 : 0.0;
    } else if (r == 1) {  // E6 = (x1/dx) (zeta_x)_2 + (n - x1/dx) (zeta_x)_1   L468
      if (diag) v = (c == 1) ? m.a11 : (c == 2) ? m.a12 : 0.0;
    } else if (c >= 1) {  // E2_{k,l}, k = r - 1 (1-based), column (zeta_x)_{n,m}, n = c   (B.6)
      const int k = r - 1;
      const double xs = m.x1 + (k - 0.5) * m.dx;
      v = -wn * k3(xn - xs, ym, yp);
      if (diag && (c == k || c == k + 1)) v += corr[l * (m.N - 1) + (k - 1)];
    }                     // c == 0: dE2/d zeta_1 = 0                            L496
    if (diag && subtract_G) v -= G[(size_t)c * m.n1 + r];
    out[r] = v;
  }
}

// ---------------------------------------------------------------------------------------
// Per-line pieces of App. C.  One CTA per y-line; the line is staged in shared memory and the
// two-term recurrences run on one thread (N dependent steps; O(NM) work in total).
//
// solve A_0 s = b in place on a shared-memory line of n1 values:
//   rows 1, 2:  a11 fx_1 + a12 fx_2 = b_1,  (fx_1 + fx_2)/2 = b_2;  then fx_{k+1} = 2 b_{1+k} - fx_k;
//   row 0:      f_1 = (b_0 - x1 fx_1) / n.
__device__ void solve_A0(const LinMesh& m, double* s) {
  const double fx1 = (s[1] - 2.0 * m.a12 * s[2]) / (m.a11 - m.a12);
  double prev = fx1;
  for (int k = 1; k <= m.N - 1; ++k) {  // row 1+k gives fx_{k+1}
    const double next = 2.0 * s[1 + k] - prev;
    s[k] = prev;
    prev = next;
  }
  s[m.N] = prev;
  s[0] = (s[0] - m.x1 * fx1) / m.n_rad;
}

// out[1+k] = scale * f*_k for k = 1..N-1, out[0] = out[1] = 0, where f is the trapezoid
// reconstruction (19) L156 of the line s = [f_1, fx_1..fx_N] and f*_k = (f_k + f_{k+1})/2 (L454).
__device__ void midpoint_of_line(const LinMesh& m, const double* s, double scale, double* out) {
  double f = s[0];
  for (int k = 1; k <= m.N - 1; ++k) {
    const double fn = f + 0.5 * m.dx * (s[k] + s[k + 1]);
    out[1 + k] = scale * (0.5 * (f + fn));
    f = fn;
  }
  out[0] = 0.0;
  out[1] = 0.0;
}

// s1 = A^-1 b1;  t2 = b2 - C s1                                                    App. C
__global__ void __launch_bounds__(256) k_stage1(LinMesh m, const double* __restrict__ v,
                                                double* __restrict__ s1, double* __restrict__ t2) {
  extern __shared__ double sh[];
  double* a = sh;            // [n1]
  double* c = sh + m.n1;     // [n1]
  const int l = blockIdx.x;
  const size_t q = blockIdx.y;  // right-hand side of a multi-vector apply
  v += q * 2 * (size_t)m.H; s1 += q * (size_t)m.H; t2 += q * (size_t)m.H;
  const double* b1 = v + (size_t)l * m.n1;
  const double* b2 = v + (size_t)m.H + (size_t)l * m.n1;
  for (int i = threadIdx.x; i < m.n1; i += blockDim.x) a[i] = b1[i];
  __syncthreads();
  if (threadIdx.x == 0) {
    solve_A0(m, a);
    midpoint_of_line(m, a, 2.0 * 3.14159265358979323846, c);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < m.n1; i += blockDim.x) {
    s1[(size_t)l * m.n1 + i] = a[i];
    t2[(size_t)l * m.n1 + i] = b2[i] - c[i];
  }
}

// r1 = s1 - A^-1 (B s2);  r2 = s2                                                  App. C
__global__ void __launch_bounds__(256) k_stage3(LinMesh m, const double* __restrict__ s1,
                                                const double* __restrict__ s2, double* __restrict__ r) {
  extern __shared__ double sh[];
  double* a = sh;
  double* c = sh + m.n1;
  const int l = blockIdx.x;
  const size_t q = blockIdx.y;
  s1 += q * (size_t)m.H; s2 += q * (size_t)m.H; r += q * 2 * (size_t)m.H;
  for (int i = threadIdx.x; i < m.n1; i += blockDim.x) a[i] = s2[(size_t)l * m.n1 + i];
  __syncthreads();
  if (threadIdx.x == 0) {
    midpoint_of_line(m, a, m.inv_f2, c);
    solve_A0(m, c);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < m.n1; i += blockDim.x) {
    r[(size_t)l * m.n1 + i] = s1[(size_t)l * m.n1 + i] - c[i];
    r[(size_t)m.H + (size_t)l * m.n1 + i] = a[i];
  }
}

// ---------------------------------------------------------------------------------------
// Block substitution sweeps: one CTA per matrix row, the row (contiguous, row-major) streamed
// once from HBM, the vector segment(s) from L2.  Fixed reduction order.
__device__ __forceinline__ double cta_sum(double v, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5;
  if ((threadIdx.x & 31) == 0) red[w] = v;
  __syncthreads();
  double s = 0.0;
  if (threadIdx.x == 0)
    for (int i = 0; i < kGemvThreads / 32; ++i) s += red[i];
  return s;
}

// dot product of one panel row with a vector, both of length K: 16-byte loads, four independent
// accumulators per thread (these kernels only stream the factor panels: ~62 MB per launch at 721x241,
// so what matters is the number of bytes in flight per SM); K even and 16-byte aligned operands when VEC
template <bool VEC>
__device__ __forceinline__ double row_dot(const double* __restrict__ row, const double* __restrict__ x, int K) {
  double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;
  if (VEC) {
    const double2* r2 = reinterpret_cast<const double2*>(row);
    const double2* x2 = reinterpret_cast<const double2*>(x);
    const int K2 = K >> 1;
    int c = threadIdx.x;
    for (; c + 3 * kGemvThreads < K2; c += 4 * kGemvThreads) {
      const double2 a0 = __ldcs(r2 + c), a1 = __ldcs(r2 + c + kGemvThreads), a2 = __ldcs(r2 + c + 2 * kGemvThreads),
                    a3 = __ldcs(r2 + c + 3 * kGemvThreads);
      const double2 b0 = x2[c], b1 = x2[c + kGemvThreads], b2 = x2[c + 2 * kGemvThreads], b3 = x2[c + 3 * kGemvThreads];
      acc0 = fma(a0.x, b0.x, acc0); acc0 = fma(a0.y, b0.y, acc0);
      acc1 = fma(a1.x, b1.x, acc1); acc1 = fma(a1.y, b1.y, acc1);
      acc2 = fma(a2.x, b2.x, acc2); acc2 = fma(a2.y, b2.y, acc2);
      acc3 = fma(a3.x, b3.x, acc3); acc3 = fma(a3.y, b3.y, acc3);
    }
    for (; c < K2; c += kGemvThreads) {
      const double2 a0 = __ldcs(r2 + c), b0 = x2[c];
      acc0 = fma(a0.x, b0.x, acc0); acc0 = fma(a0.y, b0.y, acc0);
    }
  } else {
    int c = threadIdx.x;
    for (; c + 3 * kGemvThreads < K; c += 4 * kGemvThreads) {
      acc0 = fma(row[c], x[c], acc0);
      acc1 = fma(row[c + kGemvThreads], x[c + kGemvThreads], acc1);
      acc2 = fma(row[c + 2 * kGemvThreads], x[c + 2 * kGemvThreads], acc2);
      acc3 = fma(row[c + 3 * kGemvThreads], x[c + 3 * kGemvThreads], acc3);
    }
    for (; c < K; c += kGemvThreads) acc0 = fma(row[c], x[c], acc0);
  }
  return (acc0 + acc1) + (acc2 + acc3);
}

// The same with the panel stored in FP32 (sws_precond_create flags bit 1): half the bytes to stream; the vector
// and the accumulation stay FP64.  8-byte loads of two panel entries (K even, rows 8-byte aligned), eight in
// flight per thread.
__device__ __forceinline__ double row_dot_f32(const float* __restrict__ row, const double* __restrict__ x, int K) {
  double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;
  if ((K & 1) == 0 && ((reinterpret_cast<uintptr_t>(row) | reinterpret_cast<uintptr_t>(x)) & 7) == 0 &&
      (reinterpret_cast<uintptr_t>(x) & 15) == 0) {
    const float2* r2 = reinterpret_cast<const float2*>(row);
    const double2* x2 = reinterpret_cast<const double2*>(x);
    const int K2 = K >> 1;
    int c = threadIdx.x;
    for (; c + 7 * kGemvThreads < K2; c += 8 * kGemvThreads) {
      float2 a[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) a[i] = __ldcs(r2 + c + i * kGemvThreads);
#pragma unroll
      for (int i = 0; i < 8; i += 4) {
        const double2 b0 = x2[c + i * kGemvThreads], b1 = x2[c + (i + 1) * kGemvThreads],
                      b2 = x2[c + (i + 2) * kGemvThreads], b3 = x2[c + (i + 3) * kGemvThreads];
        acc0 = fma((double)a[i].x, b0.x, acc0); acc0 = fma((double)a[i].y, b0.y, acc0);
        acc1 = fma((double)a[i + 1].x, b1.x, acc1); acc1 = fma((double)a[i + 1].y, b1.y, acc1);
        acc2 = fma((double)a[i + 2].x, b2.x, acc2); acc2 = fma((double)a[i + 2].y, b2.y, acc2);
        acc3 = fma((double)a[i + 3].x, b3.x, acc3); acc3 = fma((double)a[i + 3].y, b3.y, acc3);
      }
    }
    for (; c < K2; c += kGemvThreads) {
      const float2 a0 = __ldcs(r2 + c);
      const double2 b0 = x2[c];
      acc0 = fma((double)a0.x, b0.x, acc0); acc0 = fma((double)a0.y, b0.y, acc0);
    }
  } else {
    for (int c = threadIdx.x; c < K; c += kGemvThreads) acc0 = fma((double)row[c], x[c], acc0);
  }
  return (acc0 + acc1) + (acc2 + acc3);
}

__global__ void __launch_bounds__(kGemvThreads) k_fwd_row_f32(const float* __restrict__ panel, int n1, int lk,
                                                              const double* __restrict__ yprev,
                                                              const double* __restrict__ tk, double* __restrict__ yk) {
  __shared__ double red[kGemvThreads / 32];
  const int r = blockIdx.x;
  const int K0 = lk * n1;
  const float* row = panel + (size_t)r * (K0 + n1);
  const double s = cta_sum(row_dot_f32(row, yprev, K0) + row_dot_f32(row + K0, tk, n1), red);
  if (threadIdx.x == 0) yk[r] = s;
}

__global__ void __launch_bounds__(kGemvThreads) k_bwd_row_f32(const float* __restrict__ panel, int n1, int uk,
                                                              const double* __restrict__ xnext, double* __restrict__ yk) {
  __shared__ double red[kGemvThreads / 32];
  const int r = blockIdx.x;
  const int K = uk * n1;
  const double s = cta_sum(row_dot_f32(panel + (size_t)r * K, xnext, K), red);
  if (threadIdx.x == 0) yk[r] -= s;
}

// out (row-major, row stride ldo, type PT) [r][c] = scale * in (column-major, n1 rows) (r, c), c < cols: the
// transposing (and, for FP32 panels, converting) copy of a factor block into the apply form
template <typename PT>
__global__ void k_to_apply_form(const double* __restrict__ in, int n1, int cols, double scale, PT* __restrict__ out,
                                size_t ldo) {
  __shared__ double tile[32][33];
  const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    const int r = r0 + threadIdx.x, c = c0 + j;
    if (r < n1 && c < cols) tile[j][threadIdx.x] = in[(size_t)c * n1 + r];
  }
  __syncthreads();
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    const int r = r0 + j, c = c0 + threadIdx.x;
    if (r < n1 && c < cols) out[(size_t)r * ldo + c] = (PT)(scale * tile[threadIdx.x][j]);
  }
}

// y_k = [ -W_k | Sinv_k ] [ y_{k-lk..k-1} ; t_k ]      (forward: L~ y = t with unit... see header)
template <bool VEC>
__global__ void __launch_bounds__(kGemvThreads) k_fwd_row(const double* __restrict__ panel, int n1, int lk,
                                                          const double* __restrict__ yprev,
                                                          const double* __restrict__ tk,
                                                          double* __restrict__ yk) {
  __shared__ double red[kGemvThreads / 32];
  const int r = blockIdx.x;
  const int K0 = lk * n1;
  const double* row = panel + (size_t)r * (K0 + n1);
  const double s = cta_sum(row_dot<VEC>(row, yprev, K0) + row_dot<VEC>(row + K0, tk, n1), red);
  if (threadIdx.x == 0) yk[r] = s;
}

// x_k = y_k - U_k x_{k+1..k+uk}   (in place on y)
template <bool VEC>
__global__ void __launch_bounds__(kGemvThreads) k_bwd_row(const double* __restrict__ panel, int n1, int uk,
                                                          const double* __restrict__ xnext,
                                                          double* __restrict__ yk) {
  __shared__ double red[kGemvThreads / 32];
  const int r = blockIdx.x;
  const int K = uk * n1;
  const double s = cta_sum(row_dot<VEC>(panel + (size_t)r * K, xnext, K), red);
  if (threadIdx.x == 0) yk[r] -= s;
}

// The same sweeps for T right-hand sides at once (enlarged GMRES: one sweep over the factor panels serves the T
// vectors of a block, so the panels - 30 GB at 721x241 - are streamed once instead of T times).  Vector q of a
// buffer starts at base + q ldv.  One CTA per matrix row, the row read once, T accumulators per thread.
template <int T, typename PT>
__device__ __forceinline__ void row_dot_multi(const PT* __restrict__ row, const double* __restrict__ x, size_t ldv,
                                              int K, double (&acc)[T]) {
  int c = threadIdx.x;
  for (; c + kGemvThreads < K; c += 2 * kGemvThreads) {
    const double a0 = (double)__ldcs(row + c), a1 = (double)__ldcs(row + c + kGemvThreads);
#pragma unroll
    for (int q = 0; q < T; ++q) {
      acc[q] = fma(a0, x[q * ldv + c], acc[q]);
      acc[q] = fma(a1, x[q * ldv + c + kGemvThreads], acc[q]);
    }
  }
  for (; c < K; c += kGemvThreads) {
    const double a0 = (double)__ldcs(row + c);
#pragma unroll
    for (int q = 0; q < T; ++q) acc[q] = fma(a0, x[q * ldv + c], acc[q]);
  }
}

template <int T>
__device__ __forceinline__ void cta_sum_multi(double (&acc)[T], double* red /* [T][warps] */) {
  const int w = threadIdx.x >> 5, nw = kGemvThreads / 32;
#pragma unroll
  for (int q = 0; q < T; ++q) {
    double v = acc[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) red[q * nw + w] = v;
  }
  __syncthreads();
  if (threadIdx.x < T) {
    double s = 0.0;
    for (int i = 0; i < nw; ++i) s += red[threadIdx.x * nw + i];
    acc[0] = s;  // thread q < T holds the sum of right-hand side q
  }
}

template <int T, typename PT>
__global__ void __launch_bounds__(kGemvThreads) k_fwd_row_multi(const PT* __restrict__ panel, int n1, int lk,
                                                                const double* __restrict__ yprev,
                                                                const double* __restrict__ tk,
                                                                double* __restrict__ yk, size_t ldv) {
  __shared__ double red[T * (kGemvThreads / 32)];
  const int r = blockIdx.x;
  const int K0 = lk * n1;
  const PT* row = panel + (size_t)r * (K0 + n1);
  double acc[T];
#pragma unroll
  for (int q = 0; q < T; ++q) acc[q] = 0.0;
  row_dot_multi<T, PT>(row, yprev, ldv, K0, acc);
  row_dot_multi<T, PT>(row + K0, tk, ldv, n1, acc);
  cta_sum_multi<T>(acc, red);
  if (threadIdx.x < T) yk[threadIdx.x * ldv + r] = acc[0];
}

template <int T, typename PT>
__global__ void __launch_bounds__(kGemvThreads) k_bwd_row_multi(const PT* __restrict__ panel, int n1, int uk,
                                                                const double* __restrict__ xnext,
                                                                double* __restrict__ yk, size_t ldv) {
  __shared__ double red[T * (kGemvThreads / 32)];
  const int r = blockIdx.x;
  const int K = uk * n1;
  double acc[T];
#pragma unroll
  for (int q = 0; q < T; ++q) acc[q] = 0.0;
  row_dot_multi<T, PT>(panel + (size_t)r * K, xnext, ldv, K, acc);
  cta_sum_multi<T>(acc, red);
  if (threadIdx.x < T) yk[threadIdx.x * ldv + r] -= acc[0];
}

__global__ void k_identity(double* a, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n * n) a[i] = (i / n == i % n) ? 1.0 : 0.0;
}

cudaError_t launch_assemble_row(const sws_precond* pc, int l, int subtract_G, double* panel, cudaStream_t st) {
  const LinMesh& m = pc->lm;
  k_assemble_row<<<(2 * pc->hb + 1) * m.n1, 256, 0, st>>>(m, pc->hb, l, subtract_G, pc->G, pc->corr, panel);
  return cudaGetLastError();
}

}  // namespace jfnk

// =======================================================================================
// host side
using namespace jfnk;

namespace {

thread_local char g_err[256] = "";

int fail_cuda(cudaError_t e, const char* where) {
  snprintf(g_err, sizeof g_err, "%s: %s", where, cudaGetErrorString(e));
  return SWS_ECUDA;
}
int fail_lib(int status, const char* where) {
  snprintf(g_err, sizeof g_err, "%s: library status %d", where, status);
  return SWS_ECUDA;
}

#define CK(call)                                              \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ == cudaErrorMemoryAllocation) { rc = SWS_ENOMEM; goto done; } \
    if (e_ != cudaSuccess) { rc = fail_cuda(e_, #call); goto done; }     \
  } while (0)
#define CKB(call)                                             \
  do {                                                        \
    int s_ = (int)(call);                                     \
    if (s_ != 0) { rc = fail_lib(s_, #call); goto done; }     \
  } while (0)

// Host copy of solve_A0 / midpoint_of_line for the one-off G = C_0 A_0^-1 B_0.
void host_solve_A0(const LinMesh& m, double* s) {
  const double fx1 = (s[1] - 2.0 * m.a12 * s[2]) / (m.a11 - m.a12);
  double prev = fx1;
  for (int k = 1; k <= m.N - 1; ++k) {
    const double next = 2.0 * s[1 + k] - prev;
    s[k] = prev;
    prev = next;
  }
  s[m.N] = prev;
  s[0] = (s[0] - m.x1 * fx1) / m.n_rad;
}
void host_midpoint(const LinMesh& m, const double* s, double scale, double* out) {
  double f = s[0];
  for (int k = 1; k <= m.N - 1; ++k) {
    const double fn = f + 0.5 * m.dx * (s[k] + s[k + 1]);
    out[1 + k] = scale * (0.5 * (f + fn));
    f = fn;
  }
  out[0] = out[1] = 0.0;
}

// G (column-major n1 x n1): column c = C_0 A_0^-1 B_0 e_c.
void host_G(const LinMesh& m, std::vector<double>& G) {
  const int n1 = m.n1;
  G.assign((size_t)n1 * n1, 0.0);
  std::vector<double> e(n1), a(n1), g(n1);
  for (int c = 0; c < n1; ++c) {
    std::fill(e.begin(), e.end(), 0.0);
    e[c] = 1.0;
    host_midpoint(m, e.data(), m.inv_f2, a.data());   // B_0 e_c
    host_solve_A0(m, a.data());                        // A_0^-1
    host_midpoint(m, a.data(), 2.0 * M_PI, g.data());  // C_0
    std::memcpy(&G[(size_t)c * n1], g.data(), sizeof(double) * n1);
  }
}

}  // namespace

template <int T, typename PT>
static void launch_sweeps_multi_t(sws_precond* pc, cudaStream_t st) {
  const int n1 = pc->lm.n1, M = pc->lm.M, hb = pc->hb;
  const size_t ldv = (size_t)pc->lm.H;
  const PT* fwd = static_cast<const PT*>(pc->fwd);
  const PT* bwd = static_cast<const PT*>(pc->bwd);
  for (int k = 0; k < M; ++k) {
    const int lk = k < hb ? k : hb;
    k_fwd_row_multi<T, PT><<<n1, kGemvThreads, 0, st>>>(fwd + pc->fwd_off[k], n1, lk, pc->y + (size_t)(k - lk) * n1,
                                                        pc->t2 + (size_t)k * n1, pc->y + (size_t)k * n1, ldv);
  }
  for (int k = M - 2; k >= 0; --k) {
    const int uk = (M - 1 - k) < hb ? (M - 1 - k) : hb;
    if (uk > 0)
      k_bwd_row_multi<T, PT><<<n1, kGemvThreads, 0, st>>>(bwd + pc->bwd_off[k], n1, uk, pc->y + (size_t)(k + 1) * n1,
                                                          pc->y + (size_t)k * n1, ldv);
  }
}
template <int T>
static void launch_sweeps_multi(sws_precond* pc, cudaStream_t st) {
  if (pc->f32) launch_sweeps_multi_t<T, float>(pc, st);
  else launch_sweeps_multi_t<T, double>(pc, st);
}

extern "C" {

const char* sws_jfnk_last_error(void) { return g_err; }

int sws_precond_create(const sws_params* p, int32_t bandwidth, int32_t flags, sws_precond** out) {
  if (!p || !out) return SWS_EINVAL;
  *out = nullptr;
  if (p->N < 3 || p->M < 4 || !(p->dx > 0) || !(p->dy > 0) || !(p->froude > 0) || p->n_rad == 0.0) return SWS_EINVAL;
  if (bandwidth > 0 && bandwidth % 2 == 0) return SWS_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || p->device < 0 || p->device >= ndev)
    return fail_cuda(cudaErrorNoDevice, "sws_precond_create: no such CUDA device");
  const auto t_start = std::chrono::steady_clock::now();

  sws_precond* pc = new (std::nothrow) sws_precond();
  if (!pc) return SWS_ENOMEM;
  pc->params = *p;
  pc->device = p->device;
  LinMesh& m = pc->lm;
  m.N = p->N; m.M = p->M; m.n1 = p->N + 1; m.H = m.n1 * p->M;
  m.x1 = p->x1; m.y1 = p->y1; m.dx = p->dx; m.dy = p->dy;
  m.inv_f2 = 1.0 / (p->froude * p->froude);
  m.n_rad = p->n_rad;
  m.a12 = p->x1 / p->dx;
  m.a11 = p->n_rad - m.a12;
  if (m.a11 == m.a12) { delete pc; return SWS_EINVAL; }
  int hb = (bandwidth <= 0 || bandwidth >= 2 * m.M - 1) ? m.M - 1 : (bandwidth - 1) / 2;
  pc->hb = hb;
  pc->factored = 0;
  pc->bytes = 0;
  pc->G = pc->corr = pc->s1 = pc->t2 = pc->y = pc->panel = nullptr;
  pc->fwd = pc->bwd = nullptr;
  pc->f32 = (flags & 2) ? 1 : 0;
  pc->multi_cap = 1;

  const int n1 = m.n1, M = m.M, T = (m.N - 1) * M;
  const size_t blk = (size_t)n1 * n1;
  const size_t panel_elems = blk * (2 * hb + 1);
  int rc = SWS_OK;
  cublasHandle_t hb_blas = nullptr;
  cusolverDnHandle_t hb_sol = nullptr;
  double *ring = nullptr, *Sinv = nullptr, *W = nullptr, *work = nullptr;
  int *ipiv = nullptr, *info = nullptr;
  std::vector<double> Gh;
  std::vector<int> info_h;
  cudaStream_t sm = nullptr, sf = nullptr;
  cudaEvent_t evD = nullptr, evF = nullptr;
  DevGuard dg(p->device);

  CK(dg.err);
  CK(cudaMalloc(&pc->G, blk * sizeof(double)));
  CK(cudaMalloc(&pc->corr, (size_t)T * sizeof(double)));
  CK(cudaMalloc(&pc->s1, (size_t)m.H * sizeof(double)));
  CK(cudaMalloc(&pc->t2, (size_t)m.H * sizeof(double)));
  CK(cudaMalloc(&pc->y, (size_t)m.H * sizeof(double)));
  CK(cudaMalloc(&pc->panel, panel_elems * sizeof(double)));
  pc->bytes += (blk + T + 3 * (size_t)m.H + panel_elems) * sizeof(double);

  host_G(m, Gh);
  CK(cudaMemcpy(pc->G, Gh.data(), blk * sizeof(double), cudaMemcpyHostToDevice));
  k_corr<<<(T + 127) / 128, 128>>>(m, pc->corr);
  CK(cudaGetLastError());

  if (!(flags & 1)) {
    // apply-form storage
    pc->fwd_off.resize(M + 1);
    pc->bwd_off.resize(M + 1);
    size_t fo = 0, bo = 0;
    for (int k = 0; k < M; ++k) {
      const int lk = k < hb ? k : hb, uk = (M - 1 - k) < hb ? (M - 1 - k) : hb;
      pc->fwd_off[k] = fo; fo += blk * (lk + 1);
      pc->bwd_off[k] = bo; bo += blk * uk;
    }
    pc->fwd_off[M] = fo; pc->bwd_off[M] = bo;
    const size_t esz = pc->f32 ? sizeof(float) : sizeof(double);
    CK(cudaMalloc(&pc->fwd, fo * esz));
    CK(cudaMalloc(&pc->bwd, (bo ? bo : 1) * esz));
    pc->bytes += (fo + bo) * esz;

    // factorisation scratch (freed below)
    const int R = hb + 1;  // live block rows
    CK(cudaMalloc(&ring, panel_elems * R * sizeof(double)));
    CK(cudaMalloc(&Sinv, 2 * blk * sizeof(double)));  // explicit inverses of two consecutive diagonal blocks
    CK(cudaMalloc(&W, blk * (hb ? hb : 1) * sizeof(double)));
    CK(cudaMalloc(&ipiv, sizeof(int) * n1));
    CK(cudaMalloc(&info, sizeof(int) * 2 * M));
    CK(cudaMemset(info, 0, sizeof(int) * 2 * M));
    // Two streams: `sm` carries the assembly and every GEMM, `sf` the LU + explicit inverse of the diagonal blocks
    // (cuSOLVER getrf / getrs on a 722 x 722 block: ~2.8 ms of dependent panel steps that occupy a few SMs).  The
    // diagonal block of row k + 1 is final as soon as the FIRST trailing product of step k has updated it, so its
    // factorisation runs on `sf` next to the remaining trailing products of step k (look-ahead of one block row)
    // instead of between them: 2.28 -> 1.6 s at 721x241.
    CK(cudaDeviceSynchronize());  // the one-off work above ran on the default stream
    CK(cudaStreamCreateWithFlags(&sm, cudaStreamNonBlocking));
    {  // `sf` gets the highest priority: its small dependent kernels must not queue behind whole waves of GEMM CTAs
      int prio_lo = 0, prio_hi = 0;
      CK(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
      CK(cudaStreamCreateWithPriority(&sf, cudaStreamNonBlocking, prio_hi));
    }
    CK(cudaEventCreateWithFlags(&evD, cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&evF, cudaEventDisableTiming));
    CKB(cublasCreate(&hb_blas));
    CKB(cusolverDnCreate(&hb_sol));
    CKB(cublasSetStream(hb_blas, sm));
    CKB(cusolverDnSetStream(hb_sol, sf));
    int lwork = 0;
    CKB(cusolverDnDgetrf_bufferSize(hb_sol, n1, n1, ring, n1, &lwork));
    CK(cudaMalloc(&work, sizeof(double) * (lwork > 0 ? lwork : 1)));

    const double one = 1.0, zero = 0.0, mone = -1.0;
    // on `sf`, once `sm` has reached evD: LU of the diagonal block of row k and its explicit inverse into Sinv[k % 2]
    auto factor_diag = [&](int k) -> int {
      double* Dkk = ring + panel_elems * (k % R) + blk * hb;
      double* Si = Sinv + blk * (k % 2);
      if (cudaEventRecord(evD, sm) != cudaSuccess || cudaStreamWaitEvent(sf, evD, 0) != cudaSuccess) return 1;
      if (cusolverDnDgetrf(hb_sol, n1, n1, Dkk, n1, work, ipiv, info + 2 * k) != 0) return 2;
      k_identity<<<(int)((blk + 255) / 256), 256, 0, sf>>>(Si, n1);
      if (cudaGetLastError() != cudaSuccess) return 1;
      if (cusolverDnDgetrs(hb_sol, CUBLAS_OP_N, n1, n1, Dkk, n1, ipiv, Si, n1, info + 2 * k + 1) != 0) return 2;
      return cudaEventRecord(evF, sf) != cudaSuccess ? 1 : 0;
    };
    for (int k = 0; k < M; ++k) {
      if (k == 0) {
        for (int i = 0; i <= hb && i < M; ++i) CK(launch_assemble_row(pc, i, 1, ring + panel_elems * (i % R), sm));
        CKB(factor_diag(0));
      } else if (k + hb < M) {
        CK(launch_assemble_row(pc, k + hb, 1, ring + panel_elems * ((k + hb) % R), sm));
        if (hb == 0) CKB(factor_diag(k));  // block-diagonal case: no trailing products, row k is complete as assembled
      }
      double* Pk = ring + panel_elems * (k % R);
      const double* Sk = Sinv + blk * (k % 2);
      const int lk = k < hb ? k : hb, uk = (M - 1 - k) < hb ? (M - 1 - k) : hb;
      CK(cudaStreamWaitEvent(sm, evF, 0));  // the inverse of this row's diagonal block (recorded during step k - 1)
      // apply form of block row k: row-major [n1][(lk+1) n1] = [ -S~kk^-1 L~k,* | S~kk^-1 ] and [n1][uk n1] =
      // S~kk^-1 S~k,*, written by a transposing copy that also converts when the panels are FP32
      const int Kf = (lk + 1) * n1;
      const dim3 tb(32, 8);
      auto to_apply = [&](const double* in, int cols, double scale, size_t off_elems, size_t col0, size_t ldo, bool fwd) {
        const dim3 tg((cols + 31) / 32, (n1 + 31) / 32);
        if (pc->f32) {
          float* base = static_cast<float*>(fwd ? pc->fwd : pc->bwd) + off_elems + col0;
          k_to_apply_form<float><<<tg, tb, 0, sm>>>(in, n1, cols, scale, base, ldo);
        } else {
          double* base = static_cast<double*>(fwd ? pc->fwd : pc->bwd) + off_elems + col0;
          k_to_apply_form<double><<<tg, tb, 0, sm>>>(in, n1, cols, scale, base, ldo);
        }
      };
      if (lk > 0) {
        const double* Lk = Pk + blk * (hb - lk);  // L~k,k-lk..k-1, column-major n1 x lk n1
        CKB(cublasDgemm(hb_blas, CUBLAS_OP_N, CUBLAS_OP_N, n1, lk * n1, n1, &one, Sk, n1, Lk, n1, &zero, W, n1));
        to_apply(W, lk * n1, -1.0, pc->fwd_off[k], 0, Kf, true);
      }
      to_apply(Sk, n1, 1.0, pc->fwd_off[k], (size_t)lk * n1, Kf, true);
      CK(cudaGetLastError());
      if (uk > 0) {
        // S~kk^-1 S~k,k+1..k+uk by ONE product with the explicit inverse formed above (a getrs on this
        // wide right-hand side spends most of its time in row interchanges and triangular solves: 60 % of
        // the whole set-up when it was used here)
        const double* Uk0 = Pk + blk * (hb + 1);
        double* Uk = W;  // n1 x uk n1, column-major (W's use for the forward panel above is stream-ordered)
        CKB(cublasDgemm(hb_blas, CUBLAS_OP_N, CUBLAS_OP_N, n1, uk * n1, n1, &one, Sk, n1, Uk0, n1, &zero, Uk, n1));
        to_apply(Uk, uk * n1, 1.0, pc->bwd_off[k], 0, (size_t)uk * n1, false);
        CK(cudaGetLastError());
        for (int i = k + 1; i <= k + uk; ++i) {
          double* Pi = ring + panel_elems * (i % R);
          const double* Lik = Pi + blk * (k - i + hb);
          double* Cij = Pi + blk * (k + 1 - i + hb);
          CKB(cublasDgemm(hb_blas, CUBLAS_OP_N, CUBLAS_OP_N, n1, uk * n1, n1, &mone, Lik, n1, Uk, n1, &one, Cij, n1));
          if (i == k + 1) CKB(factor_diag(k + 1));  // row k + 1 is complete: factor its diagonal block on `sf` now
        }
      }
    }
    CK(cudaStreamSynchronize(sf));
    CK(cudaStreamSynchronize(sm));
    info_h.resize(2 * M);
    CK(cudaMemcpy(info_h.data(), info, sizeof(int) * 2 * M, cudaMemcpyDeviceToHost));
    for (int i = 0; i < 2 * M; ++i)
      if (info_h[i] != 0) {
        snprintf(g_err, sizeof g_err, "sws_precond_create: singular diagonal block of the Schur complement (line %d, info %d)",
                 i / 2, info_h[i]);
        rc = SWS_EINVAL;
        goto done;
      }
    pc->factored = 1;
  }
  CK(cudaDeviceSynchronize());

done:
  if (work) cudaFree(work);
  if (info) cudaFree(info);
  if (ipiv) cudaFree(ipiv);
  if (W) cudaFree(W);
  if (Sinv) cudaFree(Sinv);
  if (ring) cudaFree(ring);
  if (evD) cudaEventDestroy(evD);
  if (evF) cudaEventDestroy(evF);
  if (sm) cudaStreamDestroy(sm);
  if (sf) cudaStreamDestroy(sf);
  if (hb_sol) cusolverDnDestroy(hb_sol);
  if (hb_blas) cublasDestroy(hb_blas);
  if (rc != SWS_OK) {
    sws_precond_destroy(pc);
    return rc;
  }
  pc->setup_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_start).count();
  *out = pc;
  return SWS_OK;
}

// the forward and backward block sweeps of App. C on the internal vectors t2 -> y (2 M - 1 dependent launches)
static void launch_sweeps(sws_precond* pc, cudaStream_t st) {
  const int n1 = pc->lm.n1, M = pc->lm.M, hb = pc->hb;
  const bool vec = (n1 % 2) == 0;  // rows, y and t blocks then start on 16-byte boundaries
  if (pc->f32) {
    const float* fwd = static_cast<const float*>(pc->fwd);
    const float* bwd = static_cast<const float*>(pc->bwd);
    for (int k = 0; k < M; ++k) {
      const int lk = k < hb ? k : hb;
      k_fwd_row_f32<<<n1, kGemvThreads, 0, st>>>(fwd + pc->fwd_off[k], n1, lk, pc->y + (size_t)(k - lk) * n1,
                                                 pc->t2 + (size_t)k * n1, pc->y + (size_t)k * n1);
    }
    for (int k = M - 2; k >= 0; --k) {
      const int uk = (M - 1 - k) < hb ? (M - 1 - k) : hb;
      if (uk > 0)
        k_bwd_row_f32<<<n1, kGemvThreads, 0, st>>>(bwd + pc->bwd_off[k], n1, uk, pc->y + (size_t)(k + 1) * n1,
                                                   pc->y + (size_t)k * n1);
    }
    return;
  }
  const double* fwd = static_cast<const double*>(pc->fwd);
  const double* bwd = static_cast<const double*>(pc->bwd);
  for (int k = 0; k < M; ++k) {
    const int lk = k < hb ? k : hb;
    if (vec)
      k_fwd_row<true><<<n1, kGemvThreads, 0, st>>>(fwd + pc->fwd_off[k], n1, lk, pc->y + (size_t)(k - lk) * n1,
                                                   pc->t2 + (size_t)k * n1, pc->y + (size_t)k * n1);
    else
      k_fwd_row<false><<<n1, kGemvThreads, 0, st>>>(fwd + pc->fwd_off[k], n1, lk, pc->y + (size_t)(k - lk) * n1,
                                                    pc->t2 + (size_t)k * n1, pc->y + (size_t)k * n1);
  }
  for (int k = M - 2; k >= 0; --k) {
    const int uk = (M - 1 - k) < hb ? (M - 1 - k) : hb;
    if (uk > 0 && vec)
      k_bwd_row<true><<<n1, kGemvThreads, 0, st>>>(bwd + pc->bwd_off[k], n1, uk, pc->y + (size_t)(k + 1) * n1,
                                                   pc->y + (size_t)k * n1);
    else if (uk > 0)
      k_bwd_row<false><<<n1, kGemvThreads, 0, st>>>(bwd + pc->bwd_off[k], n1, uk, pc->y + (size_t)(k + 1) * n1,
                                                    pc->y + (size_t)k * n1);
  }
}

// Capture the sweeps once (on a private stream: the caller's may be the legacy default stream, which
// cannot be captured); afterwards one graph launch replaces 2 M - 1 kernel launches.
static void build_sweep_graph(sws_precond* pc) {
  pc->sweep_graph_state = -1;
  cudaStream_t cs = nullptr;
  cudaGraph_t g = nullptr;
  if (cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return; }
  if (cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
    launch_sweeps(pc, cs);
    if (cudaStreamEndCapture(cs, &g) == cudaSuccess && g &&
        cudaGraphInstantiate(&pc->sweep_graph, g, 0) == cudaSuccess)
      pc->sweep_graph_state = 1;
  }
  if (g) cudaGraphDestroy(g);
  cudaStreamDestroy(cs);
  cudaGetLastError();
}

int sws_precond_apply(sws_precond* pc, const double* v_dev, double* r_dev, void* cuda_stream) {
  if (!pc || !v_dev || !r_dev) return SWS_EINVAL;
  if (!pc->factored) return SWS_EINVAL;
  DevGuard dg(pc->device);
  if (dg.err != cudaSuccess) return fail_cuda(dg.err, "sws_precond_apply (device)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const LinMesh& m = pc->lm;
  const int n1 = m.n1, M = m.M;
  const size_t sh = 2 * (size_t)n1 * sizeof(double);
  if (pc->sweep_graph_state == 0) build_sweep_graph(pc);
  k_stage1<<<M, 256, sh, st>>>(m, v_dev, pc->s1, pc->t2);
  if (pc->sweep_graph_state == 1) {
    if (cudaGraphLaunch(pc->sweep_graph, st) != cudaSuccess) return fail_cuda(cudaGetLastError(), "sws_precond_apply (graph)");
  } else {
    launch_sweeps(pc, st);
  }
  k_stage3<<<M, 256, sh, st>>>(m, pc->s1, pc->y, r_dev);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? SWS_OK : fail_cuda(e, "sws_precond_apply");
}

int sws_precond_apply_multi(sws_precond* pc, const double* V_dev, int32_t t, double* R_dev, void* cuda_stream) {
  if (!pc || !V_dev || !R_dev || t < 1 || t > 16) return SWS_EINVAL;
  if (!pc->factored) return SWS_EINVAL;
  if (t == 1) return sws_precond_apply(pc, V_dev, R_dev, cuda_stream);
  DevGuard dg(pc->device);
  if (dg.err != cudaSuccess) return fail_cuda(dg.err, "sws_precond_apply_multi (device)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const LinMesh& m = pc->lm;
  const int n1 = m.n1, M = m.M;
  if (t > pc->multi_cap) {  // grow the internal vectors once (synchronises)
    cudaError_t e = cudaDeviceSynchronize();
    double* nb[3] = {nullptr, nullptr, nullptr};
    for (int i = 0; i < 3 && e == cudaSuccess; ++i) e = cudaMalloc(&nb[i], (size_t)16 * m.H * sizeof(double));
    if (e != cudaSuccess) {
      for (double* b : nb) if (b) cudaFree(b);
      return e == cudaErrorMemoryAllocation ? SWS_ENOMEM : fail_cuda(e, "sws_precond_apply_multi (workspace)");
    }
    cudaFree(pc->s1); cudaFree(pc->t2); cudaFree(pc->y);
    pc->s1 = nb[0]; pc->t2 = nb[1]; pc->y = nb[2];
    pc->bytes += (size_t)3 * 15 * m.H * sizeof(double);
    pc->multi_cap = 16;
    if (pc->sweep_graph) { cudaGraphExecDestroy(pc->sweep_graph); pc->sweep_graph = nullptr; }
    pc->sweep_graph_state = 0;  // the captured single-vector sweeps point at the old buffers
  }
  const size_t sh = 2 * (size_t)n1 * sizeof(double);
  int done = 0;
  while (done < t) {  // tiles of 16, 8, 4, 2, 1 right-hand sides
    const int left = t - done;
    const int T = left >= 16 ? 16 : left >= 8 ? 8 : left >= 4 ? 4 : left >= 2 ? 2 : 1;
    const double* v = V_dev + (size_t)done * 2 * m.H;
    double* r = R_dev + (size_t)done * 2 * m.H;
    k_stage1<<<dim3(M, T), 256, sh, st>>>(m, v, pc->s1, pc->t2);
    switch (T) {
      case 16: launch_sweeps_multi<16>(pc, st); break;
      case 8: launch_sweeps_multi<8>(pc, st); break;
      case 4: launch_sweeps_multi<4>(pc, st); break;
      case 2: launch_sweeps_multi<2>(pc, st); break;
      default: launch_sweeps(pc, st); break;
    }
    k_stage3<<<dim3(M, T), 256, sh, st>>>(m, pc->s1, pc->y, r);
    done += T;
  }
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? SWS_OK : fail_cuda(e, "sws_precond_apply_multi");
}

int sws_precond_block_host(sws_precond* pc, int32_t which, int32_t l, int32_t mm, double* out_host) {
  if (!pc || !out_host || l < 0 || l >= pc->lm.M || mm < 0 || mm >= pc->lm.M) return SWS_EINVAL;
  if (which < 0 || which > 1) return SWS_EINVAL;
  const int s = mm - l + pc->hb;
  if (s < 0 || s > 2 * pc->hb) return SWS_EINVAL;
  const int n1 = pc->lm.n1;
  DevGuard dg(pc->device);
  cudaError_t e = dg.err;
  if (e == cudaSuccess) e = launch_assemble_row(pc, l, which, pc->panel, nullptr);
  std::vector<double> cm((size_t)n1 * n1);
  if (e == cudaSuccess)
    e = cudaMemcpy(cm.data(), pc->panel + (size_t)s * n1 * n1, cm.size() * sizeof(double), cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) return fail_cuda(e, "sws_precond_block_host");
  for (int r = 0; r < n1; ++r)
    for (int c = 0; c < n1; ++c) out_host[(size_t)r * n1 + c] = cm[(size_t)c * n1 + r];
  return SWS_OK;
}

size_t sws_precond_bytes(const sws_precond* pc) { return pc ? pc->bytes : 0; }
int sws_precond_bandwidth(const sws_precond* pc) { return pc ? 2 * pc->hb + 1 : 0; }
double sws_precond_setup_ms(const sws_precond* pc) { return pc ? pc->setup_ms : 0.0; }

int sws_precond_destroy(sws_precond* pc) {
  if (!pc) return SWS_OK;
  DevGuard dg(pc->device);
  if (pc->sweep_graph) cudaGraphExecDestroy(pc->sweep_graph);
  void* bufs[] = {pc->G, pc->corr, pc->fwd, pc->bwd, pc->s1, pc->t2, pc->y, pc->panel};
  for (void* b : bufs)
    if (b) cudaFree(b);
  delete pc;
  return SWS_OK;
}

}  // extern "C"
