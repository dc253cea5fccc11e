// Device-resident drivers of the Jacobian-free Newton-Krylov method (section 4.1
// L205-229): right-preconditioned GMRES(m) on J(u) P^-1 (L209-215, Saad & Schultz [47]) and the
// damped Newton iteration (2), (3) L41-45 with a backtracking line search (L209).
//
// Every vector (Krylov basis, residuals, corrections) lives on the device; per iteration the
// host reads back only the new Hessenberg column and a norm (one synchronisation, next to a
// Jacobian-vector product that costs milliseconds).  E(u) and J(u) v are libsws's, called
// through its public C-ABI; P^-1 is jfnk_precond.cu.  Orthogonalisation is classical
// Gram-Schmidt applied twice (two fused multi-dot + multi-axpy passes instead of j dependent
// dot products), which spans the same Krylov space as the textbook modified Gram-Schmidt.
// All reductions have a fixed order (per-CTA partials, then a serial sum): deterministic.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <new>
#include <vector>

#include "jfnk_internal.cuh"

namespace jfnk {

__device__ __forceinline__ double block_sum(double v, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5;
  __syncthreads();  // red may still be read from the previous call
  if ((threadIdx.x & 31) == 0) red[w] = v;
  __syncthreads();
  double s = 0.0;
  if (threadIdx.x == 0)
    for (int i = 0; i < kDotThreads / 32; ++i) s += red[i];
  return s;
}
__device__ __forceinline__ double block_max(double v, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
  const int w = threadIdx.x >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[w] = v;
  __syncthreads();
  double s = 0.0;
  if (threadIdx.x == 0)
    for (int i = 0; i < kDotThreads / 32; ++i) s = fmax(s, red[i]);
  return s;
}

// partial[blk][i] = sum over the CTA's slice of V_i . w, i < nv  (V_i = V + i ld)
__global__ void __launch_bounds__(kDotThreads) k_dots(const double* __restrict__ V, size_t ld, int nv,
                                                      const double* __restrict__ w, int n,
                                                      double* __restrict__ partial) {
  __shared__ double red[kDotThreads / 32];
  for (int i = 0; i < nv; ++i) {
    const double* v = V + (size_t)i * ld;
    double a = 0.0;
    for (int idx = blockIdx.x * kDotThreads + threadIdx.x; idx < n; idx += gridDim.x * kDotThreads)
      a = fma(v[idx], w[idx], a);
    const double s = block_sum(a, red);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * nv + i] = s;
  }
}

// out[i] (+)= sum_blk partial[blk][i]
__global__ void k_dots_finish(const double* __restrict__ partial, int nblk, int nv, double* out, int accumulate) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nv) return;
  double s = 0.0;
  for (int b = 0; b < nblk; ++b) s += partial[(size_t)b * nv + i];
  out[i] = accumulate ? out[i] + s : s;
}

// w -= sum_i coef[i] V_i
__global__ void __launch_bounds__(256) k_project(double* __restrict__ w, const double* __restrict__ V, size_t ld,
                                                 int nv, const double* __restrict__ coef, int n) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n) return;
  double a = w[idx];
  for (int i = 0; i < nv; ++i) a = fma(-coef[i], V[(size_t)i * ld + idx], a);
  w[idx] = a;
}

// out = sum_i coef[i] V_i
__global__ void __launch_bounds__(256) k_lincomb(double* __restrict__ out, const double* __restrict__ V, size_t ld,
                                                 int nv, const double* __restrict__ coef, int n) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n) return;
  double a = 0.0;
  for (int i = 0; i < nv; ++i) a = fma(coef[i], V[(size_t)i * ld + idx], a);
  out[idx] = a;
}

// out = w / sqrt(*normsq)   (out unchanged when *normsq == 0: breakdown, handled by the host)
__global__ void __launch_bounds__(256) k_normalise(double* __restrict__ out, const double* __restrict__ w,
                                                   const double* __restrict__ normsq, int n) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n) return;
  const double q = *normsq;
  if (q > 0.0) out[idx] = w[idx] / sqrt(q);
}

// out = a x + b y
__global__ void __launch_bounds__(256) k_axpby(double* __restrict__ out, double a, const double* __restrict__ x,
                                               double b, const double* __restrict__ y, int n) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n) out[idx] = a * x[idx] + b * y[idx];
}

// partial[blk] = {sum e^2, max |e|}
__global__ void __launch_bounds__(kDotThreads) k_norms(const double* __restrict__ e, int n, double* __restrict__ partial) {
  __shared__ double red[kDotThreads / 32];
  double a = 0.0, mx = 0.0;
  for (int idx = blockIdx.x * kDotThreads + threadIdx.x; idx < n; idx += gridDim.x * kDotThreads) {
    const double v = e[idx];
    a = fma(v, v, a);
    mx = fmax(mx, fabs(v));
  }
  const double s = block_sum(a, red);
  const double m = block_max(mx, red);
  if (threadIdx.x == 0) {
    partial[2 * blockIdx.x] = s;
    partial[2 * blockIdx.x + 1] = m;
  }
}
__global__ void k_norms_finish(const double* __restrict__ partial, int nblk, double* out) {
  double s = 0.0, m = 0.0;
  for (int b = 0; b < nblk; ++b) {
    s += partial[2 * b];
    m = fmax(m, partial[2 * b + 1]);
  }
  out[0] = s;
  out[1] = m;
}

// Enlarged GMRES: piece c of the right-hand side, R0_c = T_c r: the entries of r that belong to the y-lines of
// group c (line l -> group floor(l t / M); the phi and zeta unknowns of a line together), zero elsewhere.
__global__ void __launch_bounds__(256) k_split(double* __restrict__ R0, const double* __restrict__ r, int n, int n1,
                                               int M, int t) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n) return;
  const int H = n1 * M;
  const int line = (idx >= H ? idx - H : idx) / n1;
  const int grp = (int)(((long long)line * t) / M);
  const double v = r[idx];
  for (int c = 0; c < t; ++c) R0[(size_t)c * n + idx] = (c == grp) ? v : 0.0;
}

}  // namespace jfnk

using namespace jfnk;

struct sws_solver {
  sws_ctx* ctx;
  sws_precond* pc;
  int device, n, m_max;
  double* V;        // [m_max + 1][n] Krylov basis
  double *w, *z, *t, *r;
  double *E, *Et, *du, *ut, *rhs;
  double *ub, *Eb;  // jv_mode 2: shifted state u + sigma v and E of it
  double* ukeep;    // sws_solver_continuation: the last converged solution
  double* partial;  // [kDotBlocks][m_max + 2]
  double* hdev;     // [2 (m_max + 1) + 2]: h1 | h2 | normsq, scratch
  double* ydev;     // [m_max]
  double* hpin;     // pinned host mirror of hdev
  // enlarged (block) GMRES, allocated at its first use
  int N, M, max_batch;
  int blk_t;        // pieces the block workspace was sized for (0: none)
  double *Zb, *Wb;  // [t][n] each: P^-1 V_j and J P^-1 V_j
  double* hblk;     // device: per column of a block [2 nv_max | 2 t | 1] orthogonalisation coefficients
  double* hblk_pin; // pinned host mirror
  size_t hblk_len;
  cudaEvent_t ev[4];
  // accounting of the current driver call
  int n_jv, n_pc, n_res;
  double ms_jv, ms_pc, ms_res;
};

namespace {

thread_local char g_err[256] = "";
int fail_cuda(cudaError_t e, const char* where) {
  snprintf(g_err, sizeof g_err, "%s: %s", where, cudaGetErrorString(e));
  return SWS_ECUDA;
}
#define RC(call)                       \
  do {                                 \
    int rc_ = (call);                  \
    if (rc_ != SWS_OK) return rc_;     \
  } while (0)
#define CU(call)                                        \
  do {                                                  \
    cudaError_t e_ = (call);                            \
    if (e_ != cudaSuccess) return fail_cuda(e_, #call); \
  } while (0)

inline int nblk(int n) { return (n + 255) / 256; }

// out = sum of squares and max of e, read back (synchronises)
int norms(sws_solver* s, const double* e, double* l2, double* linf, cudaStream_t st) {
  k_norms<<<kDotBlocks, kDotThreads, 0, st>>>(e, s->n, s->partial);
  k_norms_finish<<<1, 1, 0, st>>>(s->partial, kDotBlocks, s->hdev);
  CU(cudaMemcpyAsync(s->hpin, s->hdev, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  *l2 = std::sqrt(s->hpin[0]);
  if (linf) *linf = s->hpin[1];
  return SWS_OK;
}

int apply_pinv(sws_solver* s, const double* v, double* out, cudaStream_t st) {
  if (!s->pc) {
    CU(cudaMemcpyAsync(out, v, sizeof(double) * s->n, cudaMemcpyDeviceToDevice, st));
    return SWS_OK;
  }
  ++s->n_pc;
  return sws_precond_apply(s->pc, v, out, st);
}

// ub = fma(sigma, v, u) entry by entry, as sws_jv_batch forms its shifted states
__global__ void __launch_bounds__(256) k_shift(double* __restrict__ ub, double sigma, const double* __restrict__ v,
                                               const double* __restrict__ u, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) ub[i] = fma(sigma, v[i], u[i]);
}
// out = (Eb - E0) / sigma, eq. (25)
__global__ void __launch_bounds__(256) k_fd_quotient(double* __restrict__ out, const double* __restrict__ Eb,
                                                     const double* __restrict__ E0, double sigma, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (Eb[i] - E0[i]) / sigma;
}

// mode 2: eq. (25) with the base residual E0 = E(u) the caller already holds (the Newton driver's E_k):
// one residual evaluation per product.  unorm = ||u||_2; the shift is libsws's 1e-7 (1 + ||u||) / ||v||.
int apply_jv(sws_solver* s, const double* u, const double* v, double* out, int mode, cudaStream_t st,
             const double* E0 = nullptr, double unorm = 0.0) {
  ++s->n_jv;
  if (mode == 1) return sws_jv_batch(s->ctx, u, v, 1, nullptr, out, nullptr, nullptr, st);
  if (mode == 2) {
    double vn = 0.0;
    RC(norms(s, v, &vn, nullptr, st));
    if (vn == 0.0) {
      CU(cudaMemsetAsync(out, 0, sizeof(double) * s->n, st));
      return SWS_OK;
    }
    const double sigma = 1e-7 * (1.0 + unorm) / vn;
    k_shift<<<nblk(s->n), 256, 0, st>>>(s->ub, sigma, v, u, s->n);
    ++s->n_res;
    RC(sws_residual(s->ctx, s->ub, s->Eb, st));
    k_fd_quotient<<<nblk(s->n), 256, 0, st>>>(out, s->Eb, E0, sigma, s->n);
    return SWS_OK;
  }
  return sws_jv_apply(s->ctx, v, 1, out, st);  // the linearisation at u was formed by gmres()
}

// E0: E(u) if the caller has it (jv_mode 2 only; computed here otherwise)
int gmres(sws_solver* s, const double* u, const double* rhs, const sws_gmres_opts* o, double* d,
          sws_gmres_stats* stats, double* hist, cudaStream_t st, const double* E0 = nullptr) {
  const int n = s->n, m = o->restart;
  if (m < 1 || m > s->m_max || o->maxit < 1 || o->jv_mode < 0 || o->jv_mode > 2) return SWS_EINVAL;
  double unorm = 0.0;
  if (o->jv_mode == 2) {
    RC(norms(s, u, &unorm, nullptr, st));
    if (!E0) {  // standalone solve: the base residual, once
      ++s->n_res;
      RC(sws_residual(s->ctx, u, s->Et, st));
      E0 = s->Et;
    }
  }
  const size_t ld = (size_t)n;
  double bnorm = 0.0;
  RC(norms(s, rhs, &bnorm, nullptr, st));
  CU(cudaMemsetAsync(d, 0, sizeof(double) * n, st));
  stats->its = 0; stats->converged = 0; stats->rel_res = 0.0; stats->rhs_norm = bnorm;
  if (bnorm == 0.0) { stats->converged = 1; return SWS_OK; }
  if (o->jv_mode == 0) {  // linearise once per solve: everything of J(u) that depends on u alone
    CU(cudaEventRecord(s->ev[0], st));
    RC(sws_linearize(s->ctx, u, st));
    CU(cudaEventRecord(s->ev[1], st));
    CU(cudaStreamSynchronize(st));
    float a = 0.f;
    cudaEventElapsedTime(&a, s->ev[0], s->ev[1]);
    s->ms_jv += a;
  }
  std::vector<double> H((size_t)(m + 1) * m, 0.0), cs(m), sn(m), g(m + 1), y(m);
  auto Hm = [&](int i, int j) -> double& { return H[(size_t)i * m + j]; };
  CU(cudaMemcpyAsync(s->r, rhs, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
  int its = 0;
  double rel = 1.0;
  double beta = bnorm;
  bool first = true;
  while (its < o->maxit) {
    if (!first) RC(norms(s, s->r, &beta, nullptr, st));
    first = false;
    if (!(beta > 0.0)) { rel = 0.0; break; }  // the restart residual vanished: d is exact, nothing to normalise
    k_axpby<<<nblk(n), 256, 0, st>>>(s->V, 1.0 / beta, s->r, 0.0, s->r, n);
    std::fill(g.begin(), g.end(), 0.0);
    g[0] = beta;
    int jd = 0;
    for (int j = 0; j < m; ++j) {
      const int nv = j + 1;
      double* h1 = s->hdev;
      double* h2 = s->hdev + (m + 1);
      double* nq = s->hdev + 2 * (m + 1);
      CU(cudaEventRecord(s->ev[0], st));
      RC(apply_pinv(s, s->V + (size_t)j * ld, s->z, st));
      CU(cudaEventRecord(s->ev[1], st));
      RC(apply_jv(s, u, s->z, s->w, o->jv_mode, st, E0, unorm));
      CU(cudaEventRecord(s->ev[2], st));
      ++its;
      // classical Gram-Schmidt, twice
      k_dots<<<kDotBlocks, kDotThreads, 0, st>>>(s->V, ld, nv, s->w, n, s->partial);
      k_dots_finish<<<(nv + 127) / 128, 128, 0, st>>>(s->partial, kDotBlocks, nv, h1, 0);
      k_project<<<nblk(n), 256, 0, st>>>(s->w, s->V, ld, nv, h1, n);
      k_dots<<<kDotBlocks, kDotThreads, 0, st>>>(s->V, ld, nv, s->w, n, s->partial);
      k_dots_finish<<<(nv + 127) / 128, 128, 0, st>>>(s->partial, kDotBlocks, nv, h2, 0);
      k_project<<<nblk(n), 256, 0, st>>>(s->w, s->V, ld, nv, h2, n);
      k_dots<<<kDotBlocks, kDotThreads, 0, st>>>(s->w, ld, 1, s->w, n, s->partial);
      k_dots_finish<<<1, 128, 0, st>>>(s->partial, kDotBlocks, 1, nq, 0);
      k_normalise<<<nblk(n), 256, 0, st>>>(s->V + (size_t)(j + 1) * ld, s->w, nq, n);
      CU(cudaMemcpyAsync(s->hpin, s->hdev, sizeof(double) * (2 * (m + 1) + 1), cudaMemcpyDeviceToHost, st));
      CU(cudaStreamSynchronize(st));
      {
        float a = 0.f, b = 0.f;
        cudaEventElapsedTime(&a, s->ev[0], s->ev[1]);
        cudaEventElapsedTime(&b, s->ev[1], s->ev[2]);
        s->ms_pc += a; s->ms_jv += b;
      }
      for (int i = 0; i <= j; ++i) Hm(i, j) = s->hpin[i] + s->hpin[(m + 1) + i];
      Hm(j + 1, j) = std::sqrt(s->hpin[2 * (m + 1)]);
      for (int i = 0; i < j; ++i) {
        const double tmp = cs[i] * Hm(i, j) + sn[i] * Hm(i + 1, j);
        Hm(i + 1, j) = -sn[i] * Hm(i, j) + cs[i] * Hm(i + 1, j);
        Hm(i, j) = tmp;
      }
      // happy breakdown: w lies in the span of the basis (h_{j+1,j} = 0 up to rounding); k_normalise left
      // V_{j+1} alone, the least-squares problem is solved exactly with the j + 1 columns at hand
      double hcol = 0.0;
      for (int i = 0; i <= j; ++i) hcol = std::max(hcol, std::fabs(Hm(i, j)));
      const bool breakdown = !(Hm(j + 1, j) > 1e-300) || Hm(j + 1, j) <= 1e-15 * hcol;
      if (breakdown) Hm(j + 1, j) = 0.0;
      const double rho = std::hypot(Hm(j, j), Hm(j + 1, j));
      if (rho == 0.0) {  // J P^-1 v_j = 0: the column adds nothing; stop with what was reached
        jd = j;
        if (hist) hist[its - 1] = rel;  // the iteration was counted: its history slot holds the residual reached
        break;
      }
      cs[j] = Hm(j, j) / rho; sn[j] = Hm(j + 1, j) / rho;
      Hm(j, j) = rho; Hm(j + 1, j) = 0.0;
      g[j + 1] = -sn[j] * g[j];
      g[j] = cs[j] * g[j];
      jd = j + 1;
      rel = std::fabs(g[j + 1]) / bnorm;
      if (hist) hist[its - 1] = rel;
      if (breakdown || std::fabs(g[j + 1]) <= o->tol * bnorm || its >= o->maxit) break;
    }
    // y = R^-1 g (back substitution), d += P^-1 (V y)
    for (int i = jd - 1; i >= 0; --i) {
      double acc = g[i];
      for (int k = i + 1; k < jd; ++k) acc -= Hm(i, k) * y[k];
      y[i] = acc / Hm(i, i);
    }
    CU(cudaMemcpyAsync(s->ydev, y.data(), sizeof(double) * jd, cudaMemcpyHostToDevice, st));
    k_lincomb<<<nblk(n), 256, 0, st>>>(s->t, s->V, ld, jd, s->ydev, n);
    RC(apply_pinv(s, s->t, s->z, st));
    k_axpby<<<nblk(n), 256, 0, st>>>(d, 1.0, d, 1.0, s->z, n);
    CU(cudaStreamSynchronize(st));  // y is host memory reused by the next cycle
    if (rel <= o->tol || its >= o->maxit || jd == 0) break;
    // restart: r = rhs - J d
    RC(apply_jv(s, u, d, s->w, o->jv_mode, st, E0, unorm));
    k_axpby<<<nblk(n), 256, 0, st>>>(s->r, 1.0, rhs, -1.0, s->w, n);
  }
  stats->its = its;
  stats->rel_res = rel;
  stats->converged = rel <= o->tol ? 1 : 0;
  CU(cudaGetLastError());
  return SWS_OK;
}

// ---------------------------------------------------------------------------------------
// Enlarged (block) GMRES: the Krylov method that uses b > 1 products per iteration.
// The right-hand side is split by groups of y-lines into t pieces that sum to it, R0 = [T_1 r .. T_t r]; block
// Arnoldi builds K_m(J P^-1, R0) with ONE sws_jv_apply(V[t]) (or one sws_jv_batch) and ONE multi-vector
// preconditioner sweep per iteration; the iterate minimises ||r - J P^-1 V y|| over that space, which contains
// the plain Krylov space of the same depth.  One cycle (no restart): at most (m_max + 1) / t - 1 blocks.

int ensure_block_workspace(sws_solver* s, int t) {
  if (s->blk_t >= t) return SWS_OK;
  CU(cudaDeviceSynchronize());
  if (s->Zb) cudaFree(s->Zb);
  if (s->hblk) cudaFree(s->hblk);
  if (s->hblk_pin) cudaFreeHost(s->hblk_pin);
  s->Zb = s->Wb = s->hblk = s->hblk_pin = nullptr;
  s->blk_t = 0;
  const size_t n = (size_t)s->n;
  s->hblk_len = (size_t)t * (2 * (size_t)(s->m_max + 1) + 2 * t + 1);
  cudaError_t e = cudaMalloc(&s->Zb, 2 * (size_t)t * n * sizeof(double));
  if (e == cudaSuccess) e = cudaMalloc(&s->hblk, s->hblk_len * sizeof(double));
  if (e == cudaSuccess) e = cudaMallocHost(&s->hblk_pin, s->hblk_len * sizeof(double));
  if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? SWS_ENOMEM : fail_cuda(e, "enlarged GMRES workspace");
  s->Wb = s->Zb + (size_t)t * n;
  s->blk_t = t;
  return SWS_OK;
}

// Orthogonalise the t vectors W_c (ld n) against the nv basis vectors V (classical Gram-Schmidt, twice) and
// against one another, in order; the normalised vectors go to Q_c (Q may be W).  Coefficients of column c to
// hblk + c stride: [h1 | h2] against V, [q1 | q2] against Q_0..Q_{c-1}, then the squared norm.  No host sync.
void orth_block(sws_solver* s, double* W, int t, const double* V, int nv, double* Q, cudaStream_t st) {
  const int n = s->n, nvmax = s->m_max + 1;
  const size_t ld = (size_t)n, stride = 2 * (size_t)nvmax + 2 * t + 1;
  for (int c = 0; c < t; ++c) {
    double* w = W + (size_t)c * ld;
    double* h = s->hblk + (size_t)c * stride;
    for (int pass = 0; pass < 2; ++pass) {
      if (nv > 0) {
        double* hp = h + (size_t)pass * nvmax;
        k_dots<<<kDotBlocks, kDotThreads, 0, st>>>(V, ld, nv, w, n, s->partial);
        k_dots_finish<<<(nv + 127) / 128, 128, 0, st>>>(s->partial, kDotBlocks, nv, hp, 0);
        k_project<<<nblk(n), 256, 0, st>>>(w, V, ld, nv, hp, n);
      }
      if (c > 0) {
        double* qp = h + 2 * (size_t)nvmax + (size_t)pass * t;
        k_dots<<<kDotBlocks, kDotThreads, 0, st>>>(Q, ld, c, w, n, s->partial);
        k_dots_finish<<<1, 128, 0, st>>>(s->partial, kDotBlocks, c, qp, 0);
        k_project<<<nblk(n), 256, 0, st>>>(w, Q, ld, c, qp, n);
      }
    }
    double* nq = h + 2 * (size_t)nvmax + 2 * t;
    k_dots<<<kDotBlocks, kDotThreads, 0, st>>>(w, ld, 1, w, n, s->partial);
    k_dots_finish<<<1, 128, 0, st>>>(s->partial, kDotBlocks, 1, nq, 0);
    k_normalise<<<nblk(n), 256, 0, st>>>(Q + (size_t)c * ld, w, nq, n);
  }
}

// returns SWS_OK; *fallback = 1 when a piece of the split right-hand side vanishes (the caller runs plain GMRES)
int egmres(sws_solver* s, const double* u, const double* rhs, const sws_gmres_opts* o, double* d,
           sws_gmres_stats* stats, double* hist, cudaStream_t st, int* fallback) {
  const int n = s->n, t = o->block;
  *fallback = 0;
  if (t < 2 || t > 16 || t > s->max_batch || o->jv_mode < 0 || o->jv_mode > 2 || o->maxit < 1) return SWS_EINVAL;
  int mb = (s->m_max + 1) / t - 1;
  if (o->restart / t < mb) mb = o->restart / t;
  if (mb < 1) return SWS_EINVAL;
  RC(ensure_block_workspace(s, t));
  const size_t ld = (size_t)n;
  const int nvmax = s->m_max + 1;
  const size_t stride = 2 * (size_t)nvmax + 2 * t + 1;
  double bnorm = 0.0;
  RC(norms(s, rhs, &bnorm, nullptr, st));
  CU(cudaMemsetAsync(d, 0, sizeof(double) * n, st));
  stats->its = 0; stats->converged = 0; stats->rel_res = 0.0; stats->rhs_norm = bnorm;
  if (bnorm == 0.0) { stats->converged = 1; return SWS_OK; }
  if (o->jv_mode == 0) {
    CU(cudaEventRecord(s->ev[0], st));
    RC(sws_linearize(s->ctx, u, st));
    CU(cudaEventRecord(s->ev[1], st));
    CU(cudaStreamSynchronize(st));
    float a = 0.f;
    cudaEventElapsedTime(&a, s->ev[0], s->ev[1]);
    s->ms_jv += a;
  }
  // R0 = V_1 B
  k_split<<<nblk(n), 256, 0, st>>>(s->V, rhs, n, s->N + 1, s->M, t);
  orth_block(s, s->V, t, s->V, 0, s->V, st);
  CU(cudaMemcpyAsync(s->hblk_pin, s->hblk, s->hblk_len * sizeof(double), cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  const int rows_max = (mb + 1) * t, cols_max = mb * t;
  std::vector<double> H((size_t)rows_max * cols_max, 0.0), g(rows_max, 0.0), y(cols_max, 0.0);
  std::vector<double> rc, rs;   // Givens rotations in the order they were made ...
  std::vector<int> rr;          // ... each acting on rows (rr, rr + 1)
  auto Hm = [&](int i, int j) -> double& { return H[(size_t)i * cols_max + j]; };
  {
    // g = e_1 (x) (B 1): B[i][c] = coefficient of V_i in piece c
    for (int c = 0; c < t; ++c) {
      const double* h = s->hblk_pin + (size_t)c * stride;
      const double rcc = std::sqrt(h[2 * nvmax + 2 * t]);
      if (!(rcc > 0.0)) { *fallback = 1; return SWS_OK; }
      for (int i = 0; i < c; ++i) g[i] += h[2 * nvmax + i] + h[2 * nvmax + t + i];
      g[c] += rcc;
    }
  }
  double rel = 1.0;
  int cols = 0;  // columns of the band Hessenberg matrix that entered the least-squares problem
  bool broke = false;
  for (int j = 0; j < mb && !broke; ++j) {
    const int nv = (j + 1) * t;
    CU(cudaEventRecord(s->ev[0], st));
    if (s->pc) {
      s->n_pc += t;
      RC(sws_precond_apply_multi(s->pc, s->V + (size_t)j * t * ld, t, s->Zb, st));
    } else {
      CU(cudaMemcpyAsync(s->Zb, s->V + (size_t)j * t * ld, sizeof(double) * t * ld, cudaMemcpyDeviceToDevice, st));
    }
    CU(cudaEventRecord(s->ev[1], st));
    s->n_jv += t;
    if (o->jv_mode == 0) RC(sws_jv_apply(s->ctx, s->Zb, t, s->Wb, st));   // ONE call, t products
    else RC(sws_jv_batch(s->ctx, u, s->Zb, t, nullptr, s->Wb, nullptr, nullptr, st));
    CU(cudaEventRecord(s->ev[2], st));
    orth_block(s, s->Wb, t, s->V, nv, s->V + (size_t)nv * ld, st);
    CU(cudaMemcpyAsync(s->hblk_pin, s->hblk, s->hblk_len * sizeof(double), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    {
      float a = 0.f, b = 0.f;
      cudaEventElapsedTime(&a, s->ev[0], s->ev[1]);
      cudaEventElapsedTime(&b, s->ev[1], s->ev[2]);
      s->ms_pc += a; s->ms_jv += b;
    }
    stats->its += t;
    for (int c = 0; c < t; ++c) {
      const int col = j * t + c;
      const double* h = s->hblk_pin + (size_t)c * stride;
      for (int i = 0; i < nv; ++i) Hm(i, col) = h[i] + h[nvmax + i];
      for (int i = 0; i < c; ++i) Hm(nv + i, col) = h[2 * nvmax + i] + h[2 * nvmax + t + i];
      const double rcc = std::sqrt(h[2 * nvmax + 2 * t]);
      Hm(nv + c, col) = rcc;
      double hmax = 0.0;
      for (int i = 0; i < nv + c; ++i) hmax = std::max(hmax, std::fabs(Hm(i, col)));
      if (!(rcc > 1e-14 * hmax)) {
        // The block lost rank at this column: k_normalise left Q_c as it was (stale data of an earlier solve when the
        // squared norm is exactly 0, normalised rounding noise otherwise) and the later columns of the block were
        // projected against it.  Neither this column nor the later ones of the block enter H, the residual estimate
        // or the combination V y: the solve stops with the col columns that are orthonormal.
        broke = true;
        break;
      }
      cols = col + 1;
      for (size_t q = 0; q < rr.size(); ++q) {   // the rotations made so far
        const int r = rr[q];
        const double a = Hm(r, col), b = Hm(r + 1, col);
        Hm(r, col) = rc[q] * a + rs[q] * b;
        Hm(r + 1, col) = -rs[q] * a + rc[q] * b;
      }
      for (int r = col + t; r > col; --r) {      // zero the t entries below the diagonal, bottom up
        const double a = Hm(r - 1, col), b = Hm(r, col);
        const double rho = std::hypot(a, b);
        const double cc = rho > 0.0 ? a / rho : 1.0, ss = rho > 0.0 ? b / rho : 0.0;
        Hm(r - 1, col) = rho; Hm(r, col) = 0.0;
        const double ga = g[r - 1], gb = g[r];
        g[r - 1] = cc * ga + ss * gb;
        g[r] = -ss * ga + cc * gb;
        rr.push_back(r - 1); rc.push_back(cc); rs.push_back(ss);
      }
    }
    // least-squares residual with the first `cols` columns: the t entries of g below them
    double res2 = 0.0;
    for (int i = cols; i < cols + t; ++i) res2 += g[i] * g[i];
    rel = std::sqrt(res2) / bnorm;
    if (hist) hist[j] = rel;
    if (rel <= o->tol || stats->its + t > o->maxit) break;
  }
  for (int i = cols - 1; i >= 0; --i) {
    double acc = g[i];
    for (int k = i + 1; k < cols; ++k) acc -= Hm(i, k) * y[k];
    y[i] = Hm(i, i) != 0.0 ? acc / Hm(i, i) : 0.0;
  }
  if (cols == 0) CU(cudaMemsetAsync(s->t, 0, sizeof(double) * n, st));  // rank lost in the very first column: d = 0
  // the basis may be longer than ydev (m_max): the combination is formed in slices of m_max vectors
  for (int off = 0; off < cols; off += s->m_max) {
    const int cnt = std::min(s->m_max, cols - off);
    CU(cudaMemcpyAsync(s->ydev, y.data() + off, sizeof(double) * cnt, cudaMemcpyHostToDevice, st));
    k_lincomb<<<nblk(n), 256, 0, st>>>(off == 0 ? s->t : s->w, s->V + (size_t)off * ld, ld, cnt, s->ydev, n);
    if (off > 0) k_axpby<<<nblk(n), 256, 0, st>>>(s->t, 1.0, s->t, 1.0, s->w, n);
    CU(cudaStreamSynchronize(st));
  }
  RC(apply_pinv(s, s->t, d, st));
  CU(cudaStreamSynchronize(st));
  stats->rel_res = rel;
  stats->converged = rel <= o->tol ? 1 : 0;
  CU(cudaGetLastError());
  return SWS_OK;
}

// plain GMRES (block <= 1) or enlarged GMRES with opts->block pieces
int solve_linear(sws_solver* s, const double* u, const double* rhs, const sws_gmres_opts* o, double* d,
                 sws_gmres_stats* stats, double* hist, cudaStream_t st, const double* E0) {
  if (o->block >= 2) {
    int fallback = 0;
    RC(egmres(s, u, rhs, o, d, stats, hist, st, &fallback));
    if (!fallback) return SWS_OK;
  }
  return gmres(s, u, rhs, o, d, stats, hist, st, E0);
}

int residual(sws_solver* s, const double* u, double* E, cudaStream_t st) {
  ++s->n_res;
  CU(cudaEventRecord(s->ev[0], st));
  RC(sws_residual(s->ctx, u, E, st));
  CU(cudaEventRecord(s->ev[1], st));
  return SWS_OK;
}
void account_residual(sws_solver* s) {  // after a synchronise
  float a = 0.f;
  cudaEventElapsedTime(&a, s->ev[0], s->ev[1]);
  s->ms_res += a;
}
void reset_accounting(sws_solver* s) {
  s->n_jv = s->n_pc = s->n_res = 0;
  s->ms_jv = s->ms_pc = s->ms_res = 0.0;
}

}  // namespace

extern "C" {

const char* sws_solver_last_error(void) { return g_err; }

int sws_solver_create(sws_ctx* ctx, sws_precond* pc, int32_t max_restart, sws_solver** out) {
  if (!ctx || !out || max_restart < 1 || max_restart > 512) return SWS_EINVAL;
  *out = nullptr;
  sws_params p;
  RC(sws_get_params(ctx, &p));
  if (p.max_batch < 1) return SWS_EBATCH;
  if (pc && (pc->lm.N != p.N || pc->lm.M != p.M || pc->device != p.device)) return SWS_EINVAL;
  sws_solver* s = new (std::nothrow) sws_solver();
  if (!s) return SWS_ENOMEM;
  s->ctx = ctx; s->pc = pc; s->device = p.device;
  s->N = p.N; s->M = p.M; s->max_batch = p.max_batch;
  s->blk_t = 0; s->Zb = s->Wb = s->hblk = s->hblk_pin = nullptr; s->hblk_len = 0;
  s->n = (int)sws_num_unknowns(ctx);
  s->m_max = max_restart;
  reset_accounting(s);
  const size_t n = (size_t)s->n;
  double* base = nullptr;
  const size_t vec = (size_t)(max_restart + 1) + 12;
  DevGuard dg(p.device);
  cudaError_t e = dg.err;
  if (e == cudaSuccess) e = cudaMalloc(&base, vec * n * sizeof(double));
  if (e == cudaSuccess) e = cudaMalloc(&s->partial, sizeof(double) * kDotBlocks * (max_restart + 2));
  if (e == cudaSuccess) e = cudaMalloc(&s->hdev, sizeof(double) * (2 * (max_restart + 1) + 2));
  if (e == cudaSuccess) e = cudaMalloc(&s->ydev, sizeof(double) * max_restart);
  if (e == cudaSuccess) e = cudaMallocHost(&s->hpin, sizeof(double) * (2 * (max_restart + 1) + 2));
  for (int i = 0; i < 4 && e == cudaSuccess; ++i) e = cudaEventCreate(&s->ev[i]);
  if (e != cudaSuccess) {
    s->V = base;
    sws_solver_destroy(s);
    return e == cudaErrorMemoryAllocation ? SWS_ENOMEM : fail_cuda(e, "sws_solver_create");
  }
  s->V = base;
  double* q = base + (size_t)(max_restart + 1) * n;
  s->w = q; s->z = q + n; s->t = q + 2 * n; s->r = q + 3 * n;
  s->E = q + 4 * n; s->Et = q + 5 * n; s->du = q + 6 * n; s->ut = q + 7 * n; s->rhs = q + 8 * n;
  s->ub = q + 9 * n; s->Eb = q + 10 * n; s->ukeep = q + 11 * n;
  *out = s;
  return SWS_OK;
}

int sws_solver_gmres(sws_solver* s, const double* u_dev, const double* rhs_dev, const sws_gmres_opts* opts,
                     double* d_dev, sws_gmres_stats* stats, double* hist_host, void* cuda_stream) {
  if (!s || !u_dev || !rhs_dev || !opts || !d_dev || !stats) return SWS_EINVAL;
  DevGuard dg(s->device);
  CU(dg.err);
  reset_accounting(s);
  return solve_linear(s, u_dev, rhs_dev, opts, d_dev, stats, hist_host, (cudaStream_t)cuda_stream, nullptr);
}

int sws_solver_newton(sws_solver* s, double* u_dev, const sws_newton_opts* o, sws_newton_log* log, int32_t* nlog,
                      sws_newton_stats* stats, void* cuda_stream) {
  if (!s || !u_dev || !o || !log || !nlog || !stats) return SWS_EINVAL;
  if (o->max_newton < 0 || o->max_halvings < 0) return SWS_EINVAL;
  if (o->forcing != 0 && o->forcing != 1) return SWS_EINVAL;
  if (o->forcing == 1 && !(o->eta > 0.0 && o->eta <= o->eta_max && o->eta_max < 1.0)) return SWS_EINVAL;
  DevGuard dg(s->device);
  CU(dg.err);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const auto t0 = std::chrono::steady_clock::now();
  reset_accounting(s);
  const int n = s->n;
  sws_gmres_opts go = o->gmres;
  double eta_k = o->forcing == 1 ? o->eta_max : o->eta;
  int nl = 0, converged = 0, steps = 0;
  double fn = 0.0, finf = 0.0;
  RC(residual(s, u_dev, s->E, st));
  RC(norms(s, s->E, &fn, &finf, st));
  account_residual(s);
  for (int it = 0; it < o->max_newton; ++it) {
    if (finf <= o->ftol) { converged = 1; break; }
    k_axpby<<<nblk(n), 256, 0, st>>>(s->rhs, -1.0, s->E, 0.0, s->E, n);
    sws_gmres_stats gs;
    go.tol = eta_k;
    RC(solve_linear(s, u_dev, s->rhs, &go, s->du, &gs, nullptr, st, s->E));
    double lam = 1.0, fnt = 0.0, finft = 0.0;
    bool ok = false;
    for (int hv = 0; hv <= o->max_halvings; ++hv) {
      k_axpby<<<nblk(n), 256, 0, st>>>(s->ut, 1.0, u_dev, lam, s->du, n);
      RC(residual(s, s->ut, s->Et, st));
      RC(norms(s, s->Et, &fnt, &finft, st));
      account_residual(s);
      if (fnt < (1.0 - o->alpha * lam) * fn) { ok = true; break; }
      lam *= 0.5;
    }
    log[nl++] = sws_newton_log{it, gs.its, fn, finf, gs.rel_res, ok ? lam : 0.0};
    if (!ok) break;
    CU(cudaMemcpyAsync(u_dev, s->ut, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
    CU(cudaMemcpyAsync(s->E, s->Et, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
    if (o->forcing == 1) {  // eta_{k+1} from the decrease just obtained (sws_jfnk.h)
      double e = 0.9 * (fnt / fn) * (fnt / fn);
      const double sg = 0.9 * eta_k * eta_k;
      if (sg > 0.1) e = std::max(e, sg);
      eta_k = std::min(o->eta_max, std::max(e, o->eta));
    }
    fn = fnt; finf = finft;
    ++steps;
  }
  if (finf <= o->ftol) converged = 1;
  log[nl] = sws_newton_log{nl, 0, fn, finf, 0.0, 0.0};
  ++nl;
  CU(cudaStreamSynchronize(st));
  *nlog = nl;
  stats->steps = steps; stats->converged = converged;
  stats->residual_evals = s->n_res; stats->jv_products = s->n_jv; stats->precond_applies = s->n_pc;
  stats->ms_jv = s->ms_jv; stats->ms_precond = s->ms_pc; stats->ms_residual = s->ms_res;
  stats->ms_total = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  return SWS_OK;
}

int sws_solver_continuation(sws_solver* s, double* u_dev, const double* eps_host, int32_t n_eps,
                            const sws_newton_opts* o, sws_newton_stats* stats, int32_t* n_done, void* cuda_stream) {
  if (!s || !u_dev || !eps_host || n_eps < 1 || !o || !stats || !n_done) return SWS_EINVAL;
  DevGuard dg(s->device);
  CU(dg.err);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  *n_done = 0;
  std::vector<sws_newton_log> log((size_t)o->max_newton + 1);
  for (int i = 0; i < n_eps; ++i) {
    RC(sws_set_eps(s->ctx, eps_host[i]));
    CU(cudaMemcpyAsync(s->ukeep, u_dev, sizeof(double) * s->n, cudaMemcpyDeviceToDevice, st));
    int32_t nl = 0;
    RC(sws_solver_newton(s, u_dev, o, log.data(), &nl, &stats[i], cuda_stream));
    if (!stats[i].converged) {  // hand back the last converged solution (or the caller's guess)
      CU(cudaMemcpyAsync(u_dev, s->ukeep, sizeof(double) * s->n, cudaMemcpyDeviceToDevice, st));
      CU(cudaStreamSynchronize(st));
      break;
    }
    ++*n_done;
  }
  return SWS_OK;
}

int sws_solver_destroy(sws_solver* s) {
  if (!s) return SWS_OK;
  DevGuard dg(s->device);
  if (s->V) cudaFree(s->V);
  if (s->partial) cudaFree(s->partial);
  if (s->hdev) cudaFree(s->hdev);
  if (s->ydev) cudaFree(s->ydev);
  if (s->hpin) cudaFreeHost(s->hpin);
  if (s->Zb) cudaFree(s->Zb);
  if (s->hblk) cudaFree(s->hblk);
  if (s->hblk_pin) cudaFreeHost(s->hblk_pin);
  for (int i = 0; i < 4; ++i)
    if (s->ev[i]) cudaEventDestroy(s->ev[i]);
  delete s;
  return SWS_OK;
}

}  // extern "C"
