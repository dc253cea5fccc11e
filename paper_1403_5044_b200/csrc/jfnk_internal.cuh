// Internal declarations of libsws_jfnk (CUDA path).  Shares nothing with oracle/.
// Citations "L<n>" are lines of /root/reference/PAPER.md.
#pragma once
#include <cublas_v2.h>
#include <cuda_runtime.h>
#include <cusolverDn.h>
#include <stdint.h>

#include <vector>

#include "sws_jfnk.h"

namespace jfnk {

// Geometry and constants of the linearised problem (App. B), passed to kernels by value.
struct LinMesh {
  int N, M, n1, H;  // nodes, n1 = N + 1 unknowns per y-line and field, H = n1 M
  double x1, y1, dx, dy;
  double inv_f2;    // 1 / F^2
  double n_rad;
  // A_0 (the (N+1) x (N+1) tridiagonal block of A, identical for every line, (B.2) L462-464, (B.3)):
  //   row 0: n f_1 + x1 fx_1;  row 1: a11 fx_1 + a12 fx_2;  row 1+k: (fx_k + fx_{k+1}) / 2
  double a11, a12;  // n - x1/dx, x1/dx
};

// Entry points run on their object's device and put the caller's current device back on return.
struct DevGuard {
  int prev = -1;
  cudaError_t err;
  explicit DevGuard(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
    else prev = -1;
  }
  ~DevGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

constexpr int kGemvThreads = 256;
constexpr int kDotBlocks = 296;   // 2 CTAs per SM on 148 SMs
constexpr int kDotThreads = 256;

}  // namespace jfnk

struct sws_precond {
  sws_params params;
  jfnk::LinMesh lm;
  int hb;          // half bandwidth in blocks: |l - m| <= hb kept (L241), b = 2 hb + 1
  int factored;
  int device;
  size_t bytes;
  double setup_ms;
  // device
  double* G;       // [n1][n1] column-major: C_0 A_0^-1 B_0 (the block every diagonal block of the Schur complement loses)
  double* corr;    // [T] (sum_ij w K3 - I) / 2 per target, t = l (N-1) + (k-1)        (B.6) L499
  void* fwd;       // per block row k: row-major [n1][(lk+1) n1] = [ -S~kk^-1 L~k,k-lk..k-1 | S~kk^-1 ]
  void* bwd;       // per block row k: row-major [n1][uk n1]     = S~kk^-1 S~k,k+1..k+uk
  int f32;         // the two panels are stored in FP32 (flags bit 1): the factorisation itself is FP64
  std::vector<size_t> fwd_off, bwd_off;  // element offsets of row k's panels
  double* s1;      // [H]  A^-1 b1
  double* t2;      // [H]  b2 - C s1
  double* y;       // [H]  forward / backward substitution vector
  double* panel;   // scratch: one assembled block row (sws_precond_block_host)
  int multi_cap;   // right-hand sides s1, t2, y have room for (1, or 16 after the first sws_precond_apply_multi)
  // the 2 M dependent sweep launches of sws_precond_apply as one CUDA graph (they touch internal buffers only)
  cudaGraphExec_t sweep_graph;
  int sweep_graph_state;  // 0: not built yet, 1: built, -1: capture failed, launch directly
};

namespace jfnk {

// jfnk_precond.cu
cudaError_t launch_assemble_row(const sws_precond* pc, int l, int subtract_G, double* panel, cudaStream_t st);

}  // namespace jfnk
