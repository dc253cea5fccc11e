// libsws_debug.so (include/sws_debug.h): unit-test hooks of the all-pairs kernel's device primitives and
// the FP64 instruction-mix probes behind DESIGN.md section 6.  NOT part of the product library libsws.so:
// built only with -DSWS_BUILD_DEBUG_HOOKS, loaded by tests/ and by bench.py's measurement helpers.  The
// hooks call the very inline device functions the kernels use (sws_farfield.cuh), nothing is re-implemented.
#ifndef SWS_BUILD_DEBUG_HOOKS
#error "sws_debug.cu is the debug-hook library: compile with -DSWS_BUILD_DEBUG_HOOKS"
#endif
#include <math.h>
#include <stdio.h>

#include <vector>

#include "sws_debug.h"
#include "sws_farfield.cuh"
#include "sws_internal.cuh"

namespace sws {
cudaError_t launch_fp64_probe(int blocks, int iters, double* sink, unsigned long long* clk, cudaStream_t st);
cudaError_t launch_fp64_mix(int kind, int blocks, int iters, double* sink, unsigned long long* clk, cudaStream_t st);

// --- unit-test hook of the far-field expansion ---------------------------------------------
// out_em[i] = s2_column_em(c[i], g[i]); out_direct[i] = the plain trapezoid sum it stands for
__global__ void k_debug_s2col(EmGeom e, int M, const double* c, const double* g, int n, double* out_direct,
                              double* out_em) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  out_em[i] = s2_column_em(e, c[i], g[i]);
  double acc = 0.0;
  for (int j = 0; j < M; ++j) {
    const double yj = e.y1 + j * sqrt(e.h2);
    const double sm = yj - c[i], sp = yj + c[i];
    const double v = rsqrt_fp64(fma(sm, sm, g[i])) + rsqrt_fp64(fma(sp, sp, g[i]));
    acc += (j == 0 || j == M - 1) ? 0.5 * v : v;
  }
  out_direct[i] = acc;
}

// the three sums of the analytic Jacobian action: out[3 i + {0, 1, 2}] = {f0, f3, f3s}
__global__ void k_debug_s2col3(EmGeom e, int M, const double* c, const double* g, int n, double* out_direct,
                               double* out_em) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const Em3 r = s2_column_em3(e, c[i], g[i]);
  out_em[3 * i] = r.f0; out_em[3 * i + 1] = r.f3; out_em[3 * i + 2] = r.f3s;
  double a0 = 0.0, a3 = 0.0, a3s = 0.0;
  for (int j = 0; j < M; ++j) {
    const double yj = e.y1 + j * sqrt(e.h2);
    const double sm = yj - c[i], sp = yj + c[i];
    const double um = rsqrt_fp64(fma(sm, sm, g[i])), up = rsqrt_fp64(fma(sp, sp, g[i]));
    const double um3 = um * um * um, up3 = up * up * up;
    const double w = (j == 0 || j == M - 1) ? 0.5 : 1.0;
    a0 += w * (um + up);
    a3 += w * (um3 + up3);
    a3s += w * (sm * um3 - sp * up3);
  }
  out_direct[3 * i] = a0; out_direct[3 * i + 1] = a3; out_direct[3 * i + 2] = a3s;
}

cudaError_t launch_debug_s2col3(double y1, double dy, int M, const double* c, const double* g, int n,
                                double* out_direct, double* out_em, cudaStream_t st) {
  EmGeom e;
  e.y1 = y1; e.yM = y1 + (M - 1) * dy; e.h2 = dy * dy; e.inv_h = 1.0 / dy; e.gmin = 0.0; e.sym = (y1 == 0.0);
  k_debug_s2col3<<<(n + 127) / 128, 128, 0, st>>>(e, M, c, g, n, out_direct, out_em);
  return cudaGetLastError();
}

cudaError_t launch_debug_s2col(double y1, double dy, int M, const double* c, const double* g, int n,
                               double* out_direct, double* out_em, cudaStream_t st) {
  EmGeom e;
  e.y1 = y1; e.yM = y1 + (M - 1) * dy; e.h2 = dy * dy; e.inv_h = 1.0 / dy; e.gmin = 0.0; e.sym = (y1 == 0.0);
  k_debug_s2col<<<(n + 127) / 128, 128, 0, st>>>(e, M, c, g, n, out_direct, out_em);
  return cudaGetLastError();
}

// --- unit-test hook for the reciprocal square root --------------------------------------
__global__ void k_debug_rsqrt(const double* x, double* y, int n) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) y[i] = rsqrt_fp64(x[i]);
}

cudaError_t launch_debug_rsqrt(const double* x, double* y, int n, cudaStream_t st) {
  k_debug_rsqrt<<<(n + 255) / 256, 256, 0, st>>>(x, y, n);
  return cudaGetLastError();
}

// the variant whose seed takes its low word from the caller (rsqrt_fp64_lo, sws_farfield.cuh)
__global__ void k_debug_rsqrt_lo(const double* x, const int* lo, double* y, int n) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) y[i] = rsqrt_fp64_lo(x[i], lo[i]);
}

cudaError_t launch_debug_rsqrt_lo(const double* x, const int* lo, double* y, int n, cudaStream_t st) {
  k_debug_rsqrt_lo<<<(n + 255) / 256, 256, 0, st>>>(x, lo, y, n);
  return cudaGetLastError();
}

}  // namespace sws

static thread_local char g_dbg_err[256] = "";
static int dbg_fail(cudaError_t e, const char* where) {
  snprintf(g_dbg_err, sizeof g_dbg_err, "%s: %s", where, cudaGetErrorString(e));
  return SWS_ECUDA;
}
#define CK(call)                                        \
  do {                                                  \
    cudaError_t e_ = (call);                            \
    if (e_ != cudaSuccess) return dbg_fail(e_, #call);  \
  } while (0)
#define ON_DEVICE(dev) CK(cudaSetDevice(dev))

extern "C" {

const char* sws_debug_last_cuda_error(void) { return g_dbg_err; }

int sws_probe_fp64_peak(int32_t device, double* tflops, int32_t* sm_count, double* sm_mhz) {
  if (!tflops) return SWS_EINVAL;
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (device < 0 || device >= ndev) return SWS_EINVAL;
  ON_DEVICE(device);
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, device));
  const int sms = prop.multiProcessorCount;
  const int blocks = sms * 8, threads = 256, iters = 1 << 15;
  double* sink = nullptr;
  unsigned long long* clk = nullptr;
  CK(cudaMalloc((void**)&sink, (size_t)blocks * threads * sizeof(double)));
  CK(cudaMalloc((void**)&clk, 4 * sizeof(unsigned long long)));
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0));
  CK(cudaEventCreate(&e1));
  CK(sws::launch_fp64_probe(blocks, iters / 8, sink, clk, 0));  // warm-up
  double best = 0.0, mhz = 0.0;
  for (int rep = 0; rep < 3; ++rep) {
    CK(cudaEventRecord(e0, 0));
    CK(sws::launch_fp64_probe(blocks, iters, sink, clk, 0));
    CK(cudaEventRecord(e1, 0));
    CK(cudaEventSynchronize(e1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    unsigned long long h[4];
    CK(cudaMemcpy(h, clk, sizeof h, cudaMemcpyDeviceToHost));
    // 16 DFMA per iteration per thread, 2 flops each
    const double fl = (double)blocks * threads * (double)iters * 16.0 * 2.0;
    const double tf = fl / (ms * 1e-3) / 1e12;
    if (tf > best) {
      best = tf;
      mhz = (h[3] > h[2]) ? (double)(h[1] - h[0]) / (double)(h[3] - h[2]) * 1e3 : 0.0;
    }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  cudaFree(clk);
  *tflops = best;
  if (sm_count) *sm_count = sms;
  if (sm_mhz) *sm_mhz = mhz;
  return SWS_OK;
}

int sws_probe_fp64_mix(int32_t device, int32_t kind, int32_t warps_per_sm, double* fp64_instr_per_sm_clk,
                       double* sm_mhz) {
  if (!fp64_instr_per_sm_clk || kind < 0 || kind > 10) return SWS_EINVAL;
  if (warps_per_sm < 8 || warps_per_sm > 64 || warps_per_sm % 8) return SWS_EINVAL;
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (device < 0 || device >= ndev) return SWS_EINVAL;
  ON_DEVICE(device);
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, device));
  const int sms = prop.multiProcessorCount;
  const int blocks = sms * (warps_per_sm / 8), threads = 256, iters = kind >= 6 ? 1 << 13 : 1 << 15;
  static const int fp64_per_iter[11] = {12, 12, 12, 12, 13, 11, 48, 48, 48, 48, 48};
  double* sink = nullptr;
  unsigned long long* clk = nullptr;
  CK(cudaMalloc((void**)&sink, (size_t)blocks * threads * sizeof(double)));
  CK(cudaMalloc((void**)&clk, 4 * sizeof(unsigned long long)));
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaError_t e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  if (e == cudaSuccess) e = sws::launch_fp64_mix(kind, blocks, iters / 8, sink, clk, 0);  // warm-up
  double best = 0.0, mhz = 0.0;
  for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
    e = cudaEventRecord(e0, 0);
    if (e == cudaSuccess) e = sws::launch_fp64_mix(kind, blocks, iters, sink, clk, 0);
    if (e == cudaSuccess) e = cudaEventRecord(e1, 0);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    unsigned long long h[4] = {0, 0, 0, 0};
    if (e == cudaSuccess) e = cudaMemcpy(h, clk, sizeof h, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess || h[1] <= h[0] || h[3] <= h[2] || ms <= 0.f) break;
    // whole-launch time by CUDA events; SM clock during the loop from block 0's clock64 / globaltimer
    const double clk_mhz = (double)(h[1] - h[0]) / (double)(h[3] - h[2]) * 1e3;
    const double total = (double)fp64_per_iter[kind] * iters * threads * blocks;
    const double rate = total / (ms * 1e-3 * clk_mhz * 1e6) / sms;
    if (rate > best) { best = rate; mhz = clk_mhz; }
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(sink);
  cudaFree(clk);
  CK(e);
  *fp64_instr_per_sm_clk = best;
  if (sm_mhz) *sm_mhz = mhz;
  return SWS_OK;
}

int sws_debug_rsqrt_host(int32_t device, const double* x_host, double* y_host, int32_t n) {
  if (!x_host || !y_host || n < 1) return SWS_EINVAL;
  ON_DEVICE(device);
  double *x = nullptr, *y = nullptr;
  CK(cudaMalloc((void**)&x, (size_t)n * 8));
  CK(cudaMalloc((void**)&y, (size_t)n * 8));
  CK(cudaMemcpy(x, x_host, (size_t)n * 8, cudaMemcpyHostToDevice));
  CK(sws::launch_debug_rsqrt(x, y, n, 0));
  CK(cudaMemcpy(y_host, y, (size_t)n * 8, cudaMemcpyDeviceToHost));
  cudaFree(x);
  cudaFree(y);
  return SWS_OK;
}

int sws_debug_rsqrt_lo_host(int32_t device, const double* x_host, const int32_t* lo_host, double* y_host, int32_t n) {
  if (!x_host || !lo_host || !y_host || n < 1) return SWS_EINVAL;
  ON_DEVICE(device);
  double *x = nullptr, *y = nullptr;
  int* lo = nullptr;
  CK(cudaMalloc((void**)&x, (size_t)n * 8));
  CK(cudaMalloc((void**)&y, (size_t)n * 8));
  CK(cudaMalloc((void**)&lo, (size_t)n * 4));
  CK(cudaMemcpy(x, x_host, (size_t)n * 8, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(lo, lo_host, (size_t)n * 4, cudaMemcpyHostToDevice));
  CK(sws::launch_debug_rsqrt_lo(x, lo, y, n, 0));
  CK(cudaMemcpy(y_host, y, (size_t)n * 8, cudaMemcpyDeviceToHost));
  cudaFree(x);
  cudaFree(y);
  cudaFree(lo);
  return SWS_OK;
}

int sws_debug_s2col_host(int32_t device, double y1, double dy, int32_t M, const double* c_host,
                         const double* g_host, int32_t n, int32_t nsums, double* direct_host, double* em_host) {
  if (!c_host || !g_host || !direct_host || !em_host || n < 1 || M < 2 || !(dy > 0.0)) return SWS_EINVAL;
  if (nsums != 1 && nsums != 3) return SWS_EINVAL;
  ON_DEVICE(device);
  double* d = nullptr;
  const size_t nb = (size_t)n * 8, no = nb * nsums;
  CK(cudaMalloc((void**)&d, 2 * nb + 2 * no));
  CK(cudaMemcpy(d, c_host, nb, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(d + n, g_host, nb, cudaMemcpyHostToDevice));
  double* od = d + 2 * (size_t)n;
  double* oe = od + (size_t)n * nsums;
  cudaError_t e = nsums == 1 ? sws::launch_debug_s2col(y1, dy, M, d, d + n, n, od, oe, 0)
                             : sws::launch_debug_s2col3(y1, dy, M, d, d + n, n, od, oe, 0);
  if (e == cudaSuccess) e = cudaMemcpy(direct_host, od, no, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(em_host, oe, no, cudaMemcpyDeviceToHost);
  cudaFree(d);
  CK(e);
  return SWS_OK;
}

}  // extern "C"
