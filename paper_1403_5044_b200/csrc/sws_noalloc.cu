// sws_fd_shifts_noalloc (include/sws.h): the finite-difference shifts of eq. (25),
//     sigma_b = 1e-7 (1 + ||u||_2) / ||v_b||_2        (BASELINE.json; the paper says "a suitably-chosen shift", L221)
// for callers that are not allowed to allocate device memory.
//
// Who that is.  Every other entry point of this library needs an sws_ctx, and sws_setup cudaMalloc's the context's
// workspace.  Some programs cannot do that at the point where they need the shifts:
//   - a solver that lives inside a host application which has given ALL device memory to its own pool at start-up
//     (a simulation framework's arena, a PyTorch process running with a memory fraction): cudaMalloc then fails, or
//     takes memory the host application believes it owns;
//   - a continuation / time-stepping loop with a latency budget: cudaMalloc and cudaFree take the driver's allocation
//     lock and synchronise the device, which stalls every stream of the process in the middle of the loop;
//   - a Krylov driver that only wants the shifts (it forms u + sigma v and the quotient itself, or feeds them to
//     sws_jv_batch as sigma_host later) and has no reason to pay for a context of hundreds of MB.
// For them the reduction's scratch memory - the per-block partial sums of the two-stage 2-norm, which the context path
// keeps in its cudaMalloc'ed `norm_part` - lives in a fixed array in the library's device image instead.  The price:
// every GPU that loads libsws.so carries kNoallocScratchBytes (33,280 B) until the process exits, used or not, and the
// batch size is capped at SWS_NOALLOC_MAX_B directions per call.
//
// This file adds a code path; it changes none.  The kernels are copies of k_sumsq / k_sigma (sws_fields.cu) with the
// same block count, block size and summation order, so the shifts are bitwise those sws_jv_batch(sigma_host = NULL)
// computes and sws_last_sigma reports (tests/test_zz_no_alloc.py).
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "sws.h"

namespace {

constexpr int kBlocks = 64;    // partial sums per row (= kNormBlocks of the context path: same rounding)
constexpr int kThreads = 256;
constexpr int kMaxDevices = 64;
constexpr size_t kNoallocScratchBytes = (size_t)(SWS_NOALLOC_MAX_B + 1) * kBlocks * sizeof(double);

// The scratch: row 0 holds the block sums of u, row r >= 1 those of v_{r-1}.  ONE array per device for the whole
// process: all calls share it and it keeps whatever the last call left.  Nothing in it has to start at zero - stage 2
// reads only the (b + 1) * kBlocks slots stage 1 of the SAME call has just written (every block writes its slot, also
// when its share of the vector is empty) - so no clearing pass is needed; rows beyond b + 1 hold stale sums of earlier
// calls and are never read.
//
// In HOST code `g_scratch` is only a handle the runtime knows the symbol by: its host-side address is not a device
// address and must never be handed to a kernel.  Host code asks the runtime for the real address, once per device
// (scratch_of_device below); device code may name the array directly.
static __device__ __align__(256) double g_scratch[(SWS_NOALLOC_MAX_B + 1) * kBlocks];
static_assert(sizeof(g_scratch) == kNoallocScratchBytes && kNoallocScratchBytes == 33280, "size stated in sws.h");

std::mutex g_mu;
double* g_scratch_dev[kMaxDevices];  // device address of g_scratch on each device, resolved on first use; guarded by g_mu

thread_local char g_err[256] = "";

int fail(int code, const char* fmt, long long a = 0, long long b = 0) {
  snprintf(g_err, sizeof g_err, fmt, a, b);
  return code;
}

// Device address of this device's copy of g_scratch.  `device` must be the current device: the runtime resolves a
// symbol in the current device's copy of the module.
cudaError_t scratch_of_device(int device, double** out) {
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_scratch_dev[device]) {
    double* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_scratch);
    if (e != cudaSuccess) return e;
    g_scratch_dev[device] = p;
  }
  *out = g_scratch_dev[device];
  return cudaSuccess;
}

// Stage 1 (copy of k_sumsq): block (x, row) sums the squares of its grid-stride share of u (row 0) or v_{row-1}.
__global__ void __launch_bounds__(kThreads) k_sumsq_noalloc(const double* __restrict__ u, const double* __restrict__ V,
                                                            size_t n, double* __restrict__ part) {
  const int row = blockIdx.y;
  const double* a = row == 0 ? u : V + (size_t)(row - 1) * n;
  double s = 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    s = fma(a[i], a[i], s);
  __shared__ double sh[kThreads];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int w = kThreads / 2; w > 0; w >>= 1) {
    if (threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) part[(size_t)row * gridDim.x + blockIdx.x] = sh[0];
}

// Stage 2 (copy of k_sigma): thread r adds the block sums in index order and forms sigma_r; a zero direction gets 0.
__global__ void k_sigma_noalloc(const double* __restrict__ part, int nblk, int b, double* __restrict__ sigma) {
  const int r = threadIdx.x;
  if (r >= b) return;
  double su = 0.0, sv = 0.0;
  for (int i = 0; i < nblk; ++i) su += part[i];
  for (int i = 0; i < nblk; ++i) sv += part[(size_t)(r + 1) * nblk + i];
  sigma[r] = sv > 0.0 ? 1e-7 * (1.0 + sqrt(su)) / sqrt(sv) : 0.0;
}

}  // namespace

extern "C" {

const char* sws_noalloc_last_error(void) { return g_err; }

int sws_fd_shifts_noalloc(const double* u_dev, const double* V_dev, int64_t n, int32_t b, double* sigma_dev,
                          int32_t device, void* cuda_stream) {
  g_err[0] = 0;
  if (!u_dev || !V_dev || !sigma_dev) return fail(SWS_EINVAL, "sws_fd_shifts_noalloc: NULL pointer");
  if (n < 1 || n > (int64_t)INT32_MAX)
    return fail(SWS_EINVAL, "sws_fd_shifts_noalloc: n = %lld outside 1 .. %lld", (long long)n, (long long)INT32_MAX);
  if (b < 1 || b > SWS_NOALLOC_MAX_B)
    return fail(SWS_EBATCH,
                "sws_fd_shifts_noalloc: b = %lld directions, the built-in scratch array holds at most %lld per call "
                "(split the batch, or use sws_jv_batch with a context)",
                (long long)b, (long long)SWS_NOALLOC_MAX_B);
  if (device < 0 || device >= kMaxDevices)
    return fail(SWS_EINVAL, "sws_fd_shifts_noalloc: device %lld outside 0 .. %lld", (long long)device,
                (long long)kMaxDevices - 1);

  // run on `device`, put the caller's current device back on return (as every other entry point does)
  int prev = -1;
  cudaError_t e = cudaGetDevice(&prev);
  if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
  else prev = -1;
  double* scratch = nullptr;
  if (e == cudaSuccess) e = scratch_of_device(device, &scratch);  // first call on this device: resolves the address
  if (e == cudaSuccess) {
    cudaStream_t st = (cudaStream_t)cuda_stream;
    k_sumsq_noalloc<<<dim3(kBlocks, b + 1), kThreads, 0, st>>>(u_dev, V_dev, (size_t)n, scratch);
    e = cudaGetLastError();
    if (e == cudaSuccess) {
      k_sigma_noalloc<<<1, ((b + 31) / 32) * 32, 0, st>>>(scratch, kBlocks, b, sigma_dev);
      e = cudaGetLastError();
    }
  }
  if (prev >= 0) cudaSetDevice(prev);
  if (e != cudaSuccess) {
    snprintf(g_err, sizeof g_err, "sws_fd_shifts_noalloc: %s", cudaGetErrorString(e));
    return SWS_ECUDA;
  }
  return SWS_OK;
}

}  // extern "C"
