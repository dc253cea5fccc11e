// Measurement helper (no part of the path): a register-only DFMA loop on every SM, the
// denominator of the "alu" roofline bench.py reports.  16 independent FMA chains per
// thread so that the FP64 pipe's latency is covered many times over.
#include "sws_internal.cuh"

namespace sws {

__global__ void __launch_bounds__(256) k_fp64_probe(int iters, double* sink, unsigned long long* clk) {
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-12 * (blockIdx.x + 1);
  double r0 = 0.1, r1 = 0.2, r2 = 0.3, r3 = 0.4, r4 = 0.5, r5 = 0.6, r6 = 0.7, r7 = 0.8;
  double q0 = 1.1, q1 = 1.2, q2 = 1.3, q3 = 1.4, q4 = 1.5, q5 = 1.6, q6 = 1.7, q7 = 1.8;
  unsigned long long c0 = 0, g0 = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    c0 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
  }
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
    r0 = fma(r0, a, b); r1 = fma(r1, a, b); r2 = fma(r2, a, b); r3 = fma(r3, a, b);
    r4 = fma(r4, a, b); r5 = fma(r5, a, b); r6 = fma(r6, a, b); r7 = fma(r7, a, b);
    q0 = fma(q0, a, b); q1 = fma(q1, a, b); q2 = fma(q2, a, b); q3 = fma(q3, a, b);
    q4 = fma(q4, a, b); q5 = fma(q5, a, b); q6 = fma(q6, a, b); q7 = fma(q7, a, b);
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    unsigned long long c1 = clock64(), g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    clk[0] = c0; clk[1] = c1; clk[2] = g0; clk[3] = g1;
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] =
      ((r0 + r1) + (r2 + r3)) + ((r4 + r5) + (r6 + r7)) + ((q0 + q1) + (q2 + q3)) + ((q4 + q5) + (q6 + q7));
}

cudaError_t launch_fp64_probe(int blocks, int iters, double* sink, unsigned long long* clk,
                              cudaStream_t st) {
  k_fp64_probe<<<blocks, 256, 0, st>>>(iters, sink, clk);
  return cudaGetLastError();
}

}  // namespace sws
