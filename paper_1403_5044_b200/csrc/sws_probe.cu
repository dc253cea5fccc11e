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

// ---------------------------------------------------------------------------------------
// Instruction-mix probes behind the cycle model of DESIGN.md section 6.  Each runs 12 independent
// chains per thread, `iters` times, register only.  KIND:
//   0  DFMA with two distinct register sources      r = fma(r, r, b)
//   1  DFMA with three distinct register sources    r_i = fma(r_i, q_i, s_i)   (no operand shared between
//      neighbouring instructions, so the operand-reuse cache cannot help)
//   2  DADD, two distinct registers                 r = r + b
//   3  DMUL, two distinct registers                 r = r * a
//   4  11 two-register DFMA + 1 MUFU.RSQ64H
//   5  11 two-register DFMA + 3 integer instructions
//   6  DFMA with two distinct vector registers and one UNIFORM-register operand taken from a constant bank
//      r_i = fma(r_i, c[it], s_i)   (LDCU.64 + DFMA R, R, UR, R: the operand form of the constant-bank all-pairs kernel)
//   7-10  12 two-register DFMA + 2 more instructions that do not go to the FP64 pipe (four such rounds per iteration): 2 MUFU.RSQ64H (7),
//      2 MUFU.RSQ (FP32) (8), 2 FFMA (9), 2 LOP3 (10) - each of them costs about one cycle of FP64 issue
__constant__ double c_probe[64];

template <int KIND>
__global__ void __launch_bounds__(256) k_fp64_mix(int iters, double* sink, unsigned long long* clk) {
  const double a = 1.0 - 1e-9 * (threadIdx.x + 1), b = 1e-3 + 1e-12 * (blockIdx.x + 1);
  double r[12], q[12], s[12];
#pragma unroll
  for (int i = 0; i < 12; ++i) {
    r[i] = 0.1 + 0.01 * i + 1e-6 * threadIdx.x;
    q[i] = 0.999 - 1e-4 * i - 1e-9 * threadIdx.x;
    s[i] = 1e-4 * (i + 1) + 1e-10 * threadIdx.x;
  }
  unsigned int n0 = threadIdx.x, n1 = blockIdx.x, n2 = 12345u;
  double m0 = 1.5 + 1e-3 * threadIdx.x, m1 = 2.5 + 1e-3 * threadIdx.x;
  float f0 = 1.5f + 1e-3f * threadIdx.x, f1 = 2.5f + 1e-3f * threadIdx.x;
  unsigned long long c0 = 0, g0 = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    c0 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
  }
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
    if (KIND == 0) {
#pragma unroll
      for (int i = 0; i < 12; ++i) r[i] = fma(r[i], r[i], b);
    } else if (KIND == 1) {
#pragma unroll
      for (int i = 0; i < 12; ++i) r[i] = fma(r[i], q[i], s[i]);
    } else if (KIND == 2) {
#pragma unroll
      for (int i = 0; i < 12; ++i) r[i] = r[i] + b;
    } else if (KIND == 3) {
#pragma unroll
      for (int i = 0; i < 12; ++i) r[i] = r[i] * a;
    } else if (KIND == 4) {
      double t;
      asm volatile("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(t) : "d"(r[0] + 1.0));
#pragma unroll
      for (int i = 0; i < 10; ++i) r[i] = fma(r[i], r[i], b);
      r[10] = fma(r[10], r[10], t * 1e-3);  // DMUL + DFMA: 12 FP64 instructions + 1 DADD above, see host
    } else if (KIND == 5) {
#pragma unroll
      for (int i = 0; i < 11; ++i) r[i] = fma(r[i], r[i], b);
      n0 = n0 * 3u + n1;
      n1 = n1 + n2;
      n2 = n2 ^ n0;
    } else if (KIND == 6) {  // 4 x 12 DFMA per iteration, each round with its own uniform operand
#pragma unroll
      for (int rd = 0; rd < 4; ++rd) {
        const double cu = c_probe[(it & 15) * 4 + rd];  // uniform address: LDCU.64 into a uniform register
#pragma unroll
        for (int i = 0; i < 12; ++i) r[i] = fma(r[i], cu, s[i]);
      }
    } else {  // 4 x (12 two-register DFMA + 2 instructions of another pipe) per iteration
#pragma unroll
      for (int rd = 0; rd < 4; ++rd) {
#pragma unroll
        for (int i = 0; i < 12; ++i) r[i] = fma(r[i], r[i], b);
        if (KIND == 7) {
          asm volatile("rsqrt.approx.ftz.f64 %0, %0;" : "+d"(m0));
          asm volatile("rsqrt.approx.ftz.f64 %0, %0;" : "+d"(m1));
        } else if (KIND == 8) {
          asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(f0));
          asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(f1));
        } else if (KIND == 9) {
          asm volatile("fma.rn.f32 %0, %0, 0f3F7FF000, 0f3A000000;" : "+f"(f0));
          asm volatile("fma.rn.f32 %0, %0, 0f3F7FF000, 0f3A000000;" : "+f"(f1));
        } else {
          asm volatile("lop3.b32 %0, %0, 0x5a5a5a5a, %1, 0x96;" : "+r"(n0) : "r"(n1));
          asm volatile("lop3.b32 %0, %0, 0x5a5a5a5a, %1, 0x96;" : "+r"(n1) : "r"(n0));
        }
      }
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    unsigned long long c1 = clock64(), g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    clk[0] = c0; clk[1] = c1; clk[2] = g0; clk[3] = g1;
  }
  double acc = (double)(n0 ^ n1 ^ n2) * 1e-300 + (m0 + m1 + (double)(f0 + f1)) * 1e-300;
#pragma unroll
  for (int i = 0; i < 12; ++i) acc += r[i] + q[i] * s[i];
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

cudaError_t launch_fp64_mix(int kind, int blocks, int iters, double* sink, unsigned long long* clk, cudaStream_t st) {
  switch (kind) {
    case 0: k_fp64_mix<0><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    case 1: k_fp64_mix<1><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    case 2: k_fp64_mix<2><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    case 3: k_fp64_mix<3><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    case 4: k_fp64_mix<4><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    case 5: k_fp64_mix<5><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    case 6: k_fp64_mix<6><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    case 7: k_fp64_mix<7><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    case 8: k_fp64_mix<8><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    case 9: k_fp64_mix<9><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
    default: k_fp64_mix<10><<<blocks, 256, 0, st>>>(iters, sink, clk); break;
  }
  return cudaGetLastError();
}

cudaError_t launch_fp64_probe(int blocks, int iters, double* sink, unsigned long long* clk,
                              cudaStream_t st) {
  k_fp64_probe<<<blocks, 256, 0, st>>>(iters, sink, clk);
  return cudaGetLastError();
}

}  // namespace sws
