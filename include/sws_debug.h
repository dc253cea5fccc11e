/*
 * sws_debug.h -- C-ABI of libsws_debug.so: unit-test hooks and measurement probes.  NOT part of the
 * product library libsws.so and not needed to use it.  Built from csrc/sws_debug.cu + csrc/sws_probe.cu
 * with -DSWS_BUILD_DEBUG_HOOKS (paper_1403_5044_b200/build.py does); loaded by tests/ (the reciprocal
 * square root and the far-field expansion against long double) and by bench.py (FP64 issue-rate probes:
 * the measured denominator of the "alu" roofline).  Error codes as in sws.h.
 */
#ifndef SWS_DEBUG_H_
#define SWS_DEBUG_H_

#include "sws.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measurement helpers (no part of the path).
 * sws_probe_fp64_peak: register-only DFMA loop on every SM; reports achieved FP64
 * TFLOP/s (2 flops per DFMA), the SM count and the SM clock (MHz) read back from the
 * device clock64/globaltimer ratio. */
int sws_probe_fp64_peak(int32_t device, double* tflops, int32_t* sm_count, double* sm_mhz);

/* Instruction-mix probes behind the cycle model of DESIGN.md section 6 (register-only loops, one wave
 * of 256-thread CTAs, warps_per_sm in {8, 16, ..., 64}).  kind: 0 DFMA with two distinct register
 * sources; 1 DFMA with three distinct register sources; 2 DADD; 3 DMUL; 4 eleven two-register DFMA +
 * DADD + DMUL + one MUFU.RSQ64H (+ the move that zeroes the seed's low word); 5 eleven two-register
 * DFMA + three integer instructions; 6 DFMA with two distinct vector registers and one uniform-register operand
 * loaded from a constant bank (the operand form of the constant-bank all-pairs kernel); 7-10 twelve two-register
 * DFMA + two MUFU.RSQ64H / two FP32 MUFU.RSQ / two FFMA / two LOP3.  Reports FP64 thread-instructions per SM per clock (64 = the
 * pipe's issue limit) and the SM clock during the loop. */
int sws_probe_fp64_mix(int32_t device, int32_t kind, int32_t warps_per_sm, double* fp64_instr_per_sm_clk,
                       double* sm_mhz);

/* y[i] = the library's device reciprocal square root of x[i] (host buffers), for the
 * unit test of that primitive. */
int sws_debug_rsqrt_host(int32_t device, const double* x_host, double* y_host, int32_t n);
/* The same for the form the pair term uses for 1/R-: the seed's low 32 bits are lo_host[i] instead of zero
 * (in the kernel: whatever the low word of a dead register pair holds, so that no move follows the MUFU.RSQ64H);
 * any value must give a result within 1 ulp. */
int sws_debug_rsqrt_lo_host(int32_t device, const double* x_host, const int32_t* lo_host, double* y_host, int32_t n);

/* Unit test of the far-field expansion: for n pairs (c, g) and the column y1, y1+dy, ..., M nodes,
 * with u-+ = ((y_j -+ c)^2 + g)^-1/2, s-+ = y_j -+ c and c_j = 1/2 at both ends,
 *   nsums = 1: em_host[i]        = the library's expansion of sum_j c_j (u- + u+)        (sws_residual)
 *   nsums = 3: em_host[3i + 0..2] = the same, sum_j c_j (u-^3 + u+^3) and sum_j c_j (s- u-^3 - s+ u+^3)
 *              (the sums of the analytic Jacobian action),
 * and direct_host[...] = the same sums term by term on the device. */
int sws_debug_s2col_host(int32_t device, double y1, double dy, int32_t M, const double* c_host,
                         const double* g_host, int32_t n, int32_t nsums, double* direct_host, double* em_host);

/* Text of the last CUDA error a call of this library hit on the calling thread. */
const char* sws_debug_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SWS_DEBUG_H_ */
