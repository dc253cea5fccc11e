// Internal declarations of libsws (CUDA path, sm_100a).  Shares nothing with oracle/.
// Citations "L<n>" are lines of /root/reference/PAPER.md; "Qn" are DESIGN.md readings.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "sws.h"

namespace sws {

// One source node (x_i, y_j) of one state as the all-pairs kernel consumes it: 32 B.
// Stored TRANSPOSED, [i][j] with j fastest, so that one x-column is one contiguous
// M * 32 B run that a single bulk async copy (TMA, UBLKCP) moves into shared memory.
//   z = zeta_ij, psi = phi_ij - x_i, zx = (zeta_x)_ij, zy = (zeta_y)_ij
struct __align__(32) SrcRec {
  double z, psi, zx, zy;
};

// The same node for the FP32 pair-arithmetic variant (sws_allpairs_f32.cu), 32 B, same
// transposed layout.  zeta is a two-float number (z_hi + z_lo); fields the packed f32x2
// instructions consume as (v, v) pairs are stored twice, zeta_y negated.
struct __align__(16) SrcRecF {
  float z_hi, z_lo, psi, psi_dup;
  float zx, zx_dup, nzy, nzy_dup;
};

// One target midpoint (x_{k+1/2}, y_l) of one state (starred values, L162 / L177): 64 B.
struct __align__(32) TgtRec {
  double xs, ys;    // x*, y*
  double zs, psis;  // zeta*, phi* - x*
  double zxs;       // zeta_x*
  double A, B, C;   // 1 + zeta_x*^2, 2 zeta_x* zeta_y*, 1 + zeta_y*^2   (L177)
};

// Directional derivatives of one target's starred values for one direction (analytic Jacobian
// action, sws_jv_exact.cu): 48 B.
struct DTgtRec {
  double dzs, dpsis, dzxs;  // d zeta*, d phi*, d zeta_x*
  double dA, dB, dC;
};

struct Mesh {
  int N, M;     // nodes
  int T, S, n;  // (N-1)M targets, NM sources, 2(N+1)M unknowns
  double x1, y1, dx, dy;
  double froude, eps, n_rad;
  int dy_scheme;  // 0 spline, 1 FD
  int sym_first;  // y1 == 0: even extension across the centre line (Q3)
};

// All-pairs launch geometry (host-computed, see make_plan()).
struct PairPlan {
  int tiles;      // ceil(T / kPairThreads) target tiles
  int chunks;     // groups of source columns; one CTA = (tile, chunk, state)
  int seg_len;    // nodes of one column staged per bulk copy (<= kSegMax)
  int nseg;       // segments per column = ceil(M / seg_len)
  int cols_per_chunk;  // ceil(N / chunks)
};

constexpr int kPairThreads = 128;  // threads (= targets) per CTA of the FP32 and the linearised all-pairs kernels
constexpr int kSegMax = 256;       // max nodes staged per bulk copy (10 KB per stage)
constexpr int kStages = 2;         // staging ring depth
constexpr double kEmRadius = 8.0;  // default far-field radius of the S2 column sums, in units of dy
constexpr int kNormBlocks = 64;    // partial blocks of the 2-norm reductions

}  // namespace sws

struct sws_ctx {
  sws::Mesh mesh;
  sws_params params;
  int device;
  int sm_count;
  int max_states;       // max_batch + 1
  int chunks_user;      // 0 = auto
  int ns_user;          // states per CTA of batched all-pairs launches: 0 = library default, 1, 2
  double em_radius;     // far-field radius r of the S2 column sums in units of dy (<= 0: all direct)
  size_t ws_bytes;
  int last_launches;
  int last_states;      // states the workspace fields currently describe
  int last_lin_b;       // directions the derivative fields describe (0: none)

  // geometry (device)
  double* x;  // [N]
  double* y;  // [M]
  // spline tables (device): Thomas forward-elimination factors, data independent
  double* sp_cp;   // [M] c'_l
  double* sp_inv;  // [M] 1 / (b_l - a_l c'_{l-1})

  // per-state node planes, [state][l][k] (k fastest)
  double* zeta;
  double* phi;
  double* zx;
  double* px;
  double* zy;
  double* py;
  sws::SrcRec* src;  // [state][i][j]  (transposed)
  sws::SrcRecF* srcf;  // the same in FP32 (precision = 1 only, else NULL)
  int pair_occ;        // resident CTAs per SM of the all-pairs kernel in use
  int fused_grid;      // CTAs of the fused (cooperative) fields launch; 0: three separate launches
  unsigned int* tile_count;  // [max_states][tiles] arrival counters of the all-pairs CTAs of a target tile
  sws::TgtRec* tgt;  // [state][t], t = l (N-1) + k
  double* e2loc;     // [state][t]   2 pi (phi*-x*) + eps/rho* - zeta_x* I
  double* part;      // [state][chunk][t] partial all-pairs sums (already times dx dy)
  int part_chunks;   // chunk capacity of `part` per state
  size_t part_rows;  // capacity of `part` in rows of T doubles

  // uniform-operand (constant-bank) all-pairs path, sws_allpairs_const.cuh; NULL when a column does not fit a bank
  int const_mode;          // sws_set_const_path: -1 automatic (large meshes), 0 off, 1 on whenever a column fits
  double* acc_c;           // [bank][state][t] accumulated quadrature
  double* part_c;          // [bank][kConstMaxCols][t] column sums of the slab in flight
  unsigned int* cnt_c;     // [bank][tiles] arrival counters

  // analytic Jacobian action (max_batch > 0 only)
  double4* dsrc;          // [group][i][j][BT] {d zeta, d phi, d zeta_x, -d zeta_y}
  sws::DTgtRec* dtgt;     // [direction][t]
  double* e2lin;          // [direction][t] local part of the derivative of E2
  double4* tgtI;          // [t] {I, dI/dA, dI/dB, dI/dC} of the base state
  int lin_occ[4];         // resident CTAs per SM of k_allpairs_lin<1,4,8,16> (fused)
  int lin_occ2[4];        // the same for the directions-only kernels (sws_jv_apply)
  int lin_occ1;           // the base-sums kernel (sws_linearize)
  double* lin_sums;       // [6][t] direction-independent sums of the linearisation at lin_u
  int lin_valid;          // the base fields, tgtI and lin_sums describe the u of the last sws_linearize

  double* F0;         // [n] base residual of a batch when the caller passes no F0_dev
  double* Fpert;      // [max_batch][n] when the caller passes no Fpert_dev
  double* sigma;      // [max_batch] device
  double* norm_part;  // [max_batch + 1][kNormBlocks]
  // host-call staging (device)
  double* u_stage;    // [n]
  double* V_stage;    // [max_batch][n]
  double* out_stage;  // [2 max_batch + 1][n]
  cudaEvent_t ev0, ev1;
  int profiling;                       // sws_set_profiling
  std::vector<cudaEvent_t>* prof_events;  // pairs (before, after) of all-pairs launches
  size_t prof_used;                    // events in use (the vector only grows)
};

namespace sws {

// Launches (all asynchronous on `st`); each returns the cudaError_t of its launch.
// states = 1: base state only.  State s >= 1 is u + sigma[s-1] * V[s-1].
// lin != 0: states >= 1 are the directions v themselves (derivative fields, homogeneous rows)
// first: the first state processed (states first..states-1); sws_jv_apply skips the base state
cudaError_t launch_reconstruct(sws_ctx* c, const double* u, const double* V, int states, int lin,
                               double* F0, double* Fpert, cudaStream_t st, int first = 0);
cudaError_t launch_dy(sws_ctx* c, int states, cudaStream_t st, int first = 0);
// tgtI != NULL: base state of the analytic Jacobian action ({I, I_A, I_B, I_C} instead of e2loc)
cudaError_t launch_targets(sws_ctx* c, int states, double* F0, double* Fpert, double4* tgtI,
                           cudaStream_t st);
// dispatches on sws_params.precision (0: FP64 kernel, 1: FP32 pair arithmetic).  FP64 kernel with F0 != NULL:
// the kernel also assembles the rows E2 into F0 / Fpert (fused a6 + a9); otherwise launch_assemble follows.
cudaError_t launch_allpairs(sws_ctx* c, int states, const PairPlan& plan, cudaStream_t st, double* F0 = nullptr,
                            double* Fpert = nullptr);
cudaError_t launch_count_near(sws_ctx* c, int states, int* out, cudaStream_t st);
cudaError_t launch_allpairs_f32(sws_ctx* c, int states, const PairPlan& plan, cudaStream_t st);
cudaError_t launch_assemble(sws_ctx* c, int states, const PairPlan& plan, double* F0,
                            double* Fpert, cudaStream_t st);
cudaError_t launch_sigma(sws_ctx* c, const double* u, const double* V, int b, cudaStream_t st);
cudaError_t launch_jv_quotient(sws_ctx* c, const double* F0, const double* Fpert, int b,
                               double* JV, cudaStream_t st);

// analytic Jacobian action (sws_jv_exact.cu); BT = directions per tile (1, 4, 8 or 16)
int lin_tile(int b);
cudaError_t lin_configure(sws_ctx* c);
// mode 0: fused kernel (sws_jv_exact_batch); 1: direction-independent sums (sws_linearize);
// 2: direction sums only (sws_jv_apply)
PairPlan make_lin_plan(const sws_ctx* c, int BT, int groups, int mode);
cudaError_t launch_targets_lin(sws_ctx* c, int b, int BT, double* JV, cudaStream_t st);
cudaError_t launch_allpairs_lin(sws_ctx* c, int BT, int groups, int mode, const PairPlan& plan, cudaStream_t st);
cudaError_t launch_reduce_base(sws_ctx* c, const PairPlan& plan, cudaStream_t st);
cudaError_t launch_assemble_lin(sws_ctx* c, int b, int BT, int mode, const PairPlan& plan, double* JV,
                                cudaStream_t st);

PairPlan make_plan(const sws_ctx* c);
int max_chunks(const sws_ctx* c);
size_t allpairs_smem_bytes(const PairPlan& p, int ns);
int pair_ns(const sws_ctx* c, int states);
cudaError_t allpairs_configure(const sws_ctx* c, int* occ_out);
int pair_nt(const sws_ctx* c);
int count_near_warps(const sws_ctx* c);
cudaError_t allpairs_f32_configure(int* occ_out);
size_t allpairs_f32_smem_bytes(int seg_len);
cudaError_t fields_configure(const sws_ctx* c);
cudaError_t fused_configure(sws_ctx* c);
cudaError_t launch_fields_fused(sws_ctx* c, const double* u, const double* V, int states, double* F0, double* Fpert,
                                cudaStream_t st);
size_t reconstruct_smem_bytes(int N);

}  // namespace sws
