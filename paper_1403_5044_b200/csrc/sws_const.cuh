// Declarations of the uniform-operand ("constant-bank") all-pairs path: sws_allpairs_const.cuh (the kernel, once per
// bank) and its host side in sws_allpairs.cu.
#pragma once
#include "sws_farfield.cuh"
#include "sws_internal.cuh"

namespace sws {

constexpr int kConstBanks = 2;         // copies of the kernel, each in a module with a __constant__ bank of its own
                                       // (three and four banks were measured: no faster than two)
constexpr int kConstDoubles = 8160;    // 65,280 B of a module's 64 KB bank: y_j of the mesh + one slab of records
constexpr int kConstThreads = 64;      // threads per CTA
#ifndef SWS_CONST_NT
#define SWS_CONST_NT 1                 // targets per thread: 1, or 2 = the midpoints (k, l) and (k + 1, l) of one y-line
#endif
constexpr int kConstNT = SWS_CONST_NT;
constexpr int kConstMaxCols = 16;      // columns of a slab = CTA rows of a launch (capacity of the scratch rows)
constexpr int kConstMinCols = 4;       // the path is used only when a slab holds at least this many columns
#ifndef SWS_CONST_MIN_TARGETS
#define SWS_CONST_MIN_TARGETS 16000    // ... and the mesh has at least this many targets (226x76: 3 %, 271x91: 7 % faster
                                       // than the staged kernel, 181x61: equal)
#endif
constexpr int kConstMinTargets = SWS_CONST_MIN_TARGETS;

struct ConstArgs {
  const double* x;     // [N]
  const TgtRec* tgt;   // [T] of this state
  double* part;        // [ncols][T] scratch rows of this bank
  double* acc;         // [T] accumulated quadrature of this (bank, state)
  unsigned int* cnt;   // [tiles] arrival counters of this bank, zero between launches
  int N, M, T;
  int col0, ncols;     // the slab: columns col0 .. col0 + ncols - 1
  int cpc;             // columns per CTA: grid.y = ceil(ncols / cpc)
  int ypad;            // offset (in doubles) of the slab's records in the bank; y_j sits at [0, M)
  int first;           // first slab of this (bank, state): acc is written, not added to
  double dxdy;
  EmGeom em;
};

cudaError_t const_bank_launch_0(const ConstArgs& a, const SrcRec* slab, const double* y, int tiles, cudaStream_t st);
cudaError_t const_bank_launch_1(const ConstArgs& a, const SrcRec* slab, const double* y, int tiles, cudaStream_t st);
// resolves the bank's device address on the CURRENT device (cudaGetSymbolAddress; once per device, kept)
cudaError_t const_bank_prepare_0();
cudaError_t const_bank_prepare_1();

// target tiles (CTAs per group of columns) of a launch: 64 threads x kConstNT targets each; with two targets per thread
// the slots are (pair of x columns, y-line) and an odd last column is half empty
inline int const_tiles(int N, int M) {
  const long slots = (long)((N - 1 + kConstNT - 1) / kConstNT) * M;
  return (int)((slots + kConstThreads - 1) / kConstThreads);
}

// host side (sws_allpairs.cu)
int const_slab_cols(int M);                 // columns per slab for this M (0: a column does not fit)
int const_cols_per_cta(const sws_ctx* c);   // 4, 2 or 1: as many as leave two waves of CTAs per launch
bool const_path_active(const sws_ctx* c);   // the FP64 residual / batch of this context runs on this path
// a4 (+ a5, a6, a9 when F0 != NULL) for `states` states on the constant-bank path; asynchronous on `st`
cudaError_t launch_allpairs_const(sws_ctx* c, int states, cudaStream_t st, double* F0, double* Fpert, int* launches);
// the per-device streams / events of the path and the banks' addresses; called by sws_setup with `device` current
cudaError_t const_path_prepare(int device);

}  // namespace sws
