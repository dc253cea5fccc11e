// Step a4 with the source data in UNIFORM registers (the "constant-bank" all-pairs kernel).
//
// Why.  Every lane of a warp works on the same source node, so the node's record {zeta, phi - x, zeta_x, zeta_y}
// and y_j are warp-uniform.  The staged kernel (sws_allpairs.cu) broadcasts them from shared memory into VECTOR
// registers; the FP64 instructions that combine a per-source, a per-target and a per-pair value then read three
// distinct 64-bit vector registers, which the register file of a B200 sub-partition delivers in 3 cycles instead of
// the pipe's 2 (8 such DFMAs per pair).  An FP64 instruction can take one operand from a
// UNIFORM register instead (DFMA R, R, UR, R issues at full rate: measured 62.2 of 64 per SM per clock), and a
// uniform register is loaded from a constant bank (LDCU.64 UR, c[0x3][UR + imm]) without touching the vector
// register file or the shared-memory pipe.  With the node data in uniform registers only the two accumulating
// FMAs of a pair keep three vector sources.
//
// How.  A module's __constant__ bank holds 64 KB, i.e. one SLAB of source columns (8 columns at M = 241, 16 at
// M = 121) plus the y_j of the mesh.  The host (launch_allpairs_const, sws_allpairs.cu) walks the slabs of every
// state: device-to-device copy of the slab's records into the bank, then one launch of this kernel with
// grid = (target tiles, groups of cpc columns of the slab): one CTA = 64 targets x cpc source columns (cpc = 4, 2 or
// 1: as many as leave two waves of CTAs per launch).  There are two copies of
// this kernel in two modules (sws_allpairs_c0.cu / _c1.cu, each with its own bank) fed through two streams, so the
// copy and the tail of one slab overlap the other slab's kernel.  The CTA that completes a target tile (arrival
// counter, as in the staged kernel) adds the slab's group sums in the fixed order g = 0 .. G-1 and accumulates
// them into acc[bank][state][t]; k_finish_const (sws_allpairs.cu) forms E2 = e2_local - (acc[0] + acc[1]).
// Slab s of a state always goes to bank s mod 2, and the split into slabs depends on the mesh only: results are
// bitwise repeatable and slot b of a batch is bitwise the single evaluation of u_b.
//
// The arithmetic of a pair is pair_term() of sws_pair.cuh, the same code the staged kernel runs.
//
// This file is the body of ONE bank: it is included by sws_allpairs_c0.cu / sws_allpairs_c1.cu with
// SWS_CONST_BANK defined as 0 / 1.
#include "sws_const.cuh"
#include "sws_pair.cuh"

#ifndef SWS_CONST_BANK
#error "SWS_CONST_BANK must be 0 or 1"
#endif
#ifndef SWS_CONST_UNROLL
#define SWS_CONST_UNROLL 8  // nodes per inner-loop iteration (4 / 8 / 12: 50.9 / 49.4 / 49.8 ms per state at 721x241)
#endif
#ifndef SWS_CONST_ROTATE
#define SWS_CONST_ROTATE 1  // 0: plain unrolled loop
#endif
#ifndef SWS_CONST_MINB
#if SWS_CONST_NT == 2
#define SWS_CONST_MINB 6  // two targets per thread: 168 registers
#else
#define SWS_CONST_MINB 8  // resident CTAs per SM (caps the kernel at 128 registers)
#endif
#endif
#ifndef SWS_CONST_UNROLL2
#define SWS_CONST_UNROLL2 4  // nodes per inner-loop iteration of the two-target kernel
#endif

namespace sws {
namespace {

constexpr int kConstUnroll = SWS_CONST_UNROLL;
constexpr int kConstUnroll2 = SWS_CONST_UNROLL2;

// [0, ypad): y_j of the mesh;  [ypad, ypad + 4 M ncols): the slab's SrcRec, [column][j]
__constant__ double c_buf[kConstDoubles];

// One source column (records at c_buf[rbase + 4 j]) against one target: trapezoid half weights on the first and
// last node by peeling (Q4), in the order walk_segment() of the staged kernel takes them.
template <bool S2T>
__device__ __forceinline__ void walk_column_const(const int rbase, const int M, const TgtG& tg, const TgtS& ts,
                                                  const ColG& cg, const ColS& cs, double& col1, double& colS) {
  auto node = [&](const int j, double& o1, double& oS) {
    const double yj = c_buf[j];
    const double* r = c_buf + rbase + 4 * j;
    const double2 zp = make_double2(r[0], r[1]), sl = make_double2(r[2], r[3]);
    pair_term<S2T>(zp, sl, yj, yj - tg.ys, tg, ts, cg, cs, o1, oS);
  };
  double h1 = 0.0, hS = 0.0;
  node(0, h1, hS);
  col1 = 0.5 * h1;
  colS = 0.5 * hS;
#if SWS_CONST_ROTATE
  {
    // The first node of every unrolled group is loaded one group ahead: ptxas issues the LDCU.64 of a group at the
    // top of its body, so the group's first DADDs (y_j - y*, zeta_j - zeta*) would wait out the whole load latency
    // (short-scoreboard stalls, profiles/r2b_allpairs_const_ncu.md); with one node in flight across the back edge they
    // do not: 48.9 -> 48.6 ms per state at 721x241, 3.32 -> 3.28 ms at 361x121.  Same terms in the same order.
    struct NodeData { double yj; double2 zp, sl; };
    auto load = [&](const int j) {
      NodeData d;
      d.yj = c_buf[j];
      const double* r = c_buf + rbase + 4 * j;
      d.zp = make_double2(r[0], r[1]);
      d.sl = make_double2(r[2], r[3]);
      return d;
    };
    int j = 1;
    NodeData pre = load(j);
    for (; j + kConstUnroll <= M - 1; j += kConstUnroll) {
      const NodeData nxt = load(j + kConstUnroll < M ? j + kConstUnroll : M - 1);  // stays inside the column
      pair_term<S2T>(pre.zp, pre.sl, pre.yj, pre.yj - tg.ys, tg, ts, cg, cs, col1, colS);
#pragma unroll
      for (int u = 1; u < kConstUnroll; ++u) node(j + u, col1, colS);
      pre = nxt;
    }
    for (; j < M - 1; ++j) node(j, col1, colS);
  }
#else
#pragma unroll kConstUnroll
  for (int j = 1; j < M - 1; ++j) node(j, col1, colS);
#endif
  h1 = hS = 0.0;
  node(M - 1, h1, hS);
  col1 = fma(0.5, h1, col1);
  colS = fma(0.5, hS, colS);
}

#if SWS_CONST_NT == 2
// Two targets per thread: the midpoints (k, l) and (k + 1, l) of one y-line.  They share y*, so a node's five uniform
// loads, its y_j - y* and the loop control serve two pair terms; each target's terms and their order are those of the
// one-target kernel.
template <bool S2T>
__device__ __forceinline__ void walk_column_const2(const int rbase, const int M, const TgtG& tg, const TgtS& ts0,
                                                   const TgtS& ts1, const ColG& cg0, const ColG& cg1, const ColS& cs0,
                                                   const ColS& cs1, double& c1a, double& cSa, double& c1b, double& cSb) {
  auto node = [&](const int j, double& o1a, double& oSa, double& o1b, double& oSb) {
    const double yj = c_buf[j];
    const double* r = c_buf + rbase + 4 * j;
    const double2 zp = make_double2(r[0], r[1]), sl = make_double2(r[2], r[3]);
    const double dm = yj - tg.ys;
    pair_term<S2T>(zp, sl, yj, dm, tg, ts0, cg0, cs0, o1a, oSa);
    pair_term<S2T>(zp, sl, yj, dm, tg, ts1, cg1, cs1, o1b, oSb);
  };
  double h1a = 0.0, hSa = 0.0, h1b = 0.0, hSb = 0.0;
  node(0, h1a, hSa, h1b, hSb);
  c1a = 0.5 * h1a; cSa = 0.5 * hSa; c1b = 0.5 * h1b; cSb = 0.5 * hSb;
#pragma unroll kConstUnroll2
  for (int j = 1; j < M - 1; ++j) node(j, c1a, cSa, c1b, cSb);
  h1a = hSa = h1b = hSb = 0.0;
  node(M - 1, h1a, hSa, h1b, hSb);
  c1a = fma(0.5, h1a, c1a); cSa = fma(0.5, hSa, cSa);
  c1b = fma(0.5, h1b, c1b); cSb = fma(0.5, hSb, cSb);
}

__global__ void __launch_bounds__(kConstThreads, SWS_CONST_MINB) k_allpairs_const(const ConstArgs a) {
  const int tid = threadIdx.x, tile = blockIdx.x, g = blockIdx.y;
  // slots in TRANSPOSED order over PAIRS of x columns: slot = kk M + l, targets (2 kk, l) and (2 kk + 1, l)
  const int npc = (a.N - 1 + 1) / 2, nslots = npc * a.M;
  const int slot = tile * kConstThreads + tid;
  const int sc = slot < nslots ? slot : nslots - 1;  // ragged tail: recomputed, never stored
  const int kk = sc / a.M, l = sc - kk * a.M;
  const bool has1 = 2 * kk + 1 <= a.N - 2;           // odd N - 1: the last pair column holds one target
  const int tc0 = l * (a.N - 1) + 2 * kk, tc1 = has1 ? tc0 + 1 : tc0;
  const int t0 = slot < nslots ? tc0 : a.T, t1 = (slot < nslots && has1) ? tc1 : a.T;
  const TgtRec tr0 = a.tgt[tc0], tr1 = a.tgt[tc1];
  const TgtG tg = {tr0.ys, 2.0 * tr0.ys, 4.0 * tr0.ys};
  const TgtS ts0 = {tr0.zs, tr0.psis}, ts1 = {tr1.zs, tr1.psis};
  const double kb0 = tr0.B / (2.0 * tr0.C), kb1 = tr1.B / (2.0 * tr1.C);
  const double kg0 = tr0.A / tr0.C - kb0 * kb0, kg1 = tr1.A / tr1.C - kb1 * kb1;
  const double sfac0 = -tr0.zxs * rsqrt_fp64(tr0.C), sfac1 = -tr1.zxs * rsqrt_fp64(tr1.C);

  double tot1a = 0.0, totSa = 0.0, tot1b = 0.0, totSb = 0.0;
#pragma unroll 1
  for (int cc = 0; cc < a.cpc; ++cc) {
    const int gc = g * a.cpc + cc;
    if (gc >= a.ncols) break;
    const int i = a.col0 + gc;
    ColG cg0, cg1;
    ColS cs0, cs1;
    const double xi = __ldg(a.x + i);
    cg0.dx = xi - tr0.xs; cg0.dx2 = cg0.dx * cg0.dx;
    cg1.dx = xi - tr1.xs; cg1.dx2 = cg1.dx * cg1.dx;
    cs0.c = fma(-kb0, cg0.dx, tg.ys); cs0.g = kg0 * cg0.dx2;
    cs1.c = fma(-kb1, cg1.dx, tg.ys); cs1.g = kg1 * cg1.dx2;
    const bool far = column_is_far(fmin(cs0.g, cs1.g), a.em.gmin);  // warp-uniform: both targets of all 32 threads
    const int rbase = a.ypad + 4 * a.M * gc;
    double c1a, cSa, c1b, cSb;
    if (far) {
      walk_column_const2<false>(rbase, a.M, tg, ts0, ts1, cg0, cg1, cs0, cs1, c1a, cSa, c1b, cSb);
      cSa = s2_column_em(a.em, cs0.c, cs0.g);
      cSb = s2_column_em(a.em, cs1.c, cs1.g);
    } else {
      walk_column_const2<true>(rbase, a.M, tg, ts0, ts1, cg0, cg1, cs0, cs1, c1a, cSa, c1b, cSb);
    }
    const double ci = (i == 0 || i == a.N - 1) ? 0.5 : 1.0;  // trapezoid weight in x (Q4)
    tot1a = fma(ci, c1a, tot1a); totSa = fma(ci, cSa, totSa);
    tot1b = fma(ci, c1b, tot1b); totSb = fma(ci, cSb, totSb);
  }
  if (t0 < a.T) a.part[(size_t)g * a.T + t0] = a.dxdy * fma(sfac0, totSa, tot1a);
  if (t1 < a.T) a.part[(size_t)g * a.T + t1] = a.dxdy * fma(sfac1, totSb, tot1b);

  __shared__ int s_last;
  __threadfence();
  __syncthreads();
  if (tid == 0) {
    unsigned int* cnt = a.cnt + tile;
    const unsigned int seen = atomicAdd(cnt, 1u);
    s_last = (seen == gridDim.y - 1u);
    if (s_last) *cnt = 0u;  // ready for the next launch of this bank
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (t0 < a.T) {
    double sum = 0.0;
    for (int q = 0; q < (int)gridDim.y; ++q) sum += __ldcg(a.part + (size_t)q * a.T + t0);
    a.acc[t0] = a.first ? sum : a.acc[t0] + sum;
  }
  if (t1 < a.T) {
    double sum = 0.0;
    for (int q = 0; q < (int)gridDim.y; ++q) sum += __ldcg(a.part + (size_t)q * a.T + t1);
    a.acc[t1] = a.first ? sum : a.acc[t1] + sum;
  }
}
#else
__global__ void __launch_bounds__(kConstThreads, SWS_CONST_MINB) k_allpairs_const(const ConstArgs a) {
  const int tid = threadIdx.x, tile = blockIdx.x, g = blockIdx.y;
  // targets in TRANSPOSED order (sws_farfield.cuh): the 32 targets of a warp share one x*
  const int slot = tile * kConstThreads + tid;
  const int tc = target_of_slot(slot < a.T ? slot : a.T - 1, a.N, a.M);  // ragged tail: recomputed, never stored
  const int t = slot < a.T ? tc : a.T;
  const TgtRec tr = a.tgt[tc];
  const TgtG tg = {tr.ys, 2.0 * tr.ys, 4.0 * tr.ys};
  const TgtS ts = {tr.zs, tr.psis};
  const double kb = tr.B / (2.0 * tr.C);           // B / 2C
  const double kg = tr.A / tr.C - kb * kb;         // (4AC - B^2) / (4 C^2)
  const double sfac = -tr.zxs * rsqrt_fp64(tr.C);  // - zeta_x* / sqrt(C)

  // this CTA's columns of the slab: g cpc .. g cpc + cpc - 1
  double tot1 = 0.0, totS = 0.0;
#pragma unroll 1
  for (int cc = 0; cc < a.cpc; ++cc) {
    const int gc = g * a.cpc + cc;
    if (gc >= a.ncols) break;
    const int i = a.col0 + gc;
    ColG cg;
    ColS cs;
    cg.dx = __ldg(a.x + i) - tr.xs;
    cg.dx2 = cg.dx * cg.dx;
    cs.c = fma(-kb, cg.dx, tg.ys);
    cs.g = kg * cg.dx2;
    const bool far = column_is_far(cs.g, a.em.gmin);  // warp-uniform, as the staged kernel takes it
    const int rbase = a.ypad + 4 * a.M * gc;
    double col1, colS;
    if (far) {
      walk_column_const<false>(rbase, a.M, tg, ts, cg, cs, col1, colS);
      colS = s2_column_em(a.em, cs.c, cs.g);  // the column's S2 terms from their Euler-Maclaurin form
    } else {
      walk_column_const<true>(rbase, a.M, tg, ts, cg, cs, col1, colS);
    }
    const double ci = (i == 0 || i == a.N - 1) ? 0.5 : 1.0;  // trapezoid weight in x (Q4)
    tot1 = fma(ci, col1, tot1);
    totS = fma(ci, colS, totS);
  }
  if (t < a.T) a.part[(size_t)g * a.T + t] = a.dxdy * fma(sfac, totS, tot1);

  // the last CTA of this tile adds the slab's columns in fixed order and accumulates (no floating-point atomics)
  __shared__ int s_last;
  __threadfence();
  __syncthreads();
  if (tid == 0) {
    unsigned int* cnt = a.cnt + tile;
    const unsigned int seen = atomicAdd(cnt, 1u);
    s_last = (seen == gridDim.y - 1u);
    if (s_last) *cnt = 0u;  // ready for the next launch of this bank
  }
  __syncthreads();
  if (!s_last || t >= a.T) return;
  __threadfence();
  double sum = 0.0;
  for (int q = 0; q < (int)gridDim.y; ++q) sum += __ldcg(a.part + (size_t)q * a.T + t);
  a.acc[t] = a.first ? sum : a.acc[t] + sum;
}
#endif  // SWS_CONST_NT

}  // namespace

#define SWS_CAT2(a, b) a##b
#define SWS_CAT(a, b) SWS_CAT2(a, b)

namespace {
void* g_base_of_device[64] = {};  // the bank's device address, per device (callers hold the path's mutex)

cudaError_t bank_base(void** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  if (!g_base_of_device[dev]) {
    e = cudaGetSymbolAddress(&g_base_of_device[dev], c_buf);
    if (e != cudaSuccess) return e;
  }
  *out = g_base_of_device[dev];
  return cudaSuccess;
}
}  // namespace

cudaError_t SWS_CAT(const_bank_prepare_, SWS_CONST_BANK)() {
  void* base = nullptr;
  return bank_base(&base);
}

// Copies the slab (and, if y != NULL, the mesh's y_j) into this module's bank and launches the kernel on `st`.
cudaError_t SWS_CAT(const_bank_launch_, SWS_CONST_BANK)(const ConstArgs& a, const SrcRec* slab, const double* y,
                                                        int tiles, cudaStream_t st) {
  void* base = nullptr;
  cudaError_t e = bank_base(&base);
  if (e != cudaSuccess) return e;
  if (y) {
    e = cudaMemcpyAsync(base, y, (size_t)a.M * sizeof(double), cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return e;
  }
  e = cudaMemcpyAsync(static_cast<double*>(base) + a.ypad, slab, (size_t)a.ncols * a.M * sizeof(SrcRec),
                      cudaMemcpyDeviceToDevice, st);
  if (e != cudaSuccess) return e;
  k_allpairs_const<<<dim3(tiles, (a.ncols + a.cpc - 1) / a.cpc), kConstThreads, 0, st>>>(a);
  return cudaGetLastError();
}

}  // namespace sws
