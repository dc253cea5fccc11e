// Step a4: the all-pairs trapezoid quadrature of eq. (12) with the
// singularity subtraction of L181, for every half-mesh target and every state.
//
//   sum_{i,j} w(i,j) [ (phi_ij - phi* - x_i + x*) K1 + (zeta_x)_ij K2 - zeta_x* S2 ]
//   K1 (L107, reading Q1/Q2), K2 (L109), S2 = S2_direct + S2_image (eqs. (21),(22) L169-172),
//   w(i,j) = dx dy c_i c_j, c = 1/2 on the first/last index (L189, reading Q4).
//
// Mapping (B200): one thread = one target (two on large meshes, see kNT2MinTargets), 64 threads per CTA,
// 8 (6) CTAs per SM, targets handed out in transposed order (sws_farfield.cuh); a CTA walks a group
// of ~12 source COLUMNS (fixed x_i, all y_j).  Each column (M records of 32 B, contiguous in the
// transposed SrcRec layout) is brought into shared memory by ONE bulk async copy
// (cp.async.bulk -> UBLKCP, completion on an mbarrier), double buffered.  Every lane of a
// warp reads the same record (shared-memory broadcast), so the kernel is bound by the FP64
// pipe.  Columns at least 8 dy away from all 32 targets of a warp ("far", 97.8 % at 721x241)
// take their S2 terms - which do not depend on the source data - from the Euler-Maclaurin form of
// the column sum (sws_farfield.cuh): 28 FP64 instructions + 2 MUFU.RSQ64H per pair; the others
// sum S2 pair by pair: 44 + 4.  Everything that depends only on (target, column) - dx, dx^2 and
// the completed-square constants of S2 - is hoisted out of the j loop; the half weights are
// applied by peeling the first/last node and scaling edge columns, so the inner loop carries no
// weight multiply.  Partial sums per (state, chunk, target) are written to global memory and
// added in a fixed order by the assemble kernel: no atomics, bitwise repeatable.
#include "sws_farfield.cuh"
#include "sws_internal.cuh"
#include "sws_stage.cuh"

// build-time tuning of the all-pairs kernel (defaults measured on B200)
#ifndef SWS_PAIR_THREADS
#define SWS_PAIR_THREADS 64  // threads (= targets) per CTA of k_allpairs
#endif
#ifndef SWS_MINB
#define SWS_MINB 8  // resident CTAs per SM asked of __launch_bounds__ (caps registers at 128)
#endif
#ifndef SWS_UNROLL
#define SWS_UNROLL 8  // source nodes per inner-loop iteration
#endif

namespace sws {

constexpr int kUnroll = SWS_UNROLL;
// k_allpairs runs 64-thread CTAs, 8 per SM (16 warps per SM as with 128 x 4, but only two warps meet at
// the per-column barrier and CTAs turn over twice as often: 59.5 instead of 61.1 ms at cfg5)
constexpr int kThreads64 = SWS_PAIR_THREADS;
// Targets per thread of k_allpairs: 1, or 2 on meshes with at least kNT2MinTargets targets.  With two targets
// (kThreads64 slots apart, so usually the same x*) a thread loads every staged record once for both: 1.5
// instead of 3 shared-memory loads and half the loop overhead per pair, i.e. fewer of the non-FP64
// instructions that take issue time from the FP64 pipe: 55.4 instead of 56.8 ms at
// 721x241 with 6 CTAs of 148 registers per SM.  Small meshes keep one target per thread (more CTAs).
#ifndef SWS_NT2_MIN_TARGETS
#define SWS_NT2_MIN_TARGETS 40000
#endif
constexpr int kNT2MinTargets = SWS_NT2_MIN_TARGETS;
constexpr int kMinB2 = 6;  // resident CTAs per SM of the two-target kernel

// Per-thread constants of one target and of the current source column.
// The S2 quadratic forms are used with the square completed (C > 0):
//   A dx^2 + B dx (y-y*) + C (y-y*)^2 = C [ (y - c)^2 + g ],
//   A dx^2 - B dx (y+y*) + C (y+y*)^2 = C [ (y + c)^2 + g ],
//   c = y* - (B / 2C) dx,   g = (A/C - (B/2C)^2) dx^2 = (4AC - B^2) dx^2 / (4 C^2) > 0,
// so that each form costs one add and one two-register FMA per pair, c and g are per
// (target, column), and the common factor 1/sqrt(C) is applied once per target at the end.
struct TgtC {
  double ys, zs, psis;
  double ys2, ys4;  // 2 y*, 4 y*: the image terms follow from the direct ones (below)
};
struct ColC {
  double dx, dx2, c, g;  // x_i - x*, its square, and the S2 constants above
};

// One source node against one target: adds (phi-phi*-x+x*) K1 + zeta_x K2 to a1 and, if S2T,
// sqrt(C) S2 to aS (unit weight).  S2T = false is the far-field form: the S2 terms of the
// whole column come from s2_column_em() below, 28 FP64 instructions + 2 MUFU.RSQ64H remain.
template <bool S2T>
__device__ __forceinline__ void pair_term(const double2 zp, const double2 sl, const double yj,
                                          const TgtC& t, const ColC& c, double& a1, double& aS) {
  const double z = zp.x, psi = zp.y, zx = sl.x, zy = sl.y;
  // Image terms from the direct ones (all y >= 0, sws_setup): (y + y*)^2 = (y - y*)^2 + 4 y y* and
  // y + y* = (y - y*) + 2 y*, so y + y* itself is never formed: one DADD less per pair.  R+^2 >= R-^2, so
  // the rounding of R-^2 it inherits is below its own.
  const double dm = yj - t.ys;  // y - y*
  const double dz = z - t.zs;
  const double q = fma(dz, dz, c.dx2);
  const double Rm2 = fma(dm, dm, q);
  const double Rp2 = fma(t.ys4, yj, Rm2);
  const double rm = rsqrt_fp64(Rm2);
  const double rp = rsqrt_fp64(Rp2);
  // K1 numerators: zeta - zeta* - (x-x*) zeta_x - (y -+ y*) zeta_y, slopes at the source (Q2)
  const double n0 = fma(-c.dx, zx, dz);
  const double nm = fma(-dm, zy, n0);
  const double np = fma(-t.ys2, zy, nm);
  const double rm3 = (rm * rm) * rm;
  const double rp3 = (rp * rp) * rp;
  const double k1 = fma(np, rp3, nm * rm3);
  const double dpsi = psi - t.psis;
  a1 = fma(dpsi, k1, a1);
  a1 = fma(zx, rm + rp, a1);  // K2 = 1/R- + 1/R+
  if (S2T) {
    // S2 (eqs. (21), (22)) up to the factor 1/sqrt(C)
    const double sm = yj - c.c;
    const double sp = yj + c.c;
    const double Qm = fma(sm, sm, c.g);
    const double Qp = fma(sp, sp, c.g);
    aS += rsqrt_fp64(Qm) + rsqrt_fp64(Qp);
  }
}

// One staged segment [j0, j0 + len) of a column for the NT targets of a thread: trapezoid half weights on the
// column's first and last node by peeling (Q4), unit weights inside.  The staged record of a node is loaded
// once for the NT targets.
template <bool S2T, int NT>
__device__ __forceinline__ void walk_segment(const double2* rec, const double* yy, const int j0, const int len,
                                             const int M, const TgtC (&tg)[NT], const ColC (&cc)[NT],
                                             double (&col1)[NT], double (&colS)[NT]) {
  int jlo = 0, jhi = len;
  if (j0 == 0) {  // first node of the column: weight 1/2 in y
#pragma unroll
    for (int n = 0; n < NT; ++n) {
      double h1 = 0.0, hS = 0.0;
      pair_term<S2T>(rec[0], rec[1], yy[0], tg[n], cc[n], h1, hS);
      col1[n] = 0.5 * h1;
      colS[n] = 0.5 * hS;
    }
    jlo = 1;
  }
  const bool last = (j0 + len == M);
  if (last) jhi = len - 1;
#pragma unroll kUnroll
  for (int j = jlo; j < jhi; ++j) {
    const double2 r0 = rec[2 * j], r1 = rec[2 * j + 1];
    const double yj = yy[j];
#pragma unroll
    for (int n = 0; n < NT; ++n) pair_term<S2T>(r0, r1, yj, tg[n], cc[n], col1[n], colS[n]);
  }
  if (last && jhi >= jlo) {  // last node of the column: weight 1/2 in y
#pragma unroll
    for (int n = 0; n < NT; ++n) {
      double h1 = 0.0, hS = 0.0;
      pair_term<S2T>(rec[2 * jhi], rec[2 * jhi + 1], yy[jhi], tg[n], cc[n], h1, hS);
      col1[n] = fma(0.5, h1, col1[n]);
      colS[n] = fma(0.5, hS, colS[n]);
    }
  }
}

struct PairArgs {
  const SrcRec* src;  // [state][N][M]
  const double* x;    // [N]
  const double* y;    // [M + pad]
  const TgtRec* tgt;  // [state][T]
  double* part;       // [state][chunks][T]
  int N, M, T;
  int chunks, cols_per_chunk, seg_len, nseg;
  double dxdy;
  EmGeom em;
};

template <int MINB, int NT>
__global__ void __launch_bounds__(kThreads64, MINB) k_allpairs(const PairArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int seg_pad = a.seg_len;  // even by construction
  SrcRec* s_rec = reinterpret_cast<SrcRec*>(smem_raw);                            // [kStages][seg_pad]
  double* s_y = reinterpret_cast<double*>(s_rec + (size_t)kStages * seg_pad);     // [kStages][seg_pad]
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(s_y + (size_t)kStages * seg_pad);  // [kStages]

  const int tid = threadIdx.x;
  const int tile = blockIdx.x, chunk = blockIdx.y, state = blockIdx.z;
  // Threads take the targets in TRANSPOSED order, slot = k M + l: the 32 targets of a warp then share one
  // x* (two at most), so the columns that are near for a warp are the 2 r of one target, not 32 + 2 r
  // (near fraction 2.3 % instead of 6.5 % at 721x241).  t = l (N-1) + k is the index everything is stored by.
  // A thread owns NT targets, kThreads64 slots apart, and walks the staged records once for all of them.
  int t[NT];
  TgtC tg[NT];
  double xs[NT], kb[NT], kg[NT], sfac[NT];
#pragma unroll
  for (int n = 0; n < NT; ++n) {
    const int slot = (tile * NT + n) * kThreads64 + tid;
    const int sc = slot < a.T ? slot : a.T - 1;  // ragged tail: recompute the last target, never stored
    const int tc = target_of_slot(sc, a.N, a.M);
    t[n] = slot < a.T ? tc : a.T;
    const TgtRec tr = a.tgt[(size_t)state * a.T + tc];
    tg[n] = {tr.ys, tr.zs, tr.psis, 2.0 * tr.ys, 4.0 * tr.ys};
    xs[n] = tr.xs;
    kb[n] = tr.B / (2.0 * tr.C);                 // B / 2C
    kg[n] = tr.A / tr.C - kb[n] * kb[n];         // (4AC - B^2) / (4 C^2)
    sfac[n] = -tr.zxs * rsqrt_fp64(tr.C);
  }

  const int c0 = chunk * a.cols_per_chunk;
  const int c1 = min(a.N, c0 + a.cols_per_chunk);
  const int nitems = (c1 - c0) * a.nseg;  // (column, segment) work items of this CTA
  const SrcRec* src = a.src + (size_t)state * a.N * a.M;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&s_bar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  auto issue = [&](int q) {
    const int s = q % kStages;
    const int i = c0 + q / a.nseg, j0 = (q % a.nseg) * a.seg_len;
    const int len = min(a.seg_len, a.M - j0);
    const uint32_t rec_bytes = (uint32_t)len * (uint32_t)sizeof(SrcRec);
    const uint32_t y_bytes = (uint32_t)((len + 1) & ~1) * 8u;  // y is padded to an even count
    mbar_expect_tx(&s_bar[s], rec_bytes + y_bytes);
    bulk_g2s(s_rec + (size_t)s * seg_pad, src + (size_t)i * a.M + j0, rec_bytes, &s_bar[s]);
    bulk_g2s(s_y + (size_t)s * seg_pad, a.y + j0, y_bytes, &s_bar[s]);
  };

  if (tid == 0 && nitems > 0) issue(0);

  double tot1[NT], totS[NT];
#pragma unroll
  for (int n = 0; n < NT; ++n) tot1[n] = totS[n] = 0.0;
  for (int q = 0; q < nitems; ++q) {
    const int s = q % kStages;
    // the buffer written here was last read in iteration q-1, which ended with __syncthreads()
    if (tid == 0 && q + 1 < nitems) issue(q + 1);

    const int i = c0 + q / a.nseg, j0 = (q % a.nseg) * a.seg_len;
    const int len = min(a.seg_len, a.M - j0);
    ColC cc[NT];
    const double xi = __ldg(a.x + i);
    bool far_t = true;
#pragma unroll
    for (int n = 0; n < NT; ++n) {
      cc[n].dx = xi - xs[n];
      cc[n].dx2 = cc[n].dx * cc[n].dx;
      cc[n].c = fma(-kb[n], cc[n].dx, tg[n].ys);
      cc[n].g = kg[n] * cc[n].dx2;
      far_t = far_t && (cc[n].g >= a.em.gmin);
    }
    const double ci = (i == 0 || i == a.N - 1) ? 0.5 : 1.0;  // trapezoid weight in x (Q4)

    mbar_wait(&s_bar[s], (uint32_t)((q / kStages) & 1));

    const double2* rec = reinterpret_cast<const double2*>(s_rec + (size_t)s * seg_pad);
    const double* yy = s_y + (size_t)s * seg_pad;
    double col1[NT], colS[NT];
#pragma unroll
    for (int n = 0; n < NT; ++n) col1[n] = colS[n] = 0.0;
    if (__all_sync(0xffffffffu, far_t)) {  // warp-uniform: far for every target of the warp
      walk_segment<false, NT>(rec, yy, j0, len, a.M, tg, cc, col1, colS);
      if (j0 == 0) {
#pragma unroll
        for (int n = 0; n < NT; ++n) colS[n] = s2_column_em(a.em, cc[n].c, cc[n].g);  // the column's S2 terms, once
      }
    } else {
      walk_segment<true, NT>(rec, yy, j0, len, a.M, tg, cc, col1, colS);
    }
#pragma unroll
    for (int n = 0; n < NT; ++n) {
      tot1[n] = fma(ci, col1[n], tot1[n]);
      totS[n] = fma(ci, colS[n], totS[n]);
    }
    __syncthreads();
  }

#pragma unroll
  for (int n = 0; n < NT; ++n)
    if (t[n] < a.T)
      a.part[((size_t)state * a.chunks + chunk) * a.T + t[n]] = a.dxdy * fma(sfac[n], totS[n], tot1[n]);
}

// ---------------------------------------------------------------------------------------
// host side

constexpr int kMinB = SWS_MINB;
constexpr int kMinCtaNodes = 32;  // a CTA walks at least this many source nodes

size_t allpairs_smem_bytes(const PairPlan& p) {
  return (size_t)kStages * p.seg_len * (sizeof(SrcRec) + sizeof(double)) + kStages * sizeof(uint64_t);
}

// targets per thread of the FP64 kernel for this mesh (depends on the mesh only)
int pair_nt(const sws_ctx* c) { return c->params.precision == 0 && c->mesh.T >= kNT2MinTargets ? 2 : 1; }

cudaError_t allpairs_configure(const sws_ctx* c, int* occ_out) {
  const int smem_max = (int)(kStages * kSegMax * (sizeof(SrcRec) + sizeof(double)) + 64);
  const size_t smem_occ = kStages * kSegMax * (sizeof(SrcRec) + sizeof(double)) + kStages * sizeof(uint64_t);
  cudaError_t e = cudaFuncSetAttribute(k_allpairs<kMinB, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(k_allpairs<kMinB2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
  if (e != cudaSuccess) return e;
  int occ = 0;
  if (pair_nt(c) == 2)
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_allpairs<kMinB2, 2>, kThreads64, smem_occ);
  else
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_allpairs<kMinB, 1>, kThreads64, smem_occ);
  if (e != cudaSuccess) return e;
  *occ_out = occ > 0 ? occ : 1;
  return cudaSuccess;
}

// Choose the number of column groups.  Measured on B200: short CTAs win - at cfg5
// 19 / 61 / 121 / 241 groups give 59.5 / 59.0 / 58.8 / 58.6 ms (64-thread CTAs) - because CTAs whose
// columns are near their targets take 1.4x longer and finer pieces balance better, while every group
// costs one row of partial sums per target.  So: about kColsTarget columns per CTA, at least two waves of
// the sm_count * occupancy resident CTAs when the mesh is small, and among the candidates of that size
// the one with the least wave quantisation, cost(c) ~ ceil(CTAs / slots) * (ceil(N / c) + overhead).
// The split depends on the MESH ONLY, never on the number of states in the launch: the
// summation order of a state's quadrature is then the same in sws_residual and in every
// slot of sws_jv_batch, so a batch is bitwise a loop of single evaluations.
#ifndef SWS_COLS_TARGET
#define SWS_COLS_TARGET 12
#endif
constexpr int kColsTarget = SWS_COLS_TARGET;

PairPlan make_plan(const sws_ctx* c) {
  const Mesh& m = c->mesh;
  PairPlan p;
  const int threads = c->params.precision == 1 ? kPairThreads : kThreads64 * pair_nt(c);
  p.tiles = (m.T + threads - 1) / threads;
  p.nseg = (m.M + kSegMax - 1) / kSegMax;
  int seg = (m.M + p.nseg - 1) / p.nseg;
  p.seg_len = (seg + 1) & ~1;
  p.nseg = (m.M + p.seg_len - 1) / p.seg_len;
  const long slots = (long)c->sm_count * (c->pair_occ > 0 ? c->pair_occ : 4);
  int best = 1;
  const int cmax = max_chunks(c);
  if (c->chunks_user > 0) {
    best = c->chunks_user < cmax ? c->chunks_user : cmax;
  } else {
    int lo = (m.N + kColsTarget - 1) / kColsTarget;
    while (lo < cmax && (long)p.tiles * lo < 2 * slots) ++lo;
    if (lo > cmax) lo = cmax;
    int hi = lo + lo / 2 + 1;
    if (hi > cmax) hi = cmax;
    double best_cost = 1e300;
    for (int ch = lo; ch <= hi; ++ch) {
      const int cols = (m.N + ch - 1) / ch;
      const int used = (m.N + cols - 1) / cols;  // groups that are not empty
      if (used != ch && ch != lo) continue;
      const long ctas = (long)p.tiles * used;
      const long waves = (ctas + slots - 1) / slots;
      const double cost = (double)waves * (cols + 0.25) + 1e-3 * used;
      if (cost < best_cost) { best_cost = cost; best = used; }
    }
  }
  p.cols_per_chunk = (m.N + best - 1) / best;
  p.chunks = (m.N + p.cols_per_chunk - 1) / p.cols_per_chunk;
  return p;
}

int max_chunks(const sws_ctx* c) {
  int min_cols = (kMinCtaNodes + c->mesh.M - 1) / c->mesh.M;
  int cmax = c->mesh.N / (min_cols > 0 ? min_cols : 1);
  if (cmax < 1) cmax = 1;
  if (cmax > 256) cmax = 256;
  return cmax;
}

cudaError_t launch_allpairs(sws_ctx* c, int states, const PairPlan& plan, cudaStream_t st) {
  if (c->params.precision == 1) return launch_allpairs_f32(c, states, plan, st);
  const Mesh& m = c->mesh;
  PairArgs a;
  a.src = c->src; a.x = c->x; a.y = c->y; a.tgt = c->tgt; a.part = c->part;
  a.N = m.N; a.M = m.M; a.T = m.T;
  a.chunks = plan.chunks; a.cols_per_chunk = plan.cols_per_chunk;
  a.seg_len = plan.seg_len; a.nseg = plan.nseg;
  a.dxdy = m.dx * m.dy;
  a.em = em_geometry(c);
  dim3 grid(plan.tiles, plan.chunks, states);
  if (pair_nt(c) == 2)
    k_allpairs<kMinB2, 2><<<grid, kThreads64, allpairs_smem_bytes(plan), st>>>(a);
  else
    k_allpairs<kMinB, 1><<<grid, kThreads64, allpairs_smem_bytes(plan), st>>>(a);
  return cudaGetLastError();
}

// --- far-field statistics (bench.py: executed work of a launch) ----------------------------
// One warp = the same targets as a warp of k_allpairs (nt sets of 32 slots, kThreads64 slots apart); counts the
// columns that warp treats as near (direct S2 loop).  out[state * warps + w], warps = tiles * tpc / 32.
__global__ void k_count_near(const TgtRec* tgt, const double* x, int N, int M, int T, int nt, int tpc, int warps,
                             double gmin, int* out) {
  const int w = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32, state = blockIdx.y;
  if (w >= warps) return;
  const int wpc = tpc / 32;  // warps per CTA of the all-pairs kernel in use (tpc threads)
  const int tile = w / wpc, tid = (w % wpc) * 32 + (threadIdx.x & 31);
  double xs[2], kg[2];
  for (int n = 0; n < nt; ++n) {
    const int slot = (tile * nt + n) * tpc + tid;
    const TgtRec tr = tgt[(size_t)state * T + target_of_slot(slot < T ? slot : T - 1, N, M)];
    const double kb = tr.B / (2.0 * tr.C);
    xs[n] = tr.xs;
    kg[n] = tr.A / tr.C - kb * kb;
  }
  int near = 0;
  for (int i = 0; i < N; ++i) {
    const double xi = __ldg(x + i);
    bool far_t = true;
    for (int n = 0; n < nt; ++n) {
      const double dx = xi - xs[n];
      const double dx2 = dx * dx;
      far_t = far_t && (kg[n] * dx2 >= gmin);
    }
    if (!__all_sync(0xffffffffu, far_t)) ++near;
  }
  if ((threadIdx.x & 31) == 0) out[(size_t)state * warps + w] = near;
}

static int pair_cta_threads(const sws_ctx* c) { return c->params.precision == 1 ? kPairThreads : kThreads64; }
int count_near_warps(const sws_ctx* c) { return make_plan(c).tiles * (pair_cta_threads(c) / 32); }

cudaError_t launch_count_near(sws_ctx* c, int states, int* out, cudaStream_t st) {
  const Mesh& m = c->mesh;
  const int warps = count_near_warps(c);
  dim3 grid((warps + 3) / 4, states);
  k_count_near<<<grid, 128, 0, st>>>(c->tgt, c->x, m.N, m.M, m.T, pair_nt(c), pair_cta_threads(c), warps,
                                     em_geometry(c).gmin, out);
  return cudaGetLastError();
}

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

}  // namespace sws
