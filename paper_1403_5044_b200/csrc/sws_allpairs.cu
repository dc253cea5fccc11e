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
// the column sum (sws_farfield.cuh): 27 FP64 instructions + 2 MUFU.RSQ64H per pair; the others
// sum S2 pair by pair: 43 + 4.  Everything that depends only on (target, column) - dx, dx^2 and
// the completed-square constants of S2 - is hoisted out of the j loop; the half weights are
// applied by peeling the first/last node and scaling edge columns, so the inner loop carries no
// weight multiply.  Partial sums per (state, chunk, target) are written to global memory and
// added in a fixed order by the assemble kernel: no atomics, bitwise repeatable.
#include <mutex>

#include "sws_closed_form.cuh"
#include "sws_const.cuh"
#include "sws_farfield.cuh"
#include "sws_internal.cuh"
#include "sws_pair.cuh"
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
#ifndef SWS_MINB12
#define SWS_MINB12 6
#endif
#ifndef SWS_MINB22
#define SWS_MINB22 4
#endif
constexpr int kMinB12 = SWS_MINB12;  // ... of the one-target, two-state kernel (batches on small meshes)
constexpr int kMinB22 = SWS_MINB22;  // ... of the two-target, two-state kernel (batches on large meshes)

// One staged segment [j0, j0 + len) of a column for the NT targets x NS states of a thread: trapezoid half
// weights on the column's first and last node by peeling (Q4), unit weights inside.  A node's y_j and
// y_j - y* are formed once for the NS states (batched Jv: the states share the mesh), its staged record of
// each state is loaded once for the NT targets.  rec[m]: state m's records of this segment.
template <bool S2T, int NT, int NS>
__device__ __forceinline__ void walk_segment(const double2* const (&rec)[NS], const double* yy, const int j0,
                                             const int len, const int M, const TgtG (&tg)[NT],
                                             const TgtS (&ts)[NS][NT], const ColG (&cg)[NT],
                                             const ColS (&cs)[NS][NT], double (&col1)[NS][NT],
                                             double (&colS)[NS][NT]) {
  int jlo = 0, jhi = len;
  auto node = [&](const int j, double (&o1)[NS][NT], double (&oS)[NS][NT]) {
    const double yj = yy[j];
    double dm[NT];
#pragma unroll
    for (int n = 0; n < NT; ++n) dm[n] = yj - tg[n].ys;  // y - y*
#pragma unroll
    for (int m = 0; m < NS; ++m) {
      const double2 r0 = rec[m][2 * j], r1 = rec[m][2 * j + 1];
#pragma unroll
      for (int n = 0; n < NT; ++n) pair_term<S2T>(r0, r1, yj, dm[n], tg[n], ts[m][n], cg[n], cs[m][n], o1[m][n], oS[m][n]);
    }
  };
  if (j0 == 0) {  // first node of the column: weight 1/2 in y
    double h1[NS][NT], hS[NS][NT];
#pragma unroll
    for (int m = 0; m < NS; ++m)
#pragma unroll
      for (int n = 0; n < NT; ++n) h1[m][n] = hS[m][n] = 0.0;
    node(0, h1, hS);
#pragma unroll
    for (int m = 0; m < NS; ++m)
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        col1[m][n] = 0.5 * h1[m][n];
        colS[m][n] = 0.5 * hS[m][n];
      }
    jlo = 1;
  }
  const bool last = (j0 + len == M);
  if (last) jhi = len - 1;
#pragma unroll kUnroll
  for (int j = jlo; j < jhi; ++j) node(j, col1, colS);
  if (last && jhi >= jlo) {  // last node of the column: weight 1/2 in y
    double h1[NS][NT], hS[NS][NT];
#pragma unroll
    for (int m = 0; m < NS; ++m)
#pragma unroll
      for (int n = 0; n < NT; ++n) h1[m][n] = hS[m][n] = 0.0;
    node(jhi, h1, hS);
#pragma unroll
    for (int m = 0; m < NS; ++m)
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        col1[m][n] = fma(0.5, h1[m][n], col1[m][n]);
        colS[m][n] = fma(0.5, hS[m][n], colS[m][n]);
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
  int states;         // states of this launch (NS of them per CTA)
  int chunks, cols_per_chunk, seg_len, nseg;
  double dxdy;
  EmGeom em;
  // fused assembly (a6 + a9), tile_count != NULL: the CTA that completes a (state, target tile) - the last of
  // its `chunks` column groups to arrive - adds the partial sums in the fixed order c = 0 .. chunks-1 and writes
  // E2 = e2loc - sum into the residual; no separate assemble launch, still no floating-point atomics
  unsigned int* tile_count;  // [state][tiles], zero between launches
  double* e2loc;             // [state][T], written by CTA row 0 of this launch (a5 + a6 local part)
  double eps;
  double* F0;                // [n] residual of state 0
  double* Fpert;             // [states - 1][n]
  int n;
};

// Fused assembly, a6 + a9.  Every CTA of a (state, target tile) - its `chunks` column groups and the local row -
// counts itself in after its stores are visible; the last one adds the partial sums in the fixed order
// c = 0 .. chunks-1 (the sum and order of k_assemble) and writes E2 = e2loc - sum.
template <int NT, int NS>
__device__ __forceinline__ void arrive_and_assemble(const PairArgs& a, const int (&t)[NT], const int tile,
                                                    const int state0) {
  const int tid = threadIdx.x;
  __shared__ int s_last[NS];
  __threadfence();  // this thread's stores are visible device-wide ...
  __syncthreads();  // ... for every thread of the CTA, before the CTA counts itself in
  if (tid == 0) {
#pragma unroll
    for (int m = 0; m < NS; ++m) {
      s_last[m] = 0;
      if (state0 + m < a.states) {
        unsigned int* cnt = a.tile_count + (size_t)(state0 + m) * gridDim.x + tile;
        const unsigned int seen = atomicAdd(cnt, 1u);
        if (seen == (unsigned int)gridDim.y - 1u) {
          s_last[m] = 1;
          *cnt = 0u;  // ready for the next launch
        }
      }
    }
  }
  __syncthreads();
#pragma unroll
  for (int m = 0; m < NS; ++m) {
    if (!s_last[m]) continue;
    __threadfence();
    const int state = state0 + m;
    double* F = state == 0 ? a.F0 : a.Fpert + (size_t)(state - 1) * a.n;
#pragma unroll
    for (int n = 0; n < NT; ++n) {
      if (t[n] >= a.T) continue;
      const double* p = a.part + (size_t)state * a.chunks * a.T + t[n];
      double sum = 0.0;
      for (int c = 0; c < a.chunks; ++c) sum += __ldcg(p + (size_t)c * a.T);
      const int l = t[n] / (a.N - 1), k = t[n] - l * (a.N - 1);
      F[(size_t)(a.N + 1) * a.M + (size_t)l * (a.N + 1) + 2 + k] = __ldcg(a.e2loc + (size_t)state * a.T + t[n]) - sum;
    }
  }
}

// NS = states per CTA.  NS = 1 is the single evaluation; NS = 2 is the batched mode of sws_jv_batch: the CTA
// stages the y_j run once and one record run per state, and a thread forms y_j - y* once for its NS states.
// Every (state, target) sum goes through the same operations in the same order whatever NS is, and a column
// whose far/near decision differs between the states of a CTA is walked state by state, so that slot b of a
// batch stays bitwise sws_residual(u_b).
template <int MINB, int NT, int NS>
__global__ void __launch_bounds__(kThreads64, MINB) k_allpairs(const PairArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int seg_pad = a.seg_len;  // even by construction
  SrcRec* s_rec = reinterpret_cast<SrcRec*>(smem_raw);                                  // [kStages][NS][seg_pad]
  double* s_y = reinterpret_cast<double*>(s_rec + (size_t)kStages * NS * seg_pad);      // [kStages][seg_pad]
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(s_y + (size_t)kStages * seg_pad);       // [kStages]

  const int tid = threadIdx.x;
  // Programmatic dependent launch: this grid may have been scheduled while the kernel that produces the source /
  // target records was still in its last phase (it said so with griddepcontrol.launch_dependents); nothing of
  // global memory is touched before that kernel has completed and flushed.  A no-op otherwise.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  // With fused assembly (tile_count != NULL) CTA row y = 0 is the LOCAL row: it evaluates a5 + a6's local part
  // (the closed form I: 8 asinh per target) for the tile while the other rows walk their column groups.
  const int tile = blockIdx.x, chunk = (int)blockIdx.y - (a.tile_count ? 1 : 0), state0 = blockIdx.z * NS;
  int st[NS];  // the states of this CTA; a ragged last group recomputes the last state and stores nothing
#pragma unroll
  for (int m = 0; m < NS; ++m) st[m] = state0 + m < a.states ? state0 + m : a.states - 1;
  // Threads take the targets in TRANSPOSED order, slot = k M + l: the 32 targets of a warp then share one
  // x* (two at most), so the columns that are near for a warp are the 2 r of one target, not 32 + 2 r
  // (near fraction 2.3 % instead of 6.5 % at 721x241).  t = l (N-1) + k is the index everything is stored by.
  // A thread owns NT targets, kThreads64 slots apart, and walks the staged records once for all of them.
  int t[NT];
  TgtG tg[NT];
  TgtS ts[NS][NT];
  double xs[NT], kb[NS][NT], kg[NS][NT], sfac[NS][NT];
#pragma unroll
  for (int n = 0; n < NT; ++n) {
    const int slot = (tile * NT + n) * kThreads64 + tid;
    const int sc = slot < a.T ? slot : a.T - 1;  // ragged tail: recompute the last target, never stored
    const int tc = target_of_slot(sc, a.N, a.M);
    t[n] = slot < a.T ? tc : a.T;
#pragma unroll
    for (int m = 0; m < NS; ++m) {
      const TgtRec tr = a.tgt[(size_t)st[m] * a.T + tc];
      if (m == 0) {  // x*, y* are the mesh's: the same in every state
        tg[n] = {tr.ys, 2.0 * tr.ys, 4.0 * tr.ys};
        xs[n] = tr.xs;
      }
      ts[m][n] = {tr.zs, tr.psis};
      kb[m][n] = tr.B / (2.0 * tr.C);                    // B / 2C
      kg[m][n] = tr.A / tr.C - kb[m][n] * kb[m][n];      // (4AC - B^2) / (4 C^2)
      sfac[m][n] = -tr.zxs * rsqrt_fp64(tr.C);
    }
  }

  if (chunk < 0) {  // the local row
    const double xa = __ldg(a.x), xb = __ldg(a.x + a.N - 1), ya = __ldg(a.y), yb = __ldg(a.y + a.M - 1);
#pragma unroll
    for (int m = 0; m < NS; ++m) {
      if (state0 + m >= a.states) continue;
#pragma unroll
      for (int n = 0; n < NT; ++n)
        if (t[n] < a.T) {
          const size_t ts_ = (size_t)(state0 + m) * a.T + t[n];
          a.e2loc[ts_] = e2_local(a.tgt[ts_], a.eps, xa, xb, ya, yb);
        }
    }
    arrive_and_assemble<NT, NS>(a, t, tile, state0);
    return;
  }

  const int c0 = chunk * a.cols_per_chunk;
  const int c1 = min(a.N, c0 + a.cols_per_chunk);
  const int nitems = (c1 - c0) * a.nseg;  // (column, segment) work items of this CTA
  const size_t plane = (size_t)a.N * a.M;

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
    mbar_expect_tx(&s_bar[s], NS * rec_bytes + y_bytes);
#pragma unroll
    for (int m = 0; m < NS; ++m)
      bulk_g2s(s_rec + ((size_t)s * NS + m) * seg_pad, a.src + st[m] * plane + (size_t)i * a.M + j0, rec_bytes,
               &s_bar[s]);
    bulk_g2s(s_y + (size_t)s * seg_pad, a.y + j0, y_bytes, &s_bar[s]);
  };

  if (tid == 0 && nitems > 0) issue(0);

  double tot1[NS][NT], totS[NS][NT];
#pragma unroll
  for (int m = 0; m < NS; ++m)
#pragma unroll
    for (int n = 0; n < NT; ++n) tot1[m][n] = totS[m][n] = 0.0;
  for (int q = 0; q < nitems; ++q) {
    const int s = q % kStages;
    // the buffer written here was last read in iteration q-1, which ended with __syncthreads()
    if (tid == 0 && q + 1 < nitems) issue(q + 1);

    const int i = c0 + q / a.nseg, j0 = (q % a.nseg) * a.seg_len;
    const int len = min(a.seg_len, a.M - j0);
    ColG cg[NT];
    ColS cs[NS][NT];
    const double xi = __ldg(a.x + i);
    bool far_m[NS];
#pragma unroll
    for (int m = 0; m < NS; ++m) far_m[m] = true;
#pragma unroll
    for (int n = 0; n < NT; ++n) {
      cg[n].dx = xi - xs[n];
      cg[n].dx2 = cg[n].dx * cg[n].dx;
#pragma unroll
      for (int m = 0; m < NS; ++m) {
        cs[m][n].c = fma(-kb[m][n], cg[n].dx, tg[n].ys);
        cs[m][n].g = kg[m][n] * cg[n].dx2;
        far_m[m] = far_m[m] && (cs[m][n].g >= a.em.gmin);
      }
    }
    const double ci = (i == 0 || i == a.N - 1) ? 0.5 : 1.0;  // trapezoid weight in x (Q4)

    // warp-uniform far/near decision PER STATE (far for every target of the warp), as a single evaluation takes it
    int nfar = 0;
#pragma unroll
    for (int m = 0; m < NS; ++m) {
      far_m[m] = __all_sync(0xffffffffu, far_m[m]);
      nfar += far_m[m] ? 1 : 0;
    }

    mbar_wait(&s_bar[s], (uint32_t)((q / kStages) & 1));

    const double2* rec[NS];
#pragma unroll
    for (int m = 0; m < NS; ++m) rec[m] = reinterpret_cast<const double2*>(s_rec + ((size_t)s * NS + m) * seg_pad);
    const double* yy = s_y + (size_t)s * seg_pad;
    double col1[NS][NT], colS[NS][NT];
#pragma unroll
    for (int m = 0; m < NS; ++m)
#pragma unroll
      for (int n = 0; n < NT; ++n) col1[m][n] = colS[m][n] = 0.0;
    if (nfar == NS) {
      walk_segment<false, NT, NS>(rec, yy, j0, len, a.M, tg, ts, cg, cs, col1, colS);
    } else if (nfar == 0) {
      walk_segment<true, NT, NS>(rec, yy, j0, len, a.M, tg, ts, cg, cs, col1, colS);
    } else if (NS > 1) {  // the states disagree (a column at the edge of the radius): one state at a time
#pragma unroll
      for (int m = 0; m < NS; ++m) {
        const double2* const rec1[1] = {rec[m]};
        TgtS ts1[1][NT];
        ColS cs1[1][NT];
        double c11[1][NT], c1S[1][NT];
#pragma unroll
        for (int n = 0; n < NT; ++n) { ts1[0][n] = ts[m][n]; cs1[0][n] = cs[m][n]; c11[0][n] = c1S[0][n] = 0.0; }
        if (far_m[m]) walk_segment<false, NT, 1>(rec1, yy, j0, len, a.M, tg, ts1, cg, cs1, c11, c1S);
        else walk_segment<true, NT, 1>(rec1, yy, j0, len, a.M, tg, ts1, cg, cs1, c11, c1S);
#pragma unroll
        for (int n = 0; n < NT; ++n) { col1[m][n] = c11[0][n]; colS[m][n] = c1S[0][n]; }
      }
    }
    if (j0 == 0) {
#pragma unroll
      for (int m = 0; m < NS; ++m)
        if (far_m[m]) {
#pragma unroll
          for (int n = 0; n < NT; ++n) colS[m][n] = s2_column_em(a.em, cs[m][n].c, cs[m][n].g);  // the column's S2 terms, once
        }
    }
#pragma unroll
    for (int m = 0; m < NS; ++m)
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        tot1[m][n] = fma(ci, col1[m][n], tot1[m][n]);
        totS[m][n] = fma(ci, colS[m][n], totS[m][n]);
      }
    __syncthreads();
  }

#pragma unroll
  for (int m = 0; m < NS; ++m)
    if (state0 + m < a.states) {
#pragma unroll
      for (int n = 0; n < NT; ++n)
        if (t[n] < a.T)
          a.part[((size_t)(state0 + m) * a.chunks + chunk) * a.T + t[n]] =
              a.dxdy * fma(sfac[m][n], totS[m][n], tot1[m][n]);
    }

  if (a.tile_count != nullptr) arrive_and_assemble<NT, NS>(a, t, tile, state0);
}

// ---------------------------------------------------------------------------------------
// host side

constexpr int kMinB = SWS_MINB;
constexpr int kMinCtaNodes = 32;  // a CTA walks at least this many source nodes

size_t allpairs_smem_bytes(const PairPlan& p, int ns) {
  return (size_t)kStages * p.seg_len * (ns * sizeof(SrcRec) + sizeof(double)) + kStages * sizeof(uint64_t);
}

// targets per thread of the FP64 kernel for this mesh (depends on the mesh only)
int pair_nt(const sws_ctx* c) {
  if (const_path_active(c)) return 1;  // the constant-bank kernel: one target per thread
  return c->params.precision == 0 && c->mesh.T >= kNT2MinTargets ? 2 : 1;
}

// states per CTA of a launch with `states` states: 1 for a single evaluation; kBatchNS for a batch unless
// sws_set_states_per_cta says otherwise.  Results do not depend on it (bitwise).  Measured on B200 (DESIGN.md
// section 6, round 2): two states per CTA are 4.4-4.8 % SLOWER than one (721x241 b=16: 971 against 926 ms;
// 361x121 b=32: 127.4 against 119.0; 181x61 b=16: 4.63 against 4.42) - sharing y_j and y_j - y* saves one DADD
// and one LDS.64 of 28 + 3 per pair, the doubled register footprint (212 against 150, 148 against 114) costs
// more - so the default stays 1.
#ifndef SWS_BATCH_NS
#define SWS_BATCH_NS 1
#endif
constexpr int kBatchNS = SWS_BATCH_NS;
int pair_ns(const sws_ctx* c, int states) {
  if (states < 2 || c->params.precision != 0) return 1;
  const int want = c->ns_user > 0 ? c->ns_user : kBatchNS;
  return want >= 2 ? 2 : 1;
}

template <int MINB, int NT, int NS>
static cudaError_t configure_one(int* occ) {
  const int smem_max = (int)(kStages * kSegMax * (NS * sizeof(SrcRec) + sizeof(double)) + 64);
  const size_t smem_occ = kStages * kSegMax * (NS * sizeof(SrcRec) + sizeof(double)) + kStages * sizeof(uint64_t);
  cudaError_t e = cudaFuncSetAttribute(k_allpairs<MINB, NT, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, k_allpairs<MINB, NT, NS>, kThreads64, smem_occ);
}

cudaError_t allpairs_configure(const sws_ctx* c, int* occ_out) {
  int occ11 = 0, occ21 = 0, occ12 = 0, occ22 = 0;
  cudaError_t e = configure_one<kMinB, 1, 1>(&occ11);
  if (e == cudaSuccess) e = configure_one<kMinB2, 2, 1>(&occ21);
  if (e == cudaSuccess) e = configure_one<kMinB12, 1, 2>(&occ12);
  if (e == cudaSuccess) e = configure_one<kMinB22, 2, 2>(&occ22);
  if (e != cudaSuccess) return e;
  const int occ = pair_nt(c) == 2 ? occ21 : occ11;  // the plan is made for the single-evaluation kernel (mesh only)
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

cudaError_t launch_allpairs(sws_ctx* c, int states, const PairPlan& plan, cudaStream_t st, double* F0, double* Fpert) {
  if (c->params.precision == 1) return launch_allpairs_f32(c, states, plan, st);
  const Mesh& m = c->mesh;
  PairArgs a;
  a.src = c->src; a.x = c->x; a.y = c->y; a.tgt = c->tgt; a.part = c->part;
  a.N = m.N; a.M = m.M; a.T = m.T;
  a.states = states;
  a.chunks = plan.chunks; a.cols_per_chunk = plan.cols_per_chunk;
  a.seg_len = plan.seg_len; a.nseg = plan.nseg;
  a.dxdy = m.dx * m.dy;
  a.em = em_geometry(c);
  a.tile_count = F0 ? c->tile_count : nullptr;  // F0 given: the kernel also assembles E2 (no k_assemble launch)
  a.e2loc = c->e2loc; a.eps = m.eps; a.F0 = F0; a.Fpert = Fpert; a.n = m.n;
  const int ns = pair_ns(c, states), nt = pair_nt(c);
  dim3 grid(plan.tiles, plan.chunks + (a.tile_count ? 1 : 0), (states + ns - 1) / ns);
  const size_t smem = allpairs_smem_bytes(plan, ns);
  // launched with programmatic stream serialisation allowed: see griddepcontrol.wait at the top of the kernel
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = dim3(kThreads64); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  if (nt == 2 && ns == 2) return cudaLaunchKernelEx(&cfg, k_allpairs<kMinB22, 2, 2>, a);
  if (nt == 2) return cudaLaunchKernelEx(&cfg, k_allpairs<kMinB2, 2, 1>, a);
  if (ns == 2) return cudaLaunchKernelEx(&cfg, k_allpairs<kMinB12, 1, 2>, a);
  return cudaLaunchKernelEx(&cfg, k_allpairs<kMinB, 1, 1>, a);
}


// ---------------------------------------------------------------------------------------
// host side of the uniform-operand (constant-bank) path, sws_allpairs_const.cuh

int const_slab_cols(int M) {
  const int ypad = (M + 3) & ~3;
  int cols = (kConstDoubles - ypad) / (4 * M);
  if (cols > kConstMaxCols) cols = kConstMaxCols;
  return cols < 0 ? 0 : cols;
}

// Columns per CTA.  Measured at 721x241 / 361x121 (ms per state): 1: 50.2 / 3.41, 2: 49.4 / 3.34, 4: 49.2 / 3.33 -
// a CTA's set-up (target record, divisions) and its Euler-Maclaurin epilogues run at dependent-instruction latency,
// so longer CTAs are better as long as a launch still fills the GPU twice; 181x61: 1 is best (0.28 against 0.29 / 0.34).
int const_cols_per_cta(const sws_ctx* c) {
#ifdef SWS_CONST_CPC
  return SWS_CONST_CPC;  // build-time override for the measurements of profiles/r2_experiments.md
#endif
  const int cols = const_slab_cols(c->mesh.M);
  const long tiles = const_tiles(c->mesh.N, c->mesh.M);
  const long slots = (long)c->sm_count * 8;
  for (int cpc = 4; cpc > 1; cpc /= 2)
    if (tiles * ((cols + cpc - 1) / cpc) >= 2 * slots) return cpc;
  return 1;
}

bool const_path_active(const sws_ctx* c) {
  if (c->params.precision != 0 || !c->acc_c || c->const_mode == 0) return false;
  return c->const_mode == 1 || c->mesh.T >= kConstMinTargets;
}

// a5 + a6 + a9 after the slabs of all states: E2 = 2 pi (phi* - x*) + eps / rho* - zeta_x* I - [quadrature]
__global__ void __launch_bounds__(128) k_finish_const(const TgtRec* tgt, const double* acc, size_t bank_stride, int banks,
                                                      const double* x, const double* y, int N, int M, int T,
                                                      double eps, double* F0, double* Fpert, int n) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x, state = blockIdx.y;
  if (t >= T) return;
  const double xa = __ldg(x), xb = __ldg(x + N - 1), ya = __ldg(y), yb = __ldg(y + M - 1);
  const size_t ts = (size_t)state * T + t;
  double sum = acc[ts];
  for (int b = 1; b < banks; ++b) sum += acc[b * bank_stride + ts];  // fixed order
  double* F = state == 0 ? F0 : Fpert + (size_t)(state - 1) * n;
  const int l = t / (N - 1), k = t - l * (N - 1);
  F[(size_t)(N + 1) * M + (size_t)l * (N + 1) + 2 + k] = e2_local(tgt[ts], eps, xa, xb, ya, yb) - sum;
}

namespace {
// The two banks belong to the process (one copy per device), not to a context: every context of a device feeds
// them through the same two streams, so that slabs of different contexts can never be in a bank at the same time.
struct ConstDevice {
  bool ready = false;
  cudaStream_t stream[kConstBanks] = {};
  cudaEvent_t fork = nullptr, join[kConstBanks] = {};
};
constexpr int kMaxDevices = 64;
ConstDevice g_const_dev[kMaxDevices];
std::mutex g_const_mu;
}  // namespace

// Streams, events and bank addresses of a device: created once, by the first sws_setup on that device that allocates the
// path's workspace (so that no call - in particular no call a user is capturing into a CUDA graph - has to create them).
static cudaError_t const_device_ready(int device, ConstDevice** out) {  // the caller holds g_const_mu
  if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
  ConstDevice& d = g_const_dev[device];
  cudaError_t e = cudaSuccess;
  if (!d.ready) {
    for (int b = 0; b < kConstBanks && e == cudaSuccess; ++b) {
      if (!d.stream[b]) e = cudaStreamCreateWithFlags(&d.stream[b], cudaStreamNonBlocking);
      if (e == cudaSuccess && !d.join[b]) e = cudaEventCreateWithFlags(&d.join[b], cudaEventDisableTiming);
    }
    if (e == cudaSuccess && !d.fork) e = cudaEventCreateWithFlags(&d.fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = const_bank_prepare_0();
    if (e == cudaSuccess) e = const_bank_prepare_1();
    if (e != cudaSuccess) return e;
    d.ready = true;
  }
  *out = &d;
  return cudaSuccess;
}

cudaError_t const_path_prepare(int device) {
  std::lock_guard<std::mutex> lock(g_const_mu);
  ConstDevice* d = nullptr;
  return const_device_ready(device, &d);
}

cudaError_t launch_allpairs_const(sws_ctx* c, int states, cudaStream_t st, double* F0, double* Fpert, int* launches) {
  const Mesh& m = c->mesh;
  std::lock_guard<std::mutex> lock(g_const_mu);
  ConstDevice* dp = nullptr;
  cudaError_t e = const_device_ready(c->device, &dp);
  if (e != cudaSuccess) return e;
  ConstDevice& d = *dp;
  // A call that is being CAPTURED into a CUDA graph must not touch the two shared streams: a stream that waits on an
  // event of a capturing stream joins that capture and stays in it until cudaStreamEndCapture, and an eager call of
  // another host thread or context in that window would enqueue its slabs into the foreign capture (its F silently
  // stale).  Captured calls therefore put the copies and launches of both banks on the caller's stream itself, in the
  // same slab order: same summation order, bitwise the same result, no fork / join (and no overlap between the banks).
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if ((e = cudaStreamIsCapturing(st, &cap)) != cudaSuccess) return e;
  const bool inline_banks = cap != cudaStreamCaptureStatusNone;
  const int cols = const_slab_cols(m.M), ypad = (m.M + 3) & ~3;
  const int tiles = const_tiles(m.N, m.M);
  const int slabs = (m.N + cols - 1) / cols;
  const int banks = slabs < kConstBanks ? slabs : kConstBanks;
  // fork: both bank streams wait for what the caller's stream has enqueued so far (the fields kernels)
  if (!inline_banks) {
    if ((e = cudaEventRecord(d.fork, st)) != cudaSuccess) return e;
    for (int b = 0; b < banks; ++b)
      if ((e = cudaStreamWaitEvent(d.stream[b], d.fork, 0)) != cudaSuccess) return e;
  }
  ConstArgs a;
  a.x = c->x; a.N = m.N; a.M = m.M; a.T = m.T; a.ypad = ypad; a.dxdy = m.dx * m.dy; a.em = em_geometry(c);
  a.cpc = const_cols_per_cta(c);
  for (int s = 0; s < states && e == cudaSuccess; ++s) {
    for (int q = 0; q < slabs && e == cudaSuccess; ++q) {
      const int b = q % kConstBanks;  // slab q of a state always goes to bank q mod kConstBanks (fixed summation order)
      a.tgt = c->tgt + (size_t)s * m.T;
      a.part = c->part_c + (size_t)b * kConstMaxCols * m.T;
      a.acc = c->acc_c + ((size_t)b * c->max_states + s) * m.T;
      a.cnt = c->cnt_c + (size_t)b * tiles;
      a.col0 = q * cols;
      a.ncols = m.N - a.col0 < cols ? m.N - a.col0 : cols;
      a.first = q < kConstBanks;
      // every call puts its own y table into a bank before its first slab there: the banks belong to the process,
      // and a CUDA graph replayed by a caller may have refilled them since this context's last call
      const double* y = (s == 0 && q < kConstBanks) ? c->y : nullptr;
      const SrcRec* slab = c->src + (size_t)s * m.S + (size_t)a.col0 * m.M;
      cudaStream_t bs = inline_banks ? st : d.stream[b];
      e = b == 0 ? const_bank_launch_0(a, slab, y, tiles, bs) : const_bank_launch_1(a, slab, y, tiles, bs);
      if (e == cudaSuccess && launches) *launches += 1;
    }
  }
  // join: the caller's stream continues after both banks have drained.  Also after a failed enqueue: the bank streams
  // may already hold work that reads this context's buffers, and the caller must not run ahead of it.
  if (!inline_banks) {
    for (int b = 0; b < banks; ++b) {
      cudaError_t ej = cudaEventRecord(d.join[b], d.stream[b]);
      if (ej == cudaSuccess) ej = cudaStreamWaitEvent(st, d.join[b], 0);
      if (e == cudaSuccess) e = ej;
    }
  }
  if (e != cudaSuccess) return e;
  if (F0) {
    k_finish_const<<<dim3((m.T + 127) / 128, states), 128, 0, st>>>(c->tgt, c->acc_c, (size_t)c->max_states * m.T, banks,
                                                                 c->x, c->y, m.N, m.M, m.T, m.eps, F0, Fpert, m.n);
    if (launches) *launches += 1;
    e = cudaGetLastError();
  }
  return e;
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

}  // namespace sws
