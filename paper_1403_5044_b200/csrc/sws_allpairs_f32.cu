// Step a4 in FP32 pair arithmetic (sws_params.precision = 1; BASELINE.json config 4,
// "FP32-accumulate variant, reported separately with its measured error"; reading Q12 of
// DESIGN.md).  Same quadrature, same kernels K1/K2/S2, same
// decomposition (one thread = one target, 128 targets per CTA, source columns staged by
// bulk async copies) as sws_allpairs.cu; what changes is the arithmetic of one pair:
//
//   * the differences that cancel are formed to FP32 accuracy of the EXACT difference
//     without touching the FP64 pipe:  y_j -+ y* = ((j -+ l) dy (+ 2 y_1)) from the integer
//     mesh offsets (exact in FP32), zeta_ij - zeta* from two-float operands (hi + lo),
//     x_i - x* once per column in FP64;
//   * everything else of the pair - R^2, 1/R (MUFU.RSQ, <= 2 ulp), cubes, K1, K2, the S2
//     forms - is FP32, with the direct and the image term of each kernel in the two lanes
//     of the packed f32x2 instructions of sm_100 (FFMA2/FADD2/FMUL2);
//   * a column's terms (<= 256) are accumulated in FP32; columns are added in FP64, and the
//     per-(state, column group, target) partial goes to the same `part` buffer, so
//     everything outside a4 is the FP64 path unchanged.
//
//   * far columns (sws_farfield.cuh: sqrt(g) >= r dy for the whole warp) take their S2 column sum
//     from the FP64 Euler-Maclaurin form, exactly as the FP64 kernel does: the FP64 pipe is
//     idle here, and the pair loop drops to 2 MUFU.RSQ per pair.
//
// Bound: the XU pipe (4 MUFU.RSQ per near pair, 2 per far pair; 16 results per clock per SM), not the FP64 pipe.
// The variant is reported, never gated: tests/test_gpu_parity.py measures its error against
// the FP64 oracle.
#include "sws_farfield.cuh"
#include "sws_internal.cuh"
#include "sws_stage.cuh"

namespace sws {

namespace {

typedef unsigned long long u64;

__device__ __forceinline__ u64 pk(float lo, float hi) {
  u64 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpk(u64 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
  u64 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
  u64 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
  u64 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ float rsq(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ u64 rsq2(u64 v) {
  float a, b;
  unpk(v, a, b);
  return pk(rsq(a), rsq(b));
}

// Per-target and per-(target, column) constants, already packed (lane 0 = direct term,
// lane 1 = image term).
struct TgtF {
  u64 nzs;    // (-zeta*_hi, -zeta*_lo)
  u64 npsis;  // (-(phi*-x*), -(phi*-x*))
  u64 dy2;    // (dy, dy)
  u64 off2;   // (0, 2 y_1):  y_j - y* = (j-l) dy,  y_j + y* = (j+l) dy + 2 y_1
};
struct ColF {
  float ndx, dx2;  // -(x_i - x*), (x_i - x*)^2
  u64 kb2;         // (+kb dx, -kb dx):  s-+ = (y_j -+ y*) +- (B/2C) dx   (completed square)
  u64 g2;          // (g, g), g = (4AC - B^2) dx^2 / (4 C^2)
};

// One source node against one target.  ra = {z_hi, z_lo, psi, psi}, rb = {zx, zx, -zy, -zy};
// t2 = (j - l, j + l) as floats.  Adds the K1/K2 terms to a1 (lanes summed later) and
// sqrt(C) S2 to aS.
template <bool S2T>
__device__ __forceinline__ void pair_f32(const float4 ra, const float4 rb, const u64 t2,
                                         const TgtF& t, const ColF& c, u64& a1, u64& aS) {
  const u64 dmp = fma2(t2, t.dy2, t.off2);  // (y - y*, y + y*)
  const u64 d2 = add2(pk(ra.x, ra.y), t.nzs);
  float dh, dl;
  unpk(d2, dh, dl);
  const float dz = dh + dl;  // zeta - zeta*
  const u64 dpsi2 = add2(pk(ra.z, ra.w), t.npsis);
  const float n0 = fmaf(c.ndx, rb.x, dz);  // dz - dx zeta_x
  const float q = fmaf(dz, dz, c.dx2);
  const u64 R2 = fma2(dmp, dmp, pk(q, q));
  const u64 r = rsq2(R2);  // (1/R-, 1/R+)
  const u64 nmp = fma2(dmp, pk(rb.z, rb.w), pk(n0, n0));  // K1 numerators (Q1, Q2)
  const u64 r3 = mul2(mul2(r, r), r);
  a1 = fma2(dpsi2, mul2(nmp, r3), a1);  // (phi - phi* - x + x*) K1
  a1 = fma2(pk(rb.x, rb.y), r, a1);     // zeta_x K2
  if (S2T) {
    const u64 smp = add2(dmp, c.kb2);
    aS = add2(aS, rsq2(fma2(smp, smp, c.g2)));  // S2 up to 1/sqrt(C)
  }
}

// One staged segment of a column: half weights on the column's first and last node (Q4).
template <bool S2T>
__device__ __forceinline__ void walk_f32(const float4* rec, const int j0, const int len, const int M, const int l,
                                         const TgtF& tg, const ColF& cc, u64& col1, u64& colS) {
  const u64 one2 = pk(1.f, 1.f), half2 = pk(.5f, .5f), zero2 = pk(0.f, 0.f);
  u64 t2 = pk((float)(j0 - l), (float)(j0 + l));
  int jlo = 0, jhi = len;
  if (j0 == 0) {  // first node of the column: weight 1/2 in y
    u64 h1 = zero2, hS = zero2;
    pair_f32<S2T>(rec[0], rec[1], t2, tg, cc, h1, hS);
    col1 = mul2(half2, h1);
    colS = mul2(half2, hS);
    t2 = add2(t2, one2);
    jlo = 1;
  }
  const bool last = (j0 + len == M);
  if (last) jhi = len - 1;
#pragma unroll 4
  for (int j = jlo; j < jhi; ++j) {
    pair_f32<S2T>(rec[2 * j], rec[2 * j + 1], t2, tg, cc, col1, colS);
    t2 = add2(t2, one2);
  }
  if (last && jhi >= jlo) {  // last node of the column: weight 1/2 in y
    u64 h1 = zero2, hS = zero2;
    pair_f32<S2T>(rec[2 * jhi], rec[2 * jhi + 1], t2, tg, cc, h1, hS);
    col1 = fma2(half2, h1, col1);
    colS = fma2(half2, hS, colS);
  }
}

__device__ __forceinline__ double lanes_sum(u64 v) {
  float a, b;
  unpk(v, a, b);
  return (double)a + (double)b;
}

}  // namespace

struct PairArgsF {
  const SrcRecF* src;  // [state][N][M]
  const double* x;     // [N]
  const TgtRec* tgt;   // [state][T]
  double* part;        // [state][chunks][T]
  int N, M, T;
  int chunks, cols_per_chunk, seg_len, nseg;
  double dxdy, dy, y1;
  EmGeom em;
};

__global__ void __launch_bounds__(kPairThreads, 8) k_allpairs_f32(const PairArgsF a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int seg_pad = a.seg_len;
  SrcRecF* s_rec = reinterpret_cast<SrcRecF*>(smem_raw);                             // [kStages][seg_pad]
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(s_rec + (size_t)kStages * seg_pad);  // [kStages]

  const int tid = threadIdx.x;
  const int tile = blockIdx.x, chunk = blockIdx.y, state = blockIdx.z;
  const int slot = tile * kPairThreads + tid;  // transposed target order (sws_farfield.cuh)
  const int tc = target_of_slot(slot < a.T ? slot : a.T - 1, a.N, a.M);
  const int t = slot < a.T ? tc : a.T;
  const int l = tc / (a.N - 1);

  const TgtRec tr = a.tgt[(size_t)state * a.T + tc];
  const double xs = tr.xs;
  const double kb = tr.B / (2.0 * tr.C);
  const double kg = tr.A / tr.C - kb * kb;
  TgtF tg;
  {
    const float zh = (float)tr.zs, zl = (float)(tr.zs - (double)zh), ps = (float)tr.psis;
    const float dyf = (float)a.dy;
    tg.nzs = pk(-zh, -zl);
    tg.npsis = pk(-ps, -ps);
    tg.dy2 = pk(dyf, dyf);
    tg.off2 = pk(0.f, (float)(2.0 * a.y1));
  }
  const u64 zero2 = pk(0.f, 0.f);

  const int c0 = chunk * a.cols_per_chunk;
  const int c1 = min(a.N, c0 + a.cols_per_chunk);
  const int nitems = (c1 - c0) * a.nseg;
  const SrcRecF* src = a.src + (size_t)state * a.N * a.M;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&s_bar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  auto issue = [&](int q) {
    const int s = q % kStages;
    const int i = c0 + q / a.nseg, j0 = (q % a.nseg) * a.seg_len;
    const int len = min(a.seg_len, a.M - j0);
    const uint32_t bytes = (uint32_t)len * (uint32_t)sizeof(SrcRecF);
    mbar_expect_tx(&s_bar[s], bytes);
    bulk_g2s(s_rec + (size_t)s * seg_pad, src + (size_t)i * a.M + j0, bytes, &s_bar[s]);
  };

  if (tid == 0 && nitems > 0) issue(0);

  double tot1 = 0.0, totS = 0.0;
  for (int q = 0; q < nitems; ++q) {
    const int s = q % kStages;
    if (tid == 0 && q + 1 < nitems) issue(q + 1);

    const int i = c0 + q / a.nseg, j0 = (q % a.nseg) * a.seg_len;
    const int len = min(a.seg_len, a.M - j0);
    ColF cc;
    const double dxd = __ldg(a.x + i) - xs, dxd2 = dxd * dxd;
    const double gd = kg * dxd2;  // the S2 constants of sws_allpairs.cu, in FP64 for the far-field form
    {
      const float kbdx = (float)(kb * dxd), g = (float)gd;
      cc.ndx = -(float)dxd;
      cc.dx2 = (float)dxd2;
      cc.kb2 = pk(kbdx, -kbdx);
      cc.g2 = pk(g, g);
    }
    const double ci = (i == 0 || i == a.N - 1) ? 0.5 : 1.0;  // trapezoid weight in x (Q4)

    mbar_wait(&s_bar[s], (uint32_t)((q / kStages) & 1));

    const float4* rec = reinterpret_cast<const float4*>(s_rec + (size_t)s * seg_pad);
    u64 col1 = zero2, colS = zero2;
    double colS_far = 0.0;
    if (column_is_far(gd, a.em.gmin)) {  // warp-uniform
      walk_f32<false>(rec, j0, len, a.M, l, tg, cc, col1, colS);
      colS = zero2;
      if (j0 == 0) colS_far = s2_column_em(a.em, fma(-kb, dxd, tr.ys), gd);
    } else {
      walk_f32<true>(rec, j0, len, a.M, l, tg, cc, col1, colS);
    }
    tot1 = fma(ci, lanes_sum(col1), tot1);  // columns are added in FP64
    totS = fma(ci, lanes_sum(colS) + colS_far, totS);
    __syncthreads();
  }

  if (t < a.T)
    a.part[((size_t)state * a.chunks + chunk) * a.T + t] =
        a.dxdy * fma(-tr.zxs / sqrt(tr.C), totS, tot1);
}

// ---------------------------------------------------------------------------------------
// host side

size_t allpairs_f32_smem_bytes(int seg_len) {
  return (size_t)kStages * seg_len * sizeof(SrcRecF) + kStages * sizeof(uint64_t);
}

cudaError_t allpairs_f32_configure(int* occ_out) {
  const size_t smem = allpairs_f32_smem_bytes(kSegMax);
  cudaError_t e = cudaFuncSetAttribute(k_allpairs_f32, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)smem + 64);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_allpairs_f32, kPairThreads, smem);
  if (e != cudaSuccess) return e;
  *occ_out = occ > 0 ? occ : 1;
  return cudaSuccess;
}

cudaError_t launch_allpairs_f32(sws_ctx* c, int states, const PairPlan& plan, cudaStream_t st) {
  const Mesh& m = c->mesh;
  PairArgsF a;
  a.src = c->srcf; a.x = c->x; a.tgt = c->tgt; a.part = c->part;
  a.N = m.N; a.M = m.M; a.T = m.T;
  a.chunks = plan.chunks; a.cols_per_chunk = plan.cols_per_chunk;
  a.seg_len = plan.seg_len; a.nseg = plan.nseg;
  a.dxdy = m.dx * m.dy; a.dy = m.dy; a.y1 = m.y1;
  a.em = em_geometry(c);
  dim3 grid(plan.tiles, plan.chunks, states);
  k_allpairs_f32<<<grid, kPairThreads, allpairs_f32_smem_bytes(plan.seg_len), st>>>(a);
  return cudaGetLastError();
}

}  // namespace sws
