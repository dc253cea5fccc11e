// C-ABI of libsws (include/sws.h): context, workspace and the call sequences of
// sws_residual (steps a0-a9) and sws_jv_batch (step a10).  Host code only; the kernels
// live in sws_fields.cu and sws_allpairs.cu.  No CPU fallback anywhere: without a CUDA
// device sws_setup fails with SWS_ECUDA.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "sws_const.cuh"
#include "sws_internal.cuh"

static thread_local char g_cuda_err[256] = "";

static int cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s", where, cudaGetErrorString(e));
  return SWS_ECUDA;
}

#define CK(call)                                              \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);       \
  } while (0)

// Every entry point runs on the context's device and puts the caller's current device back on return
// (a multi-GPU PyTorch process keeps its own notion of the current device).
struct DevGuard {
  int prev = -1;
  cudaError_t err;
  explicit DevGuard(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
    else prev = -1;
  }
  ~DevGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};
#define ON_DEVICE(dev)  \
  DevGuard dev_guard_(dev); \
  CK(dev_guard_.err)

template <typename T>
static cudaError_t dev_alloc(T** p, size_t count, size_t* total) {
  size_t bytes = count * sizeof(T);
  if (bytes == 0) bytes = sizeof(T);
  *total += bytes;
  return cudaMalloc((void**)p, bytes);
}

static void free_all(sws_ctx* c) {
  void* ptrs[] = {c->x, c->y, c->sp_cp, c->sp_inv, c->zeta, c->phi, c->zx, c->px, c->zy, c->py,
                  c->src, c->srcf, c->tgt, c->e2loc, c->tile_count, c->part, c->F0, c->Fpert, c->sigma, c->norm_part,
                  c->dsrc, c->dtgt, c->e2lin, c->tgtI, c->lin_sums, c->acc_c, c->part_c, c->cnt_c,
                  c->u_stage, c->V_stage, c->out_stage};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  if (c->ev0) cudaEventDestroy(c->ev0);
  if (c->ev1) cudaEventDestroy(c->ev1);
  if (c->prof_events) {
    for (cudaEvent_t ev : *c->prof_events) cudaEventDestroy(ev);
    delete c->prof_events;
  }
}

extern "C" {

const char* sws_strerror(int code) {
  switch (code) {
    case SWS_OK: return "ok";
    case SWS_EINVAL: return "invalid argument";
    case SWS_ENOMEM: return "out of memory";
    case SWS_ECUDA: return "CUDA runtime error (see sws_last_cuda_error)";
    case SWS_EBATCH: return "batch size out of range";
    case SWS_ESTATE: return "no valid linearisation / evaluated state in the context (call sws_linearize, resp. sws_residual, first)";
    default: return "unknown error";
  }
}

const char* sws_last_cuda_error(void) { return g_cuda_err; }

int sws_setup(const sws_params* p, sws_ctx** out) {
  if (!p || !out) return SWS_EINVAL;
  *out = nullptr;
  if (p->N < 3 || p->M < 4 || !(p->dx > 0) || !(p->dy > 0) || !(p->froude > 0)) return SWS_EINVAL;
  if (!(p->y1 >= 0.0)) return SWS_EINVAL;  // eq. (12) integrates over the half plane y >= 0 and adds the images
  if (p->dy_scheme != 0 && p->dy_scheme != 1) return SWS_EINVAL;
  if (p->precision != 0 && p->precision != 1) return SWS_EINVAL;
  if (p->max_batch < 0 || p->max_batch > 1024) return SWS_EINVAL;
  if ((long long)p->N * p->M > (1ll << 30)) return SWS_EINVAL;
  if (p->M > 65535) return SWS_EINVAL;  // the O(NM) kernels put the y-line index on gridDim.y
  if (sws::reconstruct_smem_bytes(p->N) > 200 * 1024) return SWS_EINVAL;  // N <= 6400

  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (p->device < 0 || p->device >= ndev) return SWS_EINVAL;
  ON_DEVICE(p->device);

  sws_ctx* c = new (std::nothrow) sws_ctx();
  if (!c) return SWS_ENOMEM;
  memset(c, 0, sizeof *c);
  c->em_radius = sws::kEmRadius;  // far-field radius of the S2 column sums (sws_allpairs.cu, sws_set_farfield)
  c->params = *p;
  c->device = p->device;
  sws::Mesh& m = c->mesh;
  m.N = p->N; m.M = p->M;
  m.T = (p->N - 1) * p->M; m.S = p->N * p->M; m.n = 2 * (p->N + 1) * p->M;
  m.x1 = p->x1; m.y1 = p->y1; m.dx = p->dx; m.dy = p->dy;
  m.froude = p->froude; m.eps = p->eps; m.n_rad = p->n_rad;
  m.dy_scheme = p->dy_scheme;
  m.sym_first = (p->y1 == 0.0) ? 1 : 0;
  c->max_states = p->max_batch + 1;

  cudaDeviceProp prop;
  cudaError_t e = cudaGetDeviceProperties(&prop, p->device);
  if (e != cudaSuccess) { delete c; return cuda_fail(e, "cudaGetDeviceProperties"); }
  c->sm_count = prop.multiProcessorCount;

  e = p->precision == 1 ? sws::allpairs_f32_configure(&c->pair_occ) : sws::allpairs_configure(c, &c->pair_occ);
  if (e == cudaSuccess) e = sws::fields_configure(c);
  if (e == cudaSuccess) e = sws::fused_configure(c);
  if (e == cudaSuccess && p->max_batch > 0) e = sws::lin_configure(c);
  if (e != cudaSuccess) { delete c; return cuda_fail(e, "kernel configuration (is this an sm_100 device?)"); }

  // workspace
  const size_t S = m.S, T = m.T, n = m.n, st = c->max_states, mb = p->max_batch;
  // partial sums: [state][chunk][t]; capacity for the automatic plan, or 32 groups if more
  // (room for sws_set_tuning experiments), never more than the mesh allows
  int part_chunks = sws::make_plan(c).chunks;
  if (part_chunks < 32) part_chunks = 32;
  if (part_chunks > sws::max_chunks(c)) part_chunks = sws::max_chunks(c);
  if (part_chunks < sws::make_plan(c).chunks) part_chunks = sws::make_plan(c).chunks;
  c->part_chunks = part_chunks;
  c->part_rows = (size_t)part_chunks * c->max_states;
  int lin_bt = 0, lin_groups = 0;
  if (p->max_batch > 0) {
    // the analytic Jacobian action keeps [group][chunk][6 + BT] rows per target in `part`
    lin_bt = sws::lin_tile(p->max_batch);
    lin_groups = (p->max_batch + lin_bt - 1) / lin_bt;
    int lin_chunks = sws::max_chunks(c) < 32 ? sws::max_chunks(c) : 32;
    const size_t need = (size_t)lin_chunks * (6 + lin_bt) * lin_groups;
    if (need > c->part_rows) c->part_rows = need;
  }
  const size_t part_elems = c->part_rows * T;
  size_t tot = 0;
  bool ok = true;
#define ALLOC(ptr, count) ok = ok && (dev_alloc(&c->ptr, (count), &tot) == cudaSuccess)
  ALLOC(x, (size_t)m.N + 2);
  ALLOC(y, (size_t)m.M + 2);
  ALLOC(sp_cp, (size_t)m.M);
  ALLOC(sp_inv, (size_t)m.M);
  ALLOC(zeta, st * S); ALLOC(phi, st * S); ALLOC(zx, st * S);
  ALLOC(px, st * S); ALLOC(zy, st * S); ALLOC(py, st * S);
  ALLOC(src, st * S);
  if (p->precision == 1) ALLOC(srcf, st * S);
  ALLOC(tgt, st * T);
  ALLOC(e2loc, st * T);
  ALLOC(tile_count, st * ((T + 63) / 64));
  ALLOC(part, part_elems);
  ALLOC(F0, n);
  ALLOC(Fpert, mb * n);
  ALLOC(sigma, mb);
  ALLOC(norm_part, st * sws::kNormBlocks);
  ALLOC(u_stage, n);
  ALLOC(V_stage, mb * n);
  ALLOC(out_stage, (2 * mb + 1) * n);
  c->const_mode = -1;
  if (p->precision == 0 && sws::const_slab_cols(m.M) >= sws::kConstMinCols) {  // uniform-operand all-pairs path
    ALLOC(acc_c, (size_t)sws::kConstBanks * st * T);
    ALLOC(part_c, (size_t)sws::kConstBanks * sws::kConstMaxCols * T);
    ALLOC(cnt_c, (size_t)sws::kConstBanks * ((T + sws::kConstThreads - 1) / sws::kConstThreads));
  }
  if (mb > 0) {
    ALLOC(dsrc, (size_t)lin_groups * lin_bt * S);
    ALLOC(dtgt, mb * T);
    ALLOC(e2lin, mb * T);
    ALLOC(tgtI, T);
    ALLOC(lin_sums, 6 * T);
  }
#undef ALLOC
  if (!ok) {
    cudaGetLastError();
    free_all(c);
    delete c;
    return SWS_ENOMEM;
  }
  c->ws_bytes = tot;

  // mesh (L145): x_k = x_1 + (k-1) dx, y_l = y_1 + (l-1) dy, in FP64
  std::vector<double> hx(m.N + 2, 0.0), hy(m.M + 2, 0.0), cp(m.M, 0.0), inv(m.M, 0.0);
  for (int k = 0; k < m.N; ++k) hx[k] = p->x1 + (double)k * p->dx;
  for (int l = 0; l < m.M; ++l) hy[l] = p->y1 + (double)l * p->dy;
  // Thomas factors of the spline system (see k_dy): rows (a_l, b_l, c_l)
  {
    const int M = m.M;
    const double c0 = m.sym_first ? 0.0 : 2.0;  // first row: m_1 = 0, or m_1 + 2 m_2 = ...
    inv[0] = 1.0;
    cp[0] = c0;
    for (int l = 1; l < M; ++l) {
      const double a = (l == M - 1) ? 2.0 : 1.0, b = (l == M - 1) ? 1.0 : 4.0,
                   cc = (l == M - 1) ? 0.0 : 1.0;
      const double den = b - a * cp[l - 1];
      inv[l] = 1.0 / den;
      cp[l] = cc / den;
    }
  }
  e = cudaMemcpy(c->x, hx.data(), hx.size() * 8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(c->y, hy.data(), hy.size() * 8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(c->sp_cp, cp.data(), cp.size() * 8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(c->sp_inv, inv.data(), inv.size() * 8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemset(c->tile_count, 0, st * ((T + 63) / 64) * sizeof(unsigned int));
  if (e == cudaSuccess && c->cnt_c)
    e = cudaMemset(c->cnt_c, 0, (size_t)sws::kConstBanks * ((T + sws::kConstThreads - 1) / sws::kConstThreads) * sizeof(unsigned int));
  if (e == cudaSuccess && c->dsrc)  // unused direction slots of the last tile stay zero
    e = cudaMemset(c->dsrc, 0, (size_t)lin_groups * lin_bt * S * sizeof(double4));
  if (e == cudaSuccess && c->acc_c) e = sws::const_path_prepare(c->device);  // streams, events, bank addresses
  if (e == cudaSuccess) e = cudaEventCreate(&c->ev0);
  if (e == cudaSuccess) e = cudaEventCreate(&c->ev1);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  if (e != cudaSuccess) {
    free_all(c);
    delete c;
    return cuda_fail(e, "sws_setup upload");
  }
  *out = c;
  return SWS_OK;
}

int sws_destroy(sws_ctx* c) {
  if (!c) return SWS_EINVAL;
  ON_DEVICE(c->device);
  cudaDeviceSynchronize();
  free_all(c);
  delete c;
  return SWS_OK;
}

size_t sws_num_unknowns(const sws_ctx* c) { return c ? (size_t)c->mesh.n : 0; }
size_t sws_num_targets(const sws_ctx* c) { return c ? (size_t)c->mesh.T : 0; }
size_t sws_num_sources(const sws_ctx* c) { return c ? (size_t)c->mesh.S : 0; }
size_t sws_workspace_bytes(const sws_ctx* c) { return c ? c->ws_bytes : 0; }
int sws_get_params(const sws_ctx* c, sws_params* out) {
  if (!c || !out) return SWS_EINVAL;
  *out = c->params;
  return SWS_OK;
}

int sws_get_fields_host(sws_ctx* c, double* zeta_host, double* phi_host, double* zeta_y_host, double* phi_y_host,
                        void* cuda_stream) {
  if (!c) return SWS_EINVAL;
  if (c->last_states < 1) return SWS_ESTATE;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t nb = (size_t)c->mesh.S * sizeof(double);  // state 0 of each plane, [l][k]
  if (zeta_host) CK(cudaMemcpyAsync(zeta_host, c->zeta, nb, cudaMemcpyDeviceToHost, st));
  if (phi_host) CK(cudaMemcpyAsync(phi_host, c->phi, nb, cudaMemcpyDeviceToHost, st));
  if (zeta_y_host) CK(cudaMemcpyAsync(zeta_y_host, c->zy, nb, cudaMemcpyDeviceToHost, st));
  if (phi_y_host) CK(cudaMemcpyAsync(phi_y_host, c->py, nb, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return SWS_OK;
}

int sws_set_const_path(sws_ctx* c, int32_t mode) {
  if (!c || mode < -1 || mode > 1) return SWS_EINVAL;
  if (mode == 1 && !c->acc_c) return SWS_EINVAL;  // a source column does not fit a constant bank (or precision = 1)
  c->const_mode = mode;
  return SWS_OK;
}

int sws_set_eps(sws_ctx* c, double eps) {
  if (!c || eps != eps) return SWS_EINVAL;
  c->params.eps = eps;
  c->mesh.eps = eps;   // kernels take the mesh by value at launch
  c->lin_valid = 0;    // a kept linearisation belongs to the old source strength
  return SWS_OK;
}

int sws_set_farfield(sws_ctx* c, double radius_in_dy) {
  if (!c || radius_in_dy != radius_in_dy) return SWS_EINVAL;
  if (radius_in_dy > 0.0 && radius_in_dy < 6.0) return SWS_EINVAL;  // the expansion is not accurate there
  c->em_radius = radius_in_dy;
  return SWS_OK;
}

// While profiling is on: take the next (before, after) event pair and record `before`.
static int prof_begin(sws_ctx* c, cudaStream_t st, cudaEvent_t* pe0, cudaEvent_t* pe1) {
  *pe0 = *pe1 = nullptr;
  if (!c->profiling) return SWS_OK;
  if (!c->prof_events) c->prof_events = new (std::nothrow) std::vector<cudaEvent_t>();
  if (!c->prof_events) return SWS_ENOMEM;
  while (c->prof_events->size() < c->prof_used + 2) {
    cudaEvent_t ev;
    CK(cudaEventCreate(&ev));
    c->prof_events->push_back(ev);
  }
  *pe0 = (*c->prof_events)[c->prof_used];
  *pe1 = (*c->prof_events)[c->prof_used + 1];
  c->prof_used += 2;
  CK(cudaEventRecord(*pe0, st));
  return SWS_OK;
}

// a0-a9 for `states` states (state 0 = u, state s = u + sigma_{s-1} v_{s-1}).
static int run_states(sws_ctx* c, const double* u, const double* V, int states, double* F0,
                      double* Fpert, cudaStream_t st, int* launches) {
  const sws::PairPlan plan = sws::make_plan(c);
  if (c->fused_grid > 0) {  // the three O(NM) stages as phases of one cooperative launch
    CK(sws::launch_fields_fused(c, u, V, states, F0, Fpert, st));
    *launches += 1;
  } else {
    CK(sws::launch_reconstruct(c, u, V, states, 0, F0, Fpert, st));
    CK(sws::launch_dy(c, states, st));
    CK(sws::launch_targets(c, states, F0, Fpert, nullptr, st));
    *launches += 3;
  }
  cudaEvent_t pe0 = nullptr, pe1 = nullptr;
  int rc = prof_begin(c, st, &pe0, &pe1);
  if (rc != SWS_OK) return rc;
  if (sws::const_path_active(c)) {  // source data in uniform registers: one launch per slab of columns, two banks
    CK(sws::launch_allpairs_const(c, states, st, F0, Fpert, launches));
    if (pe1) CK(cudaEventRecord(pe1, st));
  } else if (c->params.precision == 0) {  // the FP64 kernel assembles E2 itself (last CTA of each target tile)
    CK(sws::launch_allpairs(c, states, plan, st, F0, Fpert));
    if (pe1) CK(cudaEventRecord(pe1, st));
    *launches += 1;
  } else {
    CK(sws::launch_allpairs(c, states, plan, st));
    if (pe1) CK(cudaEventRecord(pe1, st));
    CK(sws::launch_assemble(c, states, plan, F0, Fpert, st));
    *launches += 2;
  }
  c->last_states = states;
  c->last_lin_b = 0;
  c->lin_valid = 0;
  return SWS_OK;
}

int sws_residual(sws_ctx* c, const double* u_dev, double* F_dev, void* cuda_stream) {
  if (!c || !u_dev || !F_dev) return SWS_EINVAL;
  ON_DEVICE(c->device);
  int launches = 0;
  int rc = run_states(c, u_dev, nullptr, 1, F_dev, nullptr, (cudaStream_t)cuda_stream, &launches);
  c->last_launches = launches;
  return rc;
}

int sws_jv_batch(sws_ctx* c, const double* u_dev, const double* V_dev, int32_t b,
                 const double* sigma_host, double* JV_dev, double* Fpert_dev, double* F0_dev,
                 void* cuda_stream) {
  if (!c || !u_dev || !V_dev || !JV_dev) return SWS_EINVAL;
  if (b < 1 || b > c->params.max_batch) return SWS_EBATCH;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int launches = 0;
  if (sigma_host) {
    for (int i = 0; i < b; ++i)  // 0 is allowed (a zero direction: JV row = 0); NaN / inf are not
      if (!isfinite(sigma_host[i])) return SWS_EINVAL;
    CK(cudaMemcpyAsync(c->sigma, sigma_host, (size_t)b * sizeof(double), cudaMemcpyHostToDevice, st));
  } else {
    CK(sws::launch_sigma(c, u_dev, V_dev, b, st));
    launches += 2;
  }
  double* F0 = F0_dev ? F0_dev : c->F0;
  double* Fp = Fpert_dev ? Fpert_dev : c->Fpert;
  int rc = run_states(c, u_dev, V_dev, b + 1, F0, Fp, st, &launches);
  if (rc != SWS_OK) return rc;
  CK(sws::launch_jv_quotient(c, F0, Fp, b, JV_dev, st));
  launches += 1;
  c->last_launches = launches;
  return SWS_OK;
}

int sws_jv_exact_batch(sws_ctx* c, const double* u_dev, const double* V_dev, int32_t b, double* JV_dev,
                       void* cuda_stream) {
  if (!c || !u_dev || !V_dev || !JV_dev) return SWS_EINVAL;
  if (b < 1 || b > c->params.max_batch) return SWS_EBATCH;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int BT = sws::lin_tile(b), groups = (b + BT - 1) / BT;
  const sws::PairPlan plan = sws::make_lin_plan(c, BT, groups, 0);
  // derivative fields of every direction (states 1..b) beside the base fields (state 0);
  // the derivative radiation rows go straight to JV, the base rows to scratch
  CK(sws::launch_reconstruct(c, u_dev, V_dev, b + 1, 1, c->F0, JV_dev, st));
  CK(sws::launch_dy(c, b + 1, st));
  CK(sws::launch_targets(c, 1, c->F0, nullptr, c->tgtI, st));
  CK(sws::launch_targets_lin(c, b, BT, JV_dev, st));
  cudaEvent_t pe0 = nullptr, pe1 = nullptr;
  int rc = prof_begin(c, st, &pe0, &pe1);
  if (rc != SWS_OK) return rc;
  CK(sws::launch_allpairs_lin(c, BT, groups, 0, plan, st));
  if (pe1) CK(cudaEventRecord(pe1, st));
  CK(sws::launch_assemble_lin(c, b, BT, 0, plan, JV_dev, st));
  c->last_launches = 6;
  c->last_states = 1;
  c->last_lin_b = b;
  c->lin_valid = 0;  // the base planes now describe this u, but lin_sums does not
  return SWS_OK;
}

// Linearise once, apply many times (the shape of a Newton-Krylov step): everything that depends
// on u alone - base fields, starred values, {I, dI/dA, dI/dB, dI/dC}, and the six
// direction-independent all-pairs sums - is formed here and kept until the next call that
// overwrites the base state.
int sws_linearize(sws_ctx* c, const double* u_dev, void* cuda_stream) {
  if (!c || !u_dev) return SWS_EINVAL;
  if (c->params.max_batch < 1) return SWS_EBATCH;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const sws::PairPlan plan = sws::make_lin_plan(c, 1, 1, 1);
  CK(sws::launch_reconstruct(c, u_dev, nullptr, 1, 1, c->F0, nullptr, st));
  CK(sws::launch_dy(c, 1, st));
  CK(sws::launch_targets(c, 1, c->F0, nullptr, c->tgtI, st));
  cudaEvent_t pe0 = nullptr, pe1 = nullptr;
  int rc = prof_begin(c, st, &pe0, &pe1);
  if (rc != SWS_OK) return rc;
  CK(sws::launch_allpairs_lin(c, 1, 1, 1, plan, st));
  if (pe1) CK(cudaEventRecord(pe1, st));
  CK(sws::launch_reduce_base(c, plan, st));
  c->last_launches = 5;
  c->last_states = 1;
  c->last_lin_b = 0;
  c->lin_valid = 1;
  return SWS_OK;
}

int sws_jv_apply(sws_ctx* c, const double* V_dev, int32_t b, double* JV_dev, void* cuda_stream) {
  if (!c || !V_dev || !JV_dev) return SWS_EINVAL;
  if (b < 1 || b > c->params.max_batch) return SWS_EBATCH;
  if (!c->lin_valid) return SWS_ESTATE;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int BT = sws::lin_tile(b), groups = (b + BT - 1) / BT;
  const sws::PairPlan plan = sws::make_lin_plan(c, BT, groups, 2);
  // directions only: states 1..b of the planes; the base state (state 0) stays as linearised
  CK(sws::launch_reconstruct(c, nullptr, V_dev, b + 1, 1, c->F0, JV_dev, st, 1));
  CK(sws::launch_dy(c, b + 1, st, 1));
  CK(sws::launch_targets_lin(c, b, BT, JV_dev, st));
  cudaEvent_t pe0 = nullptr, pe1 = nullptr;
  int rc = prof_begin(c, st, &pe0, &pe1);
  if (rc != SWS_OK) return rc;
  CK(sws::launch_allpairs_lin(c, BT, groups, 2, plan, st));
  if (pe1) CK(cudaEventRecord(pe1, st));
  CK(sws::launch_assemble_lin(c, b, BT, 2, plan, JV_dev, st));
  c->last_launches = 5;
  c->last_lin_b = -b;  // direction fields of an apply (sws_time_allpairs_lin replays mode 2)
  return SWS_OK;
}

int sws_jv_exact_batch_host(sws_ctx* c, const double* u_host, const double* V_host, int32_t b,
                            double* JV_host, void* cuda_stream) {
  if (!c || !u_host || !V_host || !JV_host) return SWS_EINVAL;
  if (b < 1 || b > c->params.max_batch) return SWS_EBATCH;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t nb = (size_t)c->mesh.n * sizeof(double);
  CK(cudaMemcpyAsync(c->u_stage, u_host, nb, cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(c->V_stage, V_host, nb * b, cudaMemcpyHostToDevice, st));
  int rc = sws_jv_exact_batch(c, c->u_stage, c->V_stage, b, c->out_stage, cuda_stream);
  if (rc != SWS_OK) return rc;
  CK(cudaMemcpyAsync(JV_host, c->out_stage, nb * b, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return SWS_OK;
}

int sws_residual_host(sws_ctx* c, const double* u_host, double* F_host, void* cuda_stream) {
  if (!c || !u_host || !F_host) return SWS_EINVAL;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t nb = (size_t)c->mesh.n * sizeof(double);
  CK(cudaMemcpyAsync(c->u_stage, u_host, nb, cudaMemcpyHostToDevice, st));
  int rc = sws_residual(c, c->u_stage, c->out_stage, cuda_stream);
  if (rc != SWS_OK) return rc;
  CK(cudaMemcpyAsync(F_host, c->out_stage, nb, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return SWS_OK;
}

int sws_jv_batch_host(sws_ctx* c, const double* u_host, const double* V_host, int32_t b,
                      const double* sigma_host, double* JV_host, double* Fpert_host,
                      double* F0_host, void* cuda_stream) {
  if (!c || !u_host || !V_host || !JV_host) return SWS_EINVAL;
  if (b < 1 || b > c->params.max_batch) return SWS_EBATCH;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t n = c->mesh.n, nb = n * sizeof(double);
  CK(cudaMemcpyAsync(c->u_stage, u_host, nb, cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(c->V_stage, V_host, nb * b, cudaMemcpyHostToDevice, st));
  double* JV = c->out_stage;                              // [b][n]
  double* Fp = c->out_stage + (size_t)b * n;              // [b][n]
  double* F0 = c->out_stage + (size_t)2 * b * n;          // [n]
  int rc = sws_jv_batch(c, c->u_stage, c->V_stage, b, sigma_host, JV, Fp, F0, cuda_stream);
  if (rc != SWS_OK) return rc;
  CK(cudaMemcpyAsync(JV_host, JV, nb * b, cudaMemcpyDeviceToHost, st));
  if (Fpert_host) CK(cudaMemcpyAsync(Fpert_host, Fp, nb * b, cudaMemcpyDeviceToHost, st));
  if (F0_host) CK(cudaMemcpyAsync(F0_host, F0, nb, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return SWS_OK;
}

int sws_last_sigma(sws_ctx* c, int32_t b, double* sigma_host_out, void* cuda_stream) {
  if (!c || !sigma_host_out) return SWS_EINVAL;
  if (b < 1 || b > c->params.max_batch) return SWS_EBATCH;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CK(cudaMemcpyAsync(sigma_host_out, c->sigma, (size_t)b * sizeof(double), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return SWS_OK;
}

}  // extern "C"
