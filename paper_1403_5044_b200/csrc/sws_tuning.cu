// Timing, profiling and launch-shape calls of include/sws_tuning.h -> libsws_tuning.so.  They exist for bench.py
// --experiments, the profiles under profiles/ and the tests that assert which launch shape ran; none of them is part
// of the boundary (include/sws.h), and the product library exports none of them.  This library links against
// libsws.so and reaches the context and the launchers through the internal header.
#include <stdio.h>

#include <new>
#include <vector>

#include "sws_const.cuh"
#include "sws_internal.cuh"
#include "sws_tuning.h"

static thread_local char g_tuning_err[256] = "";

static int cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_tuning_err, sizeof g_tuning_err, "%s: %s", where, cudaGetErrorString(e));
  return SWS_ECUDA;
}

#define CK(call)                                              \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);       \
  } while (0)

// run on the context's device, put the caller's current device back on return
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

extern "C" {

const char* sws_tuning_last_cuda_error(void) { return g_tuning_err; }

int sws_last_launch_count(const sws_ctx* c) { return c ? c->last_launches : 0; }

int sws_set_tuning(sws_ctx* c, int32_t chunks) {
  if (!c || chunks < 0) return SWS_EINVAL;
  if (chunks > c->part_chunks) chunks = c->part_chunks;  // the partial-sum buffer is sized at setup
  c->chunks_user = chunks;
  return SWS_OK;
}

int sws_const_plan_info(const sws_ctx* c, int32_t out[4]) {
  if (!c || !out) return SWS_EINVAL;
  const int cols = c->acc_c ? sws::const_slab_cols(c->mesh.M) : 0;
  out[0] = sws::const_path_active(c) ? 1 : 0;
  out[1] = cols;
  out[2] = cols > 0 ? (c->mesh.N + cols - 1) / cols : 0;
  out[3] = sws::const_tiles(c->mesh.N, c->mesh.M);
  return SWS_OK;
}

int sws_set_states_per_cta(sws_ctx* c, int32_t ns) {
  if (!c || ns < 0 || ns > 2) return SWS_EINVAL;
  c->ns_user = ns;
  return SWS_OK;
}

int sws_farfield_stats(sws_ctx* c, int32_t states, double* near_fraction, void* cuda_stream) {
  if (!c || !near_fraction) return SWS_EINVAL;
  if (states < 1 || states > c->max_states || states > c->last_states) return SWS_EBATCH;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int warps = sws::count_near_warps(c);
  const size_t cnt = (size_t)states * warps;
  int* d = nullptr;
  CK(cudaMalloc((void**)&d, cnt * sizeof(int)));
  std::vector<int> h(cnt);
  cudaError_t e = sws::launch_count_near(c, states, d, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(h.data(), d, cnt * sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d);
  CK(e);
  double near = 0.0;
  for (size_t i = 0; i < cnt; ++i) near += h[i];
  *near_fraction = near / ((double)cnt * c->mesh.N);
  return SWS_OK;
}

int sws_time_allpairs_lin(sws_ctx* c, int32_t reps, float* ms_per_launch, void* cuda_stream) {
  if (!c || !ms_per_launch || reps < 1) return SWS_EINVAL;
  if (c->last_lin_b == 0) return SWS_EBATCH;  // needs the fields of a previous sws_jv_exact_batch / sws_jv_apply
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int mode = c->last_lin_b < 0 ? 2 : 0;
  const int b = c->last_lin_b < 0 ? -c->last_lin_b : c->last_lin_b, BT = sws::lin_tile(b), groups = (b + BT - 1) / BT;
  const sws::PairPlan plan = sws::make_lin_plan(c, BT, groups, mode);
  CK(sws::launch_allpairs_lin(c, BT, groups, mode, plan, st));
  CK(cudaEventRecord(c->ev0, st));
  for (int r = 0; r < reps; ++r) CK(sws::launch_allpairs_lin(c, BT, groups, mode, plan, st));
  CK(cudaEventRecord(c->ev1, st));
  CK(cudaEventSynchronize(c->ev1));
  float ms = 0.f;
  CK(cudaEventElapsedTime(&ms, c->ev0, c->ev1));
  *ms_per_launch = ms / reps;
  return SWS_OK;
}

int sws_lin_plan_info(sws_ctx* c, int32_t b, int32_t* out6) {
  if (!c || !out6) return SWS_EINVAL;
  if (b < 1 || b > c->params.max_batch) return SWS_EBATCH;
  const int BT = sws::lin_tile(b), groups = (b + BT - 1) / BT;
  const sws::PairPlan p = sws::make_lin_plan(c, BT, groups, 0);
  out6[0] = p.tiles; out6[1] = p.chunks; out6[2] = p.cols_per_chunk; out6[3] = p.seg_len; out6[4] = p.nseg;
  out6[5] = BT;
  return SWS_OK;
}

int sws_time_allpairs(sws_ctx* c, int32_t states, int32_t reps, float* ms_per_launch,
                      void* cuda_stream) {
  if (!c || !ms_per_launch || reps < 1) return SWS_EINVAL;
  if (states < 1 || states > c->max_states || states > c->last_states) return SWS_EBATCH;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const sws::PairPlan plan = sws::make_plan(c);
  auto once = [&]() -> cudaError_t {
    return sws::const_path_active(c) ? sws::launch_allpairs_const(c, states, st, nullptr, nullptr, nullptr)
                                     : sws::launch_allpairs(c, states, plan, st);
  };
  CK(once());  // warm-up
  CK(cudaEventRecord(c->ev0, st));
  for (int r = 0; r < reps; ++r) CK(once());
  CK(cudaEventRecord(c->ev1, st));
  CK(cudaEventSynchronize(c->ev1));
  float ms = 0.f;
  CK(cudaEventElapsedTime(&ms, c->ev0, c->ev1));
  *ms_per_launch = ms / reps;
  return SWS_OK;
}

int sws_time_residual(sws_ctx* c, const double* u_dev, double* F_dev, int32_t reps, float* ms_per_call,
                      void* cuda_stream) {
  if (!c || !u_dev || !F_dev || !ms_per_call || reps < 1) return SWS_EINVAL;
  ON_DEVICE(c->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = sws_residual(c, u_dev, F_dev, cuda_stream);  // warm-up
  if (rc != SWS_OK) return rc;
  CK(cudaEventRecord(c->ev0, st));
  for (int r = 0; r < reps; ++r) {
    rc = sws_residual(c, u_dev, F_dev, cuda_stream);
    if (rc != SWS_OK) return rc;
  }
  CK(cudaEventRecord(c->ev1, st));
  CK(cudaEventSynchronize(c->ev1));
  float ms = 0.f;
  CK(cudaEventElapsedTime(&ms, c->ev0, c->ev1));
  *ms_per_call = ms / reps;
  return SWS_OK;
}

int sws_set_fused_fields(sws_ctx* c, int32_t on) {
  if (!c) return SWS_EINVAL;
  if (!on) {
    c->fused_grid = 0;
    return SWS_OK;
  }
  ON_DEVICE(c->device);
  CK(sws::fused_configure(c));
  return SWS_OK;
}

int sws_set_profiling(sws_ctx* c, int32_t on) {
  if (!c) return SWS_EINVAL;
  c->profiling = on ? 1 : 0;
  return SWS_OK;
}

int sws_profile_read(sws_ctx* c, double* allpairs_ms, int32_t* launches, int32_t reset) {
  if (!c || !allpairs_ms || !launches) return SWS_EINVAL;
  ON_DEVICE(c->device);
  double tot = 0.0;
  for (size_t i = 0; i + 1 < c->prof_used; i += 2) {
    float ms = 0.f;
    CK(cudaEventSynchronize((*c->prof_events)[i + 1]));
    CK(cudaEventElapsedTime(&ms, (*c->prof_events)[i], (*c->prof_events)[i + 1]));
    tot += ms;
  }
  *allpairs_ms = tot;
  *launches = (int32_t)(c->prof_used / 2);
  if (reset) c->prof_used = 0;
  return SWS_OK;
}

int sws_plan_info(sws_ctx* c, int32_t states, int32_t* out5) {
  if (!c || !out5 || states < 1 || states > c->max_states) return SWS_EINVAL;
  const sws::PairPlan p = sws::make_plan(c);
  out5[0] = p.tiles; out5[1] = p.chunks; out5[2] = p.cols_per_chunk; out5[3] = p.seg_len; out5[4] = p.nseg;
  return SWS_OK;
}

}  // extern "C"
