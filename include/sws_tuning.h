/*
 * sws_tuning.h -- timing, profiling and launch-shape calls of libsws_tuning.so.
 *
 * NOT part of the boundary.  include/sws.h (libsws.so) is the C-ABI of the hot path; the calls below exist for
 * `bench.py --experiments`, for the ncu captures under profiles/ and for the tests that assert which launch shape
 * ran.  They act on an sws_ctx created by sws_setup (libsws.so, which this library links against) and change no
 * result: every knob here selects between launch shapes whose outputs agree bit for bit or to summation round-off,
 * as stated per call.  A production caller needs none of them.
 */
#ifndef SWS_TUNING_H_
#define SWS_TUNING_H_

#include "sws.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of kernels the last sws_residual / sws_jv_batch call launched. */
int sws_last_launch_count(const sws_ctx* ctx);

/* Time (ms, CUDA events on `cuda_stream`) of the all-pairs phase alone for `states`
 * states (1 = single residual) using the fields left by the previous call: one launch of the staged
 * kernel, or the slab launches of the constant-bank path (sws_set_const_path) without the finishing
 * kernel; used by bench.py --experiments.  Synchronises. */
int sws_time_allpairs(sws_ctx* ctx, int32_t states, int32_t reps, float* ms_per_launch,
                      void* cuda_stream);

/* Time (ms per call, CUDA events on `cuda_stream`) of `reps` back-to-back sws_residual calls issued from
 * inside the library (no binding overhead between the calls): what a compiled driver such as
 * libsws_jfnk sees on small meshes, where an evaluation takes tens of microseconds.  Synchronises. */
int sws_time_residual(sws_ctx* ctx, const double* u_dev, double* F_dev, int32_t reps, float* ms_per_call,
                      void* cuda_stream);

/* Steps a0-a3, a5-a8 run as ONE cooperative launch on meshes of up to 2^17 nodes (three phases separated by
 * grid-wide barriers) and as three launches above that.  on = 0 forces the three launches; on != 0 restores
 * the default choice.  Results do not depend on it (the phases call the same device functions). */
int sws_set_fused_fields(sws_ctx* ctx, int32_t on);

/* sws_time_allpairs for the all-pairs kernel of the analytic Jacobian action, with the fields and the batch size
 * of the previous sws_jv_exact_batch / sws_jv_apply call (SWS_EBATCH if there was none). */
int sws_time_allpairs_lin(sws_ctx* ctx, int32_t reps, float* ms_per_launch, void* cuda_stream);

/* Launch geometry of that kernel for b directions: out6 = {target tiles, column groups, columns
 * per group, nodes staged per bulk copy, segments per column, directions per tile}. */
int sws_lin_plan_info(sws_ctx* ctx, int32_t b, int32_t* out6);

/* Live timing of the dominant kernel inside ordinary calls.  While profiling is on, every
 * sws_residual / sws_jv_batch / sws_jv_exact_batch brackets its all-pairs phase (one launch of the staged kernel, or
 * the slab launches of the constant-bank path with their fork / join) with a CUDA event pair on the
 * call's stream (no synchronisation, two event records per call).  sws_profile_read
 * synchronises those events and returns the summed all-pairs time (ms) and the number of
 * phases since the last reset; reset != 0 clears the list. */
int sws_set_profiling(sws_ctx* ctx, int32_t on);
int sws_profile_read(sws_ctx* ctx, double* allpairs_ms, int32_t* launches, int32_t reset);

/* Tuning knob of the STAGED all-pairs launch: number of source-column groups a target tile's
 * quadrature is split into (0 = library default, chosen from the SM count and occupancy;
 * clamped to what the workspace was sized for).  The constant-bank path ignores it. */
int sws_set_tuning(sws_ctx* ctx, int32_t chunks);

/* Batched all-pairs launches (sws_jv_batch) let one CTA carry `ns` states: the y_j run is staged once and
 * y_j - y* is formed once per (target, node) for the ns states (north_star: "a batched mode that shares each
 * staged source tile across b perturbed states" - what the states share is the mesh geometry; the source
 * records differ).  ns = 1: one state per CTA, states on the grid's z axis; 2: two states per CTA; 0 = library
 * default (1: measured 4-5 % faster than 2 on B200).  Results do not depend on ns, bit for bit. */
int sws_set_states_per_cta(sws_ctx* ctx, int32_t ns);

/* out = {path active for this context now (0/1), columns per slab, slabs per state, target tiles (CTAs per column)} */
int sws_const_plan_info(const sws_ctx* ctx, int32_t out[4]);

/* Fraction of (warp, source column) combinations of the first `states` states of the last call
 * that take the direct S2 loop (bench.py: executed FP64 work of a launch).  Synchronises. */
int sws_farfield_stats(sws_ctx* ctx, int32_t states, double* near_fraction, void* cuda_stream);

/* The all-pairs launch geometry for `states` states: out5 = {target tiles, column groups,
 * columns per group, nodes staged per bulk copy, segments per column}. */
int sws_plan_info(sws_ctx* ctx, int32_t states, int32_t* out5);

/* This thread's message for the last SWS_ECUDA one of the calls above returned. */
const char* sws_tuning_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SWS_TUNING_H_ */
