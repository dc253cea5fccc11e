/*
 * sws.h -- C-ABI of libsws: the nonlinear residual E(u) (called F(u) in
 * BASELINE.json) of the boundary-integral discretisation of steady free-surface
 * flow past a submerged source, and batched finite-difference Jacobian-vector
 * products, on one NVIDIA B200 (sm_100a), in FP64.
 *
 * Paper: Pethiyagoda, McCue, Moroney & Back, "Jacobian-free Newton-Krylov
 * methods with GPU acceleration for computing nonlinear ship wave patterns",
 * arXiv 1403.5044.  Citations "L<n>" are lines of /root/reference/PAPER.md.
 *
 * What the path computes (section 3, App. A):
 *   u in R^{2(N+1)M}, eq. (18): per y-line l = 1..M the block
 *       [phi_{1,l}, (phi_x)_{1,l} .. (phi_x)_{N,l}], all lines; then the same for zeta.
 *   E in R^{2(N+1)M}, App. A: per line l the block [E3_l, E4_l, E1_{1..N-1,l}],
 *       all lines; then [E5_l, E6_l, E2_{1..N-1,l}].
 *   a1  x-trapezoid reconstruction of zeta, phi                       eq. (19)
 *   a2  zeta_y, phi_y by a cubic spline along y on each x-line (L160);
 *       dy_scheme = 1 selects 2nd-order finite differences instead
 *   a3  half-mesh values by two-point interpolation                    L162, L454
 *   a4  all-pairs trapezoid quadrature of K1, K2 (L107, L109), each with its
 *       y -> -y image, with the S2 singularity subtraction             eqs. (20)-(22) L164-177
 *   a5  closed-form integral I of S2 over the truncated rectangle      eq. (23)
 *   a6  integral-equation rows E2                                      eq. (12)
 *   a7  Bernoulli rows E1                                              eq. (13)
 *   a8  upstream radiation rows E3..E6, n = n_rad                      eq. (24)
 *   a9  App. A ordering                                                L421
 *   a10 J v ~ (E(u + sigma v) - E(u)) / sigma, b directions at once    eq. (25)
 * Readings of the paper where it is silent or garbled are listed in DESIGN.md.
 *
 * Conventions
 *   - Every *_dev pointer is DEVICE memory owned by the caller (e.g. a PyTorch
 *     tensor's data_ptr()), FP64, contiguous; it is never retained after the call.
 *   - Every *_host pointer is HOST memory owned by the caller.
 *   - The context owns all workspace.  sws_residual / sws_jv_batch only enqueue
 *     work on `cuda_stream` (a cudaStream_t passed as void*; NULL = the legacy
 *     default stream) and return without synchronising and without allocating.
 *   - One context must not be used from two streams at the same time.
 *   - Results are deterministic: bitwise repeatable for fixed inputs and context.
 *   - Return value: SWS_OK (0) or a negative error code; nothing throws across the
 *     ABI.  There is no CPU fallback: without a CUDA device sws_setup fails with
 *     SWS_ECUDA.
 */
#ifndef SWS_H_
#define SWS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SWS_OK 0
#define SWS_EINVAL (-1) /* bad argument (NULL pointer, N < 3, M < 4, spacing <= 0, ...) */
#define SWS_ENOMEM (-2) /* device or host allocation failed                             */
#define SWS_ECUDA (-3)  /* a CUDA runtime call failed; see sws_last_cuda_error()         */
#define SWS_EBATCH (-4) /* b < 1 or b > max_batch                                        */
#define SWS_ESTATE (-5) /* sws_jv_apply without a valid sws_linearize                    */

typedef struct sws_ctx sws_ctx; /* opaque, owned by the library */

typedef struct {
  int32_t N, M;        /* mesh nodes in x and y (N >= 3, M >= 4)                       L145 */
  double x1, y1;       /* first node; x1 = upstream truncation; y1 >= 0 (half plane of eq. (12),
                          L101), configs use y1 = 0                                    L162 */
  double dx, dy;       /* spacings Delta x, Delta y (> 0)                              L145 */
  double froude, eps;  /* Froude number F, eq. (9); source strength eq. (6)         */
  double n_rad;        /* radiation exponent n, paper value 0.05                       L189 */
  int32_t dy_scheme;   /* 0 cubic spline (L160), 1 finite differences                       */
  int32_t precision;   /* 0 = FP64 pair arithmetic; 1 = FP32 pair arithmetic (reported only) */
  int32_t max_batch;   /* largest b accepted by sws_jv_batch (0 = residual only)            */
  int32_t device;      /* CUDA ordinal                                                      */
} sws_params;

/* Validate, allocate the workspace on p->device, precompute mesh and spline tables.
 * *out receives the context.  Synchronises the device once. */
int sws_setup(const sws_params* p, sws_ctx** out);

/* F_dev[0..n) = E(u_dev[0..n)), n = 2(N+1)M.  Steps a0-a9. */
int sws_residual(sws_ctx* ctx, const double* u_dev, double* F_dev, void* cuda_stream);

/* JV_dev[b][n] (row-major) = (E(u_b) - E(u)) / sigma_b with u_b = fma(sigma_b, v_b, u)
 * entry by entry in FP64, for the b rows v_b of V_dev[b][n].  Step a10, eq. (25) L219.
 *   sigma_host  [b] shifts in pageable host memory, read during the call; NULL selects
 *               sigma_b = 1e-7 (1 + ||u||_2) / ||v_b||_2 computed on the device.  A zero direction
 *               (||v_b|| = 0) gets sigma_b = 0, E(u_b) = E(u) and the exact row JV_b = 0; a caller's
 *               sigma_b = 0 means the same; NaN / inf shifts are refused (SWS_EINVAL).
 *   Fpert_dev   [b][n] or NULL; receives E(u_b).
 *   F0_dev      [n] or NULL; receives E(u) (the base evaluation the batch performs anyway).
 * Slot b is bitwise sws_residual(u_b) and F0 is bitwise sws_residual(u): what is guaranteed to
 * 1e-10 of |E|_inf against the oracle is each E(u_b) (reading Q9 (i)).  The QUOTIENT
 * inherits the cancellation of eq. (25): two independently rounded FP64 residuals differ by
 * ~1e-13 |E| before the division by sigma ~ 1e-7, so JV_b carries a relative rounding floor of
 * 1e-9 .. 1e-7 (measured <= 1e-5 of |JV|_inf against the long-double quotient at every config;
 * the oracle's own FP64 quotient has the same floor).  Callers who need products to <= 1e-10 use
 * sws_jv_exact_batch / sws_linearize + sws_jv_apply below, which form J(u) v without a difference. */
int sws_jv_batch(sws_ctx* ctx, const double* u_dev, const double* V_dev, int32_t b,
                 const double* sigma_host, double* JV_dev, double* Fpert_dev, double* F0_dev,
                 void* cuda_stream);

/* The analytic Jacobian action: JV_dev[b][n] = J(u) v_b with J = dE/du at
 * u_dev, i.e. the sigma -> 0 limit of eq. (25), every step a0-a9 of E differentiated by
 * hand: the reconstruction (19), the spline and the midpoint averages are linear; the Bernoulli
 * row (13), the source term, the closed form I (through A, B, C, L177) and the kernels K1, K2,
 * S2 (L107-109, L169-172) are linearised about u.  No shift, no difference of two residuals:
 * the result is accurate to summation round-off (~1e-13 of |JV|_inf), where the quotient of
 * sws_jv_batch carries eps_mach / sigma ~ 1e-9..1e-7.  The pair coefficients are computed once
 * per pair for all b directions ((71 + 4 b) FP64 instructions per pair instead of 45 (b + 1)).
 * V_dev [b][n] row-major, 1 <= b <= max_batch.  Deterministic.  E(u) itself is not formed. */
int sws_jv_exact_batch(sws_ctx* ctx, const double* u_dev, const double* V_dev, int32_t b,
                       double* JV_dev, void* cuda_stream);

/* The same action split for Newton-Krylov use, where many products share one u:
 *   sws_linearize(u)      forms everything that depends on u alone (base fields, starred values,
 *                         the closed form I and its A, B, C derivatives, and the six
 *                         direction-independent all-pairs sums) and keeps it in the context;
 *   sws_jv_apply(V[b])    JV_dev[b][n] = J(u) v_b for that u: (41 + 4 b) FP64 instructions per pair
 *                         (b = 1: the cost of one residual evaluation, with no shift and no
 *                         cancellation).
 * The linearisation stays valid until the next sws_residual / sws_jv_batch / sws_jv_exact_batch /
 * sws_linearize on the same context; sws_jv_apply returns SWS_ESTATE otherwise.  Results agree with
 * sws_jv_exact_batch to summation round-off (the column split of the quadrature differs). */
int sws_linearize(sws_ctx* ctx, const double* u_dev, void* cuda_stream);
int sws_jv_apply(sws_ctx* ctx, const double* V_dev, int32_t b, double* JV_dev, void* cuda_stream);

/* The same two calls on HOST buffers: host->device copy, compute, device->host copy,
 * then a stream synchronise.  `cuda_stream` as above. */
int sws_residual_host(sws_ctx* ctx, const double* u_host, double* F_host, void* cuda_stream);
int sws_jv_batch_host(sws_ctx* ctx, const double* u_host, const double* V_host, int32_t b,
                      const double* sigma_host, double* JV_host, double* Fpert_host,
                      double* F0_host, void* cuda_stream);

int sws_jv_exact_batch_host(sws_ctx* ctx, const double* u_host, const double* V_host, int32_t b,
                            double* JV_host, void* cuda_stream);

/* The shifts the last sws_jv_batch used (device-computed or copied), after a
 * synchronise of `cuda_stream`.  sigma_host_out has room for b values. */
int sws_last_sigma(sws_ctx* ctx, int32_t b, double* sigma_host_out, void* cuda_stream);

/* The nodal fields of the state the last sws_residual / sws_jv_batch / sws_linearize call left in the
 * workspace as state 0 (= its u): zeta, phi (eq. (19)) and zeta_y, phi_y (L160), each [M][N] row-major
 * (index l N + k) into HOST buffers; any pointer may be NULL.  Synchronises `cuda_stream`.  SWS_ESTATE if
 * no call has filled the workspace yet. */
int sws_get_fields_host(sws_ctx* ctx, double* zeta_host, double* phi_host, double* zeta_y_host,
                        double* phi_y_host, void* cuda_stream);

/* Copy of the parameters the context was set up with (max_batch and device included). */
int sws_get_params(const sws_ctx* ctx, sws_params* out);

size_t sws_num_unknowns(const sws_ctx* ctx); /* 2(N+1)M */
size_t sws_num_targets(const sws_ctx* ctx);  /* (N-1)M half-mesh points */
size_t sws_num_sources(const sws_ctx* ctx);  /* NM nodes */
size_t sws_workspace_bytes(const sws_ctx* ctx);

/* The uniform-operand ("constant-bank") form of the all-pairs quadrature, step a4 (eq. (12), same pair
 * arithmetic as the staged kernel): the source records of a slab of columns are copied into a 64 KB constant bank,
 * from where the kernel takes them as uniform-register operands of its FP64 instructions (DESIGN.md section 6:
 * no three-vector-register DFMAs on the source data, no shared-memory loads); one launch per slab, two banks fed
 * through two library-owned streams that fork from and join the caller's stream (asynchronous as before).
 * mode -1 (default): used on FP64 meshes with at least 16,000 targets whose columns fit a bank at least four at a
 * time (M <= 479); 0: never (always the staged kernel); 1: whenever the columns fit (SWS_EINVAL otherwise).
 * Results are bitwise repeatable in either form and slot b of a batch is bitwise the single evaluation of u_b;
 * the two forms differ from each other in summation order only (~1e-13 of |F|).  The two banks and streams belong to
 * the process (per device): calls of any number of contexts and host threads are serialised through them.  A call may
 * be captured into a CUDA graph after one eager call.  A captured call does not fork: it keeps the copies and launches
 * of both banks on the capturing stream, in the same slab order (bitwise the same result, no overlap between the
 * banks), so the library's own streams never become part of a caller's capture and eager calls of other host threads
 * and contexts proceed normally while a capture is open.  What remains the caller's duty: a REPLAY of such a graph must
 * not run concurrently with other calls of this library on the same device (the replayed copies into the banks are not
 * ordered against them); order them with an event, or use sws_set_const_path(ctx, 0) for contexts whose calls are
 * replayed from graphs next to eager work. */
int sws_set_const_path(sws_ctx* ctx, int32_t mode);

/* Change the source strength epsilon (eq. (6)) of an existing context: the parameter of the
 * bootstrapping / continuation process of L229.  Nothing else of the set-up depends on it.  A
 * linearisation kept by sws_linearize is invalidated. */
int sws_set_eps(sws_ctx* ctx, double eps);

/* Far-field evaluation of the S2 terms (sws_allpairs.cu).  For a source
 * column whose completed-square constant g of L169-177 satisfies sqrt(g) >= radius_in_dy * dy for
 * all 32 targets of a warp, the column's S2 trapezoid sum (which does not depend on the source
 * data) is replaced by its integral (asinh) plus 7 Euler-Maclaurin end corrections, exact to
 * < 1e-16 / sqrt(g) for radius >= 8; the K1 and K2 terms are always summed pair by pair.  The S2
 * sensitivity sums of sws_jv_exact_batch / sws_linearize and the FP32 variant switch the same way.
 * radius_in_dy <= 0 switches the expansion off (every S2 term summed directly, the plain
 * definition); 0 < radius < 6 is refused (SWS_EINVAL).  Default 8. */
int sws_set_farfield(sws_ctx* ctx, double radius_in_dy);

/* The shifts of eq. (25), sigma_b = 1e-7 (1 + ||u||_2) / ||v_b||_2 (0 for a zero direction), WITHOUT a context
 * and without any allocation: sigma_dev[r] for the b rows v_r of V_dev[b][n] (row-major), r = 0 .. b-1.  The values are
 * bitwise those sws_jv_batch(sigma_host = NULL) uses and sws_last_sigma reports.
 *
 * For callers that cannot allocate device memory where they need the shifts - a solver embedded in an application
 * that handed all device memory to its own pool at start-up (cudaMalloc fails there, or takes what the application
 * thinks it owns), or a continuation / time-stepping loop that cannot afford the device-wide stall of cudaMalloc and
 * cudaFree - and for Krylov drivers that want the shifts alone and no context (sws_setup allocates the whole
 * workspace).  The call itself never calls cudaMalloc, cudaFree or a library routine that allocates.
 *
 * Where the scratch memory is: the block partial sums of the two-stage 2-norm live in ONE fixed array inside the
 * library's device image, (SWS_NOALLOC_MAX_B + 1) x 64 doubles = 33,280 bytes.  Every GPU that loads libsws.so
 * holds that array until the process exits, whether this function is called or not.  Consequences:
 *   - b > SWS_NOALLOC_MAX_B is refused with SWS_EBATCH (split the batch); n must be 1 .. 2^31 - 1.
 *   - All calls on one device share the array.  It keeps the last call's contents; no slot is read before the same
 *     call has written it, so nothing needs clearing between calls.  Two calls whose kernels can OVERLAP on the GPU
 *     (different streams without an ordering between them, or two host threads) race on it and both results are
 *     undefined: order them with an event or keep them on one stream.  Calls on different devices do not interact.
 *   - The FIRST call on each device also asks the runtime for the array's device address (cudaGetSymbolAddress, once
 *     per device, kept for the life of the process).  Make that first call eagerly, before any stream capture begins.
 * u_dev [n], V_dev [b][n], sigma_dev [b]: device memory on `device`, owned by the caller, FP64.  Asynchronous on
 * `cuda_stream`; runs on `device` and restores the caller's current device.  Returns SWS_OK, SWS_EINVAL, SWS_EBATCH or
 * SWS_ECUDA; sws_noalloc_last_error() returns this thread's message for the last failed call ("" after a success). */
#define SWS_NOALLOC_MAX_B 64
int sws_fd_shifts_noalloc(const double* u_dev, const double* V_dev, int64_t n, int32_t b, double* sigma_dev,
                          int32_t device, void* cuda_stream);
const char* sws_noalloc_last_error(void);

int sws_destroy(sws_ctx* ctx);

const char* sws_strerror(int code);
const char* sws_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SWS_H_ */
