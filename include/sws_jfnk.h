/*
 * sws_jfnk.h -- C-ABI of libsws_jfnk: the preconditioned Jacobian-free Newton-Krylov driver
 * around libsws, device resident, one NVIDIA B200, FP64.
 *
 * Paper: Pethiyagoda, McCue, Moroney & Back, arXiv 1403.5044; "L<n>" = line n of
 * /root/reference/PAPER.md.
 *
 *   preconditioner  P = [A B; C D], the Jacobian of the LINEARISED problem (section 4.2,
 *                   App. B (B.1)-(B.6) L425-503), independent of u and of epsilon, with the
 *                   dense lower-right block D kept only within block bandwidth b (blocks
 *                   (N+1) x (N+1), L241).  Stored and applied by the block factorisation of
 *                   App. C:  t2 = b2 - C A^-1 b1,  s1 = A^-1 b1,
 *                   s2 = (D - C A^-1 B)^-1 t2,  r1 = s1 - A^-1 B s2,  r2 = s2,
 *                   with A tridiagonal, B and C applied matrix-free (prefix sums), and the
 *                   block-banded Schur complement S = D - C A^-1 B factorised once.
 *   GMRES           right preconditioned (section 4.1, Saad & Schultz [47]): the Newton
 *                   correction is sought in P^-1 K_m(J P^-1, E) (L213).  J v is libsws's
 *                   analytic Jacobian action (jv_mode 0) or the difference quotient (25) L219
 *                   (jv_mode 1).
 *   Newton          damped iteration (2), (3) L41-45 with a backtracking line search (L209).
 *
 * Conventions as in sws.h: *_dev = caller-owned DEVICE memory (FP64, contiguous), *_host =
 * caller-owned HOST memory; objects own their workspace; return SWS_OK or a negative SWS_E*
 * code (sws.h); nothing throws.  Unlike sws_residual these calls SYNCHRONISE: the drivers read
 * a few scalars (norms, Hessenberg columns) back every iteration; every vector stays on the
 * device.  Results are deterministic (fixed reduction orders, no atomics).
 * Library kernels used: cuSOLVER getrf/getrs and cuBLAS gemm/geam for the one-off block LU of
 * the Schur complement (plain dense linear algebra); everything applied per iteration is this
 * library's own kernels.
 */
#ifndef SWS_JFNK_H_
#define SWS_JFNK_H_

#include "sws.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sws_precond sws_precond; /* opaque */
typedef struct sws_solver sws_solver;   /* opaque */

/* Assemble the linear Jacobian of p's mesh (N, M, x1, y1, dx, dy, froude, n_rad; eps and the
 * y-derivative scheme do not enter, App. B) on p->device, truncate D to block bandwidth
 * `bandwidth` (odd; b = 1 block diagonal, 3 block tridiagonal, ...; <= 0 or >= 2M-1 keeps all
 * of D) and factorise.  flags bit 0: do NOT factorise (the blocks stay as assembled; only
 * sws_precond_block_host is then valid).  flags bit 1: store the factor panels in FP32 (the block LU itself
 * stays FP64; the apply streams half the bytes and accumulates in FP64; P^-1 v then carries a relative error of
 * ~1e-7 x the conditioning of the Schur complement instead of ~1e-16 x: enough for a preconditioner - the GMRES
 * iteration counts of the paper's meshes are unchanged, DESIGN.md - not for a direct solve).  Synchronises.
 * SWS_ENOMEM if the band does not fit. */
int sws_precond_create(const sws_params* p, int32_t bandwidth, int32_t flags, sws_precond** out);

/* r_dev[0..n) = P^-1 v_dev[0..n), n = 2(N+1)M, App. C L511-513.  v and r may alias.
 * Asynchronous on `cuda_stream`. */
int sws_precond_apply(sws_precond* pc, const double* v_dev, double* r_dev, void* cuda_stream);

/* The same for t vectors at once (1 <= t <= 16): R_dev[q][0..n) = P^-1 V_dev[q][0..n), both [t][n] row-major.
 * The block sweeps read every factor panel once for up to 16 vectors instead of once per vector (the
 * panels are what an apply streams from HBM).  Each vector's result agrees with sws_precond_apply to
 * summation round-off.  The first call with t > 1 grows the internal vectors (synchronises once). */
int sws_precond_apply_multi(sws_precond* pc, const double* V_dev, int32_t t, double* R_dev, void* cuda_stream);

/* Block (l, m) (0-based y-lines) of the ASSEMBLED matrices, (N+1) x (N+1) row-major into
 * out_host: which = 0: D block of (B.6) and the radiation rows E5, E6; which = 1: the Schur
 * complement block D - C A^-1 B.  Needs flags bit 0 at creation and |l - m| within the band. */
int sws_precond_block_host(sws_precond* pc, int32_t which, int32_t l, int32_t m, double* out_host);

size_t sws_precond_bytes(const sws_precond* pc);    /* device memory held                     */
int sws_precond_bandwidth(const sws_precond* pc);   /* the odd block bandwidth in use         */
double sws_precond_setup_ms(const sws_precond* pc); /* wall time of assembly + factorisation  */
int sws_precond_destroy(sws_precond* pc);

typedef struct {
  double tol;       /* stop when ||rhs - J d||_2 <= tol ||rhs||_2 (Arnoldi estimate)          */
  int32_t restart;  /* Krylov dimension m before a restart (<= the solver's max_restart)      */
  int32_t maxit;    /* cap on Jacobian-vector products in total                              */
  int32_t jv_mode;  /* 0 analytic J v (sws_linearize + sws_jv_apply); 1 eq. (25) through
                       sws_jv_batch (base and shifted state evaluated per product); 2 eq. (25)
                       with the base residual E(u) the driver already holds: ONE sws_residual
                       per product, the paper's own scheme (L219), same shift sigma        */
  int32_t block;    /* 0 or 1: plain GMRES.  t in 2..16 (t <= the context's max_batch): ENLARGED GMRES - the
                       right-hand side is split by groups of y-lines into t pieces that sum to it and the block
                       Krylov space K_m(J P^-1, [T_1 r .. T_t r]) is built with ONE t-vector Jacobian action
                       (sws_jv_apply(V[t]), or sws_jv_batch for jv_mode 1, 2) and ONE t-vector preconditioner
                       sweep per iteration; the iterate minimises the residual over that space, which contains the
                       plain Krylov space of the same depth.  One cycle of at most min(restart / t,
                       (max_restart + 1) / t - 1) blocks, no restart; its, maxit and hist count / index products
                       resp. block iterations (hist[j] after block j).  Falls back to plain GMRES when a piece of
                       the right-hand side is zero.                                                       */
} sws_gmres_opts;

typedef struct {
  int32_t its;       /* Jacobian-vector products performed                                   */
  int32_t converged; /* 1 if the tolerance was met                                           */
  double rel_res;    /* last residual estimate / ||rhs||_2                                   */
  double rhs_norm;
} sws_gmres_stats;

typedef struct {
  double ftol;          /* stop when ||E(u)||_inf <= ftol                                    */
  double eta;           /* relative tolerance of each inner GMRES solve (inexact Newton L223) */
  double alpha;         /* sufficient decrease: ||E(u+lam du)|| < (1 - alpha lam) ||E(u)||   */
  int32_t max_newton;   /* cap on Newton steps                                               */
  int32_t max_halvings; /* cap on lam = 1, 1/2, 1/4, ...                                     */
  sws_gmres_opts gmres; /* tol is overridden by eta                                          */
  int32_t forcing;      /* 0: every inner solve to eta.  1: forcing term "choice 2" of Eisenstat &
                           Walker as in the survey the paper cites for its inexact Newton method
                           ([21], L223): eta_0 = eta_max, eta_k = 0.9 (||E_k||/||E_{k-1}||)^2,
                           raised to 0.9 eta_{k-1}^2 when that exceeds 0.1, clipped to [eta, eta_max] */
  double eta_max;       /* forcing = 1 only (0 < eta <= eta_max < 1)                         */
} sws_newton_opts;

typedef struct {
  int32_t newton;    /* step index k                                                         */
  int32_t gmres_its; /* J v products of step k (0 in the closing entry)                      */
  double fnorm;      /* ||E(u_k)||_2                                                         */
  double finf;       /* ||E(u_k)||_inf                                                       */
  double gmres_rel;  /* final relative residual estimate of the inner solve                 */
  double lambda;     /* accepted damping (0: none accepted / closing entry)                 */
} sws_newton_log;

typedef struct {
  int32_t steps;          /* Newton steps taken                                              */
  int32_t converged;      /* 1 if ||E||_inf <= ftol                                          */
  int32_t residual_evals; /* E(u) evaluations (sws_residual calls)                           */
  int32_t jv_products;    /* J v products                                                    */
  int32_t precond_applies;
  double ms_total;        /* wall time of the call                                           */
  double ms_jv, ms_precond, ms_residual; /* CUDA-event time of those parts                   */
} sws_newton_stats;

/* Workspace of the drivers for `ctx` (Krylov basis of max_restart + 1 vectors on ctx's device).
 * pc may be NULL (no preconditioning).  ctx needs max_batch >= 1.  Neither is owned. */
int sws_solver_create(sws_ctx* ctx, sws_precond* pc, int32_t max_restart, sws_solver** out);

/* Solve J(u) d = rhs approximately.  hist_host: [opts->maxit] relative residual estimate after
 * each product, or NULL. */
int sws_solver_gmres(sws_solver* s, const double* u_dev, const double* rhs_dev,
                     const sws_gmres_opts* opts, double* d_dev, sws_gmres_stats* stats,
                     double* hist_host, void* cuda_stream);

/* Damped Newton from u_dev (in: initial guess, out: last iterate).  log_host has room for
 * opts->max_newton + 1 entries; *nlog receives the number written. */
int sws_solver_newton(sws_solver* s, double* u_dev, const sws_newton_opts* opts,
                      sws_newton_log* log_host, int32_t* nlog, sws_newton_stats* stats,
                      void* cuda_stream);

/* The bootstrapping process of L229: for i = 0..n_eps-1 set the source strength of the solver's
 * context to eps_host[i] (sws_set_eps) and run sws_solver_newton from the previous solution
 * (u_dev in: the guess for eps_host[0], e.g. the flat state L227; out: the solution for the last
 * value reached).  stats_host has room for n_eps entries; *n_done = how many values converged
 * (the process stops at the first that does not; u_dev then holds that failed iterate's
 * predecessor, the last converged solution).  The context keeps the last epsilon it was set to. */
int sws_solver_continuation(sws_solver* s, double* u_dev, const double* eps_host, int32_t n_eps,
                            const sws_newton_opts* opts, sws_newton_stats* stats_host, int32_t* n_done,
                            void* cuda_stream);

int sws_solver_destroy(sws_solver* s);

#ifdef __cplusplus
}
#endif
#endif /* SWS_JFNK_H_ */
