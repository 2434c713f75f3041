/*
 * fe_chfsi.h -- C-ABI of the Chebyshev filtered subspace iteration around the matrix-free operator of fe_mf.h
 * (arXiv 2208.07129, Algorithm 6).  sm_100a only, no CPU fallback.
 *
 *   line 1       while ||H U - U Lambda|| > tau                  fe_chfsi_solve
 *   lines 2-17   Chebyshev filter                                fe_cheb_filter (fe_mf.h, hand-written kernels)
 *   line 18      Xo <- orthogonalize(X)                          Cholesky QR, twice: S = X^T X (cuBLAS DSYRK),
 *                                                                S = L L^T (cuSOLVER DPOTRF), X <- X L^-T (DGEMM with
 *                                                                the explicit n x n inverse)
 *   line 19      Xo^T H Xo Q = Q Lambda                          fe_mf_apply, DGEMM, cuSOLVER DSYEVD
 *   line 20      U <- Xo Q                                       DGEMM
 *                In fe_chfsi_iterate / fe_chfsi_solve the second Cholesky-QR round is folded into lines 19-20 as the
 *                generalised problem (X1^T H X1) Z = (X1^T X1) Z Lambda, U = X1 Z (cuSOLVER DSYGVD): same U, one tall
 *                DGEMM less.
 *   line 1       r_j = ||H u_j - lambda_j u_j||_2                fe_mf_apply + a column-norm kernel
 *
 * The operator is whatever the fe_mf context applies (H~ = M^-1/2 (K + M^kappa) M^-1/2 once fe_mf_set_kappa /
 * fe_mf_set_mass_scaling were called).  The dense tall-skinny algebra is library code (SURVEY.md
 * 8(f): "cuBLAS/cuSOLVER territory"); every operator application runs in the kernels of fe_mf.h.
 *
 * Multivectors are DEVICE arrays [n_dof][nvec] (vector index fastest), FP64, as in fe_mf.h.  On Dirichlet meshes the
 * eigenproblem is posed on the unconstrained DoFs (every constrained DoF is a null vector of C^T A C): the boundary
 * rows of U are zeroed on entry and stay exactly zero (the filter, the triangular solve and the rotation act row by
 * row).  All calls are enqueued on `stream` (a cudaStream_t as void*, NULL = default) except where stated; calls
 * that return host values synchronise that stream.  Return codes are fe_mf.h's FE_MF_*.
 */
#ifndef FE_CHFSI_H
#define FE_CHFSI_H

#include "fe_mf.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fe_chfsi fe_chfsi;

/* Workspace for blocks of `nvec` vectors on op's mesh: two multivectors [n_dof][nvec], three nvec x nvec matrices,
 * cuBLAS / cuSOLVER handles.  `op` must outlive the handle and is used by it (one stream at a time). */
int fe_chfsi_create(fe_chfsi **out, fe_mf_ctx *op, int nvec);
void fe_chfsi_destroy(fe_chfsi *h);
const char *fe_chfsi_last_error(const fe_chfsi *h);   /* with h == NULL: of the last failing create on this thread */

/* k-step Lanczos upper bound of the spectrum, lambda_max(T_k) + beta_k (Zhou-Saad [37]), from
 * the start vector v0_dev (DEVICE, n_dof doubles, not modified; boundary rows ignored on Dirichlet meshes).
 * bound_host: HOST.  Synchronises. */
int fe_chfsi_lanczos_bound(fe_chfsi *h, const double *v0_dev, int k, double *bound_host, void *stream);

/* Line 18 alone: X_dev <- orthonormal basis of span(X_dev), in place.  FE_MF_EINVAL if the block is numerically
 * rank deficient (the Cholesky factorisation of X^T X fails). */
int fe_chfsi_orthonormalize(fe_chfsi *h, double *X_dev, void *stream);

/* Lines 19-20 and the residuals of line 1 for an orthonormal block X_dev: U_dev <- X Q (U_dev != X_dev; X_dev is
 * left unchanged), evals_host[nvec] ascending, resid_host[nvec] = ||H u_j - lambda_j u_j||_2 (either HOST pointer may be
 * NULL).  Synchronises. */
int fe_chfsi_rayleigh_ritz(fe_chfsi *h, const double *X_dev, double *U_dev, double *evals_host, double *resid_host,
                           void *stream);

/* One pass of lines 2-20 on U_dev (in place): filter of degree m damping [lam_u, lam_max] with lower bound lam_min
 * (fe_cheb_filter's a, b, a0), orthonormalise, Rayleigh-Ritz, rotate.  Outputs as fe_chfsi_rayleigh_ritz. */
int fe_chfsi_iterate(fe_chfsi *h, double *U_dev, int m, double lam_max, double lam_u, double lam_min,
                     double *evals_host, double *resid_host, void *stream);

/* Line 1 loop: passes until the n_wanted lowest pairs have residual <= tau or max_iter passes were made.  After each
 * pass lam_min <- lowest and lam_u <- highest Ritz value of the block (the vectors beyond n_wanted are the buffer,
 * PAPER.md:977; the paper takes the bounds as data and is silent on their update: DESIGN.md).  iters_host: passes made.
 * Returns FE_MF_OK also when max_iter was reached (check resid_host). */
int fe_chfsi_solve(fe_chfsi *h, double *U_dev, int n_wanted, int m, double lam_max, double lam_u, double lam_min,
                   double tau, int max_iter, double *evals_host, double *resid_host, int *iters_host, void *stream);

/* Milliseconds (CUDA events on `stream`) spent by the last fe_chfsi_iterate in: [0] filter, [1] orthonormalisation,
 * [2] operator applications of lines 19 / 1, [3] DGEMMs of lines 19-20, [4] DSYEVD, [5] residual norms. */
int fe_chfsi_last_timings(const fe_chfsi *h, double ms_host[6]);

#ifdef __cplusplus
}
#endif
#endif
