/*
 * fe_constraints.h -- C ABI of the constraint matrices C^(t), C^(t)T of the matrix-free apply (
 * PAPER.md:288-302, section 3.2.2 "Applying the constraints"; Eq. 17 PAPER.md:270-276:
 *
 *      V = sum_t P^(t)T C^(t)T ( sum_{i_b, e} B^T Q^T A^(e) Q B ) C^(t) P^(t) U ).
 *
 * The constraints are stored "as multiple sets, and each set I comprises four arrays": the master node
 * indices M_I, the slave node indices S_I, the weight matrix W_I [ns_I][nm_I] (row-major) and the inhomogeneities b_I
 * of the slaves.  On a multivector U [ndof][nvec] (vector index innermost, as in fe_mf.h):
 *
 *      C:    U[S_I] <- W_I U[M_I] + b_I                      (hanging nodes: interpolation along faces / edges)
 *      C^T:  V[M_I] <- V[M_I] + W_I^T V[S_I],  V[S_I] <- 0   ("evaluated in the similar manner")
 *
 * Dirichlet conditions are sets without masters (nm_I = 0).  The sets must be CLOSED: every slave belongs
 * to exactly one set and no slave is a master of any set (reading 19); a master may serve several sets.  The
 * order of the sets is then immaterial.  The paper multiplies set by set with BLAS gemm; here one thread block per
 * (set, block of <= 32 vectors) evaluates the set's small dense product directly, all sets in ONE launch.
 *
 * Implemented in libfe_mf.so.  Every pointer is marked HOST or DEVICE.  Error codes are fe_mf.h's (FE_MF_OK, FE_MF_EINVAL,
 * FE_MF_ENOMEM, FE_MF_ECUDA); no exception or abort crosses the ABI.
 */
#ifndef FE_CONSTRAINTS_H
#define FE_CONSTRAINTS_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fe_constraints fe_constraints; /* opaque, library-owned; owns device copies of the four arrays */

/*
 * fe_constraints_create -- validate the sets and copy them to the device.
 *   ndof         rows of the multivectors the object will be applied to (> 0).
 *   nsets        number of sets (>= 0).
 *   master_ptr   HOST [nsets+1], master_ptr[0] = 0, non-decreasing: set I's masters are masters[master_ptr[I] .. master_ptr[I+1]).
 *   masters      HOST [master_ptr[nsets]] node indices in [0, ndof).
 *   slave_ptr    HOST [nsets+1], likewise for the slaves.
 *   slaves       HOST [slave_ptr[nsets]].
 *   weights      HOST, set after set: W_I row-major [ns_I][nm_I]; sum_I ns_I nm_I doubles (may be NULL if that is 0).
 *   inhomog      HOST [slave_ptr[nsets]] b of every slave, or NULL (all zero).
 *   cuda_device  device ordinal.
 * All arrays are copied; the caller keeps ownership.  Errors: EINVAL (null out / pointer, bad offsets, index out of
 * range, a slave in two sets, a slave that is a master), ENOMEM, ECUDA (no device).  On failure *out = NULL and
 * fe_constraints_last_error(NULL) holds the reason.
 */
int fe_constraints_create(fe_constraints **out, long long ndof, int nsets, const long long *master_ptr,
                          const long long *masters, const long long *slave_ptr, const long long *slaves,
                          const double *weights, const double *inhomog, int cuda_device);

/*
 * fe_constraints_distribute -- U <- C U (+ b unless homogeneous != 0), in place.
 *   U_dev   DEVICE [ndof][nvec] doubles, vector index innermost.  Only slave rows are written; master rows are read.
 *   nvec    >= 1.   homogeneous: 0 adds the inhomogeneities b_I, 1 leaves them out (the linear part, which is what an
 *           operator apply uses: PAPER.md Eq. 17).
 * Stream-ordered on cuda_stream, no host synchronisation.  Errors: EINVAL, ECUDA.
 */
int fe_constraints_distribute(fe_constraints *c, double *U_dev, int nvec, int homogeneous, void *cuda_stream);

/*
 * fe_constraints_distribute_transpose -- V <- C^T V, in place: master rows accumulate W_I^T V[S_I] (atomic adds: a master
 * may serve several sets, so the summation order between sets is not fixed), slave rows are zeroed.
 * Same layout, stream semantics and errors as above.
 */
int fe_constraints_distribute_transpose(fe_constraints *c, double *V_dev, int nvec, void *cuda_stream);

/* Totals: number of sets, of master entries, of slaves; any pointer may be NULL.  EINVAL if c is NULL. */
int fe_constraints_counts(const fe_constraints *c, int *nsets, long long *nmasters, long long *nslaves);

/* Message of the last failing call on c; with c == NULL, of the last failing create on this thread.  Never NULL. */
const char *fe_constraints_last_error(const fe_constraints *c);

void fe_constraints_destroy(fe_constraints *c);

#ifdef __cplusplus
}
#endif
#endif /* FE_CONSTRAINTS_H */
