/*
 * fe_mf.h -- C-ABI of the B200-native matrix-free finite-element Helmholtz multivector apply
 * and Chebyshev filter (hot path of arXiv 2208.07129).
 *
 * The library computes, entirely in hand-written sm_100a CUDA kernels and in IEEE FP64,
 *
 *     Y = A X,   A = K + sigma*M                        (Eq. 3, Eq. 6)
 *
 * for a degree-p (1..8) hexahedral GLL Lagrange discretisation with (p+1)^3 Gauss-Legendre
 * quadrature points per cell, by sum factorisation (Alg. 1
 * Alg. 2, Eq. 15): gather -> N1D x3 -> D~1D x3 -> quadrature-point scaling -> D~1D^T x3 ->
 * N1D^T x3 -> scatter-add, fused in one kernel per (cell, vector-batch) as in PAPER.md:690-740
 * (Alg. 4), plus the scaled Chebyshev three-term recurrence of PAPER.md:931-975 (Alg. 6 l.2-17)
 * with the axpby folded into the apply as in PAPER.md:1169-1174 (Eq. B.1).
 *
 * Multivector layout (all entry points): X[J*nvec + beta], J = ix + nd_x*(iy + nd_y*iz) the
 * lexicographic global node index (x fastest), beta the vector index, INNERMOST -- the paper's
 * BCV layout with one batch b = nvec (Fig. 1).  nd_d = ncells_d*p (periodic) or
 * ncells_d*p + 1 (Dirichlet; boundary nodes are counted, PAPER.md:542/820/899 DoF counts).
 *
 * Dirichlet convention (C^T A C of Eq. 6 literally): boundary entries of X are
 * ignored (read as 0), boundary entries of Y are written as 0.
 *
 * Pointers named *_dev are DEVICE pointers on the context's CUDA device; *_host are HOST
 * pointers.  The caller owns X, Y and the stream; the context owns tables, geometry and
 * workspace.  Nothing is thrown or aborted across this boundary: every call returns a code and
 * leaves a message retrievable with fe_mf_last_error().  There is no CPU fallback.
 */
#ifndef FE_MF_H
#define FE_MF_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fe_mf_ctx fe_mf_ctx; /* opaque, library-owned */

enum { FE_MF_OK = 0, FE_MF_EINVAL = 1, FE_MF_ENOMEM = 2, FE_MF_ECUDA = 3, FE_MF_EUNSUPPORTED = 4 };
enum { FE_BC_PERIODIC = 0, FE_BC_DIRICHLET = 1 };
enum { FE_GEOM_AFFINE = 0, FE_GEOM_QPOINT = 1 };

/*
 * fe_mf_create -- build a context: 1D tables N1D[q][i] = l_i(xq_q), D~1D[q][r] = l~_r'(xq_q)
 * and Gauss weights in extended precision on the host, the geometric factors
 * G^(s,d) = (J^-1 J^-T)_sd det J w_Q and G = sigma det J w_Q (mu = 1, kappa =
 * sigma), and upload them.
 *   out            receives the context (NULL on failure).
 *   ncx,ncy,ncz    cells per direction (>= 1; >= 2 in every direction if periodic).
 *   p              FE degree, 1..8; n_q = n_p = p+1.
 *   sigma          A = K + sigma*M.
 *   bc             FE_BC_PERIODIC | FE_BC_DIRICHLET (homogeneous).
 *   geom           FE_GEOM_AFFINE: one symmetric 3x3 factor per cell, J taken at the cell centre
 *                  (exact for parallelepipeds; "a linear map exists", Eq. 23);
 *                  FE_GEOM_QPOINT: 6 metric entries + 1 mass factor stored per quadrature point
 *                  from the trilinear map of the 8 cell vertices (Eq. 7c evaluated "at xi_Q").
 *   box_lo,box_hi  HOST, 3 doubles each: the box of the uniform Cartesian mesh (used when
 *                  vertices_host == NULL; must satisfy hi > lo).
 *   vertices_host  HOST, NULL or [(ncz+1)][(ncy+1)][(ncx+1)][3] doubles; copied.  For periodic
 *                  meshes the vertices on opposite box faces must match up to the box period.
 *   cuda_device    device ordinal.
 * Errors: EINVAL (null out, bad sizes/p/bc/geom, hi <= lo, non-positive det J at a quadrature
 * point), ENOMEM, ECUDA, EUNSUPPORTED (device is not sm_100).
 */
int fe_mf_create(fe_mf_ctx **out, int ncx, int ncy, int ncz, int p, double sigma, int bc, int geom,
                 const double box_lo[3], const double box_hi[3], const double *vertices_host,
                 int cuda_device);

/*
 * the distributed half of the paper (section 3.2.5, Alg. 5): the mesh is cut
 * into subdomains, one per task; a task stores its locally-owned DoFs followed by the "ghost" DoFs on the shared
 * subdomain boundary and evaluates  V = sum_t P^(t)T A^(t) P^(t) U :  ghost values of U arrive from
 * their owner (P^(t)), the task applies the cells it owns, the ghost rows of the result go back to their owner and are
 * ADDED there (P^(t)T).  Here the subdomains are z-SLABS of the structured mesh.
 *
 * fe_mf_create_slab: like fe_mf_create for ONE slab of ncz cell layers (box_lo / box_hi / vertices_host describe the
 *   slab itself).  z_open bit 0 / bit 1: the low / high z face is a CUT plane, not a boundary: no Dirichlet mask there
 *   and no periodic wrap in z.  A periodic mesh is periodic in x and y only for its slabs: z_open must be 3, and the
 *   slab has nd_z = ncz p + 1 node planes.  Multivector of a slab context: planes 0 .. ncz p of the slab, i.e. its owned
 *   planes followed by its top plane -- the ghost plane, owned by the next task (the last slab of a Dirichlet mesh owns
 *   its top plane: z_open = 1).  fe_mf_apply on such a context computes V^(t) = A^(t) U^(t) with the fused kernels;
 *   fe_cheb_filter, fe_mf_set_mass_scaling and fe_mf_mass_diagonal return EUNSUPPORTED (they need data of the
 *   neighbouring slab at every step).
 * fe_mf_halo_add: dst_dev[k] += src_dev[k], k < count (DEVICE pointers, stream-ordered): the P^(t)T step on the
 *   receiving side -- the neighbour's ghost plane of V added into the owner's first plane.
 * fe_mf_halo_pack_f32 / fe_mf_halo_unpack_f32: the mixed-precision boundary payload of PAPER.md:752 ("the boundary data
 *   communicated is recast as FP32 floats").  pack: dst_dev[k] = (float) src_dev[k], round to nearest even, on the
 *   sending side; unpack on the receiving side: dst_dev[k] = (double) src_dev[k] (add = 0: ghost values of U) or
 *   dst_dev[k] += (double) src_dev[k] (add = 1: ghost rows of V).  DEVICE pointers, count elements, stream-ordered;
 *   dst and src must not overlap.  Everything a task computes stays FP64: only the message is FP32 (half the bytes).
 * fe_mf_axpby: Z_dev[k] = beta Z_dev[k] + gamma W_dev[k], k < count (DEVICE pointers, 8-byte aligned is enough, stream-ordered;
 *   beta == 0: Z is not read and may hold anything).  The owned-rows update of a decomposed Chebyshev step
 *   (Alg. 6 l.15: X <- alpha1 V + alpha2 X - c alpha1 Y with V = the decomposed product, dd.py), which a slab
 *   context cannot fuse into its kernel because the ghost rows of V first travel to their owner.  Z and W must not overlap
 *   unless they are the same pointer.
 * Errors of the halo calls and fe_mf_axpby: EINVAL (null pointer, count < 0, add not 0 / 1), ECUDA (launch failure).
 * The exchange itself is point-to-point (two neighbours per slab): paper_2208_07129_b200/dd.py drives it with
 * torch.distributed send / recv (NCCL between GPUs; the plane to send is a contiguous block of the multivector).
 */
int fe_mf_create_slab(fe_mf_ctx **out, int ncx, int ncy, int ncz, int p, double sigma, int bc, int geom,
                      const double box_lo[3], const double box_hi[3], const double *vertices_host, int z_open,
                      int cuda_device);
int fe_mf_halo_add(double *dst_dev, const double *src_dev, long long count, void *cuda_stream);
int fe_mf_axpby(double *Z_dev, const double *W_dev, double beta, double gamma, long long count, void *cuda_stream);
int fe_mf_halo_pack_f32(float *dst_dev, const double *src_dev, long long count, void *cuda_stream);
int fe_mf_halo_unpack_f32(double *dst_dev, const float *src_dev, long long count, int add, void *cuda_stream);

/* nd_x*nd_y*nd_z including Dirichlet boundary nodes; -1 if ctx is NULL. */
long long fe_mf_ndofs(const fe_mf_ctx *ctx);

/*
 * fe_mf_apply -- Y = (K + sigma M) X for nvec vectors (Eq. 6, Eq. 17).
 *   X_dev  DEVICE, read-only, ndofs*nvec doubles, layout above.
 *   Y_dev  DEVICE, overwritten, same shape; must not alias X_dev.
 *   nvec   >= 1.
 *   cuda_stream  a cudaStream_t (NULL = default stream).  All work is enqueued on it; the call
 *                does not synchronise the host (it can be captured in a CUDA graph after a first call).
 *                A context owns the work counters of its persistent kernels: calls on ONE context must be
 *                stream-ordered (use one context per stream for concurrent applies).
 *                Pointers need only be 8-byte aligned; the TMA kernels serve 16-byte aligned pointers with an even
 *                nvec, everything else runs on kernels with plain loads and atomics (same result, slower).
 * Errors: EINVAL (null pointers, nvec < 1, aliasing), ECUDA.
 */
int fe_mf_apply(fe_mf_ctx *ctx, const double *X_dev, double *Y_dev, int nvec, void *cuda_stream);

/*
 * fe_mf_apply_bcv -- the same product on the paper's Batched Contiguous Vector layout (section 3.2.1,
 * Fig. 1): the nvec vectors in n_b = ceil(nvec / b) batches, batch i_b holding vectors i_b b .. i_b b + b_i - 1
 * (b_i = b, the last batch nvec - (n_b - 1) b) as a contiguous [ndofs][b_i] block, vector index innermost, at offset
 * ndofs * i_b * b doubles:   element (J, beta)  ->  ndofs * b * (beta / b) + J * b_i + beta % b.
 * With b >= nvec this is fe_mf_apply's layout.  One kernel launch (plus the zero fill) per batch, all on cuda_stream
 * (Eq. 17's sum over i_b); b is the caller's choice -- fe_mf_batch_width(ctx, b) tells how many vectors a thread block of
 * the kernel chosen for that width takes.  X_dev / Y_dev: DEVICE, ndofs*nvec doubles each, must not overlap.
 * Errors: EINVAL (null pointers, b < 1, nvec < 1, overlap), ECUDA.
 */
int fe_mf_apply_bcv(fe_mf_ctx *ctx, const double *X_dev, double *Y_dev, int b, int nvec, void *cuda_stream);

/*
 * fe_mf_apply_axpby -- the fused form of Eq. (B.1) without mass scaling:
 *     Z <- alpha * A * W  +  beta * Z  +  gamma * W
 * W_dev read-only, Z_dev updated in place, no aliasing.  This is the one step the Chebyshev
 * recurrence is built from (Alg. 6 l.10 and l.15).  Dirichlet: boundary rows get beta*Z + gamma*W.
 */
int fe_mf_apply_axpby(fe_mf_ctx *ctx, double alpha, const double *W_dev, double beta, double gamma,
                      double *Z_dev, int nvec, void *cuda_stream);

/*
 * fe_mf_accumulate -- Z <- Z + alpha * A * W : the fused cell kernel alone (gather ... scatter-add,
 * PAPER.md:690-740 Alg. 4) on an already initialised Z.  fe_mf_apply == (Z <- 0) + this call;
 * bench.py times it to obtain the dominant kernel's own duration.
 */
int fe_mf_accumulate(fe_mf_ctx *ctx, double alpha, const double *W_dev, double *Z_dev, int nvec,
                     void *cuda_stream);

/*
 * fe_cheb_filter -- scaled Chebyshev filter of degree m (Alg. 6 lines 2-17, garbled
 * lines reconstructed as in SURVEY.md §8(c) step 6 / DESIGN.md reading 10):
 *     e=(b-a)/2; c=(b+a)/2; s=e/(a0-c); s1=s; g=2/s1; a1=s1/e; a2=-c;  Y = a1 A X + a1 a2 X;
 *     for d=2..m: s2=1/(g-s); a1=2 s2/e; a2=-s s2;  X <- a1 A Y + a2 X - c a1 Y; swap(X,Y); s=s2;
 *   X_dev  DEVICE, input AND scratch: on return it holds iterate m-1 (for m == 1: unchanged).
 *   Y_dev  DEVICE, output: the filtered block (always delivered here).
 *   a,b    the damped interval [a, b] (a = upper bound of the wanted spectrum, b >= lambda_max);
 *   a0     lower bound of the spectrum.  Requires m >= 1, b > a, a0 < a.
 * The scalar recurrence runs on the host in double; the m fused applies are stream-ordered.
 * Errors: EINVAL, ECUDA.
 */
int fe_cheb_filter(fe_mf_ctx *ctx, double *X_dev, double *Y_dev, int nvec, int m, double a, double b,
                   double a0, void *cuda_stream);

/*
 * fe_mf_apply_host -- end-to-end convenience: same as fe_mf_apply but X_host / Y_host are HOST
 * buffers (pinned memory recommended).  Large calls on the TMA kernels are pipelined over z-slabs of the mesh: a
 * range of node planes is one contiguous block of the (z-major) multivector on both sides of the bus, so slab k+1
 * is copied in and slab k-1 copied out at the full pinned rate while the kernel runs on the cell layers of slab k
 * (three internal streams; device workspace = the whole X and Y).  Other calls stage column blocks (strided
 * copies) through a smaller workspace on two internal streams, each with its own work counter.  Returns after
 * Y_host is complete.  Errors as fe_mf_apply plus ENOMEM.
 */
int fe_mf_apply_host(fe_mf_ctx *ctx, const double *X_host, double *Y_host, int nvec);

/*
 * fe_fill_uniform -- synthetic-input generator (NOT part of the operator): fills
 * out_dev[k] = 2*((splitmix64(seed + (offset+k)*0x9E3779B97F4A7C15) >> 11) * 2^-53) - 1 for
 * k < count, bit-identical to the Python generator in paper_2208_07129_b200/inputs.py
 * (SURVEY.md §8(d)).  DEVICE pointer on the current device; stream-ordered.
 */
int fe_fill_uniform(double *out_dev, long long count, unsigned long long seed, long long offset,
                    void *cuda_stream);

/*
 * the operator of the paper's eigenproblem benchmark:
 *   H = K + M^kappa with kappa(x) given at the quadrature points, and H~ = M^-1/2 H M^-1/2 with M the mass matrix
 *   evaluated by the (p+1)-point Gauss-Lobatto-Legendre rule on the nodes, hence diagonal.
 *
 * fe_mf_set_kappa: kappa_host is a HOST array [ncells][n^3] (n = points per direction of the current rule, p + 1 unless
 *   fe_mf_set_quadrature changed it; cells x fastest, point Q = q1 + n q2 + n^2 q3 at the
 *   Gauss points of the cell: kappa_Q = kappa(x_Q)), copied; it replaces sigma in every later call
 *   (G_QQ = kappa_Q det J w_Q).  NULL restores the constant sigma.  The context must be a uniform box
 *   (FE_GEOM_AFFINE without vertices) or have been created with FE_GEOM_QPOINT, else EINVAL (one metric per cell of a
 *   vertex array has no per-point storage).  On a uniform box the fast path is kappa TOGETHER with mass scaling (the
 *   eigenproblem operator, served by the Cartesian kernels); kappa alone runs there on the general fallback kernel.
 * fe_mf_set_mass_scaling: on != 0 makes fe_mf_apply / fe_mf_apply_axpby / fe_cheb_filter / fe_mf_apply_host act
 *   with H~ instead of H: Z = alpha M^-1/2 H M^-1/2 W + beta Z + gamma W (Eq. B.1); the diagonal
 *   scaling is done inside the kernel, not in extra passes: on a uniform box M^-1/2 is a Kronecker product and is
 *   absorbed by the 1D interpolation tables (no cost); on other meshes it is applied at extraction and assembly
 *    by the full-metric kernels from a vector of n_dof doubles.  Dirichlet boundary entries of M are computed like all others and never used.
 * fe_mf_mass_diagonal: writes diag(M) (HOST array of fe_mf_ndofs doubles, node order of the multivector rows) so
 *   that the caller can map U = M^-1/2 U~.
 * All three synchronise the device (they are setup calls, not stream-ordered) and return FE_MF_* codes.
 */
int fe_mf_set_kappa(fe_mf_ctx *ctx, const double *kappa_host);

/*
 * fe_mf_set_quadrature: nq Gauss points per direction instead of n_p = p + 1 (the paper also
 * benchmarks n_q = n_p + 2); p + 1 <= nq <= 12, else EINVAL; nq = p + 1 restores the default.
 * Everything else keeps its meaning (N becomes n_q x n_p, the gradients are taken by collocation on the n_q points,
 * D = D~ N of PAPER.md:188, per-point geometry and kappa live on the n_q^3 points).  On affine cells with constant
 * kappa the result does not change (the n_p-point rule is already exact there).  A kappa array set before belongs
 * to the points of the old rule and is dropped (constant sigma again): call fe_mf_set_kappa afterwards with
 * [ncells][nq^3] values.  With nq = p + 3 the calls run on an even-odd line-task kernel with compile-time sizes, with any
 * other nq != p + 1 on one plain kernel (rectangular tables, loads and atomics).
 * Synchronises the device.
 */
int fe_mf_set_quadrature(fe_mf_ctx *ctx, int nq);
int fe_mf_set_mass_scaling(fe_mf_ctx *ctx, int on);
int fe_mf_mass_diagonal(fe_mf_ctx *ctx, double *out_host);

/*
 * fe_probe_peaks -- box peaks for the roofline (BASELINE.json north_star: "peaks measured on the box
 * by a stream/DGEMM microbenchmark"): FP64 FMA-chain rate in TFLOP/s (2 flops per DFMA) and FP64
 * stream-copy bandwidth in GB/s (read + write bytes), best of 5 after one warm-up, on cuda_device's
 * default stream.  Synchronises the host.  HOST output pointers.
 */
int fe_probe_peaks(double *fp64_tflops, double *hbm_gbs, int cuda_device);

/* Introspection used by bench.py / tests: vectors per thread block chosen for this nvec, the
 * number of kernel launches the last call enqueued, and the dominant kernel's name. */
int fe_mf_batch_width(const fe_mf_ctx *ctx, int nvec);
/* Nodes per direction nd[3] (HOST), boundary condition FE_BC_* and the CUDA device of the context. */
int fe_mf_shape(const fe_mf_ctx *ctx, int nd[3], int *bc, int *cuda_device);
const char *fe_mf_kernel_name(const fe_mf_ctx *ctx, int nvec);   /* static string, never NULL */
int fe_mf_last_launch_count(const fe_mf_ctx *ctx);

/* Select a kernel variant (0 = default: chosen from degree, geometry and nvec).  For tests and profiling only:
 * 1 general fallback kernel (with n_q != n_p: loads and atomics on every cell instead of TMA), 2 one-vector-per-thread
 * Cartesian kernel (LDG/RED), 7 full-metric TMA kernel on a Cartesian mesh, 8 plane kernel (p = 6), 10 / 11 line
 * kernel with 16 / 8 vectors per block; 22 / 23 fe_mf_apply_host in column chunks only / in z-slabs whatever the size.  Returns EINVAL if unknown. */
int fe_mf_set_variant(fe_mf_ctx *ctx, int variant);

/* Message of the last failing call on ctx; with ctx == NULL, of the last failing fe_mf_create on
 * this thread.  Never NULL. */
const char *fe_mf_last_error(const fe_mf_ctx *ctx);

void fe_mf_destroy(fe_mf_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* FE_MF_H */
