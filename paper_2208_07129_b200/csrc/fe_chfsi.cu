// C-ABI of include/fe_chfsi.h: Chebyshev filtered subspace iteration (Alg. 6) around the
// matrix-free operator of libfe_mf.so.  The operator applications and the filter are fe_mf.h calls (hand-written
// kernels); the tall-skinny dense algebra of lines 18-20 is cuBLAS / cuSOLVER; the residual norms and the constraint
// projection are two small kernels here.  sm_100a only.
#include "../../include/fe_chfsi.h"

#include <cublas_v2.h>
#include <cuda_runtime.h>
#include <cusolverDn.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

struct fe_chfsi {
  fe_mf_ctx* op = nullptr;
  int nvec = 0, nd[3] = {0, 0, 0}, bc = 0, device = 0;
  long long ndof = 0;
  cublasHandle_t blas = nullptr;
  cusolverDnHandle_t sol = nullptr;
  double *Y = nullptr, *W = nullptr;        // multivectors [ndof][nvec]
  double *S = nullptr, *T = nullptr;        // nvec x nvec (column-major for the libraries)
  double *lam = nullptr, *res = nullptr;    // nvec
  double* work = nullptr; int lwork = 0; int* info = nullptr;
  double* lv = nullptr;                     // 3 Lanczos vectors, allocated on first use
  cudaEvent_t ev[8] = {};
  cudaEvent_t ev_end = nullptr;
  double ms[6] = {0, 0, 0, 0, 0, 0};
  int gram_depth = 1;   // measured (n = 1024): 0 -> 61 ms, 1 -> 47 ms, 2 -> 63 ms, 3 -> 110 ms per Gram matrix
  std::string err;
};

static thread_local std::string g_chfsi_create_err = "";

namespace {

int fail(fe_chfsi* h, int code, const std::string& msg) {
  if (h) h->err = msg; else g_chfsi_create_err = msg;
  return code;
}

#define CH_CUDA(h, call)                                                                       \
  do {                                                                                         \
    cudaError_t e_ = (call);                                                                   \
    if (e_ != cudaSuccess) return fail((h), FE_MF_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
  } while (0)
#define CH_BLAS(h, call)                                                                       \
  do {                                                                                         \
    cublasStatus_t s_ = (call);                                                                \
    if (s_ != CUBLAS_STATUS_SUCCESS) return fail((h), FE_MF_ECUDA, std::string(#call) + ": cuBLAS status " + std::to_string((int)s_)); \
  } while (0)
#define CH_SOL(h, call)                                                                        \
  do {                                                                                         \
    cusolverStatus_t s_ = (call);                                                              \
    if (s_ != CUSOLVER_STATUS_SUCCESS) return fail((h), FE_MF_ECUDA, std::string(#call) + ": cuSOLVER status " + std::to_string((int)s_)); \
  } while (0)
#define CH_OP(h, call)                                                                         \
  do {                                                                                         \
    int rc_ = (call);                                                                          \
    if (rc_ != FE_MF_OK) return fail((h), rc_, std::string(#call) + ": " + fe_mf_last_error((h)->op)); \
  } while (0)

struct DevGuard {
  int prev = -1; bool ok = false;
  explicit DevGuard(int dev) { if (cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess) ok = true; }
  ~DevGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Constrained (Dirichlet boundary) rows of a multivector <- 0: the eigenproblem lives on the unconstrained DoFs
__global__ void zero_boundary_rows(double* __restrict__ U, int ndx, int ndy, int ndz, int nvec) {
  const long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (node >= (long long)ndx * ndy * ndz) return;
  const int ix = (int)(node % ndx), iy = (int)((node / ndx) % ndy), iz = (int)(node / ((long long)ndx * ndy));
  if (ix == 0 || ix == ndx - 1 || iy == 0 || iy == ndy - 1 || iz == 0 || iz == ndz - 1) {
    double* row = U + node * nvec;
    for (int c = 0; c < nvec; ++c) row[c] = 0.0;
  }
}

// out[c] += sum over the block's rows of (HU[r][c] - lam[c] U[r][c])^2   (line 1 of Alg. 6, squared column norms)
__global__ void residual_sq_kernel(const double* __restrict__ HU, const double* __restrict__ U,
                                   const double* __restrict__ lam, double* __restrict__ out, long long ndof, int nvec,
                                   int cw, long long rows_per_block) {
  const int col0 = threadIdx.x % cw, rsub = threadIdx.x / cw, rstep = blockDim.x / cw;
  const long long r0 = (long long)blockIdx.x * rows_per_block;
  const long long r1 = r0 + rows_per_block < ndof ? r0 + rows_per_block : ndof;
  for (int c = col0; c < nvec; c += cw) {
    const double l = lam[c];
    double acc = 0.0;
    for (long long r = r0 + rsub; r < r1; r += rstep) {
      const double d = fma(-l, U[r * nvec + c], HU[r * nvec + c]);
      acc = fma(d, d, acc);
    }
    if (acc != 0.0) atomicAdd(out + c, acc);
  }
}

// largest eigenvalue of the symmetric tridiagonal (alpha, beta) by bisection on the Sturm count
double tridiag_lambda_max(const std::vector<double>& a, const std::vector<double>& b) {
  const int n = (int)a.size();
  double lo = a[0], hi = a[0];
  for (int i = 0; i < n; ++i) {
    const double r = (i > 0 ? std::fabs(b[i - 1]) : 0.0) + (i + 1 < n ? std::fabs(b[i]) : 0.0);
    lo = std::fmin(lo, a[i] - r); hi = std::fmax(hi, a[i] + r);
  }
  auto count_below = [&](double x) {   // number of eigenvalues < x
    int cnt = 0; double q = 1.0;
    for (int i = 0; i < n; ++i) {
      const double off = (i > 0) ? b[i - 1] * b[i - 1] : 0.0;
      q = a[i] - x - (i > 0 ? off / q : 0.0);
      if (q == 0.0) q = 1e-300;
      if (q < 0.0) ++cnt;
    }
    return cnt;
  };
  for (int it = 0; it < 200 && hi - lo > 4e-16 * std::fmax(std::fabs(lo), std::fabs(hi)); ++it) {
    const double mid = 0.5 * (lo + hi);
    if (count_below(mid) >= n) hi = mid; else lo = mid;
  }
  return 0.5 * (lo + hi);
}

int zero_constrained(fe_chfsi* h, double* U, int nvec, cudaStream_t st) {
  if (h->bc != FE_BC_DIRICHLET) return FE_MF_OK;
  const long long nodes = h->ndof;
  zero_boundary_rows<<<(unsigned)((nodes + 255) / 256), 256, 0, st>>>(U, h->nd[0], h->nd[1], h->nd[2], nvec);
  CH_CUDA(h, cudaGetLastError());
  return FE_MF_OK;
}

// Lower triangle of S = X^T X for the tall block (column-major n x k view A with leading dimension lda; S n x n with
// leading dimension lds).  cuBLAS DSYRK runs this shape at the time of the full DGEMM (61 vs 53 ms for n = 1024,
// k = 884736), i.e. at half the FP64 peak; splitting the columns in two halves turns half of the work into a DGEMM at
// full rate: [S11 . ; S21 S22] with S11, S22 by recursion and S21 = A2 A1^T.
int gram_lower(fe_chfsi* h, const double* A, int lda, int n, int k, double* S, int lds, int depth) {
  const double one = 1.0, zero = 0.0;
  if (depth == 0 || n < 256 || (n & 1)) {
    CH_BLAS(h, cublasDsyrk(h->blas, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_N, n, k, &one, A, lda, &zero, S, lds));
    return FE_MF_OK;
  }
  const int n1 = n / 2;
  int rc = gram_lower(h, A, lda, n1, k, S, lds, depth - 1);
  if (rc == FE_MF_OK) rc = gram_lower(h, A + n1, lda, n - n1, k, S + n1 + (size_t)n1 * lds, lds, depth - 1);
  if (rc != FE_MF_OK) return rc;
  CH_BLAS(h, cublasDgemm(h->blas, CUBLAS_OP_N, CUBLAS_OP_T, n - n1, n1, k, &one, A + n1, lda, A, lda, &zero, S + n1, lds));
  return FE_MF_OK;
}

__global__ void set_identity(double* __restrict__ A, int n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < (long long)n * n) A[i] = (i / n == i % n) ? 1.0 : 0.0;
}

// Cholesky QR, one round (X row-major [ndof][nvec] = column-major nvec x ndof): S = X^T X, S = L L^T,
// dst <- X L^-T (dst != X).  The triangular solve of the tall block is done as a DGEMM with the explicit n x n
// inverse L^-1 (measured on the B200, n = 1024, n_dof = 884736: DTRSM 95 ms, DGEMM 53 ms; the second round removes
// what the explicit inverse loses).  h->T holds L^-1 afterwards.
int cholqr_round(fe_chfsi* h, const double* X, double* dst, cudaStream_t st) {
  const int n = h->nvec, k = (int)h->ndof;
  const double one = 1.0, zero = 0.0;
  {
    const int rc = gram_lower(h, X, n, n, k, h->S, n, h->gram_depth);
    if (rc != FE_MF_OK) return rc;
  }
  CH_SOL(h, cusolverDnDpotrf(h->sol, CUBLAS_FILL_MODE_LOWER, n, h->S, n, h->work, h->lwork, h->info));
  int info = 0;
  CH_CUDA(h, cudaMemcpyAsync(&info, h->info, sizeof(int), cudaMemcpyDeviceToHost, st));
  CH_CUDA(h, cudaStreamSynchronize(st));
  if (info != 0)
    return fail(h, FE_MF_EINVAL, "orthonormalisation: X^T X is not positive definite (block numerically rank deficient, potrf info " +
                                     std::to_string(info) + ")");
  set_identity<<<(unsigned)(((long long)n * n + 255) / 256), 256, 0, st>>>(h->T, n);
  CH_CUDA(h, cudaGetLastError());
  CH_BLAS(h, cublasDtrsm(h->blas, CUBLAS_SIDE_LEFT, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_N, CUBLAS_DIAG_NON_UNIT, n, n, &one,
                         h->S, n, h->T, n));                                                     // T = L^-1
  CH_BLAS(h, cublasDgemm(h->blas, CUBLAS_OP_N, CUBLAS_OP_N, n, k, n, &one, h->T, n, X, n, &zero, dst, n));
  return FE_MF_OK;
}

int set_stream(fe_chfsi* h, cudaStream_t st) {
  CH_BLAS(h, cublasSetStream(h->blas, st));
  CH_SOL(h, cusolverDnSetStream(h->sol, st));
  return FE_MF_OK;
}

int orthonormalize_impl(fe_chfsi* h, double* X, cudaStream_t st) {
  // twice: the first round leaves ||X^T X - I|| ~ eps cond(X)^2, the second brings it to eps  (X -> W -> X)
  int rc = cholqr_round(h, X, h->W, st);
  if (rc == FE_MF_OK) rc = cholqr_round(h, h->W, X, st);
  return rc;
}

// h->res[c] = || HU[:,c] - lam[c] U[:,c] ||^2  (device)
int residual_norms(fe_chfsi* h, const double* HU, const double* U, cudaStream_t st) {
  const int n = h->nvec;
  CH_CUDA(h, cudaMemsetAsync(h->res, 0, sizeof(double) * n, st));
  int cw = 1;
  while (cw * 2 <= n && cw < 256) cw *= 2;
  const long long blocks = 148LL * 8;
  const long long rpb = (h->ndof + blocks - 1) / blocks;
  residual_sq_kernel<<<(unsigned)((h->ndof + rpb - 1) / rpb), 256, 0, st>>>(HU, U, h->lam, h->res, h->ndof, n, cw, rpb);
  CH_CUDA(h, cudaGetLastError());
  return FE_MF_OK;
}

int rayleigh_ritz_impl(fe_chfsi* h, const double* X, double* U, double* evals_host, double* resid_host, cudaStream_t st) {
  const int n = h->nvec, k = (int)h->ndof;
  const double one = 1.0, zero = 0.0;
  CH_CUDA(h, cudaEventRecord(h->ev[2], st));
  CH_OP(h, fe_mf_apply(h->op, X, h->W, n, st));                                                   // W = H Xo
  CH_CUDA(h, cudaEventRecord(h->ev[3], st));
  // T = Xo^T (H Xo)  (line 19); cuSOLVER reads the lower triangle
  CH_BLAS(h, cublasDgemm(h->blas, CUBLAS_OP_N, CUBLAS_OP_T, n, n, k, &one, X, n, h->W, n, &zero, h->T, n));
  CH_CUDA(h, cudaEventRecord(h->ev[4], st));
  CH_SOL(h, cusolverDnDsyevd(h->sol, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, h->T, n, h->lam, h->work,
                             h->lwork, h->info));
  int info = 0;
  CH_CUDA(h, cudaMemcpyAsync(&info, h->info, sizeof(int), cudaMemcpyDeviceToHost, st));
  CH_CUDA(h, cudaEventRecord(h->ev[5], st));
  // U = Xo Q  (line 20): U^T = Q^T Xo^T
  CH_BLAS(h, cublasDgemm(h->blas, CUBLAS_OP_T, CUBLAS_OP_N, n, k, n, &one, h->T, n, X, n, &zero, U, n));
  CH_CUDA(h, cudaEventRecord(h->ev[6], st));
  CH_OP(h, fe_mf_apply(h->op, U, h->W, n, st));                                                   // W = H U
  CH_CUDA(h, cudaEventRecord(h->ev[7], st));
  {
    const int rc = residual_norms(h, h->W, U, st);
    if (rc != FE_MF_OK) return rc;
  }
  CH_CUDA(h, cudaEventRecord(h->ev[0], st));   // reused as the end mark
  std::vector<double> r(n);
  if (evals_host) CH_CUDA(h, cudaMemcpyAsync(evals_host, h->lam, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
  CH_CUDA(h, cudaMemcpyAsync(r.data(), h->res, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
  CH_CUDA(h, cudaStreamSynchronize(st));
  if (info != 0) return fail(h, FE_MF_ECUDA, "cusolverDnDsyevd did not converge (info " + std::to_string(info) + ")");
  if (resid_host) for (int j = 0; j < n; ++j) resid_host[j] = std::sqrt(r[j]);
  float t = 0.f;
  cudaEventElapsedTime(&t, h->ev[2], h->ev[3]); h->ms[2] = t;
  cudaEventElapsedTime(&t, h->ev[6], h->ev[7]); h->ms[2] += t;
  cudaEventElapsedTime(&t, h->ev[3], h->ev[4]); h->ms[3] = t;
  cudaEventElapsedTime(&t, h->ev[5], h->ev[6]); h->ms[3] += t;
  cudaEventElapsedTime(&t, h->ev[4], h->ev[5]); h->ms[4] = t;
  cudaEventElapsedTime(&t, h->ev[7], h->ev[0]); h->ms[5] = t;
  return FE_MF_OK;
}

}  // namespace

extern "C" int fe_chfsi_create(fe_chfsi** out, fe_mf_ctx* op, int nvec) {
  if (!out) return fail(nullptr, FE_MF_EINVAL, "out is NULL");
  *out = nullptr;
  if (!op) return fail(nullptr, FE_MF_EINVAL, "op is NULL");
  if (nvec < 1) return fail(nullptr, FE_MF_EINVAL, "nvec must be >= 1");
  fe_chfsi* h = new (std::nothrow) fe_chfsi();
  if (!h) return fail(nullptr, FE_MF_ENOMEM, "out of host memory");
  h->op = op; h->nvec = nvec; h->ndof = fe_mf_ndofs(op);
  if (getenv("FE_CHFSI_GRAM_DEPTH")) h->gram_depth = atoi(getenv("FE_CHFSI_GRAM_DEPTH"));
  fe_mf_shape(op, h->nd, &h->bc, &h->device);
  if (h->ndof > 2147483647LL || (long long)nvec > h->ndof) {
    delete h;
    return fail(nullptr, FE_MF_EINVAL, "need nvec <= n_dof <= 2^31 - 1 (32-bit library dimensions)");
  }
  DevGuard guard(h->device);
  if (!guard.ok) { delete h; return fail(nullptr, FE_MF_ECUDA, "cudaSetDevice failed"); }
  bool ok = cublasCreate(&h->blas) == CUBLAS_STATUS_SUCCESS && cusolverDnCreate(&h->sol) == CUSOLVER_STATUS_SUCCESS;
  const size_t mv = (size_t)h->ndof * nvec * sizeof(double), mm = (size_t)nvec * nvec * sizeof(double);
  ok = ok && cudaMalloc(&h->Y, mv) == cudaSuccess && cudaMalloc(&h->W, mv) == cudaSuccess;
  ok = ok && cudaMalloc(&h->S, mm) == cudaSuccess && cudaMalloc(&h->T, mm) == cudaSuccess;
  ok = ok && cudaMalloc(&h->lam, nvec * sizeof(double)) == cudaSuccess && cudaMalloc(&h->res, nvec * sizeof(double)) == cudaSuccess;
  ok = ok && cudaMalloc(&h->info, sizeof(int)) == cudaSuccess;
  int l1 = 0, l2 = 0;
  if (ok) {
    ok = cusolverDnDpotrf_bufferSize(h->sol, CUBLAS_FILL_MODE_LOWER, nvec, h->S, nvec, &l1) == CUSOLVER_STATUS_SUCCESS &&
         cusolverDnDsyevd_bufferSize(h->sol, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, nvec, h->T, nvec, h->lam, &l2) ==
             CUSOLVER_STATUS_SUCCESS;
    int l3 = 0;
    ok = ok && cusolverDnDsygvd_bufferSize(h->sol, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, nvec,
                                           h->T, nvec, h->S, nvec, h->lam, &l3) == CUSOLVER_STATUS_SUCCESS;
    h->lwork = l1 > l2 ? l1 : l2;
    if (l3 > h->lwork) h->lwork = l3;
    if (h->lwork < 1) h->lwork = 1;
    ok = ok && cudaMalloc(&h->work, (size_t)h->lwork * sizeof(double)) == cudaSuccess;
  }
  for (int i = 0; ok && i < 8; ++i) ok = cudaEventCreate(&h->ev[i]) == cudaSuccess;
  ok = ok && cudaEventCreate(&h->ev_end) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    fe_chfsi_destroy(h);
    return fail(nullptr, FE_MF_ENOMEM, "workspace allocation or cuBLAS/cuSOLVER initialisation failed");
  }
  *out = h;
  return FE_MF_OK;
}

extern "C" void fe_chfsi_destroy(fe_chfsi* h) {
  if (!h) return;
  DevGuard guard(h->device);
  if (h->blas) cublasDestroy(h->blas);
  if (h->sol) cusolverDnDestroy(h->sol);
  double* bufs[] = {h->Y, h->W, h->S, h->T, h->lam, h->res, h->work, h->lv};
  for (double* b : bufs) if (b) cudaFree(b);
  if (h->info) cudaFree(h->info);
  for (int i = 0; i < 8; ++i) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
  if (h->ev_end) cudaEventDestroy(h->ev_end);
  delete h;
}

extern "C" const char* fe_chfsi_last_error(const fe_chfsi* h) { return h ? h->err.c_str() : g_chfsi_create_err.c_str(); }

extern "C" int fe_chfsi_lanczos_bound(fe_chfsi* h, const double* v0_dev, int k, double* bound_host, void* stream) {
  if (!h) return FE_MF_EINVAL;
  if (!v0_dev || !bound_host || k < 1) return fail(h, FE_MF_EINVAL, "need v0_dev, bound_host, k >= 1");
  DevGuard guard(h->device);
  if (!guard.ok) return fail(h, FE_MF_ECUDA, "cudaSetDevice failed");
  cudaStream_t st = (cudaStream_t)stream;
  int rc = set_stream(h, st);
  if (rc != FE_MF_OK) return rc;
  const int n = (int)h->ndof;
  if (!h->lv && cudaMalloc(&h->lv, 3 * (size_t)n * sizeof(double)) != cudaSuccess) {
    h->lv = nullptr;
    return fail(h, FE_MF_ENOMEM, "cudaMalloc (Lanczos vectors) failed");
  }
  double *v = h->lv, *vp = h->lv + n, *w = h->lv + 2 * (size_t)n;
  CH_CUDA(h, cudaMemcpyAsync(v, v0_dev, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
  CH_CUDA(h, cudaMemsetAsync(vp, 0, sizeof(double) * n, st));
  rc = zero_constrained(h, v, 1, st);
  if (rc != FE_MF_OK) return rc;
  double nrm = 0.0;
  CH_BLAS(h, cublasDnrm2(h->blas, n, v, 1, &nrm));
  if (!(nrm > 0.0)) return fail(h, FE_MF_EINVAL, "Lanczos start vector is zero");
  double s = 1.0 / nrm;
  CH_BLAS(h, cublasDscal(h->blas, n, &s, v, 1));
  std::vector<double> al, be;
  double beta = 0.0;
  for (int j = 0; j < k; ++j) {
    CH_OP(h, fe_mf_apply(h->op, v, w, 1, st));
    double mb = -beta, alpha = 0.0;
    CH_BLAS(h, cublasDaxpy(h->blas, n, &mb, vp, 1, w, 1));
    CH_BLAS(h, cublasDdot(h->blas, n, v, 1, w, 1, &alpha));
    double ma = -alpha;
    CH_BLAS(h, cublasDaxpy(h->blas, n, &ma, v, 1, w, 1));
    CH_BLAS(h, cublasDnrm2(h->blas, n, w, 1, &beta));
    al.push_back(alpha); be.push_back(beta);
    if (beta == 0.0) break;
    s = 1.0 / beta;
    CH_BLAS(h, cublasDscal(h->blas, n, &s, w, 1));
    double* t = vp; vp = v; v = w; w = t;
  }
  std::vector<double> off(be.begin(), be.end() - 1);
  *bound_host = tridiag_lambda_max(al, off) + be.back();
  return FE_MF_OK;
}

extern "C" int fe_chfsi_orthonormalize(fe_chfsi* h, double* X_dev, void* stream) {
  if (!h) return FE_MF_EINVAL;
  if (!X_dev) return fail(h, FE_MF_EINVAL, "X_dev is NULL");
  DevGuard guard(h->device);
  if (!guard.ok) return fail(h, FE_MF_ECUDA, "cudaSetDevice failed");
  cudaStream_t st = (cudaStream_t)stream;
  int rc = set_stream(h, st);
  if (rc == FE_MF_OK) rc = orthonormalize_impl(h, X_dev, st);
  return rc;
}

extern "C" int fe_chfsi_rayleigh_ritz(fe_chfsi* h, const double* X_dev, double* U_dev, double* evals_host,
                                      double* resid_host, void* stream) {
  if (!h) return FE_MF_EINVAL;
  if (!X_dev || !U_dev || X_dev == U_dev) return fail(h, FE_MF_EINVAL, "need distinct X_dev and U_dev");
  DevGuard guard(h->device);
  if (!guard.ok) return fail(h, FE_MF_ECUDA, "cudaSetDevice failed");
  cudaStream_t st = (cudaStream_t)stream;
  int rc = set_stream(h, st);
  if (rc == FE_MF_OK) rc = rayleigh_ritz_impl(h, X_dev, U_dev, evals_host, resid_host, st);
  return rc;
}

extern "C" int fe_chfsi_iterate(fe_chfsi* h, double* U_dev, int m, double lam_max, double lam_u, double lam_min,
                                double* evals_host, double* resid_host, void* stream) {
  if (!h) return FE_MF_EINVAL;
  if (!U_dev) return fail(h, FE_MF_EINVAL, "U_dev is NULL");
  DevGuard guard(h->device);
  if (!guard.ok) return fail(h, FE_MF_ECUDA, "cudaSetDevice failed");
  cudaStream_t st = (cudaStream_t)stream;
  int rc = set_stream(h, st);
  if (rc != FE_MF_OK) return rc;
  rc = zero_constrained(h, U_dev, h->nvec, st);
  if (rc != FE_MF_OK) return rc;
  const int n = h->nvec, k = (int)h->ndof;
  const double one = 1.0, zero = 0.0;
  CH_CUDA(h, cudaEventRecord(h->ev[0], st));
  CH_OP(h, fe_cheb_filter(h->op, U_dev, h->Y, n, m, lam_u, lam_max, lam_min, st));              // lines 2-17: Y
  CH_CUDA(h, cudaEventRecord(h->ev[1], st));
  // line 18, first Cholesky-QR round: X1 = Y L1^-T -> W.  The second round is folded into lines 19-20: with
  // S2 = X1^T X1 = L2 L2^T (= I up to eps cond(Y)^2) the orthonormal block is Xo = X1 L2^-T, and
  // Xo^T H Xo Q = Q Lambda, U = Xo Q  <=>  (X1^T H X1) Z = S2 Z Lambda, Z^T S2 Z = I, U = X1 Z  (Z = L2^-T Q),
  // which DSYGVD solves: one tall DGEMM and the DTRSM of the second round are saved.
  rc = cholqr_round(h, h->Y, h->W, st);
  if (rc != FE_MF_OK) return rc;
  rc = gram_lower(h, h->W, n, n, k, h->S, n, h->gram_depth);                                       // S2
  if (rc != FE_MF_OK) return rc;
  CH_CUDA(h, cudaEventRecord(h->ev[2], st));
  CH_OP(h, fe_mf_apply(h->op, h->W, h->Y, n, st));                                                // Y = H X1
  CH_CUDA(h, cudaEventRecord(h->ev[3], st));
  CH_BLAS(h, cublasDgemm(h->blas, CUBLAS_OP_N, CUBLAS_OP_T, n, n, k, &one, h->W, n, h->Y, n, &zero, h->T, n));   // X1^T H X1
  CH_CUDA(h, cudaEventRecord(h->ev[4], st));
  CH_SOL(h, cusolverDnDsygvd(h->sol, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, h->T, n,
                             h->S, n, h->lam, h->work, h->lwork, h->info));                       // line 19
  int info = 0;
  CH_CUDA(h, cudaMemcpyAsync(&info, h->info, sizeof(int), cudaMemcpyDeviceToHost, st));
  CH_CUDA(h, cudaEventRecord(h->ev[5], st));
  CH_BLAS(h, cublasDgemm(h->blas, CUBLAS_OP_T, CUBLAS_OP_N, n, k, n, &one, h->T, n, h->W, n, &zero, U_dev, n));  // line 20
  CH_CUDA(h, cudaEventRecord(h->ev[6], st));
  CH_OP(h, fe_mf_apply(h->op, U_dev, h->Y, n, st));                                               // Y = H U
  CH_CUDA(h, cudaEventRecord(h->ev[7], st));
  rc = residual_norms(h, h->Y, U_dev, st);                                                        // line 1
  if (rc != FE_MF_OK) return rc;
  cudaEvent_t end = h->ev_end;
  CH_CUDA(h, cudaEventRecord(end, st));
  std::vector<double> r(n);
  if (evals_host) CH_CUDA(h, cudaMemcpyAsync(evals_host, h->lam, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
  CH_CUDA(h, cudaMemcpyAsync(r.data(), h->res, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
  CH_CUDA(h, cudaStreamSynchronize(st));
  if (info != 0)
    return fail(h, info > n ? FE_MF_EINVAL : FE_MF_ECUDA,
                info > n ? "orthonormalisation: second-round Gram matrix not positive definite" : "cusolverDnDsygvd did not converge");
  if (resid_host) for (int j = 0; j < n; ++j) resid_host[j] = std::sqrt(r[j]);
  auto el = [](cudaEvent_t a, cudaEvent_t b) { float t = 0.f; cudaEventElapsedTime(&t, a, b); return (double)t; };
  h->ms[0] = el(h->ev[0], h->ev[1]);
  h->ms[1] = el(h->ev[1], h->ev[2]);
  h->ms[2] = el(h->ev[2], h->ev[3]) + el(h->ev[6], h->ev[7]);
  h->ms[3] = el(h->ev[3], h->ev[4]) + el(h->ev[5], h->ev[6]);
  h->ms[4] = el(h->ev[4], h->ev[5]);
  h->ms[5] = el(h->ev[7], end);
  return FE_MF_OK;
}

extern "C" int fe_chfsi_solve(fe_chfsi* h, double* U_dev, int n_wanted, int m, double lam_max, double lam_u,
                              double lam_min, double tau, int max_iter, double* evals_host, double* resid_host,
                              int* iters_host, void* stream) {
  if (!h) return FE_MF_EINVAL;
  if (n_wanted < 1 || n_wanted > h->nvec || h->nvec < 2 || max_iter < 1 || !(tau > 0.0))
    return fail(h, FE_MF_EINVAL, "need 1 <= n_wanted <= nvec, nvec >= 2, max_iter >= 1, tau > 0");
  std::vector<double> lam(h->nvec), res(h->nvec);
  int it = 0;
  for (it = 1; it <= max_iter; ++it) {
    const int rc = fe_chfsi_iterate(h, U_dev, m, lam_max, lam_u, lam_min, lam.data(), res.data(), stream);
    if (rc != FE_MF_OK) return rc;
    double worst = 0.0;
    for (int j = 0; j < n_wanted; ++j) worst = std::fmax(worst, res[j]);
    if (worst <= tau) break;
    lam_min = lam[0]; lam_u = lam[h->nvec - 1];
  }
  if (it > max_iter) it = max_iter;
  if (evals_host) std::memcpy(evals_host, lam.data(), sizeof(double) * h->nvec);
  if (resid_host) std::memcpy(resid_host, res.data(), sizeof(double) * h->nvec);
  if (iters_host) *iters_host = it;
  return FE_MF_OK;
}

extern "C" int fe_chfsi_last_timings(const fe_chfsi* h, double ms_host[6]) {
  if (!h || !ms_host) return FE_MF_EINVAL;
  for (int i = 0; i < 6; ++i) ms_host[i] = h->ms[i];
  return FE_MF_OK;
}
