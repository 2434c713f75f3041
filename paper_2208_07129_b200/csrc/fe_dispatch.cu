// Kernel selection and the stream-ordered entry points of include/fe_mf.h (host code only; the kernels live in the
// fe_tu_*.cu translation units and are reached through the launchers declared in fe_ctx.h).
//
// Kernels:
//   kind 8  fe_apply_cart_plane  uniform Cartesian cells, p = 6: one n x n plane of one vector per thread
//   kind 9  fe_apply_cart_line   uniform Cartesian cells, any p: one line of two vectors per thread
//   kind 6  fe_apply_gen_tma     full symmetric metric (per-q-point or per-cell geometry)
//   kind 2  fe_apply_cart        Cartesian, odd nvec or unaligned pointers (LDG gather / RED scatter)
//   kind 3  fe_apply_cart<CELLS> Cartesian, 1-3 vectors: the tile slots hold several cells of an x-row
//   kind 1  fe_apply_general     anything else (nvec = 1, odd nvec with a full metric): plain contractions
//   kind 11 fe_apply_oi / fe_apply_general_oi   n_q != n_p points per direction
// fe_mf_set_variant forces a kind for tests and profiling: 1 -> kind 1, 2 -> kind 2, 7 -> kind 6 on a Cartesian
// mesh, 8 -> plane, 10 -> line with 16-vector blocks, 11 -> line with 8-vector blocks; 22 / 23 -> fe_mf_apply_host always in
// column chunks / in z-slabs whatever the size.
#include <cstring>

#include "fe_ctx.h"

using fe_host::fail;
using fe_host::DeviceGuard;

namespace {

// ---- tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn lookup_encode_tiled() {
  void* p = nullptr;
  cudaDriverEntryPointQueryResult q;
  EncodeTiledFn fn = nullptr;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
      q == cudaDriverEntryPointSuccess)
    fn = (EncodeTiledFn)p;
  (void)cudaGetLastError();
  return fn;
}
EncodeTiledFn encode_tiled_fn() {
  static const EncodeTiledFn fn = lookup_encode_tiled();   // a driver entry point: process-wide, initialised once (thread-safe)
  return fn;
}

// 4-D FP64 tensor map of a multivector [z][y][x][beta] with box (bv, n, n, n): the numbers come from fe::tensor_map_desc
// (fe_params.h: trimming for Dirichlet meshes, cut planes of slabs, the pad node of the 8-vector line kernels)
bool make_tensor_map(CUtensorMap* tm, const fe_mf_ctx* c, const void* base, int nvec, int bv, int trim = 0, int padx = 0) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  fe::TensorMapDesc d;
  if (!fe::tensor_map_desc(d, c->ndx, c->ndy, c->ndz, c->n, c->zopen, nvec, bv, trim, padx)) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)d.dims[0], (cuuint64_t)d.dims[1], (cuuint64_t)d.dims[2], (cuuint64_t)d.dims[3]};
  const cuuint64_t strides[3] = {(cuuint64_t)d.strides[0], (cuuint64_t)d.strides[1], (cuuint64_t)d.strides[2]};
  base = (const char*)base + d.base_offset;
  const cuuint32_t box[4] = {(cuuint32_t)d.box[0], (cuuint32_t)d.box[1], (cuuint32_t)d.box[2], (cuuint32_t)d.box[3]};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int line_bv(const fe_mf_ctx* c, int nvec) {
  if (c->p == 8 || c->variant == 11 || nvec <= 8) return 8;
  if (c->p == 7 && c->variant != 10) return 8;
  return 16;
}

// ---- which kernel serves (ctx, nvec, pointers)
int pick_kernel(const fe_mf_ctx* c, int nvec, const void* W, const void* Z) {
  if (c->nq_oi) return 11;   // n_q != n_p: only the plain kernel with rectangular tables
  if (c->variant == 1) return 1;
  // NEXT-1 operator: a uniform box with mass scaling runs on the Cartesian TMA kernels instantiated with EIG (kappa per
  // point, M^-1/2 inside the interpolation tables); kappa without mass scaling on such a context only on the general
  // kernel; every other mesh on the full-metric kernels (kinds 6, 1), which read d = diag(M)^-1/2 from memory
  const bool msc = c->mass_scaled;
  const bool eig = msc && c->geom_mode == 0;
  if (c->kappa_dev && !msc) return 1;
  const bool diag = (!msc || eig) && (c->geom_mode == 0) && c->ug[1] == 0.0 && c->ug[2] == 0.0 && c->ug[4] == 0.0;
  const bool aligned = ((((uintptr_t)W) | ((uintptr_t)Z)) & 15) == 0;
  const bool tma_ok = !(nvec & 1) && aligned && encode_tiled_fn() &&
                      (unsigned long long)nvec * 8ULL * c->ndx * c->ndy < (1ULL << 40) &&
                      c->ncells * ((nvec + 7) / 8) < (1LL << 31);
  const bool trim_ok = (c->bc != FE_BC_DIRICHLET) || (c->ndx >= 3 && c->ndy >= 3 && c->ndz >= 3);
  if (eig) {   // kinds 8 / 9 or the general kernel (which then reads d and kappa from memory)
    if (!tma_ok || !trim_ok || nvec < 4 || c->variant == 2 || c->variant == 7) return 1;
  } else {
    if ((!diag || c->variant == 7) && tma_ok) return 6;
    if (!diag) return 1;
    if (nvec < 4) return 3;
    if (!tma_ok || c->variant == 2) return 2;
    if (!trim_ok) return 2;
  }
  if (c->variant == 10 || c->variant == 11) return 9;
  if (c->variant == 8 && c->p == 6) return 8;
  // plane kernel: 16 vectors per block; worth it when the last block of vectors is mostly full
  const int tail = nvec % 16;
  if (c->p == 6 && nvec >= 12 && (tail == 0 || tail >= 12)) return 8;
  return 9;
}
int kernel_bv(const fe_mf_ctx* c, int kind, int nvec) {
  switch (kind) {
    case 1: return fe_host::general_bv(c->p, nvec);
    case 2: return 8;
    case 3: return nvec;
    case 6: return fe_host::gen_bv(c, nvec);
    case 8: return 16;
    case 11: return fe_host::oi_bv(c->nq_oi, nvec);
    default: return line_bv(c, nvec);
  }
}

fe::ApplyParams make_params(const fe_mf_ctx* c, const double* W, double* Z, double alpha, int nvec, int bv) {
  fe::ApplyParams P;
  P.W = W; P.Z = Z; P.geom = c->geom_dev;
  for (int k = 0; k < 7; ++k) P.ug[k] = c->ug[k];
  P.alpha = alpha;
  P.ncx = c->ncx; P.ncy = c->ncy; P.ncz = c->ncz;
  P.ndx = c->ndx; P.ndy = c->ndy; P.ndz = c->ndz;
  P.nvec = nvec; P.bv = bv; P.nvb = (nvec + bv - 1) / bv;
  P.dirichlet = (c->bc == FE_BC_DIRICHLET) ? 1 : 0;
  P.zopen = c->zopen;
  P.geom_mode = c->geom_mode;
  P.nsm = c->nsm;
  P.geom_stride = c->geom_stride;
  P.item_ctr = fe_host::item_counter(c);
  P.item0 = 0; P.item_count = 0;
  P.idw = 0.0;
  P.dscale = c->mass_scaled ? c->dscale_dev : nullptr;
  P.kappa = c->kappa_dev;
  if (P.kappa) P.ug[6] = c->detj0;   // mass factor = det J * kappa_Q
  return P;
}

// Can this kernel add a multiple of W (identity term, partition-of-unity weights) in the same pass?  The Cartesian
// plane and line kernels, at every node they write: all nodes on periodic meshes, the interior nodes on Dirichlet
// meshes (the boundary nodes never enter a tile: callers treat them separately).
bool kind_adds_identity(const fe_mf_ctx* c, int kind) { return (kind == 8 && c->p == 6) || kind == 9; }

// Z += alpha * A * W  (Z already initialised); idw != 0 (only if kind_adds_identity): Z += alpha A W + idw W in one
// launch.  Counts launches into c->last_launches.
int launch_accumulate(fe_mf_ctx* c, double alpha, const double* W, double* Z, int nvec, cudaStream_t st, double idw = 0.0,
                      int item0 = 0, int item_count = 0) {
  const int kind = pick_kernel(c, nvec, W, Z);
  const int bv = kernel_bv(c, kind, nvec);
  fe::ApplyParams P = make_params(c, W, Z, alpha, nvec, bv);
  P.idw = idw;
  P.item0 = item0; P.item_count = item_count;   // persistent kernels only (kinds 6, 8, 9): a range of cell layers
  if (c->ncells * (long long)P.nvb > 2147483647LL) return fail(c, FE_MF_EINVAL, "grid too large");
  cudaError_t e = cudaErrorInvalidValue;
  CUtensorMap tw, tz;
  if (kind == 6 || kind == 8 || kind == 9) {
    // Cartesian kernels on Dirichlet meshes: boundary nodes are out of bounds of the maps (see make_tensor_map)
    const bool trim = (kind != 6) && (c->bc == FE_BC_DIRICHLET);
    const int padx = (kind == 9) ? fe_host::line_padx(c->p, bv) : 0;
    if (!make_tensor_map(&tw, c, W, nvec, bv, trim ? 2 : 0, padx) || !make_tensor_map(&tz, c, Z, nvec, bv, trim ? 1 : 0, padx))
      return fail(c, FE_MF_ECUDA, "cuTensorMapEncodeTiled failed");
  }
  if (kind == 8 || kind == 9 || kind == 2 || kind == 3)
    for (int k = 0; k < 7; ++k) P.ug[k] *= alpha;   // Cartesian kernels: the result is linear in the metric constants
  if ((kind == 8 || kind == 9) && c->mass_scaled) {
    // EIG kernels: diag(M)^-1/2 = (det J)^-1/2 kron diag(w~)^-1/2; the tables carry the second factor (both sides)
    for (int k = 0; k < 7; ++k) P.ug[k] /= c->detj0;
    P.dscale = nullptr;
  }
  if (kind == 11) {
    // the compile-time kernel takes its tiles through TMA under the same conditions as the other TMA kernels
    const bool aligned = ((((uintptr_t)W) | ((uintptr_t)Z)) & 15) == 0;
    const bool use_tma = fe_host::oi_compile_time_kernel(c, nvec) && !(nvec & 1) && aligned && c->variant != 1 &&
                         make_tensor_map(&tw, c, W, nvec, bv, 0, 0) && make_tensor_map(&tz, c, Z, nvec, bv, 0, 0);
    e = fe_host::launch_oi(c, P, use_tma ? &tw : nullptr, use_tma ? &tz : nullptr, st);
  } else if (kind == 6) {
    e = fe_host::launch_gen(c, P, tw, tz, st);
  } else if (kind == 8) {
    e = fe_host::launch_plane(c, P, tw, tz, st);
  } else if (kind == 9) {
    e = (bv == 16) ? fe_host::launch_line16(c, P, tw, tz, st) : fe_host::launch_line8(c, P, tw, tz, st);
  } else if (kind == 3) {
    P.alpha = 1.0;
    e = fe_host::launch_cart_cells(c, P, st);
  } else if (kind == 2) {
    P.alpha = 1.0;
    e = fe_host::launch_cart(c, P, st);
  } else {
    e = fe_host::launch_general(c, P, st);
  }
  if (e != cudaSuccess) return fail(c, FE_MF_ECUDA, std::string("apply kernel launch: ") + cudaGetErrorString(e));
  c->last_launches += 1;
  return FE_MF_OK;
}

// Z <- beta*Z + gamma*W, stream-ordered (S1 / the axpby half of S9).
int launch_init(fe_mf_ctx* c, double* Z, const double* W, double beta, double gamma, size_t count, cudaStream_t st) {
  if (beta == 0.0 && gamma == 0.0) {
    FE_CUDA(c, cudaMemsetAsync(Z, 0, count * sizeof(double), st));   // a driver memset: not counted as a kernel launch
    return FE_MF_OK;
  }
  if (beta == 0.0) FE_CUDA(c, fe_host::launch_scale_copy(Z, W, gamma, count, st));
  else FE_CUDA(c, fe_host::launch_axpby(Z, W, beta, gamma, count, st));
  c->last_launches += 1;
  return FE_MF_OK;
}

int check_io(fe_mf_ctx* c, const double* W, const double* Z, int nvec) {
  if (!c) return FE_MF_EINVAL;
  if (!W || !Z) return fail(c, FE_MF_EINVAL, "null device pointer");
  if (nvec < 1) return fail(c, FE_MF_EINVAL, "nvec must be >= 1");
  const size_t bytes = (size_t)c->ndof * nvec * sizeof(double);
  const char* a = (const char*)W; const char* b = (const char*)Z;
  if (a < b + bytes && b < a + bytes) return fail(c, FE_MF_EINVAL, "input and output alias");
  return FE_MF_OK;
}

}  // namespace

extern "C" int fe_mf_apply_axpby(fe_mf_ctx* ctx, double alpha, const double* W_dev, double beta, double gamma,
                                 double* Z_dev, int nvec, void* cuda_stream) {
  int rc = check_io(ctx, W_dev, Z_dev, nvec);
  if (rc) return rc;
  DeviceGuard guard(ctx->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  ctx->last_launches = 0;
  const size_t count = (size_t)ctx->ndof * nvec;
  const int kind = pick_kernel(ctx, nvec, W_dev, Z_dev);
  if (kind_adds_identity(ctx, kind) && gamma != 0.0 && ctx->bc == FE_BC_PERIODIC && !ctx->zopen) {
    // the kernel adds gamma W itself (IDENT): the separate pass only has to scale Z (or zero it)
    if (beta == 0.0) {
      FE_CUDA(ctx, cudaMemsetAsync(Z_dev, 0, count * sizeof(double), st));
    } else if (beta != 1.0) {
      FE_CUDA(ctx, fe_host::launch_scale(Z_dev, beta, count, st));
      ctx->last_launches += 1;
    }
    return launch_accumulate(ctx, alpha, W_dev, Z_dev, nvec, st, gamma);
  }
  rc = launch_init(ctx, Z_dev, W_dev, beta, gamma, count, st);
  if (rc) return rc;
  return launch_accumulate(ctx, alpha, W_dev, Z_dev, nvec, st);
}

extern "C" int fe_mf_accumulate(fe_mf_ctx* ctx, double alpha, const double* W_dev, double* Z_dev, int nvec,
                                void* cuda_stream) {
  int rc = check_io(ctx, W_dev, Z_dev, nvec);
  if (rc) return rc;
  DeviceGuard guard(ctx->device);
  ctx->last_launches = 0;
  return launch_accumulate(ctx, alpha, W_dev, Z_dev, nvec, (cudaStream_t)cuda_stream);
}

extern "C" int fe_mf_apply(fe_mf_ctx* ctx, const double* X_dev, double* Y_dev, int nvec, void* cuda_stream) {
  return fe_mf_apply_axpby(ctx, 1.0, X_dev, 0.0, 0.0, Y_dev, nvec, cuda_stream);
}

// BCV layout (Fig. 1): n_b = ceil(nvec / b) batches, batch i_b = the [ndof][b_i] block of vectors
// i_b b .. i_b b + b_i - 1 stored contiguously at offset ndof * i_b * b.  Each batch is a multivector of the simple
// layout, so the batched apply is one fe_mf_apply per batch on the same stream (Eq. 17's sum over i_b).
extern "C" int fe_mf_apply_bcv(fe_mf_ctx* ctx, const double* X_dev, double* Y_dev, int b, int nvec, void* cuda_stream) {
  if (!ctx) return FE_MF_EINVAL;
  if (!X_dev || !Y_dev) return fail(ctx, FE_MF_EINVAL, "null device pointer");
  if (b < 1 || nvec < 1) return fail(ctx, FE_MF_EINVAL, "b and nvec must be >= 1");
  const size_t total = (size_t)ctx->ndof * nvec;
  if (X_dev < Y_dev + total && Y_dev < X_dev + total) return fail(ctx, FE_MF_EINVAL, "X and Y must not overlap");
  int launches = 0;
  for (int v0 = 0; v0 < nvec; v0 += b) {
    const int bi = (v0 + b <= nvec) ? b : (nvec - v0);
    const size_t off = (size_t)ctx->ndof * v0;
    const int rc = fe_mf_apply(ctx, X_dev + off, Y_dev + off, bi, cuda_stream);
    if (rc) return rc;
    launches += ctx->last_launches;
  }
  ctx->last_launches = launches;
  return FE_MF_OK;
}

namespace {

// The scale factors s_k of the one-launch-per-step form of the recurrence (see fe_cheb_filter): s_0 = s_1 = 1,
// s_{k+1} = b_k s_{k-1} with b_k = -sigma sigma_2.  |s_k| shrinks like |b|^(k/2); with a narrow damping interval far
// from a0 (|sigma| << 1) it underflows long before m = 200 and a_k s_k / s_{k+1} becomes 0/0.  True if every s_k of a
// degree-m filter stays a comfortably normal number.
bool scaled_recurrence_is_safe(int m, double e, double c, double a0) {
  double sigma = e / (a0 - c);
  const double gamma = 2.0 / sigma;
  double s_prev = 1.0, s_cur = 1.0;
  for (int d = 2; d <= m; ++d) {
    const double sigma2 = 1.0 / (gamma - sigma);
    const double s_next = -sigma * sigma2 * s_prev;
    if (!(std::fabs(s_next) > 1e-250) || !(std::fabs(s_next) < 1e250)) return false;
    s_prev = s_cur; s_cur = s_next;
    sigma = sigma2;
  }
  return true;
}

}  // namespace

extern "C" int fe_cheb_filter(fe_mf_ctx* ctx, double* X_dev, double* Y_dev, int nvec, int m, double a, double b,
                              double a0, void* cuda_stream) {
  int rc = check_io(ctx, X_dev, Y_dev, nvec);
  if (rc) return rc;
  if (ctx->zopen) return fail(ctx, FE_MF_EUNSUPPORTED, "fe_cheb_filter on a slab context: every step needs a halo exchange (use fe_mf_apply_axpby per step)");
  if (m < 1) return fail(ctx, FE_MF_EINVAL, "m must be >= 1");
  if (!(b > a)) return fail(ctx, FE_MF_EINVAL, "need b > a (inverted or empty damping interval)");
  if (!(a0 < a)) return fail(ctx, FE_MF_EINVAL, "need a0 < a");
  DeviceGuard guard(ctx->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t count = (size_t)ctx->ndof * nvec;
  int launches = 0;
  // Alg. 6 lines 2-9 (garbled lines per DESIGN.md reading 10)
  const double e = (b - a) / 2.0;
  const double c = (b + a) / 2.0;
  double sigma = e / (a0 - c);
  const double sigma1 = sigma;
  const double gamma = 2.0 / sigma1;
  double alpha1 = sigma1 / e;
  double alpha2 = -c;
  double* X = X_dev; double* Y = Y_dev;
  if (c != 0.0 && kind_adds_identity(ctx, pick_kernel(ctx, nvec, X_dev, Y_dev)) && scaled_recurrence_is_safe(m, e, c, a0)) {
    // The same recurrence, X_1 = a_0 (A - cI) X_0, X_{k+1} = a_k (A - cI) X_k + b_k X_{k-1}  (a_0 = sigma_1/e,
    // a_k = 2 sigma_2/e, b_k = -sigma sigma_2), in the scaled variables X_k = s_k U_k with s_0 = s_1 = 1,
    // s_{k+1} = b_k s_{k-1}:   U_{k+1} = U_{k-1} + (a_k s_k / s_{k+1}) (A - cI) U_k.
    // Every step is then ONE accumulate launch into the buffer of U_{k-1} (the kernels add the -cI part with
    // partition-of-unity weights): no axpby pass.  s_m and s_{m-1} are applied once at the end.  (Filters whose s_k
    // would leave the normal range -- checked above on the host -- take the unscaled path below.)  Dirichlet meshes:
    // the kernels neither read nor write the boundary nodes, whose entries obey the scalar recurrence with A = 0
    // (q_k); X_dev keeps the input there until the final kernel writes q_m x0 and q_{m-1} x0.
    FE_CUDA(ctx, cudaMemsetAsync(Y, 0, count * sizeof(double), st));
    ctx->last_launches = 0;
    rc = launch_accumulate(ctx, alpha1, X, Y, nvec, st, -c * alpha1);
    if (rc) return rc;
    launches += ctx->last_launches;
    double s_prev = 1.0, s_cur = 1.0;
    double q_prev = 1.0, q_cur = -c * alpha1;   // the same recurrence at a boundary node of a Dirichlet mesh: (A X) = 0 there
    double* Uprev = X; double* Ucur = Y;
    for (int d = 2; d <= m; ++d) {
      const double sigma2 = 1.0 / (gamma - sigma);
      alpha1 = 2.0 * sigma2 / e;
      alpha2 = -sigma * sigma2;
      const double s_next = alpha2 * s_prev;
      const double al = alpha1 * s_cur / s_next;
      const double q_next = -c * alpha1 * q_cur + alpha2 * q_prev;
      q_prev = q_cur; q_cur = q_next;
      ctx->last_launches = 0;
      rc = launch_accumulate(ctx, al, Ucur, Uprev, nvec, st, -c * al);
      if (rc) return rc;
      launches += ctx->last_launches;
      double* t = Uprev; Uprev = Ucur; Ucur = t;
      s_prev = s_cur; s_cur = s_next;
      sigma = sigma2;
    }
    // Y_dev <- s_m U_m, X_dev <- s_{m-1} U_{m-1}
    const int swap = (Ucur != Y_dev) ? 1 : 0;
    const int bnd = (ctx->bc == FE_BC_DIRICHLET) ? 1 : 0;
    if (swap || bnd || s_cur != 1.0 || s_prev != 1.0) {
      FE_CUDA(ctx, fe_host::launch_scale2(X_dev, Y_dev, s_prev, s_cur, swap, count, bnd, q_prev, q_cur, ctx->ndx, ctx->ndy,
                                          ctx->ndz, nvec, st));
      launches += 1;
    }
    ctx->last_launches = launches;
    return FE_MF_OK;
  }
  // line 10: Y <- alpha1 A X + alpha1 alpha2 X
  rc = fe_mf_apply_axpby(ctx, alpha1, X, 0.0, alpha1 * alpha2, Y, nvec, cuda_stream);
  if (rc) return rc;
  launches += ctx->last_launches;
  for (int d = 2; d <= m; ++d) {
    const double sigma2 = 1.0 / (gamma - sigma);
    alpha1 = 2.0 * sigma2 / e;
    alpha2 = -sigma * sigma2;
    // line 15: X <- alpha1 A Y + alpha2 X - c alpha1 Y ; line 16: swap
    rc = fe_mf_apply_axpby(ctx, alpha1, Y, alpha2, -(c * alpha1), X, nvec, cuda_stream);
    if (rc) return rc;
    launches += ctx->last_launches;
    double* t = X; X = Y; Y = t;
    sigma = sigma2;
  }
  if (Y != Y_dev) {  // m even: the result sits in the caller's X buffer; exchange contents
    FE_CUDA(ctx, fe_host::launch_swap(X_dev, Y_dev, count, st));
    launches += 1;
  }
  ctx->last_launches = launches;
  return FE_MF_OK;
}

namespace {

// fe_mf_apply_host, pipelined over z-SLABS of the mesh (the persistent TMA kernels only: they take item ranges).
// The multivector is z-major, so a range of node planes is ONE contiguous block on both sides of the bus: the copies
// run at the full pinned rate (55 GB/s each way measured on the box, 49 GB/s with both directions busy), whereas a
// column chunk is a strided 2-D copy of 128-byte rows (the column-chunk path below: 29 GB/s each way).  Chunk k =
// cell layers lay[k] .. lay[k+1]: its kernel (an item range of the one persistent kernel) needs the node planes up to
// lay[k+1] p, starts when their copy has landed, and leaves planes lay[k] p .. lay[k+1] p - 1 of Y final (the top
// plane also receives from chunk k+1; on a periodic mesh plane 0 also from the last chunk, so it travels last).
// Three internal streams: H2D, kernels, D2H.  Needs the whole X and Y on the device (2 ndof nvec doubles).
int apply_host_slabs(fe_mf_ctx* ctx, const double* X_host, double* Y_host, int nvec, int nchunks) {
  const size_t total = (size_t)ctx->ndof * nvec;
  if (ctx->ws_elems < total) {
    if (ctx->ws_x) cudaFree(ctx->ws_x);
    if (ctx->ws_y) cudaFree(ctx->ws_y);
    ctx->ws_x = ctx->ws_y = nullptr; ctx->ws_elems = 0;
    if (cudaMalloc(&ctx->ws_x, total * sizeof(double)) != cudaSuccess || cudaMalloc(&ctx->ws_y, total * sizeof(double)) != cudaSuccess) {
      if (ctx->ws_x) cudaFree(ctx->ws_x);
      ctx->ws_x = nullptr; (void)cudaGetLastError();
      return FE_MF_ENOMEM;   // the caller falls back to the column-chunk path
    }
    ctx->ws_elems = total;
  }
  for (cudaStream_t& s_ : ctx->hs)
    if (!s_) FE_CUDA(ctx, cudaStreamCreateWithFlags(&s_, cudaStreamNonBlocking));
  while ((int)ctx->hev.size() < 2 * nchunks) {
    cudaEvent_t ev;
    FE_CUDA(ctx, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    ctx->hev.push_back(ev);
  }
  cudaStream_t sin = ctx->hs[0], sk = ctx->hs[1], sout = ctx->hs[2];
  double *dx = ctx->ws_x, *dy = ctx->ws_y;
  const size_t plane = (size_t)ctx->ndx * ctx->ndy * nvec;
  const bool periodic = ctx->bc == FE_BC_PERIODIC && !ctx->zopen;
  const int kind = pick_kernel(ctx, nvec, dx, dy);
  const int bv = kernel_bv(ctx, kind, nvec);
  const long long layer_items = (long long)ctx->ncx * ctx->ncy * ((nvec + bv - 1) / bv);
  FE_CUDA(ctx, cudaMemsetAsync(dy, 0, total * sizeof(double), sk));
  int first_in = 0, launches = 0, rc = FE_MF_OK;
  for (int k = 0; k < nchunks && rc == FE_MF_OK; ++k) {
    const int l0 = (int)((long long)ctx->ncz * k / nchunks), l1 = (int)((long long)ctx->ncz * (k + 1) / nchunks);
    int last_in = l1 * ctx->p;                             // top node plane the chunk's cells read
    if (last_in > ctx->ndz - 1) last_in = ctx->ndz - 1;    // periodic: the top plane of the last layer is plane 0, copied first
    if (last_in >= first_in) {
      FE_CUDA(ctx, cudaMemcpyAsync(dx + (size_t)first_in * plane, X_host + (size_t)first_in * plane,
                                   (size_t)(last_in - first_in + 1) * plane * sizeof(double), cudaMemcpyHostToDevice, sin));
      first_in = last_in + 1;
    }
    FE_CUDA(ctx, cudaEventRecord(ctx->hev[2 * k], sin));
    FE_CUDA(ctx, cudaStreamWaitEvent(sk, ctx->hev[2 * k], 0));
    ctx->ctrl_slot = 1;
    ctx->last_launches = 0;
    rc = launch_accumulate(ctx, 1.0, dx, dy, nvec, sk, 0.0, (int)(l0 * layer_items), (int)((l1 - l0) * layer_items));
    ctx->ctrl_slot = 0;
    if (rc) break;
    launches += ctx->last_launches;
    FE_CUDA(ctx, cudaEventRecord(ctx->hev[2 * k + 1], sk));
    FE_CUDA(ctx, cudaStreamWaitEvent(sout, ctx->hev[2 * k + 1], 0));
    // planes final after this chunk: lay[k] p .. lay[k+1] p - 1 (the last chunk: up to the end); periodic plane 0 waits
    int o0 = l0 * ctx->p, o1 = (k == nchunks - 1) ? ctx->ndz - 1 : l1 * ctx->p - 1;
    if (periodic && k == 0) o0 = 1;
    if (o1 >= o0)
      FE_CUDA(ctx, cudaMemcpyAsync(Y_host + (size_t)o0 * plane, dy + (size_t)o0 * plane, (size_t)(o1 - o0 + 1) * plane * sizeof(double),
                                   cudaMemcpyDeviceToHost, sout));
    if (periodic && k == nchunks - 1)
      FE_CUDA(ctx, cudaMemcpyAsync(Y_host, dy, plane * sizeof(double), cudaMemcpyDeviceToHost, sout));
  }
  for (cudaStream_t s_ : ctx->hs) FE_CUDA(ctx, cudaStreamSynchronize(s_));
  if (rc) return rc;
  ctx->last_launches = launches;
  return FE_MF_OK;
}

}  // namespace

extern "C" int fe_mf_apply_host(fe_mf_ctx* ctx, const double* X_host, double* Y_host, int nvec) {
  if (!ctx) return FE_MF_EINVAL;
  if (!X_host || !Y_host) return fail(ctx, FE_MF_EINVAL, "null host pointer");
  if (nvec < 1) return fail(ctx, FE_MF_EINVAL, "nvec must be >= 1");
  DeviceGuard guard(ctx->device);
  {
    // large outputs on the persistent TMA kernels: z-slab pipeline with contiguous copies (variant 22 switches it off)
    const int kind = pick_kernel(ctx, nvec, nullptr, nullptr);
    const size_t bytes = (size_t)ctx->ndof * nvec * sizeof(double);
    int nchunks = ctx->ncz < 12 ? ctx->ncz : 12;
    const long long layer_items = (long long)ctx->ncx * ctx->ncy * ((nvec + kernel_bv(ctx, kind, nvec) - 1) / kernel_bv(ctx, kind, nvec));
    const bool force = ctx->variant == 23;   // tests: the slab pipeline on meshes of any size
    while (!force && nchunks > 1 && (long long)(ctx->ncz / nchunks) * layer_items < 2LL * 2 * ctx->nsm) --nchunks;   // >= 2 items per resident block
    if ((kind == 6 || kind == 8 || kind == 9) && ctx->variant != 22 &&
        (force ? nchunks >= 2 : (nchunks >= 3 && bytes >= ((size_t)32 << 20)))) {
      const int rc = apply_host_slabs(ctx, X_host, Y_host, nvec, nchunks);
      if (rc != FE_MF_ENOMEM) return rc;
    }
  }
  // column chunks: copies of chunk k+1 / k-1 overlap the kernels of chunk k on two streams
  // (at least 16 columns = 128-byte rows per chunk: strided host copies with 64-byte rows ran at half the rate;
  // measured on config 2: 1 chunk 42 ms, 2 chunks of 16 columns 30 ms, 4 chunks of 8 columns 43 ms)
  int cw = (nvec + 3) / 4;
  if (cw < 16) cw = 16;
  cw = (cw + 3) / 4 * 4;
  if (cw > nvec) cw = nvec;
  const int nchunks = (nvec + cw - 1) / cw;
  const size_t per = (size_t)ctx->ndof * cw;
  const int nbuf = nchunks > 1 ? 2 : 1;
  if (ctx->ws_elems < per * nbuf) {
    if (ctx->ws_x) cudaFree(ctx->ws_x);
    if (ctx->ws_y) cudaFree(ctx->ws_y);
    ctx->ws_x = ctx->ws_y = nullptr; ctx->ws_elems = 0;
    if (cudaMalloc(&ctx->ws_x, per * nbuf * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&ctx->ws_y, per * nbuf * sizeof(double)) != cudaSuccess) {
      if (ctx->ws_x) cudaFree(ctx->ws_x);
      ctx->ws_x = nullptr; (void)cudaGetLastError();
      return fail(ctx, FE_MF_ENOMEM, "device workspace allocation failed");
    }
    ctx->ws_elems = per * nbuf;
  }
  for (cudaStream_t& s_ : ctx->hs)
    if (!s_) FE_CUDA(ctx, cudaStreamCreateWithFlags(&s_, cudaStreamNonBlocking));
  int launches = 0, rc = FE_MF_OK;
  for (int k = 0; k < nchunks && rc == FE_MF_OK; ++k) {
    const int c0 = k * cw, w = (c0 + cw <= nvec) ? cw : (nvec - c0);
    cudaStream_t st = ctx->hs[k & 1];
    double* dx = ctx->ws_x + (size_t)(k % nbuf) * per;
    double* dy = ctx->ws_y + (size_t)(k % nbuf) * per;
    FE_CUDA(ctx, cudaMemcpy2DAsync(dx, (size_t)w * 8, X_host + c0, (size_t)nvec * 8, (size_t)w * 8, (size_t)ctx->ndof,
                                   cudaMemcpyHostToDevice, st));
    // the two internal streams run concurrently: each has its own work counter (a context's counter slot 0 belongs
    // to the caller's stream; a counter reset on one stream must never land under a running kernel of the other)
    ctx->ctrl_slot = 1 + (k & 1);
    rc = fe_mf_apply(ctx, dx, dy, w, st);
    ctx->ctrl_slot = 0;
    if (rc) break;
    launches += ctx->last_launches;
    FE_CUDA(ctx, cudaMemcpy2DAsync(Y_host + c0, (size_t)nvec * 8, dy, (size_t)w * 8, (size_t)w * 8, (size_t)ctx->ndof,
                                   cudaMemcpyDeviceToHost, st));
  }
  FE_CUDA(ctx, cudaStreamSynchronize(ctx->hs[0]));
  FE_CUDA(ctx, cudaStreamSynchronize(ctx->hs[1]));
  if (rc) return rc;
  ctx->last_launches = launches;
  return FE_MF_OK;
}

extern "C" int fe_fill_uniform(double* out_dev, long long count, unsigned long long seed, long long offset,
                               void* cuda_stream) {
  if (!out_dev || count < 0) return FE_MF_EINVAL;
  if (count == 0) return FE_MF_OK;
  return fe_host::launch_fill_uniform(out_dev, count, seed, offset, (cudaStream_t)cuda_stream) == cudaSuccess ? FE_MF_OK : FE_MF_ECUDA;
}

extern "C" int fe_mf_halo_add(double* dst_dev, const double* src_dev, long long count, void* cuda_stream) {
  if (!dst_dev || !src_dev || count < 0) return FE_MF_EINVAL;
  if (count == 0) return FE_MF_OK;
  return fe_host::launch_axpby(dst_dev, src_dev, 1.0, 1.0, (size_t)count, (cudaStream_t)cuda_stream) == cudaSuccess ? FE_MF_OK : FE_MF_ECUDA;
}

extern "C" int fe_mf_axpby(double* Z_dev, const double* W_dev, double beta, double gamma, long long count, void* cuda_stream) {
  if (!Z_dev || !W_dev || count < 0) return FE_MF_EINVAL;
  if (count == 0) return FE_MF_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // beta == 0: Z is not read (it may hold anything, NaN included)
  const cudaError_t e = (beta == 0.0) ? fe_host::launch_scale_copy(Z_dev, W_dev, gamma, (size_t)count, st)
                                      : fe_host::launch_axpby(Z_dev, W_dev, beta, gamma, (size_t)count, st);
  return e == cudaSuccess ? FE_MF_OK : FE_MF_ECUDA;
}

extern "C" int fe_mf_halo_pack_f32(float* dst_dev, const double* src_dev, long long count, void* cuda_stream) {
  if (!dst_dev || !src_dev || count < 0) return FE_MF_EINVAL;
  if (count == 0) return FE_MF_OK;
  return fe_host::launch_halo_pack_f32(dst_dev, src_dev, (size_t)count, (cudaStream_t)cuda_stream) == cudaSuccess ? FE_MF_OK : FE_MF_ECUDA;
}

extern "C" int fe_mf_halo_unpack_f32(double* dst_dev, const float* src_dev, long long count, int add, void* cuda_stream) {
  if (!dst_dev || !src_dev || count < 0 || (add != 0 && add != 1)) return FE_MF_EINVAL;
  if (count == 0) return FE_MF_OK;
  return fe_host::launch_halo_unpack_f32(dst_dev, src_dev, (size_t)count, add, (cudaStream_t)cuda_stream) == cudaSuccess ? FE_MF_OK : FE_MF_ECUDA;
}

extern "C" int fe_mf_batch_width(const fe_mf_ctx* ctx, int nvec) {
  if (!ctx || nvec < 1) return -1;
  const int kind = pick_kernel(ctx, nvec, nullptr, nullptr);
  return kernel_bv(ctx, kind, nvec);
}

extern "C" const char* fe_mf_kernel_name(const fe_mf_ctx* ctx, int nvec) {
  if (!ctx || nvec < 1) return "";
  switch (pick_kernel(ctx, nvec, nullptr, nullptr)) {
    case 1: return "fe_apply_general";
    case 2: return "fe_apply_cart";
    case 3: return "fe_apply_cart<CELLS>";
    case 6: return "fe_apply_gen_tma";
    case 8: return "fe_apply_cart_plane";
    case 11: return fe_host::oi_compile_time_kernel(ctx, nvec) ? "fe_apply_oi" : "fe_apply_general_oi";
    default: return "fe_apply_cart_line";
  }
}

extern "C" int fe_mf_last_launch_count(const fe_mf_ctx* ctx) { return ctx ? ctx->last_launches : -1; }

extern "C" int fe_mf_set_variant(fe_mf_ctx* ctx, int variant) {
  if (!ctx) return FE_MF_EINVAL;
  const bool known = variant == 0 || variant == 1 || variant == 2 || variant == 7 || variant == 8 || variant == 10 || variant == 11 || variant == 22 || variant == 23;
  if (!known) return fail(ctx, FE_MF_EINVAL, "unknown kernel variant");
  ctx->variant = variant;
  return FE_MF_OK;
}
