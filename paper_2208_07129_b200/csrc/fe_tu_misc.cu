// Kernel translation unit: the general fallback kernel (plain contractions, any geometry, any nvec), the even-odd
// Cartesian kernel with loads and atomics (odd nvec, unaligned pointers, 1-3 vectors), the streaming kernels of S1 / S9
// and the input generator.
#include "fe_ctx.h"
#include "fe_kernels.cuh"
#include "fe_kernels_eo.cuh"
#include "fe_kernels_stream.cuh"

namespace fe_host {

cudaError_t upload_tables_misc(const fe::HostTables& t) {
  const int p = t.p, n = p + 1;
  cudaError_t e = cudaMemcpyToSymbol(fe::c_N, t.N, sizeof(double) * n * n, sizeof(double) * fe::KMAXN * fe::KMAXN * p);
  if (e == cudaSuccess) e = cudaMemcpyToSymbol(fe::c_D, t.D, sizeof(double) * n * n, sizeof(double) * fe::KMAXN * fe::KMAXN * p);
  if (e == cudaSuccess) e = cudaMemcpyToSymbol(fe::c_w, t.w, sizeof(double) * n, sizeof(double) * fe::KMAXN * p);
  if (e == cudaSuccess) e = cudaMemcpyToSymbol(fe::c_eo, t.eo, sizeof(t.eo), sizeof(fe::EoTab) * 5 * p);
  return e;
}

// ---- general fallback, 4 tiles of n^3*bv doubles; keep >= 2 blocks per SM resident
int general_bv(int p, int nvec) {
  const int nn = (p + 1) * (p + 1) * (p + 1);
  int bv = 32;
  while (bv > 1 && ((size_t)4 * nn * bv * 8 > kMaxSmem / 2 - 1024 || bv > nvec)) bv >>= 1;
  return bv;
}

template <int PDEG>
static cudaError_t launch_general_p(fe_mf_ctx* c, const fe::ApplyParams& prm, cudaStream_t st) {
  constexpr int NN = (PDEG + 1) * (PDEG + 1) * (PDEG + 1);
  const size_t smem = (size_t)4 * NN * prm.bv * sizeof(double);
  cudaError_t e = ensure_smem(c, fe::fe_apply_general<PDEG>, smem);
  if (e != cudaSuccess) return e;
  fe::fe_apply_general<PDEG><<<(unsigned)(c->ncells * prm.nvb), 256, smem, st>>>(prm);
  return cudaGetLastError();
}
cudaError_t launch_general(fe_mf_ctx* c, const fe::ApplyParams& P, cudaStream_t st) {
  cudaError_t e = cudaErrorInvalidValue;
#define FE_CALL(p_) launch_general_p<p_>(c, P, st)
  FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  return e;
}

// ---- even-odd Cartesian kernel, one vector per thread, 8 vectors per block
template <int PDEG>
struct CartCfg {
  static constexpr int BV = 8, N = PDEG + 1;
  static constexpr int TASKS = N * N * BV;
  static constexpr int NT = (PDEG >= 5) ? TASKS / 2 : (TASKS < 32 ? 32 : TASKS);
  static constexpr size_t SMEM = (size_t)2 * fe::Tile<PDEG, BV>::SIZE * sizeof(double);
  static constexpr int BY_SMEM = (int)((kMaxSmem - 1024) / (SMEM + 1024));
  static constexpr int BY_THREADS = 2048 / NT;
  static constexpr int MINB0 = BY_SMEM < BY_THREADS ? BY_SMEM : BY_THREADS;
  static constexpr int MINB = MINB0 > 4 ? 4 : (MINB0 < 1 ? 1 : MINB0);
};

template <int PDEG>
static cudaError_t launch_cart_p(fe_mf_ctx* c, const fe::ApplyParams& prm, cudaStream_t st) {
  using C = CartCfg<PDEG>;
  auto kern = fe::fe_apply_cart<PDEG, C::BV, C::NT, C::MINB>;
  cudaError_t e = ensure_smem(c, kern, C::SMEM);
  if (e != cudaSuccess) return e;
  kern<<<(unsigned)(c->ncells * prm.nvb), C::NT, C::SMEM, st>>>(prm);
  return cudaGetLastError();
}
cudaError_t launch_cart(fe_mf_ctx* c, const fe::ApplyParams& P, cudaStream_t st) {
  cudaError_t e = cudaErrorInvalidValue;
#define FE_CALL(p_) launch_cart_p<p_>(c, P, st)
  FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  return e;
}

// the same kernel with the 8 tile slots holding 1-3 vectors of 8 / nvec consecutive cells of an x-row
template <int PDEG>
static cudaError_t launch_cart_cells_p(fe_mf_ctx* c, const fe::ApplyParams& prm, cudaStream_t st) {
  using C = CartCfg<PDEG>;
  auto kern = fe::fe_apply_cart<PDEG, C::BV, C::NT, C::MINB, true>;
  cudaError_t e = ensure_smem(c, kern, C::SMEM);
  if (e != cudaSuccess) return e;
  const int cb = C::BV / prm.nvec;                      // cells per block
  const long long groups = (c->ncx + cb - 1) / cb;
  const long long grid = groups * c->ncy * c->ncz;
  if (grid > 2147483647LL) return cudaErrorInvalidValue;
  kern<<<(unsigned)grid, C::NT, C::SMEM, st>>>(prm);
  return cudaGetLastError();
}
cudaError_t launch_cart_cells(fe_mf_ctx* c, const fe::ApplyParams& P, cudaStream_t st) {
  cudaError_t e = cudaErrorInvalidValue;
#define FE_CALL(p_) launch_cart_cells_p<p_>(c, P, st)
  FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  return e;
}

// ---- streaming kernels
static int stream_grid(size_t count) {
  size_t b = (count + 255) / 256;
  if (b > 148 * 16) b = 148 * 16;
  if (b < 1) b = 1;
  return (int)b;
}
static bool aligned16(const void* a, const void* b = nullptr) { return ((((uintptr_t)a) | ((uintptr_t)b)) & 15) == 0; }

cudaError_t launch_axpby(double* Z, const double* W, double beta, double gamma, size_t count, cudaStream_t st) {
  if (aligned16(Z, W)) fe::fe_axpby_kernel<<<stream_grid(count / 2 + 1), 256, 0, st>>>(Z, W, beta, gamma, count);
  else fe::fe_axpby_scalar_kernel<<<stream_grid(count), 256, 0, st>>>(Z, W, beta, gamma, count);
  return cudaGetLastError();
}
cudaError_t launch_scale_copy(double* Z, const double* W, double gamma, size_t count, cudaStream_t st) {
  fe::fe_scale_copy_kernel<<<stream_grid(count), 256, 0, st>>>(Z, W, gamma, count);
  return cudaGetLastError();
}
cudaError_t launch_scale(double* Z, double beta, size_t count, cudaStream_t st) {
  if (aligned16(Z)) fe::fe_scale_kernel<<<stream_grid(count / 2 + 1), 256, 0, st>>>(Z, beta, count);
  else fe::fe_axpby_scalar_kernel<<<stream_grid(count), 256, 0, st>>>(Z, Z, beta, 0.0, count);
  return cudaGetLastError();
}
cudaError_t launch_scale2(double* A, double* B, double sa, double sb, int swap, size_t count, int bnd, double qa, double qb,
                          int ndx, int ndy, int ndz, int nvec, cudaStream_t st) {
  fe::fe_scale2_kernel<<<stream_grid(count), 256, 0, st>>>(A, B, sa, sb, swap, count, bnd, qa, qb, ndx, ndy, ndz, nvec);
  return cudaGetLastError();
}
cudaError_t launch_swap(double* A, double* B, size_t count, cudaStream_t st) {
  fe::fe_swap_kernel<<<stream_grid(count), 256, 0, st>>>(A, B, count);
  return cudaGetLastError();
}
cudaError_t launch_halo_pack_f32(float* dst, const double* src, size_t count, cudaStream_t st) {
  fe::fe_halo_pack_f32_kernel<<<stream_grid(count), 256, 0, st>>>(dst, src, count);
  return cudaGetLastError();
}
cudaError_t launch_halo_unpack_f32(double* dst, const float* src, size_t count, int add, cudaStream_t st) {
  fe::fe_halo_unpack_f32_kernel<<<stream_grid(count), 256, 0, st>>>(dst, src, count, add);
  return cudaGetLastError();
}
cudaError_t launch_fill_uniform(double* out, long long count, unsigned long long seed, long long offset, cudaStream_t st) {
  fe::fe_fill_uniform_kernel<<<stream_grid((size_t)count), 256, 0, st>>>(out, count, seed, offset);
  return cudaGetLastError();
}

}  // namespace fe_host
