// Kernel translation unit: n_q != n_p Gauss points per direction (fe_kernels_oi.cuh and the
// run-time-n_q fallback fe_apply_general_oi of fe_kernels.cuh).
#include <cstring>

#include "fe_ctx.h"
#include "fe_kernels_oi.cuh"

namespace fe_host {

cudaError_t upload_tables_oi(const double* pack, size_t count, size_t offset_doubles) {
  return cudaMemcpyToSymbol(fe::c_oi, pack, count * sizeof(double), offset_doubles * sizeof(double));
}

int oi_bv(int nq, int nvec) {
  // the compile-time kernel is instantiated for 2 and 4 vectors per block; 2 wherever three such blocks fit an SM
  int bv = ((size_t)3 * ((size_t)4 * nq * nq * nq * 2 * 8 + 4096) <= kMaxSmem) ? 2 : 4;
  while (bv > 1 && ((size_t)4 * nq * nq * nq * bv * 8 > kMaxSmem / 2 - 4096 || bv > nvec)) bv >>= 1;
  return bv;
}
bool oi_compile_time_kernel(const fe_mf_ctx* c, int nvec) { return c->nq_oi == c->p + 3 && oi_bv(c->nq_oi, nvec) >= 2; }

template <int PDEG>
static cudaError_t launch_oi_p(fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap* tw, const CUtensorMap* tz, cudaStream_t st) {
  const int nq = c->nq_oi;
  fe::OiParams O{nq, c->oi_N, c->oi_D, c->oi_w, c->oi_geom, c->oi_geom_stride};
  const size_t smem = ((size_t)4 * nq * nq * nq * prm.bv + (size_t)nq * (PDEG + 1) + (size_t)nq * nq) * sizeof(double);
  if (nq == PDEG + 3 && (prm.bv == 2 || prm.bv == 4)) {   // the paper's n_q = n_p + 2: compile-time sizes, line tasks
    // 2-vector blocks, three or four per SM, where four tiles fit that often (n_q <= 10 / n_q <= 9): measured faster
    // than two 4-vector blocks (p = 6: 25.4 -> 27.2 with three)
    constexpr size_t TB2 = (size_t)4 * (PDEG + 3) * (PDEG + 3) * (PDEG + 3) * 2 * 8 + 4096;
    constexpr int MB = 4 * TB2 <= kMaxSmem ? 4 : (3 * TB2 <= kMaxSmem ? 3 : 2);
    auto kern = prm.bv == 4 ? fe::fe_apply_oi<PDEG, PDEG + 3, 4> : fe::fe_apply_oi<PDEG, PDEG + 3, 2, MB>;
    cudaError_t e = ensure_smem(c, kern, smem);
    if (e != cudaSuccess) return e;
    // cells take their tile through TMA when the call meets the TMA conditions (tw / tz non-NULL); otherwise they
    // gather with loads and scatter with atomics inside the same kernel
    CUtensorMap dummy;
    memset(&dummy, 0, sizeof(dummy));
    const int use_tma = (tw && tz) ? 1 : 0;
    kern<<<(unsigned)(c->ncells * prm.nvb), 256, smem, st>>>(use_tma ? *tw : dummy, use_tma ? *tz : dummy, prm, O, use_tma);
    return cudaGetLastError();
  }
  cudaError_t e = ensure_smem(c, fe::fe_apply_general_oi<PDEG>, smem);
  if (e != cudaSuccess) return e;
  fe::fe_apply_general_oi<PDEG><<<(unsigned)(c->ncells * prm.nvb), 256, smem, st>>>(prm, O);
  return cudaGetLastError();
}

cudaError_t launch_oi(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap* tw, const CUtensorMap* tz, cudaStream_t st) {
  cudaError_t e = cudaErrorInvalidValue;
#define FE_CALL(p_) launch_oi_p<p_>(c, P, tw, tz, st)
  FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  return e;
}

}  // namespace fe_host
