// Kernel translation unit: the plane kernel of uniform Cartesian cells at p = 6 (fe_kernels_plane.cuh).
#include "fe_ctx.h"
#include "fe_kernels_plane.cuh"

namespace fe_host {

cudaError_t upload_tables_plane(const fe::HostTables& t) {
  return cudaMemcpyToSymbol(fe::c_eo2, t.eo2, sizeof(t.eo2), sizeof(fe::EoTab2) * fe::MAT_COUNT * t.p);
}

// one thread = one n x n plane of one vector, 16 vectors per block
template <int PDEG> struct PlaneCfg;
template <> struct PlaneCfg<6> { static constexpr int BV = 16, NT = 128, MINB = 2; };

template <int PDEG, bool IDENT, bool EIG>
static cudaError_t launch_plane_v(fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap& tw, const CUtensorMap& tz,
                                  cudaStream_t st) {
  using C = PlaneCfg<PDEG>;
  constexpr size_t SMEM = (size_t)2 * fe::DenseTile<PDEG, C::BV>::PITCH + 64;
  auto kern = fe::fe_apply_cart_plane<PDEG, C::BV, C::NT, C::MINB, IDENT, EIG>;
  long long grid = 0;
  const long long nitems = prm.item_count ? prm.item_count : c->ncells * prm.nvb;
  cudaError_t e = persistent_grid(c, kern, C::NT, SMEM, nitems, grid);
  if (e == cudaSuccess) e = reset_counter(c, st);
  if (e != cudaSuccess) return e;
  kern<<<(unsigned)grid, C::NT, SMEM, st>>>(tw, tz, prm, (int)nitems);
  return cudaGetLastError();
}

cudaError_t launch_plane(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap& tw, const CUtensorMap& tz, cudaStream_t st) {
  if (c->p != 6) return cudaErrorInvalidValue;
  if (P.kappa)   // eigenproblem operator (EIG)
    return P.idw != 0.0 ? launch_plane_v<6, true, true>(c, P, tw, tz, st) : launch_plane_v<6, false, true>(c, P, tw, tz, st);
  return P.idw != 0.0 ? launch_plane_v<6, true, false>(c, P, tw, tz, st) : launch_plane_v<6, false, false>(c, P, tw, tz, st);
}

}  // namespace fe_host
