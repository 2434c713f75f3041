// Kernel translation unit: the persistent TMA kernel for a full symmetric metric (fe_kernels_gen.cuh).
#include "fe_ctx.h"
#include "fe_kernels_gen.cuh"

namespace fe_host {

cudaError_t upload_tables_gen(const fe::HostTables& t) {
  return cudaMemcpyToSymbol(fe::c_eo, t.eo, sizeof(t.eo), sizeof(fe::EoTab) * 5 * t.p);
}

template <int PDEG> struct GenCfg;
template <> struct GenCfg<1> { static constexpr int BV = 8, NT = 32, MINB = 4; };
template <> struct GenCfg<2> { static constexpr int BV = 8, NT = 64, MINB = 4; };
template <> struct GenCfg<3> { static constexpr int BV = 8, NT = 64, MINB = 4; };
template <> struct GenCfg<4> { static constexpr int BV = 8, NT = 128, MINB = 3; };
template <> struct GenCfg<5> { static constexpr int BV = 8, NT = 160, MINB = 2; };
template <> struct GenCfg<6> { static constexpr int BV = 8, NT = 128, MINB = 3; };
template <> struct GenCfg<7> { static constexpr int BV = 8, NT = 256, MINB = 1; };
template <> struct GenCfg<8> { static constexpr int BV = 4, NT = 192, MINB = 2; };


template <int PDEG, bool MSC>
static cudaError_t launch_gen_p(fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap& tw, const CUtensorMap& tz,
                                cudaStream_t st) {
  using C = GenCfg<PDEG>;
  constexpr int NN = (PDEG + 1) * (PDEG + 1) * (PDEG + 1);
  constexpr size_t SMEM = (size_t)3 * fe::DenseTile<PDEG, C::BV>::PITCH + ((size_t)7 * NN * 8 + 15) / 16 * 16 + 64;
  auto kern = fe::fe_apply_gen_tma<PDEG, C::BV, C::NT, C::MINB, MSC>;
  const long long nitems = prm.item_count ? prm.item_count : c->ncells * prm.nvb;
  long long grid = 0;
  cudaError_t e = persistent_grid(c, kern, C::NT, SMEM, nitems, grid);
  if (e == cudaSuccess) e = reset_counter(c, st);
  if (e != cudaSuccess) return e;
  kern<<<(unsigned)grid, C::NT, SMEM, st>>>(tw, tz, prm, (int)nitems);
  return cudaGetLastError();
}

int gen_bv(const fe_mf_ctx* c, int) { return c->p == 8 ? 4 : 8; }

cudaError_t launch_gen(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap& tw, const CUtensorMap& tz, cudaStream_t st) {
  cudaError_t e = cudaErrorInvalidValue;
  if (P.dscale) {
#define FE_CALL(p_) launch_gen_p<p_, true>(c, P, tw, tz, st)
    FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  } else {
#define FE_CALL(p_) launch_gen_p<p_, false>(c, P, tw, tz, st)
    FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  }
  return e;
}

}  // namespace fe_host
