// Included by fe_tu_line16.cu / fe_tu_line8.cu: launcher of one line-kernel configuration.
template <int PDEG, int CFG, bool IDENT, bool EIG>
static cudaError_t launch_line_v(fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap& tw, const CUtensorMap& tz,
                                 cudaStream_t st) {
  using C = LineCfg<CFG>;
  constexpr int PADX = line_padx(PDEG, C::BV);
  constexpr size_t SMEM = (size_t)2 * fe::DenseTile<PDEG, C::BV, PADX>::PITCH + 64;
  auto kern = fe::fe_apply_cart_line<PDEG, C::BV, C::NT, C::MINB, PADX, IDENT, EIG>;
  const long long nitems = prm.item_count ? prm.item_count : c->ncells * prm.nvb;
  long long grid = 0;
  cudaError_t e = persistent_grid(c, kern, C::NT, SMEM, nitems, grid);
  if (e == cudaSuccess) e = reset_counter(c, st);
  if (e != cudaSuccess) return e;
  kern<<<(unsigned)grid, C::NT, SMEM, st>>>(tw, tz, prm, (int)nitems);
  return cudaGetLastError();
}

template <int PDEG, int CFG>
static cudaError_t launch_line_p(fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap& tw, const CUtensorMap& tz,
                                 cudaStream_t st) {
  if (prm.kappa)
    return prm.idw != 0.0 ? launch_line_v<PDEG, CFG, true, true>(c, prm, tw, tz, st)
                          : launch_line_v<PDEG, CFG, false, true>(c, prm, tw, tz, st);
  return prm.idw != 0.0 ? launch_line_v<PDEG, CFG, true, false>(c, prm, tw, tz, st)
                        : launch_line_v<PDEG, CFG, false, false>(c, prm, tw, tz, st);
}
