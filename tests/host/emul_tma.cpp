// Test helper: the persistent TMA kernels of libfe_mf.so -- fe_apply_cart_plane (csrc/fe_kernels_plane.cuh),
// fe_apply_cart_line (csrc/fe_kernels_line.cuh) and fe_apply_gen_tma (csrc/fe_kernels_gen.cuh) -- compiled from their EXACT
// source and run on CPU threads.  tests/host/shim/cuda.h supplies CUtensorMap as plain numbers and host versions of the
// PTX wrappers (mbarrier, bulk tensor load with zero fill, bulk tensor reduce-add with clipping, the item counter); the
// numbers of the tensor maps come from the product's fe::tensor_map_desc (csrc/fe_params.h), tables and geometry from
// the product's host code (emul_common.h), launch parameters are restated from csrc/fe_dispatch.cu (launch_accumulate) and
// the fe_tu_*.cu launchers (block sizes, tile sizes).  A few blocks run one after another, so both the first item of a
// block and the items handed out by the counter are exercised.  tests/test_host_emulation.py compares with the oracle.
//   usage: tests/host/emul_common.h ; KERNEL = plane | line16 | line8 | gen
#include "../../paper_2208_07129_b200/csrc/fe_kernels_plane.cuh"
#include "../../paper_2208_07129_b200/csrc/fe_kernels_line.cuh"
#include "../../paper_2208_07129_b200/csrc/fe_kernels_gen.cuh"
#include "emul_common.h"

namespace fe { alignas(1024) unsigned char smem_raw[256 * 1024]; }   // the dynamic shared memory of the running block

static constexpr int line_padx(int p, int bv) { return ((bv == 8 || bv == 4) && (p + 1) % 2 == 0 && p >= 3) ? 1 : 0; }   // fe_ctx.h

static int g_item_counter = 0;

template <typename Kernel>
static void launch(EmulSetup& s, int bv, int nt, size_t smem_bytes, bool cartesian, int padx, Kernel kernel) {
  if (smem_bytes > sizeof(fe::smem_raw) || smem_bytes > 232448) { fprintf(stderr, "shared memory %zu too large\n", smem_bytes); exit(8); }
  emul_set_bv(s, bv);
  if (cartesian)                          // launch_accumulate, kinds 8 / 9: the result is linear in the metric constants
    for (int k = 0; k < 7; ++k) s.P.ug[k] *= s.alpha;
  if (cartesian && !s.dscale.empty()) {   // launch_accumulate, EIG kernels: diag(M)^-1/2 = (det J)^-1/2 kron diag(w~)^-1/2, the tables carry the second factor
    for (int k = 0; k < 7; ++k) s.P.ug[k] /= s.detj0;
    s.P.dscale = nullptr;
  }
  const bool trim = cartesian && s.bc == 1;
  const CUtensorMap tw = make_map(s, s.X.data(), bv, trim ? 2 : 0, padx), tz = make_map(s, s.Y.data(), bv, trim ? 1 : 0, padx);
  g_item_counter = 0;
  s.P.item_ctr = &g_item_counter;
  const long long nitems = emul_item_range(s);
  const unsigned grid = (unsigned)(nitems < 3 ? nitems : 3);
  const fe::ApplyParams P = s.P;
  emul_launch(grid, 1, (unsigned)nt, [&] { kernel(tw, tz, P, (int)nitems); });
  fe::emul_check_nothing_pending();
}

// IDENT / EIG instantiations are chosen the way launch_plane / launch_line_p do: EIG if kappa is set, IDENT if idw != 0
template <int PDEG, int BV, int NT, bool IDENT, bool EIG>
static void run_line(EmulSetup& s) {
  constexpr int PADX = line_padx(PDEG, BV);
  launch(s, BV, NT, (size_t)2 * fe::DenseTile<PDEG, BV, PADX>::PITCH + 64, true, PADX,
         [](const CUtensorMap& a, const CUtensorMap& b, const fe::ApplyParams& P, int n) { fe::fe_apply_cart_line<PDEG, BV, NT, 1, PADX, IDENT, EIG>(a, b, P, n); });
}
template <int PDEG, int BV, int NT>
static void run_line_i(EmulSetup& s) {
  const bool eig = !s.kappa.empty(), ident = s.idw != 0.0;
  if (eig) { if (ident) run_line<PDEG, BV, NT, true, true>(s); else run_line<PDEG, BV, NT, false, true>(s); }
  else { if (ident) run_line<PDEG, BV, NT, true, false>(s); else run_line<PDEG, BV, NT, false, false>(s); }
}

template <bool IDENT, bool EIG>
static void run_plane_v(EmulSetup& s) {
  launch(s, 16, 128, (size_t)2 * fe::DenseTile<6, 16>::PITCH + 64, true, 0,
         [](const CUtensorMap& a, const CUtensorMap& b, const fe::ApplyParams& P, int n) { fe::fe_apply_cart_plane<6, 16, 128, 2, IDENT, EIG>(a, b, P, n); });
}
static void run_plane(EmulSetup& s) {
  const bool eig = !s.kappa.empty(), ident = s.idw != 0.0;
  if (eig) { if (ident) run_plane_v<true, true>(s); else run_plane_v<false, true>(s); }
  else { if (ident) run_plane_v<true, false>(s); else run_plane_v<false, false>(s); }
}

template <int PDEG, int BV, int NT>
static void run_gen(EmulSetup& s) {   // launch_gen: MSC if d is given
  constexpr int NN = (PDEG + 1) * (PDEG + 1) * (PDEG + 1);
  constexpr size_t SMEM = (size_t)3 * fe::DenseTile<PDEG, BV>::PITCH + ((size_t)7 * NN * 8 + 15) / 16 * 16 + 64;
  if (!s.dscale.empty())
    launch(s, BV, NT, SMEM, false, 0,
           [](const CUtensorMap& a, const CUtensorMap& b, const fe::ApplyParams& P, int n) { fe::fe_apply_gen_tma<PDEG, BV, NT, 1, true>(a, b, P, n); });
  else
    launch(s, BV, NT, SMEM, false, 0,
           [](const CUtensorMap& a, const CUtensorMap& b, const fe::ApplyParams& P, int n) { fe::fe_apply_gen_tma<PDEG, BV, NT, 1, false>(a, b, P, n); });
}

int main(int argc, char** argv) {
  EmulSetup s;
  emul_setup(s, argc, argv);
  const int p = s.p;
  std::memcpy(fe::c_eo[p], s.eo, sizeof(s.eo));       // upload_tables_gen
  std::memcpy(fe::c_eo2[p], s.eo2, sizeof(s.eo2));    // upload_tables_plane / _line16 / _line8
  if (s.nvec & 1) return 4;                           // pick_kernel: the TMA kernels take an even nvec
  if (s.kernel != "gen" && s.geom_mode != 0) return 4;
  bool ok = true;
  // block sizes: PlaneCfg (fe_tu_plane.cu), LineCfg (fe_tu_line16.cu, fe_tu_line8.cu), GenCfg (fe_tu_gen.cu)
  if (s.kernel == "plane" && p == 6) run_plane(s);
  else if (s.kernel == "line16" && p == 1) run_line_i<1, 16, 32>(s);
  else if (s.kernel == "line16" && p == 2) run_line_i<2, 16, 96>(s);
  else if (s.kernel == "line16" && p == 3) run_line_i<3, 16, 128>(s);
  else if (s.kernel == "line16" && p == 5) run_line_i<5, 16, 160>(s);
  else if (s.kernel == "line16" && p == 6) run_line_i<6, 16, 256>(s);
  else if (s.kernel == "line8" && p == 1) run_line_i<1, 8, 32>(s);
  else if (s.kernel == "line8" && p == 2) run_line_i<2, 8, 64>(s);
  else if (s.kernel == "line8" && p == 3) run_line_i<3, 8, 64>(s);
  else if (s.kernel == "line8" && p == 4) run_line_i<4, 8, 128>(s);
  else if (s.kernel == "line8" && p == 7) run_line_i<7, 8, 128>(s);
  else if (s.kernel == "gen" && p == 1) run_gen<1, 8, 32>(s);
  else if (s.kernel == "gen" && p == 2) run_gen<2, 8, 64>(s);
  else if (s.kernel == "gen" && p == 3) run_gen<3, 8, 64>(s);
  else if (s.kernel == "gen" && p == 5) run_gen<5, 8, 160>(s);
  else if (s.kernel == "gen" && p == 8) run_gen<8, 4, 192>(s);
  else ok = false;
  if (!ok) { fprintf(stderr, "no instantiation for %s p=%d\n", s.kernel.c_str(), p); return 5; }
  return emul_write(s);
}
