// Test helper: the two apply kernels of libfe_mf.so that need neither TMA nor inline PTX -- fe_apply_general (plain sum
// factorisation, any geometry: csrc/fe_kernels.cuh) and fe_apply_cart (even-odd, uniform Cartesian cells, also in its
// cells-as-slots mode for 1-3 vectors: csrc/fe_kernels_eo.cuh) -- compiled from their EXACT source with
// tests/host/shim/cuda_runtime.h and run on CPU threads, one block after another.  Tables and geometry are built by the
// product's host code (csrc/fe_tables.h, csrc/fe_eo_tables.h) the way fe_mf_create does; the kernel parameters are set the
// way csrc/fe_dispatch.cu (make_params, launch_accumulate) and csrc/fe_tu_misc.cu (grid, block, tile sizes) do.
// tests/test_host_emulation.py compares the output with the oracle.
//   usage: tests/host/emul_common.h ; KERNEL = general | cart | cells
#include "../../paper_2208_07129_b200/csrc/fe_kernels.cuh"
#include "../../paper_2208_07129_b200/csrc/fe_kernels_eo.cuh"
#include "emul_common.h"

namespace fe { double smem[1 << 18]; }   // the dynamic shared memory of the running block (blocks run one at a time)

// mirrors CartCfg of csrc/fe_tu_misc.cu
template <int PDEG>
struct CartCfg {
  static constexpr int BV = 8, N = PDEG + 1, TASKS = N * N * BV;
  static constexpr int NT = (PDEG >= 5) ? TASKS / 2 : (TASKS < 32 ? 32 : TASKS);
};

template <int PDEG>
static void run(const std::string& kernel, const fe::ApplyParams& P, long long ncells) {
  using C = CartCfg<PDEG>;
  if (kernel == "general") {
    emul_launch((unsigned)(ncells * P.nvb), 1, 256, [&] { fe::fe_apply_general<PDEG>(P); });
  } else if (kernel == "cart") {
    emul_launch((unsigned)(ncells * P.nvb), 1, C::NT, [&] { fe::fe_apply_cart<PDEG, C::BV, C::NT, 1, false>(P); });
  } else {
    const int cb = C::BV / P.nvec;
    const long long groups = (P.ncx + cb - 1) / cb;
    emul_launch((unsigned)(groups * P.ncy * P.ncz), 1, C::NT, [&] { fe::fe_apply_cart<PDEG, C::BV, C::NT, 1, true>(P); });
  }
}

int main(int argc, char** argv) {
  EmulSetup s;
  emul_setup(s, argc, argv);
  const int p = s.p, n = s.n;
  // what upload_tables_misc puts into constant memory
  std::memcpy(fe::c_N[p], s.tab.N, sizeof(double) * n * n);
  std::memcpy(fe::c_D[p], s.tab.Dt, sizeof(double) * n * n);
  std::memcpy(fe::c_w[p], s.tab.w, sizeof(double) * n);
  std::memcpy(fe::c_eo[p], s.eo, sizeof(s.eo));
  if (s.kernel == "general") {             // general_bv of fe_tu_misc.cu
    int bv = 32;
    while (bv > 1 && ((size_t)4 * s.nn * bv * 8 > 232448 / 2 - 1024 || bv > s.nvec)) bv >>= 1;
    emul_set_bv(s, bv);
    if (s.geom_mode == 0) s.P.geom = nullptr;
  } else {
    if (s.geom_mode != 0) return 4;        // the Cartesian kernel reads the uniform metric only
    if (s.kernel == "cells" && (s.nvec < 1 || s.nvec > 3)) return 4;
    emul_set_bv(s, 8);
    for (int k = 0; k < 7; ++k) s.P.ug[k] *= s.alpha;   // launch_accumulate, kinds 2 / 3: alpha inside the metric constants,
    s.P.alpha = 1.0;                                    // P.alpha = 1
  }
  const fe::ApplyParams& P = s.P;
  switch (p) {
    case 1: run<1>(s.kernel, P, s.ncells); break;
    case 2: run<2>(s.kernel, P, s.ncells); break;
    case 3: run<3>(s.kernel, P, s.ncells); break;
    case 4: run<4>(s.kernel, P, s.ncells); break;
    case 5: run<5>(s.kernel, P, s.ncells); break;
    case 6: run<6>(s.kernel, P, s.ncells); break;
    default: return 5;
  }
  return emul_write(s);
}
