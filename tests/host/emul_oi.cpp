// Test helper: the kernels of the n_q != n_p rule -- fe_apply_oi (compile-time sizes, n_q = n_p + 2:
// csrc/fe_kernels_oi.cuh) in its loads / atomics mode and fe_apply_general_oi (any n_q: csrc/fe_kernels.cuh) -- from their
// exact source on CPU threads.  Tables from the product's csrc/fe_oi_tables.h, per-point geometry the way
// fe_mf_set_quadrature builds it, launch parameters restated from csrc/fe_tu_oi.cu and launch_accumulate (kind 11).
//   usage: tests/host/emul_common.h ; KERNEL = oi (loads / atomics) | oi_tma (cell tile by bulk tensor copies) | general_oi ; nq=N required
#include "../../paper_2208_07129_b200/csrc/fe_kernels_oi.cuh"
#include "../../paper_2208_07129_b200/csrc/fe_oi_tables.h"
#include "emul_common.h"

namespace fe {
double smem[1 << 18];
alignas(128) unsigned char smem_oi[256 * 1024];
}

template <int PDEG>
static void run(EmulSetup& s, const fe::OiParams& O, int bv) {
  emul_set_bv(s, bv);
  const fe::ApplyParams P = s.P;
  const unsigned grid = (unsigned)(s.ncells * P.nvb);
  CUtensorMap dummy;
  std::memset(&dummy, 0, sizeof(dummy));
  if (s.kernel == "oi" || s.kernel == "oi_tma") {
    if (O.nq != PDEG + 3 || (bv != 2 && bv != 4)) { fprintf(stderr, "the compile-time kernel needs nq = p + 3 and 2 or 4 vectors per block\n"); exit(4); }
    const int use_tma = s.kernel == "oi_tma" ? 1 : 0;
    if (use_tma && (s.nvec & 1)) { fprintf(stderr, "the bulk-tensor mode needs an even nvec\n"); exit(4); }
    const CUtensorMap tw = use_tma ? make_map(s, s.X.data(), bv, 0, 0) : dummy, tz = use_tma ? make_map(s, s.Y.data(), bv, 0, 0) : dummy;
    if (bv == 4) emul_launch(grid, 1, 256, [&] { fe::fe_apply_oi<PDEG, PDEG + 3, 4>(tw, tz, P, O, use_tma); });
    else emul_launch(grid, 1, 256, [&] { fe::fe_apply_oi<PDEG, PDEG + 3, 2>(tw, tz, P, O, use_tma); });
    fe::emul_check_nothing_pending();
  } else {
    emul_launch(grid, 1, 256, [&] { fe::fe_apply_general_oi<PDEG>(P, O); });
  }
}

int main(int argc, char** argv) {
  EmulSetup s;
  emul_setup(s, argc, argv);
  const int p = s.p, nq = s.nq;
  if (nq < p + 1 || nq > 12) return 4;
  fe_host::OiTables t;
  fe_host::make_oi_tables(p, nq, t);
  if (!t.pack.empty()) std::memcpy(fe::c_oi + fe::oi_offset(p), t.pack.data(), t.pack.size() * sizeof(double));   // upload_tables_oi
  // per-point metric at the nq^3 points: fe_mf_set_quadrature
  std::vector<double> G;
  const size_t nn = (size_t)nq * nq * nq;
  if (s.geom_mode == 2) {
    G.assign(7 * nn * (size_t)s.ncells, 0.0);
    for (int ez = 0; ez < s.ncz; ++ez)
      for (int ey = 0; ey < s.ncy; ++ey)
        for (int ex = 0; ex < s.ncx; ++ex) {
          double v[8][3], J[3][3], m[7];
          for (int k = 0; k < 8; ++k) {
            const int vx = ex + (k & 1), vy = ey + ((k >> 1) & 1), vz = ez + ((k >> 2) & 1);
            const double* q = s.verts.data() + 3 * ((size_t)vx + (size_t)(s.ncx + 1) * ((size_t)vy + (size_t)(s.ncy + 1) * vz));
            v[k][0] = q[0]; v[k][1] = q[1]; v[k][2] = q[2];
          }
          double* g = G.data() + ((size_t)ex + (size_t)s.ncx * ((size_t)ey + (size_t)s.ncy * ez)) * 7 * nn;
          for (int q3 = 0; q3 < nq; ++q3)
            for (int q2 = 0; q2 < nq; ++q2)
              for (int q1 = 0; q1 < nq; ++q1) {
                const double x3[3] = {(double)t.xq[q1], (double)t.xq[q2], (double)t.xq[q3]};
                fe::trilinear_jacobian(v, x3, J);
                if (!fe::metric_from_jacobian(J, m)) return 3;
                const size_t Q = (size_t)q1 + (size_t)nq * (q2 + (size_t)nq * q3);
                for (int k = 0; k < 6; ++k) g[(size_t)k * nn + Q] = m[k];
                g[6 * nn + Q] = s.sigma * m[6];
              }
        }
  }
  const fe::OiParams O{nq, t.N.data(), t.D.data(), t.w.data(), G.empty() ? nullptr : G.data(), (long long)(7 * nn)};
  // oi_bv of fe_tu_oi.cu
  int bv = ((size_t)3 * ((size_t)4 * nn * 2 * 8 + 4096) <= 232448) ? 2 : 4;
  while (bv > 1 && ((size_t)4 * nn * bv * 8 > 232448 / 2 - 4096 || bv > s.nvec)) bv >>= 1;
  switch (p) {
    case 2: run<2>(s, O, bv); break;
    case 3: run<3>(s, O, bv); break;
    case 4: run<4>(s, O, bv); break;
    case 6: run<6>(s, O, bv); break;
    default: return 5;
  }
  return emul_write(s);
}
