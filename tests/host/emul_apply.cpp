// Test helper: the two apply kernels of libfe_mf.so that need neither TMA nor inline PTX -- fe_apply_general (plain sum
// factorisation, any geometry: csrc/fe_kernels.cuh) and fe_apply_cart (even-odd, uniform Cartesian cells, also in its
// cells-as-slots mode for 1-3 vectors: csrc/fe_kernels_eo.cuh) -- compiled from their EXACT source with
// tests/host/shim/cuda_runtime.h and run on CPU threads, one block after another.  Tables and geometry are built by the
// product's host code (csrc/fe_tables.h, csrc/fe_eo_tables.h) the way fe_mf_create does; the kernel parameters are set the
// way csrc/fe_dispatch.cu (make_params, launch_accumulate) and csrc/fe_tu_misc.cu (grid, block, tile sizes) do.
// tests/test_host_emulation.py compares the output with the oracle.
//   usage: emul_apply KERNEL p ncx ncy ncz bc zopen geom_mode nvec sigma lox loy loz hix hiy hiz X.bin Y.bin [verts.bin]
//          KERNEL = general | cart | cells ; bc 0 periodic / 1 Dirichlet ; geom_mode 0 uniform box, 1 per cell, 2 per q-point
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>

#include "../../paper_2208_07129_b200/csrc/fe_kernels.cuh"
#include "../../paper_2208_07129_b200/csrc/fe_kernels_eo.cuh"
#include "../../paper_2208_07129_b200/csrc/fe_eo_tables.h"

namespace fe { double smem[1 << 18]; }   // the dynamic shared memory of the running block (blocks run one at a time)

static std::vector<double> read_bin(const char* path, size_t count) {
  std::vector<double> v(count);
  FILE* f = fopen(path, "rb");
  if (!f || fread(v.data(), sizeof(double), count, f) != count) { fprintf(stderr, "cannot read %zu doubles from %s\n", count, path); exit(2); }
  fclose(f);
  return v;
}

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
  if (argc < 19) { fprintf(stderr, "usage: see the header of emul_apply.cpp\n"); return 2; }
  const std::string kernel = argv[1];
  const int p = atoi(argv[2]), ncx = atoi(argv[3]), ncy = atoi(argv[4]), ncz = atoi(argv[5]);
  const int bc = atoi(argv[6]), zopen = atoi(argv[7]), geom_mode = atoi(argv[8]), nvec = atoi(argv[9]);
  const double sigma = atof(argv[10]);
  double lo[3], hi[3], h[3];
  for (int d = 0; d < 3; ++d) { lo[d] = atof(argv[11 + d]); hi[d] = atof(argv[14 + d]); }
  const int nc[3] = {ncx, ncy, ncz};
  for (int d = 0; d < 3; ++d) h[d] = (hi[d] - lo[d]) / nc[d];
  const int n = p + 1, nn = n * n * n, add = bc ? 1 : 0;
  // sizes: fe_mf.cu create_impl
  const int ndx = ncx * p + add, ndy = ncy * p + add, ndz = ncz * p + (zopen ? 1 : add);
  const long long ndof = (long long)ndx * ndy * ndz, ncells = (long long)ncx * ncy * ncz;
  std::vector<double> X = read_bin(argv[17], (size_t)ndof * nvec), Y((size_t)ndof * nvec, 0.0), verts;
  if (geom_mode != 0) verts = read_bin(argv[19], (size_t)3 * (ncx + 1) * (ncy + 1) * (ncz + 1));

  // tables: what upload_tables_misc puts into constant memory
  const fe::Tables1D tab = fe::make_tables(p);
  fe::EoTab eo[5];
  fe::EoTab2 eo2[fe::MAT_COUNT];
  fe_host::make_eo_tables(tab, eo, eo2);
  std::memcpy(fe::c_N[p], tab.N, sizeof(double) * n * n);
  std::memcpy(fe::c_D[p], tab.Dt, sizeof(double) * n * n);
  std::memcpy(fe::c_w[p], tab.w, sizeof(double) * n);
  std::memcpy(fe::c_eo[p], eo, sizeof(eo));

  // geometry: fe_mf.cu create_impl
  fe::ApplyParams P;
  std::memset(&P, 0, sizeof(P));
  std::vector<double> G;
  const double centre[3] = {0.0, 0.0, 0.0};
  auto cell_vertices = [&](int ex, int ey, int ez, double v[8][3]) {
    for (int k = 0; k < 8; ++k) {
      const int vx = ex + (k & 1), vy = ey + ((k >> 1) & 1), vz = ez + ((k >> 2) & 1);
      if (!verts.empty()) {
        const double* s = verts.data() + 3 * ((size_t)vx + (size_t)(ncx + 1) * ((size_t)vy + (size_t)(ncy + 1) * vz));
        v[k][0] = s[0]; v[k][1] = s[1]; v[k][2] = s[2];
      } else {
        v[k][0] = lo[0] + h[0] * vx; v[k][1] = lo[1] + h[1] * vy; v[k][2] = lo[2] + h[2] * vz;
      }
    }
  };
  if (geom_mode == 0) {
    double v[8][3], J[3][3];
    cell_vertices(0, 0, 0, v);
    fe::trilinear_jacobian(v, centre, J);
    if (!fe::metric_from_jacobian(J, P.ug)) return 3;
    P.ug[6] *= sigma;
    P.geom_stride = 7;
  } else {
    const bool perq = geom_mode == 2;
    const size_t per_cell = perq ? (((size_t)7 * nn + 1) & ~(size_t)1) : 7;
    P.geom_stride = (long long)per_cell;
    G.assign(per_cell * (size_t)ncells, 0.0);
    for (int ez = 0; ez < ncz; ++ez)
      for (int ey = 0; ey < ncy; ++ey)
        for (int ex = 0; ex < ncx; ++ex) {
          double v[8][3], J[3][3], m[7];
          cell_vertices(ex, ey, ez, v);
          double* g = G.data() + ((size_t)ex + (size_t)ncx * ((size_t)ey + (size_t)ncy * ez)) * per_cell;
          if (!perq) {
            fe::trilinear_jacobian(v, centre, J);
            if (!fe::metric_from_jacobian(J, m)) return 3;
            for (int k = 0; k < 6; ++k) g[k] = m[k];
            g[6] = sigma * m[6];
          } else {
            for (int q3 = 0; q3 < n; ++q3)
              for (int q2 = 0; q2 < n; ++q2)
                for (int q1 = 0; q1 < n; ++q1) {
                  const double xi[3] = {tab.xq[q1], tab.xq[q2], tab.xq[q3]};
                  fe::trilinear_jacobian(v, xi, J);
                  if (!fe::metric_from_jacobian(J, m)) return 3;
                  const int Q = q1 + n * (q2 + n * q3);
                  for (int k = 0; k < 6; ++k) g[(size_t)k * nn + Q] = m[k];
                  g[(size_t)6 * nn + Q] = sigma * m[6];
                }
          }
        }
    P.geom = G.data();
  }
  // parameters: fe_dispatch.cu make_params / launch_accumulate (alpha = 1)
  int bv;
  if (kernel == "general") {             // general_bv of fe_tu_misc.cu
    bv = 32;
    while (bv > 1 && ((size_t)4 * nn * bv * 8 > 232448 / 2 - 1024 || bv > nvec)) bv >>= 1;
  } else {
    bv = 8;
    if (geom_mode != 0) return 4;        // the Cartesian kernel reads the uniform metric only
    if (kernel == "cells" && (nvec < 1 || nvec > 3)) return 4;
  }
  P.W = X.data(); P.Z = Y.data();
  P.alpha = 1.0;
  P.ncx = ncx; P.ncy = ncy; P.ncz = ncz; P.ndx = ndx; P.ndy = ndy; P.ndz = ndz;
  P.nvec = nvec; P.bv = bv; P.nvb = (nvec + bv - 1) / bv;
  P.dirichlet = bc ? 1 : 0; P.zopen = zopen; P.geom_mode = geom_mode; P.nsm = 148;
  switch (p) {
    case 1: run<1>(kernel, P, ncells); break;
    case 2: run<2>(kernel, P, ncells); break;
    case 3: run<3>(kernel, P, ncells); break;
    case 4: run<4>(kernel, P, ncells); break;
    case 5: run<5>(kernel, P, ncells); break;
    case 6: run<6>(kernel, P, ncells); break;
    default: return 5;
  }
  FILE* f = fopen(argv[18], "wb");
  if (!f || fwrite(Y.data(), sizeof(double), Y.size(), f) != Y.size()) return 6;
  fclose(f);
  return 0;
}
