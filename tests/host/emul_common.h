// Shared by emul_apply.cpp and emul_tma.cpp (test helpers): command line, input files, the tables and the geometry built by
// the product's host code (csrc/fe_tables.h, csrc/fe_eo_tables.h) the way fe_mf_create does (csrc/fe_mf.cu create_impl),
// and the kernel parameters the way csrc/fe_dispatch.cu make_params does (alpha = 1).
//   usage: PROGRAM KERNEL p ncx ncy ncz bc zopen geom_mode nvec sigma lox loy loz hix hiy hiz X.bin Y.bin [verts.bin|-] [key=value ...]
//          bc 0 periodic / 1 Dirichlet ; geom_mode 0 uniform box, 1 per cell, 2 per q-point (1, 2 need verts.bin)
//          alpha=c        Z += c A W instead of Z += A W (fe_mf_accumulate; the Cartesian kernels take it inside the metric constants)
//          z0=FILE        initial contents of Z (default: zeros)
//          idw=c          Z = A W + c W (the identity term of the Cartesian TMA kernels, periodic meshes)
//          kappa=FILE     kappa at the quadrature points [cell][n^3] of a uniform box (fe_mf_set_kappa); sigma is then unused
//          dscale=FILE    d = diag(M)^-1/2 [ndof] (fe_mf_set_mass_scaling): Z = d.(A (d.W)); on a uniform box with kappa the
//                         Cartesian TMA kernels run their EIG instantiation instead (d inside the tables)
//          nq=N           N Gauss points per direction instead of p + 1 (emul_oi.cpp; fe_mf_set_quadrature)
//          layers=l0:l1   only the cells of layers l0 <= ez < l1 (the item ranges of fe_mf_apply_host's z-slab pipeline)
#pragma once
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../paper_2208_07129_b200/csrc/fe_params.h"
#include "../../paper_2208_07129_b200/csrc/fe_tables.h"
#include "../../paper_2208_07129_b200/csrc/fe_eo_tables.h"

struct EmulSetup {
  std::string kernel, out_path;
  int p, n, nn, ncx, ncy, ncz, bc, zopen, geom_mode, nvec;
  int ndx, ndy, ndz;
  long long ndof, ncells;
  double sigma, idw = 0.0, detj0 = 1.0, alpha = 1.0;
  int layer0 = 0, layer1 = -1, nq = 0;
  std::vector<double> X, Y, verts, G, kappa, dscale;
  fe::Tables1D tab;
  fe::EoTab eo[5];
  fe::EoTab2 eo2[fe::MAT_COUNT];
  fe::ApplyParams P;
};

inline std::vector<double> emul_read_bin(const char* path, size_t count) {
  std::vector<double> v(count);
  FILE* f = fopen(path, "rb");
  if (!f || fread(v.data(), sizeof(double), count, f) != count) { fprintf(stderr, "cannot read %zu doubles from %s\n", count, path); exit(2); }
  fclose(f);
  return v;
}

inline void emul_setup(EmulSetup& s, int argc, char** argv) {
  if (argc < 19) { fprintf(stderr, "usage: see tests/host/emul_common.h\n"); exit(2); }
  s.kernel = argv[1];
  s.p = atoi(argv[2]); s.ncx = atoi(argv[3]); s.ncy = atoi(argv[4]); s.ncz = atoi(argv[5]);
  s.bc = atoi(argv[6]); s.zopen = atoi(argv[7]); s.geom_mode = atoi(argv[8]); s.nvec = atoi(argv[9]);
  s.sigma = atof(argv[10]);
  double lo[3], hi[3], h[3];
  for (int d = 0; d < 3; ++d) { lo[d] = atof(argv[11 + d]); hi[d] = atof(argv[14 + d]); }
  s.out_path = argv[18];
  std::string kappa_path, dscale_path, z0_path;
  for (int a = 20; a < argc; ++a) {
    const std::string kv = argv[a];
    if (kv.rfind("idw=", 0) == 0) s.idw = atof(kv.c_str() + 4);
    else if (kv.rfind("alpha=", 0) == 0) s.alpha = atof(kv.c_str() + 6);
    else if (kv.rfind("z0=", 0) == 0) z0_path = kv.substr(3);
    else if (kv.rfind("kappa=", 0) == 0) kappa_path = kv.substr(6);
    else if (kv.rfind("dscale=", 0) == 0) dscale_path = kv.substr(7);
    else if (kv.rfind("nq=", 0) == 0) s.nq = atoi(kv.c_str() + 3);
    else if (kv.rfind("layers=", 0) == 0) { if (sscanf(kv.c_str() + 7, "%d:%d", &s.layer0, &s.layer1) != 2) exit(2); }
    else { fprintf(stderr, "unknown option %s\n", kv.c_str()); exit(2); }
  }
  const int nc[3] = {s.ncx, s.ncy, s.ncz};
  for (int d = 0; d < 3; ++d) h[d] = (hi[d] - lo[d]) / nc[d];
  const int p = s.p, n = p + 1, nn = n * n * n, add = s.bc ? 1 : 0, ncx = s.ncx, ncy = s.ncy, ncz = s.ncz;
  s.n = n; s.nn = nn;
  // sizes: create_impl
  s.ndx = ncx * p + add; s.ndy = ncy * p + add; s.ndz = ncz * p + (s.zopen ? 1 : add);
  s.ndof = (long long)s.ndx * s.ndy * s.ndz; s.ncells = (long long)ncx * ncy * ncz;
  s.X = emul_read_bin(argv[17], (size_t)s.ndof * s.nvec);
  if (z0_path.empty()) s.Y.assign((size_t)s.ndof * s.nvec, 0.0);
  else s.Y = emul_read_bin(z0_path.c_str(), (size_t)s.ndof * s.nvec);
  if (s.geom_mode != 0) s.verts = emul_read_bin(argv[19], (size_t)3 * (ncx + 1) * (ncy + 1) * (ncz + 1));
  const size_t npts = s.nq ? (size_t)s.nq * s.nq * s.nq : (size_t)nn;   // points per cell of the rule in force
  if (!kappa_path.empty()) s.kappa = emul_read_bin(kappa_path.c_str(), npts * s.ncells);
  if (!dscale_path.empty()) s.dscale = emul_read_bin(dscale_path.c_str(), (size_t)s.ndof);
  s.tab = fe::make_tables(p);
  fe_host::make_eo_tables(s.tab, s.eo, s.eo2);

  fe::ApplyParams& P = s.P;
  std::memset(&P, 0, sizeof(P));
  const double centre[3] = {0.0, 0.0, 0.0};
  auto cell_vertices = [&](int ex, int ey, int ez, double v[8][3]) {
    for (int k = 0; k < 8; ++k) {
      const int vx = ex + (k & 1), vy = ey + ((k >> 1) & 1), vz = ez + ((k >> 2) & 1);
      if (!s.verts.empty()) {
        const double* q = s.verts.data() + 3 * ((size_t)vx + (size_t)(ncx + 1) * ((size_t)vy + (size_t)(ncy + 1) * vz));
        v[k][0] = q[0]; v[k][1] = q[1]; v[k][2] = q[2];
      } else {
        v[k][0] = lo[0] + h[0] * vx; v[k][1] = lo[1] + h[1] * vy; v[k][2] = lo[2] + h[2] * vz;
      }
    }
  };
  if (s.geom_mode == 0) {
    double v[8][3], J[3][3];
    cell_vertices(0, 0, 0, v);
    fe::trilinear_jacobian(v, centre, J);
    if (!fe::metric_from_jacobian(J, P.ug)) exit(3);
    s.detj0 = P.ug[6];
    P.ug[6] *= s.sigma;
    P.geom_stride = 7;
    s.G.assign(P.ug, P.ug + 7);            // the full-metric TMA kernel reads the uniform metric from memory
  } else {
    const bool perq = s.geom_mode == 2;
    const size_t per_cell = perq ? (((size_t)7 * nn + 1) & ~(size_t)1) : 7;
    P.geom_stride = (long long)per_cell;
    s.G.assign(per_cell * (size_t)s.ncells, 0.0);
    for (int ez = 0; ez < ncz; ++ez)
      for (int ey = 0; ey < ncy; ++ey)
        for (int ex = 0; ex < ncx; ++ex) {
          double v[8][3], J[3][3], m[7];
          cell_vertices(ex, ey, ez, v);
          double* g = s.G.data() + ((size_t)ex + (size_t)ncx * ((size_t)ey + (size_t)ncy * ez)) * per_cell;
          if (!perq) {
            fe::trilinear_jacobian(v, centre, J);
            if (!fe::metric_from_jacobian(J, m)) exit(3);
            for (int k = 0; k < 6; ++k) g[k] = m[k];
            g[6] = s.sigma * m[6];
          } else {
            for (int q3 = 0; q3 < n; ++q3)
              for (int q2 = 0; q2 < n; ++q2)
                for (int q1 = 0; q1 < n; ++q1) {
                  const double xi[3] = {s.tab.xq[q1], s.tab.xq[q2], s.tab.xq[q3]};
                  fe::trilinear_jacobian(v, xi, J);
                  if (!fe::metric_from_jacobian(J, m)) exit(3);
                  const int Q = q1 + n * (q2 + n * q3);
                  for (int k = 0; k < 6; ++k) g[(size_t)k * nn + Q] = m[k];
                  g[(size_t)6 * nn + Q] = s.sigma * m[6];
                }
          }
        }
  }
  P.geom = s.G.data();
  P.W = s.X.data(); P.Z = s.Y.data();
  P.alpha = s.alpha;
  P.ncx = ncx; P.ncy = ncy; P.ncz = ncz; P.ndx = s.ndx; P.ndy = s.ndy; P.ndz = s.ndz;
  P.nvec = s.nvec;
  P.dirichlet = s.bc ? 1 : 0; P.zopen = s.zopen; P.geom_mode = s.geom_mode; P.nsm = 148;
  P.idw = s.idw;
  // make_params: kappa on a uniform box -> the mass factor is det J * kappa_Q; d = diag(M)^-1/2
  if (!s.kappa.empty()) {
    if (s.geom_mode != 0) { fprintf(stderr, "kappa= needs a uniform box here\n"); exit(2); }
    P.kappa = s.kappa.data();
    P.ug[6] = s.detj0;
  }
  if (!s.dscale.empty()) P.dscale = s.dscale.data();
}

// the persistent kernels: a range of cell layers as an item range (fe_dispatch.cu apply_host_slabs)
inline long long emul_item_range(EmulSetup& s) {
  const long long layer_items = (long long)s.ncx * s.ncy * s.P.nvb;
  if (s.layer1 < 0) return s.ncells * s.P.nvb;
  s.P.item0 = (int)(s.layer0 * layer_items);
  s.P.item_count = (int)((s.layer1 - s.layer0) * layer_items);
  return s.P.item_count;
}

inline void emul_set_bv(EmulSetup& s, int bv) { s.P.bv = bv; s.P.nvb = (s.nvec + bv - 1) / bv; }

inline int emul_write(const EmulSetup& s) {
  FILE* f = fopen(s.out_path.c_str(), "wb");
  if (!f || fwrite(s.Y.data(), sizeof(double), s.Y.size(), f) != s.Y.size()) return 6;
  fclose(f);
  return 0;
}

#ifdef FE_TMA_WRAPPERS_PROVIDED   // programs that include tests/host/shim/cuda.h: the tensor map as the product computes its numbers
inline CUtensorMap make_map(const EmulSetup& s, double* base, int bv, int trim, int padx) {
  fe::TensorMapDesc d;
  if (!fe::tensor_map_desc(d, s.ndx, s.ndy, s.ndz, s.n, s.zopen, s.nvec, bv, trim, padx)) { fprintf(stderr, "tensor_map_desc refused\n"); exit(7); }
  CUtensorMap tm;
  tm.base = reinterpret_cast<double*>(reinterpret_cast<char*>(base) + d.base_offset);
  for (int k = 0; k < 4; ++k) { tm.dims[k] = d.dims[k]; tm.box[k] = d.box[k]; }
  for (int k = 0; k < 3; ++k) tm.strides[k] = d.strides[k];
  return tm;
}
#endif
