// Host code, no CUDA: the tables of an n_q-point Gauss rule with n_q != n_p points per direction (
// PAPER.md:798, 869) that fe_mf_set_quadrature uploads.  A header of its own so that the host-only tests build the same
// tables (tests/host/emul_oi.cpp).
#pragma once
#include <cstddef>
#include <vector>

#include "fe_tables.h"

namespace fe_host {

struct OiTables {
  std::vector<double> N;      // [nq][n]   N[q][i] = l_i(xq_q) on the GLL nodes
  std::vector<double> D;      // [nq][nq]  D~[q][r] = l~_r'(xq_q), the collocation derivative on the quadrature points
  std::vector<double> w;      // [nq]
  std::vector<double> pack;   // nq == p + 3 only: even / odd halves [Ne | No | De | Do] for the constant-memory table c_oi
  long double xq[16];         // the quadrature points
};

// p + 1 <= nq <= 12 (checked by the caller)
inline void make_oi_tables(int p, int nq, OiTables& t) {
  const int n = p + 1;
  // tables of the nq-point rule in long double
  long double xi[16], w[16], c[16];
  long double* xq = t.xq;
  fe::gll_nodes(p, xi);
  fe::gauss_legendre(nq, xq, w);
  std::vector<double>&hN = t.N, &hD = t.D, &hw = t.w;
  hN.assign((size_t)nq * n, 0.0); hD.assign((size_t)nq * nq, 0.0); hw.assign(nq, 0.0);
  for (int q = 0; q < nq; ++q) {
    hw[q] = (double)w[q];
    for (int i = 0; i < n; ++i) {
      long double v = 1.0L;
      for (int j = 0; j < n; ++j) if (j != i) v *= (xq[q] - xi[j]) / (xi[i] - xi[j]);
      hN[(size_t)q * n + i] = (double)v;
    }
  }
  for (int r = 0; r < nq; ++r) { c[r] = 1.0L; for (int j = 0; j < nq; ++j) if (j != r) c[r] *= (xq[r] - xq[j]); }
  for (int q = 0; q < nq; ++q)
    for (int r = 0; r < nq; ++r) {
      long double v = 0.0L;
      if (q != r) v = (c[q] / c[r]) / (xq[q] - xq[r]);
      else for (int j = 0; j < nq; ++j) if (j != q) v += 1.0L / (xq[q] - xq[j]);
      hD[(size_t)q * nq + r] = (double)v;
    }
  t.pack.clear();
  if (nq == p + 3) {   // the compile-time kernel of n_q = n_p + 2 reads its tables from constant memory
    // even / odd halves [Ne | No | De | Do] (layout: fe_kernels_oi.cuh, c_oi), halved in long double from the symmetrised pair
    std::vector<double>& pack = t.pack;
    auto halves = [&](const std::vector<double>& M, int R, int C, double sgn) {
      const int hR = (R + 1) / 2, hC = (C + 1) / 2;
      for (int part = 0; part < 2; ++part)
        for (int o = 0; o < hR; ++o)
          for (int i = 0; i < hC; ++i) {
            // the centro-(anti)symmetry is enforced exactly: entry (o, i) is averaged with its image (R-1-o, C-1-i)
            const long double a = 0.5L * ((long double)M[(size_t)o * C + i] + sgn * (long double)M[(size_t)(R - 1 - o) * C + (C - 1 - i)]);
            const long double b = 0.5L * ((long double)M[(size_t)o * C + (C - 1 - i)] + sgn * (long double)M[(size_t)(R - 1 - o) * C + i]);
            pack.push_back((double)(part == 0 ? 0.5L * (a + b) : 0.5L * (a - b)));
          }
    };
    halves(hN, nq, n, 1.0);
    halves(hD, nq, nq, -1.0);
  }
}

}  // namespace fe_host
