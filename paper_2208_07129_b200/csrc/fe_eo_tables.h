// Host code, no CUDA: the even-odd half tables that fe_mf_create uploads into the constant memory of the kernel
// translation units (S0 of SURVEY.md 8(a)).  A header of its own so that the host-only tests can build the same tables
// (tests/host/emul_apply.cpp, tests/test_host_tables.py).
#pragma once
#include <cmath>
#include <cstring>

#include "fe_params.h"
#include "fe_tables.h"

namespace fe_host {

// Even-odd half tables of the sqrt(w)-rescaled matrices: kind 0 Ns = diag(sqrt w) N,
// 1 Ns^T, 2 Ds = diag(sqrt w) D~ diag(1/sqrt w), 3 Ds^T.
inline void make_eo_tables(const fe::Tables1D& t, fe::EoTab out[5], fe::EoTab2 out2[fe::MAT_COUNT]) {
  const int n = t.n, h = n / 2, m = n / 2;
  long double M[6][fe::MAXN * fe::MAXN];
  for (int q = 0; q < n; ++q)
    for (int i = 0; i < n; ++i) {
      const long double sq = sqrtl(t.wl[q]), si = sqrtl(t.wl[i]);
      const long double ns = sq * t.Nl[q * n + i];
      const long double ds = sq * t.Dl[q * n + i] / si;
      M[0][q * n + i] = ns; M[1][i * n + q] = ns;
      M[2][q * n + i] = ds; M[3][i * n + q] = ds;
    }
  // M[4] = Ds^T Ds / 2: the 1D stiffness operator at the quadrature points that the Cartesian kernels apply as ONE
  // even-odd contraction (constant diagonal metric: Ds^T g Ds = g Ds^T Ds); symmetric and centro-symmetric
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      long double acc = 0.0L;
      for (int q = 0; q < n; ++q) acc += M[2][q * n + i] * M[2][q * n + j];
      M[4][i * n + j] = 0.5L * acc;
    }
  // M[5] = Ns diag(w~)^-1/2, w~ = the (p+1)-point Gauss-Lobatto weights with the two end weights doubled (a face
  // node of a uniform mesh belongs to two cells per direction): on a uniform box diag(M)^-1/2 of the GLL-lumped mass
  // matrix is (1/det J)^1/2 times the Kronecker product of diag(w~)^-1/2, so that the mass scaling of
  // H~ = M^-1/2 H M^-1/2 is absorbed by the interpolation tables and costs nothing in the kernels
  {
    long double xl[fe::MAXN];
    fe::gll_nodes(t.p, xl);
    for (int i = 0; i < n; ++i) {
      long double pn, pm;
      fe::legendre(t.p, xl[i], pn, pm);
      long double wg = 2.0L / ((long double)t.p * (t.p + 1) * pn * pn);
      if (i == 0 || i == n - 1) wg *= 2.0L;
      const long double si = 1.0L / sqrtl(wg);
      for (int q = 0; q < n; ++q) M[5][q * n + i] = M[0][q * n + i] * si;
    }
  }
  fe::EoTab tabs[6];
  for (int k = 0; k < 6; ++k) {
    std::memset(&tabs[k], 0, sizeof(fe::EoTab));
    for (int q = 0; q < h; ++q) {
      for (int i = 0; i < h; ++i) {
        tabs[k].P[q * h + i] = (double)(0.5L * (M[k][q * n + i] + M[k][q * n + (n - 1 - i)]));
        tabs[k].Mn[q * h + i] = (double)(0.5L * (M[k][q * n + i] - M[k][q * n + (n - 1 - i)]));
      }
      if (n & 1) tabs[k].Pm[q] = (double)M[k][q * n + m];
    }
    if (n & 1) {
      for (int i = 0; i < h; ++i) tabs[k].mid[i] = (double)M[k][m * n + i];
      tabs[k].midm = (double)M[k][m * n + m];
    }
  }
  for (int k = 0; k < 5; ++k) out[k] = tabs[k];
  // the plane / line kernels' tables: Ns, Ds (the transposes reuse them) and Ds^T Ds / 2, plus the halved middle
  // column / row
  const int src[fe::MAT_COUNT] = {0, 2, 4, 5};   // MAT_NS, MAT_DS, MAT_SH, MAT_NSS
  for (int k2 = 0; k2 < fe::MAT_COUNT; ++k2) {
    const fe::EoTab& s = tabs[src[k2]];
    fe::EoTab2& d = out2[k2];
    std::memset(&d, 0, sizeof(fe::EoTab2));
    for (int i = 0; i < 16; ++i) { d.P[i] = s.P[i]; d.Mn[i] = s.Mn[i]; }
    for (int i = 0; i < 4; ++i) { d.Pm[i] = s.Pm[i]; d.mid[i] = s.mid[i]; d.Pmh[i] = 0.5 * s.Pm[i]; d.midh[i] = 0.5 * s.mid[i]; }
    d.midm = s.midm; d.midmh = 0.5 * s.midm;
  }
}

}  // namespace fe_host
