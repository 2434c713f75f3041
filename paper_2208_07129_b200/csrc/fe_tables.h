// Host-side setup (S0 of SURVEY.md §8(a)): 1D nodes, quadrature and Lagrange tables in extended
// precision, and the geometric factors of PAPER.md:124/128.  Plain C++ (no CUDA); shares nothing
// with oracle/.
#pragma once
#include <cmath>
#include <vector>

namespace fe {

constexpr int MAXN = 9;  // p <= 8

struct Tables1D {
  int p = 0, n = 0;
  double xi[MAXN];           // GLL nodes
  double xq[MAXN];           // Gauss-Legendre points
  double w[MAXN];            // Gauss-Legendre weights
  double N[MAXN * MAXN];     // N[q*n+i]  = l_i(xq_q)
  double Dt[MAXN * MAXN];    // Dt[q*n+r] = l~_r'(xq_q)
  long double Nl[MAXN * MAXN], Dl[MAXN * MAXN], wl[MAXN];  // the same before rounding to double
};

inline void legendre(int n, long double x, long double& pn, long double& pnm1) {
  long double p0 = 1.0L, p1 = x;
  if (n == 0) { pn = 1.0L; pnm1 = 0.0L; return; }
  for (int k = 2; k <= n; ++k) {
    long double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k;
    p0 = p1; p1 = p2;
  }
  pn = p1; pnm1 = p0;
}

// GLL nodes: +-1 and the roots of P_p', Newton with the Legendre ODE for P_p''.
inline void gll_nodes(int p, long double* x) {
  const long double pi = 3.14159265358979323846264338327950288L;
  x[0] = -1.0L; x[p] = 1.0L;
  for (int k = 1; k < p; ++k) {
    long double t = -cosl(pi * k / p);
    for (int it = 0; it < 100; ++it) {
      long double pn, pm; legendre(p, t, pn, pm);
      long double d1 = p * (t * pn - pm) / (t * t - 1.0L);
      long double d2 = (2.0L * t * d1 - (long double)p * (p + 1) * pn) / (1.0L - t * t);
      long double dt = d1 / d2;
      t -= dt;
      if (fabsl(dt) < 1e-19L) break;
    }
    x[k] = t;
  }
  for (int k = 0; k <= p / 2; ++k) {  // exact anti-symmetry
    long double s = (x[p - k] - x[k]) / 2.0L;
    x[k] = -s; x[p - k] = s;
  }
}

inline void gauss_legendre(int n, long double* x, long double* w) {
  const long double pi = 3.14159265358979323846264338327950288L;
  for (int k = 0; k < n; ++k) {
    long double t = -cosl(pi * (k + 0.75L) / (n + 0.5L));
    long double d1 = 0;
    for (int it = 0; it < 100; ++it) {
      long double pn, pm; legendre(n, t, pn, pm);
      d1 = n * (t * pn - pm) / (t * t - 1.0L);
      long double dt = pn / d1;
      t -= dt;
      if (fabsl(dt) < 1e-19L) break;
    }
    long double pn, pm; legendre(n, t, pn, pm);
    d1 = n * (t * pn - pm) / (t * t - 1.0L);
    x[k] = t;
    w[k] = 2.0L / ((1.0L - t * t) * d1 * d1);
  }
  for (int k = 0; k < n / 2; ++k) {
    long double s = (x[n - 1 - k] - x[k]) / 2.0L, ww = (w[k] + w[n - 1 - k]) / 2.0L;
    x[k] = -s; x[n - 1 - k] = s; w[k] = w[n - 1 - k] = ww;
  }
  if (n & 1) x[n / 2] = 0.0L;
}

inline Tables1D make_tables(int p) {
  Tables1D t; t.p = p; t.n = p + 1;
  const int n = p + 1;
  long double xi[MAXN], xq[MAXN], w[MAXN];
  gll_nodes(p, xi);
  gauss_legendre(n, xq, w);
  for (int i = 0; i < n; ++i) { t.xi[i] = (double)xi[i]; t.xq[i] = (double)xq[i]; t.w[i] = (double)w[i]; t.wl[i] = w[i]; }
  // N[q][i] = prod_{j != i} (xq_q - xi_j)/(xi_i - xi_j)
  for (int q = 0; q < n; ++q)
    for (int i = 0; i < n; ++i) {
      long double v = 1.0L;
      for (int j = 0; j < n; ++j) if (j != i) v *= (xq[q] - xi[j]) / (xi[i] - xi[j]);
      t.Nl[q * n + i] = v;
    }
  // Dt[q][r] = l~_r'(xq_q) on the quadrature points: barycentric form
  long double c[MAXN];
  for (int r = 0; r < n; ++r) { c[r] = 1.0L; for (int j = 0; j < n; ++j) if (j != r) c[r] *= (xq[r] - xq[j]); }
  for (int q = 0; q < n; ++q)
    for (int r = 0; r < n; ++r) {
      long double v = 0.0L;
      if (q != r) v = (c[q] / c[r]) / (xq[q] - xq[r]);
      else for (int j = 0; j < n; ++j) if (j != q) v += 1.0L / (xq[q] - xq[j]);
      t.Dl[q * n + r] = v;
    }
  // enforce the exact centro-(anti)symmetry the even-odd kernels assume (reading 14)
  for (int q = 0; q < n; ++q)
    for (int i = 0; i < n; ++i) {
      int q2 = n - 1 - q, i2 = n - 1 - i;
      if (q * n + i < q2 * n + i2) {
        long double a = 0.5L * (t.Nl[q * n + i] + t.Nl[q2 * n + i2]);
        t.Nl[q * n + i] = t.Nl[q2 * n + i2] = a;
        long double d = 0.5L * (t.Dl[q * n + i] - t.Dl[q2 * n + i2]);
        t.Dl[q * n + i] = d; t.Dl[q2 * n + i2] = -d;
      } else if (q * n + i == q2 * n + i2) {
        t.Dl[q * n + i] = 0.0L;  // centre of an odd-n table
      }
    }
  for (int k = 0; k < n * n; ++k) { t.N[k] = (double)t.Nl[k]; t.Dt[k] = (double)t.Dl[k]; }
  return t;
}

// Trilinear Jacobian J[a][c] = dx_a/dxi_c at reference point xi; vertex v = v1 + 2 v2 + 4 v3 at
// corner (2v1-1, 2v2-1, 2v3-1) (reference cell [-1,1]^3).
inline void trilinear_jacobian(const double v[8][3], const double xi[3], double J[3][3]) {
  for (int a = 0; a < 3; ++a) for (int c = 0; c < 3; ++c) J[a][c] = 0.0;
  for (int k = 0; k < 8; ++k) {
    double s[3] = {(k & 1) ? 1.0 : -1.0, (k & 2) ? 1.0 : -1.0, (k & 4) ? 1.0 : -1.0};
    double f[3] = {0.5 * (1 + s[0] * xi[0]), 0.5 * (1 + s[1] * xi[1]), 0.5 * (1 + s[2] * xi[2])};
    double d[3] = {0.5 * s[0] * f[1] * f[2], 0.5 * s[1] * f[0] * f[2], 0.5 * s[2] * f[0] * f[1]};
    for (int a = 0; a < 3; ++a) for (int c = 0; c < 3; ++c) J[a][c] += v[k][a] * d[c];
  }
}

// out[0..5] = (J^-1 J^-T)_{00,01,02,11,12,22} * det J, out[6] = det J.  Returns false if det J <= 0.
inline bool metric_from_jacobian(const double J[3][3], double out[7]) {
  double c00 = J[1][1] * J[2][2] - J[1][2] * J[2][1];
  double c01 = J[1][2] * J[2][0] - J[1][0] * J[2][2];
  double c02 = J[1][0] * J[2][1] - J[1][1] * J[2][0];
  double det = J[0][0] * c00 + J[0][1] * c01 + J[0][2] * c02;
  if (!(det > 0.0)) return false;
  double inv[3][3];  // inv = J^-1
  inv[0][0] = c00 / det;
  inv[1][0] = c01 / det;
  inv[2][0] = c02 / det;
  inv[0][1] = (J[0][2] * J[2][1] - J[0][1] * J[2][2]) / det;
  inv[1][1] = (J[0][0] * J[2][2] - J[0][2] * J[2][0]) / det;
  inv[2][1] = (J[0][1] * J[2][0] - J[0][0] * J[2][1]) / det;
  inv[0][2] = (J[0][1] * J[1][2] - J[0][2] * J[1][1]) / det;
  inv[1][2] = (J[0][2] * J[1][0] - J[0][0] * J[1][2]) / det;
  inv[2][2] = (J[0][0] * J[1][1] - J[0][1] * J[1][0]) / det;
  int k = 0;
  for (int s = 0; s < 3; ++s)
    for (int d = s; d < 3; ++d) {
      double g = 0.0;
      for (int a = 0; a < 3; ++a) g += inv[s][a] * inv[d][a];   // (J^-1 J^-T)_sd
      out[k++] = g * det;
    }
  out[6] = det;
  return true;
}

}  // namespace fe
