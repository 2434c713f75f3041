// Test helper (host only, no CUDA): prints the 1-D tables and the geometric factors that fe_mf_create computes on the host
// (S0 of SURVEY.md 8(a); paper_2208_07129_b200/csrc/fe_tables.h) so that tests/test_host_tables.py can compare them with the
// oracle without a GPU.   usage: dump_tables <p>
#include <cstdio>
#include <cstdlib>

#include "../../paper_2208_07129_b200/csrc/fe_tables.h"

int main(int argc, char** argv) {
  const int p = argc > 1 ? atoi(argv[1]) : 3;
  const fe::Tables1D t = fe::make_tables(p);
  const int n = p + 1;
  printf("xi");  for (int i = 0; i < n; ++i) printf(" %.17g", t.xi[i]);  printf("\n");
  printf("xq");  for (int i = 0; i < n; ++i) printf(" %.17g", t.xq[i]);  printf("\n");
  printf("w");   for (int i = 0; i < n; ++i) printf(" %.17g", t.w[i]);   printf("\n");
  printf("N");   for (int k = 0; k < n * n; ++k) printf(" %.17g", t.N[k]);  printf("\n");
  printf("Dt");  for (int k = 0; k < n * n; ++k) printf(" %.17g", t.Dt[k]); printf("\n");
  // a distorted cell: metric factors at one reference point
  const double v[8][3] = {{0, 0, 0}, {1.1, 0.05, -0.02}, {0.03, 0.9, 0.04}, {1.0, 1.05, 0.1},
                          {-0.05, 0.02, 1.2}, {1.08, 0.0, 1.1}, {0.1, 1.0, 1.15}, {1.2, 0.95, 1.3}};
  const double xi[3] = {0.3, -0.55, 0.8};
  double J[3][3], m[7];
  fe::trilinear_jacobian(v, xi, J);
  const bool ok = fe::metric_from_jacobian(J, m);
  printf("J");  for (int a = 0; a < 3; ++a) for (int c = 0; c < 3; ++c) printf(" %.17g", J[a][c]);  printf("\n");
  printf("metric %d", ok ? 1 : 0);  for (int k = 0; k < 7; ++k) printf(" %.17g", m[k]);  printf("\n");
  return 0;
}
