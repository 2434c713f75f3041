// Test helper: the two kernels of paper_2208_07129_b200/csrc/fe_constraints.cu (their exact source, cut out between the
// [device-code-begin] / [device-code-end] markers into emul_constraints_kernels.inc by tests/test_host_emulation.py), run
// on CPU threads and compared with plain loops over the sets.  Prints "name nvec maxerr" lines.
#include <cstdio>
#include <random>

#include "cuda_runtime.h"
constexpr int kThreads = 256;
constexpr int kVecBlock = 32;
#include "emul_constraints_kernels.inc"

int main() {
  std::mt19937_64 rng(7);
  std::uniform_real_distribution<double> U(-1, 1);
  for (int nvec : {1, 5, 32, 40}) {
    const long long ndof = 600;
    const int nsets = 9;
    std::vector<long long> perm(ndof);
    for (long long i = 0; i < ndof; ++i) perm[i] = i;
    std::shuffle(perm.begin(), perm.end(), rng);
    std::vector<long long> mp{0}, sp{0}, wp{0}, ms, sl;
    std::vector<double> W, b;
    long long k = 0;
    for (int I = 0; I < nsets; ++I) {      // slaves from perm[0..300), masters from perm[300..600): closed sets; set 0 has no masters
      const int ns = 1 + (int)(rng() % 30), nm = I == 0 ? 0 : 1 + (int)(rng() % 12);
      for (int s = 0; s < ns; ++s) sl.push_back(perm[k++]);
      for (int m = 0; m < nm; ++m) ms.push_back(perm[300 + (rng() % 300)]);
      for (int e = 0; e < ns * nm; ++e) W.push_back(U(rng));
      for (int s = 0; s < ns; ++s) b.push_back(U(rng));
      mp.push_back((long long)ms.size()); sp.push_back((long long)sl.size()); wp.push_back((long long)W.size());
    }
    if (k > 300) return 2;
    SetArrays A{mp.data(), sp.data(), wp.data(), ms.data(), sl.data(), W.data(), b.data()};
    std::vector<double> X(ndof * nvec);
    for (auto& v : X) v = U(rng);
    const unsigned gy = (nvec + kVecBlock - 1) / kVecBlock;
    for (int hom = 0; hom < 2; ++hom) {
      std::vector<double> got = X, ref = X;
      emul_launch(nsets, gy, kThreads, [&] { fe_constraints_distribute_kernel(A, got.data(), nvec, hom); });
      for (int I = 0; I < nsets; ++I)
        for (long long s = sp[I]; s < sp[I + 1]; ++s)
          for (int v = 0; v < nvec; ++v) {
            double acc = hom ? 0.0 : b[s];
            const long long nm = mp[I + 1] - mp[I];
            for (long long m = 0; m < nm; ++m) acc += W[wp[I] + (s - sp[I]) * nm + m] * X[ms[mp[I] + m] * nvec + v];
            ref[sl[s] * nvec + v] = acc;
          }
      double e = 0;
      for (size_t i = 0; i < ref.size(); ++i) e = std::max(e, std::fabs(ref[i] - got[i]));
      printf("distribute_hom%d %d %.3e\n", hom, nvec, e);
    }
    std::vector<double> got = X, ref = X;
    emul_launch(nsets, gy, kThreads, [&] { fe_constraints_transpose_kernel(A, got.data(), nvec); });
    for (int I = 0; I < nsets; ++I) {
      const long long nm = mp[I + 1] - mp[I];
      for (long long m = 0; m < nm; ++m)
        for (int v = 0; v < nvec; ++v) {
          double acc = 0;
          for (long long s = sp[I]; s < sp[I + 1]; ++s) acc += W[wp[I] + (s - sp[I]) * nm + m] * X[sl[s] * nvec + v];
          ref[ms[mp[I] + m] * nvec + v] += acc;
        }
    }
    for (size_t s = 0; s < sl.size(); ++s)
      for (int v = 0; v < nvec; ++v) ref[sl[s] * nvec + v] = 0;
    double e = 0;
    for (size_t i = 0; i < ref.size(); ++i) e = std::max(e, std::fabs(ref[i] - got[i]));
    printf("transpose %d %.3e\n", nvec, e);
  }
  return 0;
}
