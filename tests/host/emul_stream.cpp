// Test helper: the streaming kernels of paper_2208_07129_b200/csrc/fe_kernels_stream.cuh (included as they are, with
// tests/host/shim/cuda_runtime.h standing in for the CUDA header) on CPU threads: the FP32 halo payload pair, the two
// axpby kernels (vectorised and scalar), scale, scale-copy and swap, on odd counts and small grids so that the
// grid-stride loops and the tails are exercised.  Prints "name count mismatches" lines.
#include <cstdio>
#include <cstring>
#include <random>

#include "../../paper_2208_07129_b200/csrc/fe_kernels_stream.cuh"

template <typename T>
static long long mismatches(const std::vector<T>& a, const std::vector<T>& b) {
  long long n = 0;
  for (size_t i = 0; i < a.size(); ++i) n += std::memcmp(&a[i], &b[i], sizeof(T)) != 0;
  return n;
}

int main() {
  std::mt19937_64 rng(11);
  std::uniform_real_distribution<double> U(-1, 1);
  for (size_t count : {(size_t)1, (size_t)2, (size_t)255, (size_t)1001, (size_t)4096}) {
    const unsigned grid = count < 600 ? 1 : 3, nt = 64;       // fewer threads than elements: the stride loops wrap
    std::vector<double> src(count), acc(count);
    for (auto& v : src) v = U(rng) * std::pow(10.0, (int)(rng() % 60) - 30);
    for (auto& v : acc) v = U(rng);
    // FP32 payload
    std::vector<float> p32(count + 1, 7.0f), r32(count + 1, 7.0f);
    emul_launch(grid, 1, nt, [&] { fe::fe_halo_pack_f32_kernel(p32.data(), src.data(), count); });
    for (size_t i = 0; i < count; ++i) r32[i] = (float)src[i];
    printf("pack %zu %lld\n", count, mismatches(p32, r32));
    std::vector<double> d(count + 1, -3.0), rd(count + 1, -3.0);
    emul_launch(grid, 1, nt, [&] { fe::fe_halo_unpack_f32_kernel(d.data(), p32.data(), count, 0); });
    for (size_t i = 0; i < count; ++i) rd[i] = (double)r32[i];
    printf("unpack %zu %lld\n", count, mismatches(d, rd));
    std::vector<double> a = acc, ra = acc;
    emul_launch(grid, 1, nt, [&] { fe::fe_halo_unpack_f32_kernel(a.data(), p32.data(), count, 1); });
    for (size_t i = 0; i < count; ++i) ra[i] = acc[i] + (double)r32[i];
    printf("unpack_add %zu %lld\n", count, mismatches(a, ra));
    // axpby (vectorised and scalar), scale, scale-copy, swap
    const double beta = 0.75, gamma = -1.5;
    std::vector<double> z = acc, zs = acc, rz = acc;
    emul_launch(grid, 1, nt, [&] { fe::fe_axpby_kernel(z.data(), src.data(), beta, gamma, count); });
    emul_launch(grid, 1, nt, [&] { fe::fe_axpby_scalar_kernel(zs.data(), src.data(), beta, gamma, count); });
    for (size_t i = 0; i < count; ++i) rz[i] = beta * acc[i] + gamma * src[i];
    printf("axpby %zu %lld\n", count, mismatches(z, rz));
    printf("axpby_scalar %zu %lld\n", count, mismatches(zs, rz));
    z = acc;
    emul_launch(grid, 1, nt, [&] { fe::fe_scale_kernel(z.data(), beta, count); });
    for (size_t i = 0; i < count; ++i) rz[i] = acc[i] * beta;
    printf("scale %zu %lld\n", count, mismatches(z, rz));
    z = acc;
    emul_launch(grid, 1, nt, [&] { fe::fe_scale_copy_kernel(z.data(), src.data(), gamma, count); });
    for (size_t i = 0; i < count; ++i) rz[i] = gamma * src[i];
    printf("scale_copy %zu %lld\n", count, mismatches(z, rz));
    std::vector<double> s1 = src, s2 = acc;
    emul_launch(grid, 1, nt, [&] { fe::fe_swap_kernel(s1.data(), s2.data(), count); });
    printf("swap %zu %lld\n", count, mismatches(s1, acc) + mismatches(s2, src));
  }
  return 0;
}
