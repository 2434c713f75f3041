// Box peaks for the roofline (north_star: "peaks measured on the box by a stream/DGEMM
// microbenchmark"): FP64 FMA-chain throughput and FP64 stream-copy bandwidth.
#include "../../include/fe_mf.h"

#include <cuda_runtime.h>

namespace {

template <int ITERS>
__global__ void probe_dfma(double* out, double a, double b) {
  double acc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i] = threadIdx.x * 1e-3 + i;
  for (int it = 0; it < ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = fma(acc[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += acc[i];
  if (s == 12345.678) out[0] = s;
}

__global__ void probe_copy(double2* __restrict__ dst, const double2* __restrict__ src, size_t n2) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; i < n2; i += stride) dst[i] = src[i];
}

}  // namespace

extern "C" int fe_probe_peaks(double* fp64_tflops, double* hbm_gbs, int cuda_device) {
  if (!fp64_tflops || !hbm_gbs) return FE_MF_EINVAL;
  if (cudaSetDevice(cuda_device) != cudaSuccess) return FE_MF_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return FE_MF_ECUDA;
  const int nsm = prop.multiProcessorCount;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double* out = nullptr;
  if (cudaMalloc(&out, 64) != cudaSuccess) return FE_MF_ENOMEM;
  constexpr int IT = 8192;
  const int threads = 512, blocks = nsm * 2;
  float best = 1e30f;
  for (int r = 0; r < 6; ++r) {
    cudaEventRecord(e0);
    probe_dfma<IT><<<blocks, threads>>>(out, 1.0000001, 1e-9);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (r > 0 && ms < best) best = ms;
  }
  *fp64_tflops = 2.0 * 8 * IT * (double)threads * blocks / (best * 1e-3) * 1e-12;
  cudaFree(out);
  const size_t bytes = (size_t)1 << 31;  // 2 GiB each way
  double2 *a = nullptr, *b = nullptr;
  if (cudaMalloc(&a, bytes) != cudaSuccess || cudaMalloc(&b, bytes) != cudaSuccess) {
    if (a) cudaFree(a);
    (void)cudaGetLastError();
    return FE_MF_ENOMEM;
  }
  cudaMemset(a, 0, bytes); cudaMemset(b, 0, bytes);
  best = 1e30f;
  for (int r = 0; r < 6; ++r) {
    cudaEventRecord(e0);
    probe_copy<<<nsm * 16, 512>>>(b, a, bytes / 16);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (r > 0 && ms < best) best = ms;
  }
  *hbm_gbs = 2.0 * (double)bytes / (best * 1e-3) * 1e-9;
  cudaFree(a); cudaFree(b);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return cudaGetLastError() == cudaSuccess ? FE_MF_OK : FE_MF_ECUDA;
}
