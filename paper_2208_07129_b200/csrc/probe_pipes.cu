// Box probe (standalone program, NOT part of libfe_mf.so): does the FP64 tensor-core instruction (DMMA, PTX
// mma.sync.m8n8k4.f64) add FP64 throughput on top of the FP64 FMA pipe on this GPU, and how well do the FP64 pipe and
// the shared-memory pipe overlap?  BASELINE.json's north_star allows FP64 tensor cores "only if ncu shows the batched
// contractions are compute-bound"; the kernels are FP64-bound at p = 6, 7, so the question is whether DMMA is a second
// pipe.  DESIGN.md section 5 quotes the output (profiles/r2_probe_pipes.md holds the raw text and the command).
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/probe_pipes paper_2208_07129_b200/csrc/probe_pipes.cu
//   /tmp/probe_pipes
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA error %s at %s:%d\n", cudaGetErrorString(e_), __FILE__, __LINE__); exit(1); } } while (0)

constexpr int ITERS = 4096;

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// MODE 0: 8 independent DFMA chains per thread.  MODE 1: 4 independent DMMA chains (8 accumulator registers).
// MODE 2: both interleaved in every warp (8 DFMA + 4 DMMA per iteration).  MODE 3: even warps DFMA, odd warps DMMA.
template <int MODE>
__global__ void probe_fp64(double* out, double a, double b) {
  double f[8], d[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { f[i] = threadIdx.x * 1e-3 + i; d[i] = threadIdx.x * 1e-4 + i; }
  const bool do_fma = MODE == 0 || MODE == 2 || (MODE == 3 && ((threadIdx.x >> 5) & 1) == 0);
  const bool do_mma = MODE == 1 || MODE == 2 || (MODE == 3 && ((threadIdx.x >> 5) & 1) == 1);
  for (int it = 0; it < ITERS; ++it) {
    if (do_fma) {
#pragma unroll
      for (int i = 0; i < 8; ++i) f[i] = fma(f[i], a, b);
    }
    if (do_mma) {
#pragma unroll
      for (int i = 0; i < 4; ++i) dmma(d[2 * i], d[2 * i + 1], a, b);
    }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += f[i] + d[i];
  if (s == 12345.678) out[0] = s;
}

// Shared-memory loads (LDS.128, conflict-free) with FPL FP64 FMAs per load: how far do the two pipes overlap?
template <int FPL>
__global__ void probe_lds_fma(double* out, double a, double b) {
  __shared__ double2 buf[2048];
  for (int i = threadIdx.x; i < 2048; i += blockDim.x) buf[i] = make_double2(i, -i);
  __syncthreads();
  double f[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) f[i] = threadIdx.x + i;
  int idx = threadIdx.x;
  for (int it = 0; it < ITERS; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const double2 v = buf[(idx + u * 256) & 2047];
      f[u] = fma(v.y, 1e-300, fma(v.x, 1e-300, f[u]));   // consumes the load (2 DFMA)
#pragma unroll
      for (int k = 0; k < FPL - 2; ++k) f[(u + k + 1) & 7] = fma(f[(u + k + 1) & 7], a, b);
    }
    idx = (idx + 32) & 2047;
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += f[i];
  if (s == 12345.678) out[0] = s;
}

template <typename K>
float time_kernel(K kern, int blocks, int threads, double* out) {
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  float best = 1e30f;
  for (int r = 0; r < 5; ++r) {
    CK(cudaEventRecord(e0));
    kern<<<blocks, threads>>>(out, 1.0000001, 1e-9);
    CK(cudaEventRecord(e1)); CK(cudaEventSynchronize(e1));
    float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
    if (r > 0 && ms < best) best = ms;
  }
  CK(cudaGetLastError());
  return best;
}

int main() {
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, 0));
  const int nsm = prop.multiProcessorCount;
  int clk_khz = 0;
  CK(cudaDeviceGetAttribute(&clk_khz, cudaDevAttrClockRate, 0));
  printf("device %s, %d SMs, max SM clock %.0f MHz; nominal FP64 FMA peak = SMs x 64 FMA/clk x 2 x clock = %.2f TFLOP/s\n",
         prop.name, nsm, clk_khz / 1e3, nsm * 64.0 * 2.0 * clk_khz * 1e3 / 1e12);
  double* out;
  CK(cudaMalloc(&out, 64));
  const int threads = 512, blocks = nsm * 2;   // 32 warps per SM
  const double lanes = (double)threads * blocks;
  const double fma_flops = 2.0 * 8 * ITERS * lanes;                 // 8 DFMA per thread and iteration
  const double mma_flops = 2.0 * 8 * 8 * 4 * 4.0 * ITERS * (lanes / 32);   // 4 DMMA (8x8x4) per warp and iteration
  float t;
  t = time_kernel(probe_fp64<0>, blocks, threads, out);
  printf("DFMA only                      : %7.3f ms  %6.2f TFLOP/s\n", t, fma_flops / (t * 1e-3) / 1e12);
  t = time_kernel(probe_fp64<1>, blocks, threads, out);
  printf("DMMA m8n8k4 only               : %7.3f ms  %6.2f TFLOP/s\n", t, mma_flops / (t * 1e-3) / 1e12);
  t = time_kernel(probe_fp64<2>, blocks, threads, out);
  printf("DFMA + DMMA in every warp      : %7.3f ms  %6.2f TFLOP/s (sum of both)   [a second pipe would keep the DFMA-only time]\n", t,
         (fma_flops + mma_flops) / (t * 1e-3) / 1e12);
  t = time_kernel(probe_fp64<3>, blocks, threads, out);
  printf("even warps DFMA, odd warps DMMA: %7.3f ms  %6.2f TFLOP/s (sum of both)\n", t, (0.5 * fma_flops + 0.5 * mma_flops) / (t * 1e-3) / 1e12);
  // shared memory alone and with FP64 work
  const double lds_bytes = 16.0 * 4 * ITERS * lanes;
  t = time_kernel(probe_lds_fma<2>, blocks, threads, out);
  printf("LDS.128 + 2 DFMA per load      : %7.3f ms  %6.1f B/clk/SM shared, %5.2f TFLOP/s\n", t,
         lds_bytes / (t * 1e-3) / nsm / (clk_khz * 1e3), 2.0 * 2 * 4 * ITERS * lanes / (t * 1e-3) / 1e12);
  t = time_kernel(probe_lds_fma<4>, blocks, threads, out);
  printf("LDS.128 + 4 DFMA per load      : %7.3f ms  %6.1f B/clk/SM shared, %5.2f TFLOP/s\n", t,
         lds_bytes / (t * 1e-3) / nsm / (clk_khz * 1e3), 2.0 * 4 * 4 * ITERS * lanes / (t * 1e-3) / 1e12);
  t = time_kernel(probe_lds_fma<8>, blocks, threads, out);
  printf("LDS.128 + 8 DFMA per load      : %7.3f ms  %6.1f B/clk/SM shared, %5.2f TFLOP/s\n", t,
         lds_bytes / (t * 1e-3) / nsm / (clk_khz * 1e3), 2.0 * 8 * 4 * ITERS * lanes / (t * 1e-3) / 1e12);
  t = time_kernel(probe_lds_fma<16>, blocks, threads, out);
  printf("LDS.128 + 16 DFMA per load     : %7.3f ms  %6.1f B/clk/SM shared, %5.2f TFLOP/s\n", t,
         lds_bytes / (t * 1e-3) / nsm / (clk_khz * 1e3), 2.0 * 16 * 4 * ITERS * lanes / (t * 1e-3) / 1e12);
  cudaFree(out);
  return 0;
}
