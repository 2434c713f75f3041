// Host stand-in for <cuda_runtime.h>, used ONLY by tests/test_host_emulation.py: enough of the CUDA execution model to
// run simple kernels of the library on CPU threads -- one std::thread per CUDA thread of a block, a std::barrier for
// __syncthreads(), blocks one after another.  No GPU semantics beyond that (no warps, no memory model).
#pragma once
#include <algorithm>
#include <barrier>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <mutex>
#include <thread>
#include <vector>

struct double2 { double x, y; };
struct EmulDim3 { unsigned x = 1, y = 1, z = 1; };
inline thread_local EmulDim3 blockIdx, threadIdx, blockDim, gridDim;
inline std::barrier<>* emul_barrier = nullptr;
inline std::mutex emul_atomic_mutex;

#define FE_HOST_EMULATION 1
#define __global__
#define __device__
#define __host__
#define __constant__
#define __shared__                       // "extern __shared__ double smem[]" becomes a plain extern array the test program defines
#define __forceinline__ inline
#define __launch_bounds__(...)
#define __grid_constant__
#define __align__(n)                     // the test program defines the shared-memory array with the alignment
template <typename T>
inline T __ldg(const T* p) { return *p; }
#define __syncthreads() emul_barrier->arrive_and_wait()
using std::min;
using std::max;

inline double atomicAdd(double* p, double v) {
  std::lock_guard<std::mutex> lock(emul_atomic_mutex);
  const double old = *p;
  *p = old + v;
  return old;
}
inline float __double2float_rn(double x) { return static_cast<float>(x); }   // IEEE round to nearest even on the host

// launch f() on a grid of gx x gy blocks of nt threads
template <typename F>
void emul_launch(unsigned gx, unsigned gy, unsigned nt, F f) {
  for (unsigned by = 0; by < gy; ++by)
    for (unsigned bx = 0; bx < gx; ++bx) {
      std::barrier<> bar(nt);
      emul_barrier = &bar;
      std::vector<std::thread> threads;
      for (unsigned t = 0; t < nt; ++t)
        threads.emplace_back([=] {
          blockIdx.x = bx; blockIdx.y = by; threadIdx.x = t;
          blockDim.x = nt; gridDim.x = gx; gridDim.y = gy;
          f();
        });
      for (auto& th : threads) th.join();
    }
}
