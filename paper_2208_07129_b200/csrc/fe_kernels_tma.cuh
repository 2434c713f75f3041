// Device code, part 4: building blocks of the persistent TMA kernels (fe_kernels_plane.cuh, fe_kernels_line.cuh,
// fe_kernels_gen.cuh): mbarrier / bulk-tensor PTX wrappers, the dense tile layout of a TMA box, the task loop.
//   * a cell tile [z][y][x][beta] is fetched by ONE 4-D tensor-map bulk copy (cp.async.bulk.tensor, SASS UTMALDG)
//     issued by one thread and tracked by an mbarrier; the result tile leaves through ONE bulk tensor reduction
//     (cp.reduce.async.bulk.tensor ... add, f64; SASS UTMAREDG): no per-thread address arithmetic, LDG or RED;
//   * out-of-range box elements (vector tail, periodic wrap, Dirichlet boundary) are zero-filled on load and
//     clipped on reduce by the TMA unit.  A reduction must not START at a negative coordinate (it faults).
#pragma once
#include <cuda.h>

#include "fe_kernels_cart2.cuh"

// A statically allocated shared-memory variable of a kernel.  (The host-thread builds of the tests define __shared__ away
// so that "extern __shared__ T name[]" becomes a plain extern array; a static variable then needs "static" instead.)
#ifdef FE_HOST_EMULATION
#define FE_STATIC_SHARED static
#else
#define FE_STATIC_SHARED __shared__
#endif

namespace fe {

// The PTX wrappers.  FE_TMA_WRAPPERS_PROVIDED: tests/host/shim/cuda.h supplies host stand-ins with the same names and
// semantics (tests/test_host_emulation.py runs the kernels on CPU threads); never defined in a CUDA build.
#ifndef FE_TMA_WRAPPERS_PROVIDED
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!done);
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_reduce_add_4d(const CUtensorMap* tm, const void* src, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.reduce.async.bulk.tensor.4d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
      ::"l"(tm), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
// 1-D bulk copy global -> shared, completion on an mbarrier (bytes and both addresses multiples of 16)
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_all0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// after mbar_init, before the barrier is used by the async proxy
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// the dynamic item counter: returns the old value (asm volatile: the compiler must not move it, nor anything that
// depends on the result, across the surrounding code)
__device__ __forceinline__ unsigned item_counter_next(int* ctr) {
  unsigned old;
  asm volatile("atom.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(ctr) : "memory");
  return old;
}
#endif  // FE_TMA_WRAPPERS_PROVIDED

// PADX = 1: the box carries one extra node per x-row (the first node of the next cell's interior, never used).
// With 8 vectors per block a node is 64 bytes, and for even n all x-lines of a dense tile start a multiple of
// 128 bytes apart, so the two lines that share a 128-byte wavefront always collide (measured at p = 7: a third of
// all shared-memory wavefronts were conflict replays); the extra node makes the row pitch an odd multiple of 64.
template <int PDEG, int BV, int PADX = 0>
struct DenseTile {
  static constexpr int N = PDEG + 1;
  static constexpr int XP = (N + PADX) * BV;          // dense: the TMA box layout
  static constexpr int SIZE = N * N * XP;             // doubles
  static constexpr int BYTES = SIZE * 8;
  static constexpr int PITCH = (BYTES + 127) / 128 * 128;   // placement of the second tile
  template <int DIR>
  static __device__ __forceinline__ void line(int l, int& base, int& stride) {
    const int a = l % N, b = l / N;
    if (DIR == 0) { base = (b * N + a) * XP; stride = BV; }
    else if (DIR == 1) { base = b * N * XP + a * BV; stride = XP; }
    else { base = b * XP + a * BV; stride = N * XP; }
  }
};

// Task loop of one phase: ROUNDS rounds of NT tasks; in the last (partial) round the tasks are rotated over
// the warps by `rot` so that the SM sub-partition (warp % 4) that gets the extra warp-task differs between
// the blocks resident on one SM and between successive items (FP64 issue is per sub-partition).
#define FE_FOR_TASKS(t)                                                                          \
  _Pragma("unroll 1") for (int r_ = 0, t = 0; r_ < ROUNDS; ++r_)                                  \
    if ((t = (r_ < ROUNDS - 1 || !ROTATE) ? tid + r_ * NT : r_ * NT + rot_tid), t < TASKS)

}  // namespace fe
