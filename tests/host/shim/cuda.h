// Host stand-in for <cuda.h>, used ONLY by tests/test_host_emulation.py: CUtensorMap as plain numbers and host versions
// of the PTX wrappers of csrc/fe_kernels_tma.cuh (same names, same semantics, executed synchronously by the calling
// thread), so that the persistent TMA kernels run on CPU threads from their exact source.
//   mbarrier   a 64-bit word: low half = number of completed phases, high half = bytes still expected in the current one
//   bulk load  copies the box at once, zero-fills out-of-range elements, then completes its bytes on the barrier
//   reduce     adds the in-range elements of the box; a box that STARTS at a negative coordinate aborts (the device faults)
// The device runs the bulk copies asynchronously.  Two legal extremes are modelled: by default a copy happens AT ISSUE
// (the earliest moment: a prefetch into a tile that some thread still needs clobbers it, the result goes wrong);
// with -DFE_EMUL_LAZY_TMA it happens AS LATE AS the kernel's own synchronisation allows -- a load when a thread waits on
// its mbarrier, a reduction when the issuing thread calls tma_wait_read0 / tma_wait_all0 -- so a missing wait reads a
// tile that has not arrived or reduces a tile that has been overwritten (the result goes wrong), and a block that ends
// with copies still pending aborts.
#pragma once
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <mutex>
#include <utility>
#include <vector>

#include "cuda_runtime.h"

#define FE_TMA_WRAPPERS_PROVIDED 1

struct CUtensorMap {
  double* base;                    // the map's origin (multivector base + TensorMapDesc::base_offset)
  unsigned long long dims[4];      // elements: beta, x, y, z
  unsigned long long strides[3];   // bytes: x, y, z
  unsigned box[4];
};

inline double2 make_double2(double x, double y) { return double2{x, y}; }

namespace fe {

inline std::atomic_ref<uint64_t> emul_bar(uint64_t* bar) { return std::atomic_ref<uint64_t>(*bar); }
inline void emul_complete_tx(uint64_t* bar, uint64_t bytes) {
  auto b = emul_bar(bar);
  uint64_t old = b.load(), upd;
  do {
    if ((old >> 32) < bytes) { fprintf(stderr, "emulation: more bytes completed than expected on an mbarrier\n"); abort(); }
    upd = old - (bytes << 32);
    if ((upd >> 32) == 0) upd += 1;          // all expected bytes have landed: the phase completes
  } while (!b.compare_exchange_weak(old, upd));
}
#ifdef FE_EMUL_LAZY_TMA
inline std::mutex emul_pending_mutex;
inline std::vector<std::pair<uint64_t*, std::function<void()>>> emul_pending_loads;   // (mbarrier, the copy)
inline std::vector<std::function<void()>> emul_pending_reductions;
inline void emul_flush_loads(uint64_t* bar) {
  std::lock_guard<std::mutex> lock(emul_pending_mutex);
  for (size_t k = 0; k < emul_pending_loads.size();) {
    if (emul_pending_loads[k].first == bar) { emul_pending_loads[k].second(); emul_pending_loads.erase(emul_pending_loads.begin() + k); }
    else ++k;
  }
}
inline void emul_flush_reductions() {
  std::lock_guard<std::mutex> lock(emul_pending_mutex);
  for (auto& f : emul_pending_reductions) f();
  emul_pending_reductions.clear();
}
inline void emul_check_nothing_pending() {
  std::lock_guard<std::mutex> lock(emul_pending_mutex);
  if (!emul_pending_loads.empty() || !emul_pending_reductions.empty()) { fprintf(stderr, "emulation: a block ended with bulk copies pending\n"); abort(); }
}
#else
inline void emul_check_nothing_pending() {}
#endif
inline void mbar_init(uint64_t* bar, int) { emul_bar(bar).store(0); }
inline void mbar_init_fence() {}
inline void mbar_expect_tx(uint64_t* bar, uint32_t bytes) { emul_bar(bar).fetch_add((uint64_t)bytes << 32); }
inline void mbar_wait(uint64_t* bar, uint32_t parity) {
#ifdef FE_EMUL_LAZY_TMA
  while (true) {
    emul_flush_loads(bar);
    if (((uint32_t)emul_bar(bar).load(std::memory_order_acquire) & 1u) != parity) break;
    std::this_thread::yield();
  }
#else
  while (((uint32_t)emul_bar(bar).load(std::memory_order_acquire) & 1u) == parity) std::this_thread::yield();
#endif
}
inline long long emul_tm_offset(const CUtensorMap* tm, const long long c[4]) {   // in doubles; -1 if out of range
  for (int d = 0; d < 4; ++d)
    if (c[d] < 0 || c[d] >= (long long)tm->dims[d]) return -1;
  return c[0] + (long long)(c[1] * tm->strides[0] + c[2] * tm->strides[1] + c[3] * tm->strides[2]) / 8;
}
inline void emul_do_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3) {
  if (((uintptr_t)dst & 127) != 0) { fprintf(stderr, "emulation: bulk tensor destination not 128-byte aligned\n"); abort(); }
  double* d = static_cast<double*>(dst);
  size_t k = 0;
  for (unsigned i3 = 0; i3 < tm->box[3]; ++i3)
    for (unsigned i2 = 0; i2 < tm->box[2]; ++i2)
      for (unsigned i1 = 0; i1 < tm->box[1]; ++i1)
        for (unsigned i0 = 0; i0 < tm->box[0]; ++i0) {
          const long long c[4] = {c0 + (long long)i0, c1 + (long long)i1, c2 + (long long)i2, c3 + (long long)i3};
          const long long off = emul_tm_offset(tm, c);
          d[k++] = off < 0 ? 0.0 : tm->base[off];
        }
  emul_complete_tx(bar, (uint64_t)k * 8);
}
inline void emul_do_reduce_add_4d(const CUtensorMap* tm, const void* src, int c0, int c1, int c2, int c3) {
  if (c0 < 0 || c1 < 0 || c2 < 0 || c3 < 0) { fprintf(stderr, "emulation: bulk tensor reduction starts at a negative coordinate\n"); abort(); }
  if (((uintptr_t)src & 127) != 0) { fprintf(stderr, "emulation: bulk tensor source not 128-byte aligned\n"); abort(); }
  const double* s = static_cast<const double*>(src);
  size_t k = 0;
  for (unsigned i3 = 0; i3 < tm->box[3]; ++i3)
    for (unsigned i2 = 0; i2 < tm->box[2]; ++i2)
      for (unsigned i1 = 0; i1 < tm->box[1]; ++i1)
        for (unsigned i0 = 0; i0 < tm->box[0]; ++i0, ++k) {
          const long long c[4] = {c0 + (long long)i0, c1 + (long long)i1, c2 + (long long)i2, c3 + (long long)i3};
          const long long off = emul_tm_offset(tm, c);
          if (off >= 0) atomicAdd(tm->base + off, s[k]);
        }
}
inline void emul_do_bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  if ((((uintptr_t)dst | (uintptr_t)src | bytes) & 15) != 0) { fprintf(stderr, "emulation: bulk copy not 16-byte aligned\n"); abort(); }
  std::memcpy(dst, src, bytes);
  emul_complete_tx(bar, bytes);
}
#ifdef FE_EMUL_LAZY_TMA
inline void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3) {
  const CUtensorMap m = *tm;
  std::lock_guard<std::mutex> lock(emul_pending_mutex);
  emul_pending_loads.emplace_back(bar, [=] { emul_do_load_4d(dst, &m, bar, c0, c1, c2, c3); });
}
inline void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  std::lock_guard<std::mutex> lock(emul_pending_mutex);
  emul_pending_loads.emplace_back(bar, [=] { emul_do_bulk_load(dst, src, bytes, bar); });
}
inline void tma_reduce_add_4d(const CUtensorMap* tm, const void* src, int c0, int c1, int c2, int c3) {
  const CUtensorMap m = *tm;
  std::lock_guard<std::mutex> lock(emul_pending_mutex);
  emul_pending_reductions.push_back([=] { emul_do_reduce_add_4d(&m, src, c0, c1, c2, c3); });
}
inline void tma_wait_read0() { emul_flush_reductions(); }
inline void tma_wait_all0() { emul_flush_reductions(); }
#else
inline void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3) { emul_do_load_4d(dst, tm, bar, c0, c1, c2, c3); }
inline void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) { emul_do_bulk_load(dst, src, bytes, bar); }
inline void tma_reduce_add_4d(const CUtensorMap* tm, const void* src, int c0, int c1, int c2, int c3) { emul_do_reduce_add_4d(tm, src, c0, c1, c2, c3); }
inline void tma_wait_read0() {}
inline void tma_wait_all0() {}
#endif
inline void tma_commit() {}
inline void fence_async_smem() {}
inline unsigned item_counter_next(int* ctr) { return (unsigned)std::atomic_ref<int>(*ctr).fetch_add(1); }

}  // namespace fe
