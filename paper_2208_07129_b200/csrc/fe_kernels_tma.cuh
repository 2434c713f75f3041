// Device code, part 4: persistent Cartesian kernel with TMA gather and TMA reduce-scatter.
//
// Same fused even-odd pass structure as fe_apply_cart2, but
//   * the cell tile [z][y][x][beta] is fetched by ONE 4-D tensor-map bulk copy (cp.async.bulk.tensor,
//     SASS UTMALDG) issued by one thread and tracked by an mbarrier, and the result tile leaves through
//     ONE bulk tensor reduction (cp.reduce.async.bulk.tensor ... add, f64; SASS UTMAREDG): no per-thread
//     address arithmetic, predicates, LDG or RED in the steady state;
//   * blocks are persistent (grid = resident blocks) and prefetch the next item's tile into tile A as soon
//     as phase 4 has consumed it, so the gather latency hides behind phases 5-6 and the reduction drains
//     behind phases 0-1 of the next item;
//   * out-of-range box elements (vector tail, periodic wrap) are zero-filled on load and clipped on
//     reduce by the TMA unit; Dirichlet nodes are masked in registers; the few periodic wrap-around
//     elements of the last cell in each direction are patched with direct LDG / RED.
#pragma once
#include <cuda.h>

#include "fe_kernels_cart2.cuh"

namespace fe {

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

template <int PDEG, int BV>
struct DenseTile {
  static constexpr int N = PDEG + 1;
  static constexpr int XP = N * BV;                   // dense: the TMA box layout
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

// timing experiments (never used by the product path): DBG 1 = no FP64 work, DBG 2 = no block barriers
#define FE_SYNC() do { if (DBG != 2) __syncthreads(); } while (0)
template <int PDEG, int MAT, bool TRANS, int DBG, typename T>
__device__ __forceinline__ void eo2d(const T (&x)[PDEG + 1], T (&y)[PDEG + 1]) {
  if (DBG == 1) {
#pragma unroll
    for (int i = 0; i <= PDEG; ++i) y[i] = x[i];
  } else {
    eo2<PDEG, MAT, TRANS>(x, y);
  }
}
template <int PDEG, int DBG, typename T>
__device__ __forceinline__ void kterm2d(const T (&t)[PDEG + 1], T (&r)[PDEG + 1], double g) {
  if (DBG == 1) {
#pragma unroll
    for (int i = 0; i <= PDEG; ++i) r[i] = r[i] + vmul(g, t[i]);
  } else {
    kterm2<PDEG>(t, r, g);
  }
}
// Task loop of one phase: ROUNDS rounds of NT tasks; in the last (partial) round the tasks are rotated over
// the warps by `rot` so that the SM sub-partition (warp % 4) that gets the extra warp-task differs between
// the blocks resident on one SM and between successive items (FP64 issue is per sub-partition).
#define FE_FOR_TASKS(t)                                                                          \
  _Pragma("unroll 1") for (int r_ = 0, t = 0; r_ < ROUNDS; ++r_)                                  \
    if ((t = (r_ < ROUNDS - 1 || !ROTATE) ? tid + r_ * NT : r_ * NT + rot_tid), t < TASKS)

template <int PDEG, int BV, int NT, int MINB, bool TMA_OUT, int DBG = 0>
__global__ void __launch_bounds__(NT, MINB)
fe_apply_cart_tma(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmZ,
                  const ApplyParams P, int nitems) {
  using TL = DenseTile<PDEG, BV>;
  constexpr int N = PDEG + 1, NL = N * N, TPL = BV / 2, TASKS = NL * TPL;
  constexpr int ROUNDS = (TASKS + NT - 1) / NT;
  constexpr bool ROTATE = (NT % 32 == 0) && (NT >= 128);
  constexpr int NW = NT / 32;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* A = reinterpret_cast<double*>(smem_raw);
  double* B = reinterpret_cast<double*>(smem_raw + TL::PITCH);
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * TL::PITCH);
  const int tid = threadIdx.x;
  const double gxx = P.ug[0], gyy = P.ug[3], gzz = P.ug[5], gm = P.ug[6];
  const long long nvec = P.nvec;
  const bool dirichlet = P.dirichlet != 0;

  if (tid == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  FE_SYNC();

  int item = blockIdx.x;
  if (tid == 0 && item < nitems) {
    const int vb = item % P.nvb, cell = item / P.nvb;
    const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
    mbar_expect_tx(bar, TL::BYTES);
    tma_load_4d(A, &tmW, bar, vb * BV, ex * PDEG, ey * PDEG, ez * PDEG);
  }
  uint32_t parity = 0;
  int rot = (blockIdx.x / P.nsm) & 3;
  for (; item < nitems; item += gridDim.x, rot = (rot + 1) & 3) {
    const int rot_tid = ROTATE ? ((((tid >> 5) + NW - rot) % NW) << 5) + (tid & 31) : tid;
    const int vb = item % P.nvb, cell = item / P.nvb;
    const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
    const int v0 = vb * BV;
    // periodic wrap of the last cell in a direction / Dirichlet boundary cells
    const bool wx = !dirichlet && ex == P.ncx - 1, wy = !dirichlet && ey == P.ncy - 1, wz = !dirichlet && ez == P.ncz - 1;
    const bool special = dirichlet ? (ex == 0 || ex == P.ncx - 1 || ey == 0 || ey == P.ncy - 1 || ez == 0 || ez == P.ncz - 1)
                                   : (wx || wy || wz);
    mbar_wait(bar, parity);
    parity ^= 1u;

    // phase 0: Ns along x, in place in A; boundary masking / wrap patching
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 x[N], y[N];
      lds_line2<N>(A + base + b2, stride, x);
      if (special) {
        const int i2 = l % N, i3 = l / N;
        if (dirichlet) {
          const int iy = ey * PDEG + i2, iz = ez * PDEG + i3;
          if (iy == 0 || iy == P.ndy - 1 || iz == 0 || iz == P.ndz - 1) {
#pragma unroll
            for (int i = 0; i < N; ++i) x[i] = {0.0, 0.0};
          }
          if (ex == 0) x[0] = {0.0, 0.0};
          if (ex == P.ncx - 1) x[N - 1] = {0.0, 0.0};
        } else if ((v0 + b2) < P.nvec) {
          int iy = ey * PDEG + i2, iz = ez * PDEG + i3;
          const bool line_wrapped = (iy >= P.ndy) || (iz >= P.ndz);
          if (iy >= P.ndy) iy -= P.ndy;
          if (iz >= P.ndz) iz -= P.ndz;
          const long long row = (long long)P.ndx * ((long long)iy + (long long)P.ndy * iz);
          const double* src = P.W + (row + (long long)ex * PDEG) * nvec + v0 + b2;
          if (line_wrapped) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
              long long off = (long long)i * nvec;
              if (wx && i == N - 1) off -= (long long)P.ndx * nvec;
              const double2 d = __ldg(reinterpret_cast<const double2*>(src + off));
              x[i] = {d.x, d.y};
            }
          } else if (wx) {
            const double2 d = __ldg(reinterpret_cast<const double2*>(src + (long long)(PDEG - P.ndx) * nvec));
            x[N - 1] = {d.x, d.y};
          }
        }
      }
      eo2d<PDEG, MAT_NS, false, DBG>(x, y);
      sts_line2<N>(A + base + b2, stride, y);
    }
    FE_SYNC();
    // phase 1: Ns along y, in place
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<1>(l, base, stride);
      v2 x[N], y[N];
      lds_line2<N>(A + base + b2, stride, x);
      eo2d<PDEG, MAT_NS, false, DBG>(x, y);
      sts_line2<N>(A + base + b2, stride, y);
    }
    if (TMA_OUT && tid == 0) tma_wait_read0();     // the previous item's reduction has finished reading tile B
    FE_SYNC();
    // phase 2: Ns along z -> T (A); R = gm*T + Ds^T gzz Ds T along z -> B
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<2>(l, base, stride);
      v2 x[N], tq[N], r[N];
      lds_line2<N>(A + base + b2, stride, x);
      eo2d<PDEG, MAT_NS, false, DBG>(x, tq);
      sts_line2<N>(A + base + b2, stride, tq);
#pragma unroll
      for (int i = 0; i < N; ++i) r[i] = vmul(gm, tq[i]);
      kterm2d<PDEG, DBG>(tq, r, gzz);
      sts_line2<N>(B + base + b2, stride, r);
    }
    FE_SYNC();
    // phase 3: R += Ds^T gxx Ds T along x
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 tq[N], r[N];
      lds_line2<N>(A + base + b2, stride, tq);
      lds_line2<N>(B + base + b2, stride, r);
      kterm2d<PDEG, DBG>(tq, r, gxx);
      sts_line2<N>(B + base + b2, stride, r);
    }
    FE_SYNC();
    // phase 4: R += Ds^T gyy Ds T along y, then Ns^T along y, in place in B
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<1>(l, base, stride);
      v2 tq[N], r[N], u[N];
      lds_line2<N>(A + base + b2, stride, tq);
      lds_line2<N>(B + base + b2, stride, r);
      kterm2d<PDEG, DBG>(tq, r, gyy);
      eo2d<PDEG, MAT_NS, true, DBG>(r, u);
      sts_line2<N>(B + base + b2, stride, u);
    }
    FE_SYNC();
    // tile A is free: prefetch the next item's tile (overlaps phases 5-6)
    if (tid == 0) {
      const int nxt = item + gridDim.x;
      if (nxt < nitems) {
        const int nvb_ = nxt % P.nvb, ncell = nxt / P.nvb;
        const int nex = ncell % P.ncx, ney = (ncell / P.ncx) % P.ncy, nez = ncell / (P.ncx * P.ncy);
        mbar_expect_tx(bar, TL::BYTES);
        tma_load_4d(A, &tmW, bar, nvb_ * BV, nex * PDEG, ney * PDEG, nez * PDEG);
      }
    }
    // phase 5: Ns^T along x, in place
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 x[N], y[N];
      lds_line2<N>(B + base + b2, stride, x);
      eo2d<PDEG, MAT_NS, true, DBG>(x, y);
      sts_line2<N>(B + base + b2, stride, y);
    }
    FE_SYNC();
    // phase 6: Ns^T along z, in place; Dirichlet rows zeroed; wrap-around elements scattered by RED
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<2>(l, base, stride);
      v2 x[N], y[N];
      lds_line2<N>(B + base + b2, stride, x);
      eo2d<PDEG, MAT_NS, true, DBG>(x, y);
      if (!TMA_OUT) {
        // direct scatter-add from registers (RED.F64): saves the tile write + TMA read of the result
        const int i1 = l % N, i2 = l / N;
        int ix = ex * PDEG + i1, iy = ey * PDEG + i2;
        bool live = (v0 + b2) < P.nvec;
        bool first_ok = true, last_ok = true;
        const long long plane = (long long)P.ndx * P.ndy * nvec;
        long long last_off = (long long)PDEG * plane;
        if (dirichlet) {
          if (ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1) live = false;
          first_ok = (ez != 0); last_ok = (ez != P.ncz - 1);
        } else {
          if (ix >= P.ndx) ix -= P.ndx;
          if (iy >= P.ndy) iy -= P.ndy;
          if (wz) last_off -= (long long)P.ndz * plane;
        }
        if (live) {
          double* dst = P.Z + ((long long)ix + (long long)P.ndx * iy) * nvec + (long long)ez * PDEG * plane + v0 + b2;
#pragma unroll
          for (int i = 0; i < N; ++i) {
            const bool ok = (i == 0 ? first_ok : (i == N - 1 ? last_ok : true));
            const long long off = (i == N - 1) ? last_off : (long long)i * plane;
            if (ok) { atomicAdd(dst + off, y[i].a); atomicAdd(dst + off + 1, y[i].b); }
          }
        }
        continue;
      }
      if (special) {
        const int i1 = l % N, i2 = l / N;
        int ix = ex * PDEG + i1, iy = ey * PDEG + i2;
        if (dirichlet) {
          if (ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1) {
#pragma unroll
            for (int i = 0; i < N; ++i) y[i] = {0.0, 0.0};
          }
          if (ez == 0) y[0] = {0.0, 0.0};
          if (ez == P.ncz - 1) y[N - 1] = {0.0, 0.0};
        } else if ((v0 + b2) < P.nvec) {
          const bool line_wrapped = (ix >= P.ndx) || (iy >= P.ndy);
          if (ix >= P.ndx) ix -= P.ndx;
          if (iy >= P.ndy) iy -= P.ndy;
          const long long plane = (long long)P.ndx * P.ndy * nvec;
          double* dst = P.Z + ((long long)ix + (long long)P.ndx * iy) * nvec + (long long)ez * PDEG * plane + v0 + b2;
          if (line_wrapped) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
              long long off = (long long)i * plane;
              if (wz && i == N - 1) off -= (long long)P.ndz * plane;
              atomicAdd(dst + off, y[i].a); atomicAdd(dst + off + 1, y[i].b);
            }
          } else if (wz) {
            const long long off = (long long)(PDEG - P.ndz) * plane;
            atomicAdd(dst + off, y[N - 1].a); atomicAdd(dst + off + 1, y[N - 1].b);
          }
        }
      }
      sts_line2<N>(B + base + b2, stride, y);
    }
    if (TMA_OUT) {
      fence_async_smem();
      FE_SYNC();
      if (tid == 0) {
        tma_reduce_add_4d(&tmZ, B, v0, ex * PDEG, ey * PDEG, ez * PDEG);
        tma_commit();
      }
    }
  }
  if (TMA_OUT && tid == 0) tma_wait_all0();
}

}  // namespace fe
