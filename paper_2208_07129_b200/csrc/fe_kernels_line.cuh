// Device code, part 7: persistent Cartesian LINE kernel, second generation (replaces fe_apply_cart_tma where a
// whole plane per thread does not fit: p = 7, 8, and small vector counts).
//
// One thread = one line of the cell tile for TWO vectors (v2).  Same seven passes as fe_apply_cart_tma
//   x: Ns | y: Ns | z: Ns, T -> A, R = gm T + Kz T -> B | x: R += Kx T | y: R += Ky T, Ns^T | x: Ns^T | z: Ns^T
// but with the fused even/odd operator chains of fe_kernels_plane.cuh (no combine followed by split, the
// quadrature-point factor folded into the accumulate FMA), the Dirichlet boundary handled by the tensor maps
// (interior map on load, trimmed map on reduce) and the periodic wrap by face fix-ups on the shared-memory tile,
// so the pass bodies are branch-free.
#pragma once
#include "fe_kernels_plane.cuh"

namespace fe {

// IDENT: Z += alpha A W + idw W in the same pass (see fe_apply_cart_plane): the identity part is added in ph6 on
// the nodal result, with partition-of-unity weights, from the nodal values of W re-read through L2.
// EIG: see fe_apply_cart_plane (kappa per quadrature point, mass-scaled interpolation tables).
template <int PDEG, int BV, int NT, int MINB, int PADX, bool IDENT, bool EIG = false>
__global__ void __launch_bounds__(NT, MINB)
fe_apply_cart_line(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmZ,
                   const __grid_constant__ ApplyParams P, int nitems) {
  using TL = DenseTile<PDEG, BV, PADX>;
  constexpr int N = PDEG + 1, H = N / 2, HH = H > 0 ? H : 1, NL = N * N, TPL = BV / 2, TASKS = NL * TPL;
  constexpr int ROUNDS = (TASKS + NT - 1) / NT;
  constexpr int NSM = EIG ? MAT_NSS : MAT_NS;
  constexpr bool ROTATE = (NT % 32 == 0) && (NT >= 128) && (TASKS % NT != 0);
  constexpr int NW = NT / 32;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* A = reinterpret_cast<double*>(smem_raw);
  double* B = reinterpret_cast<double*>(smem_raw + TL::PITCH);
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * TL::PITCH);
  int* s_next = reinterpret_cast<int*>(bar + 1);
  const int tid = threadIdx.x;
  const bool dirichlet = P.dirichlet != 0;
  const int org = dirichlet ? -1 : 0;   // see fe_apply_cart_plane: interior input map on Dirichlet meshes
  const int orgz = (dirichlet && !(P.zopen & 1)) ? -1 : 0;
  const double g2x = 2.0 * P.ug[0], g2y = 2.0 * P.ug[3], g4y = 4.0 * P.ug[3], g4z = 4.0 * P.ug[5], gm = P.ug[6];

  if (tid == 0) {
    mbar_init(bar, 1);
    mbar_init_fence();
  }
  if (PADX) {   // the pad node of every x-row of the result tile is reduced into Z too: it must stay zero
    for (int e = tid; e < N * N * BV; e += NT) B[(e / BV) * TL::XP + N * BV + e % BV] = 0.0;
    fence_async_smem();
  }
  __syncthreads();
  int item = blockIdx.x;
  if (tid == 0 && item < nitems) {
    const int vb = (item + P.item0) % P.nvb, cell = (item + P.item0) / P.nvb;
    const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
    mbar_expect_tx(bar, TL::BYTES);
    tma_load_4d(A, &tmW, bar, vb * BV, ex * PDEG + org, ey * PDEG + org, ez * PDEG + orgz);
  }
  uint32_t parity = 0;
  int rot = (blockIdx.x / P.nsm) & 3;
  // items are handed out dynamically after the first one (co-resident blocks do not run at the same speed)
  for (; item < nitems; rot = (rot + 1) & 3) {
    unsigned nxt_raw = 0;
    if (tid == 0) nxt_raw = item_counter_next(P.item_ctr);
    const int rot_tid = ROTATE ? ((((tid >> 5) + NW - rot) % NW) << 5) + (tid & 31) : tid;
    const int vb = (item + P.item0) % P.nvb, cell = (item + P.item0) / P.nvb;
    const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
    const int v0 = vb * BV;
    const bool wx = !dirichlet && ex == P.ncx - 1, wy = !dirichlet && ey == P.ncy - 1, wz = !dirichlet && !P.zopen && ez == P.ncz - 1;
    const bool special = wx || wy || wz;
    const bool zlow = ez == 0 && !(P.zopen & 1);
    const bool dlow = dirichlet && (ex == 0 || ey == 0 || zlow);
    mbar_wait(bar, parity);
    parity ^= 1u;
    if (special) {
      plane_wrap_fixup<PDEG, BV, NT, false, PADX>(A, P, tid, ex, ey, ez, v0, wx, wy, wz);
      __syncthreads();
    }
    // ph0: Ns along x, in place in A
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 x[N];
      lds_line2<N>(A + base + b2, stride, x);
      eo_full<PDEG, NSM, false>(x, x);
      sts_line2<N>(A + base + b2, stride, x);
    }
    __syncthreads();
    // ph1: Ns along y, in place
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<1>(l, base, stride);
      v2 x[N];
      lds_line2<N>(A + base + b2, stride, x);
      eo_full<PDEG, NSM, false>(x, x);
      sts_line2<N>(A + base + b2, stride, x);
    }
    if (tid == 0) tma_wait_read0();     // the previous item's reduction has finished reading tile B
    __syncthreads();
    // ph2: T = Ns_z A -> A ; R = gm T + gzz Ds^T Ds T -> B  (the Ds chain starts from the even/odd parts of T)
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<2>(l, base, stride);
      v2 x[N], tq[N], xp[HH], xm[HH], u[HH], v[HH], m, u2[HH], vv[HH], m2;
      double gq[N];   // gm kappa_Q along the z-line l = i1 + N i2
      if (EIG) {
        const double* kp = P.kappa + (size_t)cell * (N * N * N) + l;
#pragma unroll
        for (int q = 0; q < N; ++q) gq[q] = gm * __ldg(kp + q * N * N);
      }
      lds_line2<N>(A + base + b2, stride, x);
      eo_split<N>(x, xp, xm);
      eo_mult<PDEG, NSM, false, false>(xp, xm, x[H], u, v, m);
      eo_combine<N, false>(u, v, m, tq);
      sts_line2<N>(A + base + b2, stride, tq);
      eo_dtd_eo<PDEG>(u, v, m, u2, vv, m2);
      v2 r[N];
#pragma unroll
      for (int q = 0; q < H; ++q) {
        r[q] = vfma(g4z, u2[q] + vv[q], vmul(EIG ? gq[q] : gm, tq[q]));
        r[N - 1 - q] = vfma(g4z, vv[q] - u2[q], vmul(EIG ? gq[N - 1 - q] : gm, tq[N - 1 - q]));
      }
      if (N & 1) r[H] = vfma(g4z, m2, vmul(EIG ? gq[H] : gm, tq[H]));
      sts_line2<N>(B + base + b2, stride, r);
    }
    __syncthreads();
    // ph3: R += gxx Ds^T Ds T along x
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 tq[N], r[N], u2[HH], vv[HH], m2;
      lds_line2<N>(A + base + b2, stride, tq);
      lds_line2<N>(B + base + b2, stride, r);
      eo_dtd<PDEG>(tq, u2, vv, m2);
#pragma unroll
      for (int q = 0; q < H; ++q) {
        r[q] = vfma(g2x, u2[q] + vv[q], r[q]);
        r[N - 1 - q] = vfma(g2x, vv[q] - u2[q], r[N - 1 - q]);
      }
      if (N & 1) r[H] = vfma(g2x, m2, r[H]);
      sts_line2<N>(B + base + b2, stride, r);
    }
    __syncthreads();
    // ph4: R += gyy Ds^T Ds T along y, then Ns^T along y (accumulated in the even/odd basis), in place in B
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<1>(l, base, stride);
      v2 tq[N], c[N], u2[HH], vv[HH], m2, rp[HH], rm[HH], u[HH], v[HH], m, rc;
      lds_line2<N>(A + base + b2, stride, tq);
      lds_line2<N>(B + base + b2, stride, c);
      eo_dtd<PDEG>(tq, u2, vv, m2);
      eo_split<N>(c, rp, rm);
#pragma unroll
      for (int q = 0; q < H; ++q) { rp[q] = vfma(g4y, vv[q], rp[q]); rm[q] = vfma(g4y, u2[q], rm[q]); }
      vzero(rc);
      if (N & 1) rc = vfma(g2y, m2, c[H]);
      eo_mult<PDEG, NSM, true, false>(rp, rm, rc, u, v, m);
      eo_combine<N, false>(u, v, m, c);
      sts_line2<N>(B + base + b2, stride, c);
    }
    __syncthreads();
    // tile A is free: prefetch the next item's tile (overlaps ph5-ph6)
    if (tid == 0) {
      const int nxt = (int)(gridDim.x + nxt_raw);
      *s_next = nxt;
      if (nxt < nitems) {
        const int nvb_ = (nxt + P.item0) % P.nvb, ncell = (nxt + P.item0) / P.nvb;
        const int nex = ncell % P.ncx, ney = (ncell / P.ncx) % P.ncy, nez = ncell / (P.ncx * P.ncy);
        mbar_expect_tx(bar, TL::BYTES);
        tma_load_4d(A, &tmW, bar, nvb_ * BV, nex * PDEG + org, ney * PDEG + org, nez * PDEG + orgz);
      }
    }
    // ph5: Ns^T along x, in place
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 x[N];
      lds_line2<N>(B + base + b2, stride, x);
      eo_full<PDEG, NSM, true>(x, x);
      sts_line2<N>(B + base + b2, stride, x);
    }
    __syncthreads();
    // ph6: Ns^T along z, in place; low Dirichlet faces zeroed (the reduction cannot start at a negative coordinate)
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<2>(l, base, stride);
      v2 x[N], wv[N];
      if (IDENT) {   // the z-line (i1, i2) of W in global memory (issued first: in flight during the contraction)
        const int i1 = l % N, i2 = l / N;
        int ixw = ex * PDEG + i1, iyw = ey * PDEG + i2;
        if (ixw >= P.ndx) ixw -= P.ndx;
        if (iyw >= P.ndy) iyw -= P.ndy;
        const bool wlive = (v0 + b2) < P.nvec;
        const long long zstep = (long long)P.ndx * P.ndy * P.nvec;
        const double* q = P.W + ((long long)ixw + (long long)P.ndx * ((long long)iyw + (long long)P.ndy * ez * PDEG)) * P.nvec + v0 + b2;
        const long long zwrap = wz ? (long long)P.ndz * zstep : 0;
#pragma unroll
        for (int j = 0; j < N; ++j) {
          double2 d = make_double2(0.0, 0.0);
          if (wlive) d = __ldg(reinterpret_cast<const double2*>(q + j * zstep - (j == N - 1 ? zwrap : 0)));
          wv[j] = {d.x, d.y};
        }
      }
      lds_line2<N>(B + base + b2, stride, x);
      eo_full<PDEG, NSM, true>(x, x);
      if (IDENT) {
        const int i1 = l % N, i2 = l / N;
        double wl = P.idw;
        if (i1 == 0 || i1 == N - 1) wl *= 0.5;
        if (i2 == 0 || i2 == N - 1) wl *= 0.5;
#pragma unroll
        for (int j = 0; j < N; ++j) x[j] = vfma((j == 0 || j == N - 1) ? 0.5 * wl : wl, wv[j], x[j]);
      }
      if (dlow) {
        const int i1 = l % N, i2 = l / N;
        if ((ex == 0 && i1 == 0) || (ey == 0 && i2 == 0)) {
#pragma unroll
          for (int i = 0; i < N; ++i) x[i] = {0.0, 0.0};
        }
        if (zlow) x[0] = {0.0, 0.0};
      }
      sts_line2<N>(B + base + b2, stride, x);
    }
    fence_async_smem();
    __syncthreads();
    if (special) plane_wrap_fixup<PDEG, BV, NT, true, PADX>(B, P, tid, ex, ey, ez, v0, wx, wy, wz);
    if (tid == 0) {
      tma_reduce_add_4d(&tmZ, B, v0, ex * PDEG, ey * PDEG, ez * PDEG);
      tma_commit();
    }
    item = *s_next;   // written before the barrier that ended ph6
  }
  if (tid == 0) tma_wait_all0();
}

}  // namespace fe
