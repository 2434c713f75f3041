// Device code, part 8: persistent Cartesian KRONECKER kernel -- uniform box, constant kappa.
//
// On a cell whose metric is constant and diagonal and whose mass factor is constant, the quadrature stage of Alg. 2
// factorises along with the basis: with the 1D matrices M1 = Ns^T Ns (= N^T W N) and
// K1 = (Ds Ns)^T (Ds Ns) (= D^T W D), both evaluated with the SAME n_q-point rule as everywhere else,
//   A_e = gxx K1 x M1 x M1 + gyy M1 x K1 x M1 + gzz M1 x M1 x K1 + gm M1 x M1 x M1        (x = Kronecker product)
// which is exactly N^T..D^T G D..N of Eq. 8-9 for such a cell, regrouped.  (Same kind of host precomputation as
// D = D~ N of PAPER.md:188 and as the merged Ds^T Ds of the line kernel, taken one step further.)  Sum factorisation
// then needs 7 one-dimensional contractions per point instead of 9 and 3 passes over the tile instead of 7:
//
//   ph0  x-lines : a = M1 x -> T0 (in place) ; b = K1 x -> T1
//   ph1  y-lines : c = M1 a -> T0 ; s = gxx M1 b + gyy K1 a + gm c -> T1
//   ph2  z-lines : out = M1 s + gzz K1 c (+ identity term, IDENT) -> T1 ; TMA reduce-add T1 -> Z
//
// 10 tile accesses per point (line kernel: 17), ~60 FP64 instructions per DoF*vec at p = 6 (line / plane kernel: 79).
// M1 and K1 are symmetric and centro-symmetric: the even-odd primitives of fe_kernels_plane.cuh apply unchanged.
// Three tiles rotate per item (input / scratch+result / prefetch target): the input tile is transformed in place and
// read until ph2, so the next item's tile is fetched into the third one (issued after ph0's barrier).
// Everything else (one thread = one line of two vectors, dynamic items, Dirichlet through the tensor maps, periodic
// wrap fix-ups on the tile, pad node, IDENT) is the line kernel's.
#pragma once
#include "fe_kernels_line.cuh"

namespace fe {

// one line of the tile for VPT = 1 (double) or 2 (v2) vectors
template <int N> __device__ __forceinline__ void lds_line(const double* s, int stride, v2 (&x)[N]) { lds_line2<N>(s, stride, x); }
template <int N> __device__ __forceinline__ void sts_line(double* s, int stride, const v2 (&x)[N]) { sts_line2<N>(s, stride, x); }
// (the one-vector overloads of lds_line / sts_line are those of fe_kernels_eo.cuh)
__device__ __forceinline__ void ldg_vec(const double* q, bool live, v2& w) {
  double2 d = make_double2(0.0, 0.0);
  if (live) d = __ldg(reinterpret_cast<const double2*>(q));
  w = {d.x, d.y};
}
__device__ __forceinline__ void ldg_vec(const double* q, bool live, double& w) { w = live ? __ldg(q) : 0.0; }
template <int VPT> struct KronVec { using type = v2; };
template <> struct KronVec<1> { using type = double; };

// VPT: vectors per thread (2: 128-bit tile accesses, fewer instructions; 1: half the registers, more warps)
template <int PDEG, int BV, int NT, int MINB, int PADX, bool IDENT, int VPT = 2>
__global__ void __launch_bounds__(NT, MINB)
fe_apply_cart_kron(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmZ,
                   const __grid_constant__ ApplyParams P, int nitems) {
  using TL = DenseTile<PDEG, BV, PADX>;
  using V = typename KronVec<VPT>::type;
  constexpr int N = PDEG + 1, H = N / 2, HH = H > 0 ? H : 1, NL = N * N, TPL = BV / VPT, TASKS = NL * TPL;
  constexpr int ROUNDS = (TASKS + NT - 1) / NT;
  constexpr bool ROTATE = (NT % 32 == 0) && (NT >= 128) && (TASKS % NT != 0);
  constexpr int NW = NT / 32;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* T0 = reinterpret_cast<double*>(smem_raw);                    // input of this item
  double* T1 = reinterpret_cast<double*>(smem_raw + TL::PITCH);        // scratch, then the result
  double* T2 = reinterpret_cast<double*>(smem_raw + 2 * TL::PITCH);    // prefetch target
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 3 * TL::PITCH);
  int* s_next = reinterpret_cast<int*>(bar + 1);
  const int tid = threadIdx.x;
  const bool dirichlet = P.dirichlet != 0;
  const int org = dirichlet ? -1 : 0;   // see fe_apply_cart_plane: interior input map on Dirichlet meshes
  const double gx = P.ug[0], gy = P.ug[3], gz = P.ug[5], gm = P.ug[6];

  if (tid == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  int item = blockIdx.x;
  if (tid == 0 && item < nitems) {
    const int vb = item % P.nvb, cell = item / P.nvb;
    const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
    mbar_expect_tx(bar, TL::BYTES);
    tma_load_4d(T0, &tmW, bar, vb * BV, ex * PDEG + org, ey * PDEG + org, ez * PDEG + org);
  }
  uint32_t parity = 0;
  // the warps that carry tasks differ between the blocks resident on one SM by two warps (complementary footprints on
  // the four sub-partitions) and move by one warp per item
  int rot = ((blockIdx.x / P.nsm) * 2) % NW;
  // items are handed out dynamically after the first one (co-resident blocks do not run at the same speed)
  for (; item < nitems; rot = (rot + 1) % NW) {
    const int rot_tid = ROTATE ? ((((tid >> 5) + NW - rot) % NW) << 5) + (tid & 31) : tid;
    const int vb = item % P.nvb, cell = item / P.nvb;
    const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
    const int v0 = vb * BV;
    const bool wx = !dirichlet && ex == P.ncx - 1, wy = !dirichlet && ey == P.ncy - 1, wz = !dirichlet && ez == P.ncz - 1;
    const bool special = wx || wy || wz;
    const bool dlow = dirichlet && (ex == 0 || ey == 0 || ez == 0);
    int* const nslot = s_next + (parity & 1u);   // two slots: slow threads still read the previous item's
    if (tid == 0) {
      unsigned nxt_raw = 0;
      asm volatile("atom.global.add.u32 %0, [%1], 1;" : "=r"(nxt_raw) : "l"(P.item_ctr) : "memory");
      *nslot = (int)(gridDim.x + nxt_raw);   // read by all threads after the barriers below
      tma_wait_read0();                      // the previous item's reduction has finished reading what is now T2
    }
    mbar_wait(bar, parity);
    parity ^= 1u;
    if (special) {
      plane_wrap_fixup<PDEG, BV, NT, false, PADX>(T0, P, tid, ex, ey, ez, v0, wx, wy, wz);
      __syncthreads();
    }
    // ph0: x-lines: a = M1 x -> T0 in place, b = K1 x -> T1 (the pad node of the result tile is zeroed here)
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * VPT, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      V x[N], xp[HH], xm[HH], u[HH], v[HH], m;
      lds_line<N>(T0 + base + b2, stride, x);
      eo_split<N>(x, xp, xm);
      const V xc = x[H];
      eo_mult<PDEG, MAT_M1, false, false>(xp, xm, xc, u, v, m);
      eo_combine<N, false>(u, v, m, x);
      sts_line<N>(T0 + base + b2, stride, x);
      eo_mult<PDEG, MAT_K1, false, false>(xp, xm, xc, u, v, m);
      eo_combine<N, false>(u, v, m, x);
      sts_line<N>(T1 + base + b2, stride, x);
      if (PADX) { V z; vzero(z); V zz[1] = {z}; sts_line<1>(T1 + base + b2 + N * stride, stride, zz); }
    }
    __syncthreads();
    // every thread is past the mbarrier wait (a thread still polling the old phase must not see two phases complete):
    // arm the barrier for the next item's tile and fetch it into T2; the copy overlaps ph1 and ph2
    if (tid == 0) {
      const int nxt = *nslot;
      if (nxt < nitems) {
        const int nvb_ = nxt % P.nvb, ncell = nxt / P.nvb;
        const int nex = ncell % P.ncx, ney = (ncell / P.ncx) % P.ncy, nez = ncell / (P.ncx * P.ncy);
        mbar_expect_tx(bar, TL::BYTES);
        tma_load_4d(T2, &tmW, bar, nvb_ * BV, nex * PDEG + org, ney * PDEG + org, nez * PDEG + org);
      }
    }
    // ph1: y-lines: c = M1 a -> T0 ; s = gx M1 b + gy K1 a + gm c -> T1
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * VPT, l = t / TPL;
      int base, stride; TL::template line<1>(l, base, stride);
      // ordered for register pressure: the b-line is consumed (gx M1 b) before the a-line is loaded
      V us[HH], vs[HH], ms;
      {
        V b[N], bp[HH], bm[HH], ue[HH], ve[HH], me;
        lds_line<N>(T1 + base + b2, stride, b);
        eo_split<N>(b, bp, bm);
        eo_mult<PDEG, MAT_M1, false, false>(bp, bm, b[H], ue, ve, me);
#pragma unroll
        for (int q = 0; q < H; ++q) { us[q] = vmul(gx, ue[q]); vs[q] = vmul(gx, ve[q]); }
        vzero(ms);
        if (N & 1) ms = vmul(gx, me);
      }
      V a[N], ap[HH], am[HH], uc[HH], vc[HH], mc;
      lds_line<N>(T0 + base + b2, stride, a);
      eo_split<N>(a, ap, am);
      {
        V ud[HH], vd[HH], md;
        eo_mult<PDEG, MAT_K1, false, false>(ap, am, a[H], ud, vd, md);
#pragma unroll
        for (int q = 0; q < H; ++q) { us[q] = vfma(gy, ud[q], us[q]); vs[q] = vfma(gy, vd[q], vs[q]); }
        if (N & 1) ms = vfma(gy, md, ms);
      }
      eo_mult<PDEG, MAT_M1, false, false>(ap, am, a[H], uc, vc, mc);
#pragma unroll
      for (int q = 0; q < H; ++q) { us[q] = vfma(gm, uc[q], us[q]); vs[q] = vfma(gm, vc[q], vs[q]); }
      if (N & 1) ms = vfma(gm, mc, ms);
      eo_combine<N, false>(uc, vc, mc, a);
      V b[N];
      eo_combine<N, false>(us, vs, ms, b);
      sts_line<N>(T0 + base + b2, stride, a);
      sts_line<N>(T1 + base + b2, stride, b);
    }
    __syncthreads();
    // ph2: z-lines: out = M1 s + gz K1 c (+ idw w W), in place in T1; low Dirichlet faces zeroed (the reduction
    // cannot start at a negative coordinate)
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * VPT, l = t / TPL;
      int base, stride; TL::template line<2>(l, base, stride);
      V c[N], s[N], cp[HH], cm[HH], sp[HH], sm[HH], u[HH], v[HH], m, uk[HH], vk[HH], mk, wv[N];
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
        for (int j = 0; j < N; ++j) ldg_vec(q + j * zstep - (j == N - 1 ? zwrap : 0), wlive, wv[j]);
      }
      lds_line<N>(T0 + base + b2, stride, c);
      lds_line<N>(T1 + base + b2, stride, s);
      eo_split<N>(c, cp, cm);
      eo_split<N>(s, sp, sm);
      eo_mult<PDEG, MAT_M1, false, false>(sp, sm, s[H], u, v, m);
      eo_mult<PDEG, MAT_K1, false, false>(cp, cm, c[H], uk, vk, mk);
#pragma unroll
      for (int q = 0; q < H; ++q) { u[q] = vfma(gz, uk[q], u[q]); v[q] = vfma(gz, vk[q], v[q]); }
      if (N & 1) m = vfma(gz, mk, m);
      eo_combine<N, false>(u, v, m, s);
      if (IDENT) {
        const int i1 = l % N, i2 = l / N;
        double wl = P.idw;
        if (i1 == 0 || i1 == N - 1) wl *= 0.5;
        if (i2 == 0 || i2 == N - 1) wl *= 0.5;
#pragma unroll
        for (int j = 0; j < N; ++j) s[j] = vfma((j == 0 || j == N - 1) ? 0.5 * wl : wl, wv[j], s[j]);
      }
      if (dlow) {
        const int i1 = l % N, i2 = l / N;
        if ((ex == 0 && i1 == 0) || (ey == 0 && i2 == 0)) {
#pragma unroll
          for (int i = 0; i < N; ++i) vzero(s[i]);
        }
        if (ez == 0) vzero(s[0]);
      }
      sts_line<N>(T1 + base + b2, stride, s);
    }
    fence_async_smem();
    __syncthreads();
    if (special) plane_wrap_fixup<PDEG, BV, NT, true, PADX>(T1, P, tid, ex, ey, ez, v0, wx, wy, wz);
    if (tid == 0) {
      tma_reduce_add_4d(&tmZ, T1, v0, ex * PDEG, ey * PDEG, ez * PDEG);
      tma_commit();
    }
    item = *nslot;
    { double* t_ = T0; T0 = T2; T2 = T1; T1 = t_; }   // (input, result, prefetch) <- (prefetch, old input, old result)
  }
  if (tid == 0) tma_wait_all0();
}

}  // namespace fe
