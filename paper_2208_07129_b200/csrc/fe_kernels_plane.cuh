// Device code, part 6: "plane" kernels -- one thread owns a whole n x n plane of the cell tile for ONE vector.
//
// Why: with line tasks (fe_kernels_tma.cuh) every 1D contraction is a shared-memory round trip (18 tile
// accesses per point) and the shared-memory pipe (128 B/clk/SM) is as loaded as the FP64 pipe, with seven
// block barriers per cell.  A thread that holds an n x n plane in registers applies the contractions of
// TWO directions between one load and one store:
//
//   P1  xy-plane (i3 fixed):  A <- Ns_y Ns_x A                                       (S3, dims 1-2)
//   P2  z-lines of an xz-plane: T = Ns_z A -> A ;  R = gm T + Ds_z^T gzz Ds_z T -> B  (S3 dim 3, S4-S6 z-part)
//   P3  xy-plane: R += Ds_x^T gxx Ds_x T + Ds_y^T gyy Ds_y T ; B <- Ns_x^T Ns_y^T R   (S4-S6 x,y; S7 dims 1-2)
//   P4  z-lines: B <- Ns_z^T B                                                        (S7 dim 3) -> TMA reduce (S8)
//
// 11 thread tile accesses per point (+2 by the TMA unit) and 4 barriers per cell.  Consecutive 1D operators
// on the same line stay in the even/odd basis (no combine followed by split), and the quadrature-point
// factor is folded into the accumulate FMA: 94.8 FP64 instructions per DoF*vector at p = 6 instead of 111.8.
//
// Even/odd algebra (derived from the centro-symmetry M[n-1-q][n-1-i] = s M[q][i], reading 14):
//   split:    xp_i = x_i + x_{n-1-i},  xm_i = x_i - x_{n-1-i},  xc = x_mid
//   mult:     u = P xp + Pm xc,  v = Mn xm,  m = mid . xp + midm xc  (s = +1)   |   m = mid . xm  (s = -1)
//   combine:  y_q = u_q + v_q,  y_{n-1-q} = s (u_q - v_q),  y_mid = m
// so y_q + y_{n-1-q} = 2u (s=+1) or 2v (s=-1) and y_q - y_{n-1-q} = 2v or 2u: the (u, v, m) of one operator
// feed the next one directly; the missing factor 2 on (xp, xm) relative to xc is absorbed by halved
// middle-column tables (HALF) and by the scalar of the final accumulate.
#pragma once
#include "fe_kernels_tma.cuh"

#ifndef FE_ZLOOP_PRAGMA   // the z-line loops of P2 / P4: rolled (small code) or unrolled (loads hoisted)
#define FE_ZLOOP_PRAGMA _Pragma("unroll 1")
#endif

namespace fe {

static __constant__ EoTab2 c_eo2[KMAXN][MAT_COUNT];   // [p][MAT_NS | MAT_DS | MAT_SH | MAT_NSS]

// The primitives are generic in the value type T: double (one vector per thread, plane kernels) or v2 (two
// vectors per thread, line kernels).
__device__ __forceinline__ double vmul(double c, double x) { return c * x; }
__device__ __forceinline__ double vfma(double c, double x, double y) { return fma(c, x, y); }
__device__ __forceinline__ void vzero(double& x) { x = 0.0; }
__device__ __forceinline__ void vzero(v2& x) { x = {0.0, 0.0}; }

template <int N, typename T>
__device__ __forceinline__ void eo_split(const T (&x)[N], T (&xp)[N / 2 > 0 ? N / 2 : 1], T (&xm)[N / 2 > 0 ? N / 2 : 1]) {
#pragma unroll
  for (int i = 0; i < N / 2; ++i) { xp[i] = x[i] + x[N - 1 - i]; xm[i] = x[i] - x[N - 1 - i]; }
}

// (u, v, m) of y = M x (or M^T x) from (xp, xm, xc).  HALF: (xp, xm) carry half their true value relative to
// xc; the outputs are then half the true (u, v, m).
template <int PDEG, int MAT, bool TRANS, bool HALF, typename T>
__device__ __forceinline__ void eo_mult(const T (&xp)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1],
                                        const T (&xm)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1], T xc,
                                        T (&u)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1],
                                        T (&v)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1], T& m) {
  constexpr int N = PDEG + 1, H = N / 2;
  constexpr bool ODD = (N & 1) != 0, ANTI = (MAT == MAT_DS);
  const EoTab2& t = c_eo2[PDEG][MAT];
#pragma unroll
  for (int q = 0; q < H; ++q) {
    T a = vmul(!TRANS ? t.P[q * H] : (ANTI ? t.Mn[q] : t.P[q]), xp[0]);
#pragma unroll
    for (int i = 1; i < H; ++i) a = vfma(!TRANS ? t.P[q * H + i] : (ANTI ? t.Mn[i * H + q] : t.P[i * H + q]), xp[i], a);
    if (ODD) a = vfma(!TRANS ? (HALF ? t.Pmh[q] : t.Pm[q]) : (HALF ? t.midh[q] : t.mid[q]), xc, a);
    T b = vmul(!TRANS ? t.Mn[q * H] : (ANTI ? t.P[q] : t.Mn[q]), xm[0]);
#pragma unroll
    for (int i = 1; i < H; ++i) b = vfma(!TRANS ? t.Mn[q * H + i] : (ANTI ? t.P[i * H + q] : t.Mn[i * H + q]), xm[i], b);
    u[q] = a; v[q] = b;
  }
  vzero(m);
  if (ODD) {
    if (ANTI) {
      T c = vmul(!TRANS ? t.mid[0] : t.Pm[0], xm[0]);
#pragma unroll
      for (int i = 1; i < H; ++i) c = vfma(!TRANS ? t.mid[i] : t.Pm[i], xm[i], c);
      m = c;
    } else {
      T c = vmul(HALF ? t.midmh : t.midm, xc);
#pragma unroll
      for (int i = 0; i < H; ++i) c = vfma(!TRANS ? t.mid[i] : t.Pm[i], xp[i], c);
      m = c;
    }
  }
}

template <int N, bool ANTI, typename T>
__device__ __forceinline__ void eo_combine(const T (&u)[N / 2 > 0 ? N / 2 : 1], const T (&v)[N / 2 > 0 ? N / 2 : 1], T m, T (&y)[N]) {
#pragma unroll
  for (int q = 0; q < N / 2; ++q) { y[q] = u[q] + v[q]; y[N - 1 - q] = ANTI ? (v[q] - u[q]) : (u[q] - v[q]); }
  if (N & 1) y[N / 2] = m;
}

// y = M x or M^T x, complete (split, mult, combine); x and y may be the same array.
template <int PDEG, int MAT, bool TRANS, typename T>
__device__ __forceinline__ void eo_full(const T (&x)[PDEG + 1], T (&y)[PDEG + 1]) {
  constexpr int N = PDEG + 1, HH = N / 2 > 0 ? N / 2 : 1;
  T xp[HH], xm[HH], u[HH], v[HH], m;
  eo_split<N>(x, xp, xm);
  eo_mult<PDEG, MAT, TRANS, false>(xp, xm, x[N / 2], u, v, m);
  eo_combine<N, MAT == MAT_DS>(u, v, m, y);
}

// (u2, v2, m2) = HALF of the even/odd parts of Ds^T Ds t, from the line t, in the convention of an
// anti-symmetric-type product: y_q = 2 (u2_q + v2_q), y_{n-1-q} = 2 (v2_q - u2_q), y_mid = 2 m2.
// On Cartesian cells the metric factor is constant along a line, so Ds^T g Ds = g (Ds^T Ds) and the 1D operator
// S/2 = Ds^T Ds / 2 (host-precomputed like D = D~ N of PAPER.md:188; symmetric type) is applied as ONE contraction.
template <int PDEG, typename T>
__device__ __forceinline__ void eo_dtd(const T (&t)[PDEG + 1], T (&u2)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1],
                                       T (&v2)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1], T& m2) {
  constexpr int N = PDEG + 1, HH = N / 2 > 0 ? N / 2 : 1;
  T tp[HH], tm[HH];
  eo_split<N>(t, tp, tm);
  eo_mult<PDEG, MAT_SH, false, false>(tp, tm, t[N / 2], v2, u2, m2);   // (u, v) of a symmetric type swap roles
}
// The same from the even/odd parts (u, v, m) of t itself (as eo_mult leaves them: half of x+ / x-): QUARTER of
// the even/odd parts of Ds^T Ds t.
template <int PDEG, typename T>
__device__ __forceinline__ void eo_dtd_eo(const T (&u)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1],
                                          const T (&v)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1], T m,
                                          T (&u2)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1],
                                          T (&v2)[(PDEG + 1) / 2 > 0 ? (PDEG + 1) / 2 : 1], T& m2) {
  eo_mult<PDEG, MAT_SH, false, true>(u, v, m, v2, u2, m2);
}

// Periodic wrap fix-ups of the last cell in a direction, done cooperatively on the shared-memory tile so that
// the plane phases stay branch-free: only the (up to three) wrapped faces i_d = N-1 are visited.
// IN (OUT = false): fetch the wrap-around nodes the TMA box could not reach (it zero-filled them).
// OUT: RED the wrap-around nodes that the clipped TMA reduction will not store.
template <int PDEG, int BV, int NT, bool OUT, int PADX = 0>
__device__ __forceinline__ void plane_wrap_fixup(double* tile, const ApplyParams& P, int tid, int ex, int ey, int ez, int v0,
                                                 bool wx, bool wy, bool wz) {
  constexpr int N = PDEG + 1, HB = BV / 2, FACE = N * N * HB;
  const long long nvec = P.nvec;
  constexpr int IT = (FACE + NT - 1) / NT;
#pragma unroll
  for (int f = 0; f < 3; ++f) {
    if (!(f == 0 ? wx : (f == 1 ? wy : wz))) continue;
    // all the loads of a thread are issued before the first store (one L2 round trip per face instead of IT)
    double2 val[IT];
    double2* dst[IT];
#pragma unroll
    for (int it = 0; it < IT; ++it) {
      const int r = tid + it * NT;
      dst[it] = nullptr;
      if (r >= FACE) continue;
      const int b2 = (r % HB) * 2, a = (r / HB) % N, b = r / (HB * N);
      int i1, i2, i3;
      if (f == 0) { i1 = N - 1; i2 = a; i3 = b; }
      else if (f == 1) { i2 = N - 1; i1 = a; i3 = b; if (wx && i1 == N - 1) continue; }
      else { i3 = N - 1; i1 = a; i2 = b; if ((wx && i1 == N - 1) || (wy && i2 == N - 1)) continue; }
      if ((v0 + b2) >= P.nvec) continue;
      int ix = ex * PDEG + i1, iy = ey * PDEG + i2, iz = ez * PDEG + i3;
      if (ix >= P.ndx) ix -= P.ndx;
      if (iy >= P.ndy) iy -= P.ndy;
      if (iz >= P.ndz) iz -= P.ndz;
      const long long g = ((long long)ix + (long long)P.ndx * ((long long)iy + (long long)P.ndy * iz)) * nvec + v0 + b2;
      double2* s = reinterpret_cast<double2*>(tile + ((i3 * N + i2) * (N + PADX) + i1) * BV + b2);
      if (!OUT) {
        val[it] = __ldg(reinterpret_cast<const double2*>(P.W + g));
        dst[it] = s;
      } else {
        const double2 d = *s;
        atomicAdd(P.Z + g, d.x); atomicAdd(P.Z + g + 1, d.y);
      }
    }
    if (!OUT) {
#pragma unroll
      for (int it = 0; it < IT; ++it)
        if (dst[it]) *dst[it] = val[it];
    }
  }
}

// Z (+)= A W on uniform Cartesian cells (diagonal constant metric; alpha folded into P.ug).  One block = one
// cell x BV vectors per item, persistent; thread (k, beta) = plane k of vector beta.
// IDENT (periodic meshes): Z += alpha A W + idw W in the same pass.  The identity part is added cell by cell with
// partition-of-unity weights (a node on a cell face in a direction is shared by two cells: weight 1/2 per
// direction) in P4, on the nodal result, from the nodal values of W re-read through L2 (the tile that held them was
// transformed in place).  The shifted operator A - cI of the Chebyshev recurrence then costs no separate pass.
// EIG: the operator of the paper's eigenproblem on a uniform box, H~ = M^-1/2 (K + M^kappa) M^-1/2:
// kappa is read per quadrature point (P.kappa [cell][n^3]) and the interpolation passes use the
// mass-scaled tables MAT_NSS (the constant (1/det J) of M^-1 is folded into the metric constants by the host).
template <int PDEG, int BV, int NT, int MINB, bool IDENT, bool EIG = false>
__global__ void __launch_bounds__(NT, MINB)
fe_apply_cart_plane(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmZ,
                    const __grid_constant__ ApplyParams P, int nitems) {
  using TL = DenseTile<PDEG, BV>;
  constexpr int N = PDEG + 1, H = N / 2, HH = H > 0 ? H : 1;
  constexpr int S1 = BV, S2 = N * BV, S3 = N * N * BV;   // element strides along x, y, z
  constexpr int NSM = EIG ? MAT_NSS : MAT_NS;
  static_assert(N * BV <= NT && NT % 128 == 0, "one plane task per thread; whole warps on every sub-partition");
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* A = reinterpret_cast<double*>(smem_raw);
  double* B = reinterpret_cast<double*>(smem_raw + TL::PITCH);
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * TL::PITCH);
  int* s_next = reinterpret_cast<int*>(bar + 1);
  const int tid = threadIdx.x;
  const int beta = tid % BV, k = tid / BV;
  const bool active = k < N;
  // Dirichlet: the input tensor map covers the INTERIOR nodes only (origin = node (1,1,1)), so boundary nodes are
  // out of bounds for the TMA unit and arrive as zeros (X read as 0).  A bulk tensor REDUCTION faults on negative
  // coordinates (measured on sm_100a), so the output map keeps its origin at node 0 and drops only the last
  // node per direction (clipped); the low boundary faces are zeroed in registers in P4 (Y rows stay 0).
  const bool dirichlet = P.dirichlet != 0;
  const int org = dirichlet ? -1 : 0;
  const int orgz = (dirichlet && !(P.zopen & 1)) ? -1 : 0;   // a slab's low cut plane is inside the input map
  const double g2x = 2.0 * P.ug[0], g2y = 2.0 * P.ug[3], g4y = 4.0 * P.ug[3], g4z = 4.0 * P.ug[5], gm = P.ug[6];
  if (tid == 0) {
    mbar_init(bar, 1);
    mbar_init_fence();
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
  // Items are handed out dynamically (the first one is blockIdx.x): co-resident blocks do not run at the same
  // speed (the warp arbiter favours one of them), and a static round-robin would leave the slow ones behind.
  while (item < nitems) {
    const int vb = (item + P.item0) % P.nvb, cell = (item + P.item0) / P.nvb;
    const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
    const int v0 = vb * BV;
    const bool wx = !dirichlet && ex == P.ncx - 1, wy = !dirichlet && ey == P.ncy - 1, wz = !dirichlet && !P.zopen && ez == P.ncz - 1;
    const bool special = wx || wy || wz;
    const bool zlow = ez == 0 && !(P.zopen & 1);   // the low z face is a Dirichlet boundary (not a cut plane)
    const bool dlow = dirichlet && (ex == 0 || ey == 0 || zlow);
    // the next item: consumed later, latency hidden (asm volatile: the compiler must not schedule anything that
    // depends on the result up here)
    unsigned nxt_raw = 0;
    if (tid == 0) nxt_raw = item_counter_next(P.item_ctr);
    mbar_wait(bar, parity);
    parity ^= 1u;
    if (special) {
      plane_wrap_fixup<PDEG, BV, NT, false>(A, P, tid, ex, ey, ez, v0, wx, wy, wz);
      __syncthreads();
    }

    // P1: xy-plane i3 = k: Ns along x (rows) then along y (columns), in registers
    if (active) {
      double* a = A + k * S3 + beta;
      double r[N][N];
#pragma unroll
      for (int j = 0; j < N; ++j)
#pragma unroll
        for (int i = 0; i < N; ++i) r[j][i] = a[j * S2 + i * S1];
#pragma unroll
      for (int j = 0; j < N; ++j) eo_full<PDEG, NSM, false>(r[j], r[j]);
#pragma unroll
      for (int i = 0; i < N; ++i) {
        double c[N];
#pragma unroll
        for (int j = 0; j < N; ++j) c[j] = r[j][i];
        eo_full<PDEG, NSM, false>(c, c);
#pragma unroll
        for (int j = 0; j < N; ++j) a[j * S2 + i * S1] = c[j];
      }
    }
    if (tid == 0) {
      tma_wait_read0();   // the previous item's reduction has finished reading tile B
    }
    __syncthreads();

    // P2: z-lines (i1, i2 = k): T = Ns_z A -> A ; R = gm T + 4 gzz (DtD T)/4 -> B
    if (active) {
      double xn[N];   // software pipeline: the next line is in flight while this one is computed
#pragma unroll
      for (int j = 0; j < N; ++j) xn[j] = A[k * S2 + beta + j * S3];
FE_ZLOOP_PRAGMA
      for (int i = 0; i < N; ++i) {
        double* a = A + k * S2 + i * S1 + beta;
        double* b = B + k * S2 + i * S1 + beta;
        double x[N], tq[N], xp[HH], xm[HH], u[HH], v[HH], m, u2[HH], v2[HH], m2;
        double gq[N];   // gm kappa_Q along the z-line (i, k, .): shared by the block's vectors, L1-resident
        if (EIG) {
          const double* kp = P.kappa + (size_t)cell * (N * N * N) + i + N * k;
#pragma unroll
          for (int q = 0; q < N; ++q) gq[q] = __ldg(kp + q * N * N);
        }
#pragma unroll
        for (int j = 0; j < N; ++j) x[j] = xn[j];
        if (i + 1 < N) {
#pragma unroll
          for (int j = 0; j < N; ++j) xn[j] = a[S1 + j * S3];
        }
        eo_split<N>(x, xp, xm);
        eo_mult<PDEG, NSM, false, false>(xp, xm, x[H], u, v, m);
        eo_combine<N, false>(u, v, m, tq);
#pragma unroll
        for (int j = 0; j < N; ++j) a[j * S3] = tq[j];
        eo_dtd_eo<PDEG>(u, v, m, u2, v2, m2);                          // quarter of Ds^T Ds T
#pragma unroll
        for (int q = 0; q < H; ++q) {
          b[q * S3] = fma(g4z, u2[q] + v2[q], (EIG ? gm * gq[q] : gm) * tq[q]);
          b[(N - 1 - q) * S3] = fma(g4z, v2[q] - u2[q], (EIG ? gm * gq[N - 1 - q] : gm) * tq[N - 1 - q]);
        }
        if (N & 1) b[H * S3] = fma(g4z, m2, (EIG ? gm * gq[H] : gm) * tq[H]);
      }
    }
    __syncthreads();

    // P3: xy-plane i3 = k: R += Kx T (rows) ; R += Ky T, Ns^T along y (columns) ; Ns^T along x (rows)
    {
      const double* a = A + k * S3 + beta;
      double* b = B + k * S3 + beta;
      double r[N][N];
      if (active) {
#pragma unroll
        for (int j = 0; j < N; ++j)
#pragma unroll
          for (int i = 0; i < N; ++i) r[j][i] = b[j * S2 + i * S1];
#pragma unroll
        for (int j = 0; j < N; ++j) {
          double t[N], u2[HH], v2[HH], m2;
#pragma unroll
          for (int i = 0; i < N; ++i) t[i] = a[j * S2 + i * S1];
          eo_dtd<PDEG>(t, u2, v2, m2);
#pragma unroll
          for (int q = 0; q < H; ++q) {
            r[j][q] = fma(g2x, u2[q] + v2[q], r[j][q]);
            r[j][N - 1 - q] = fma(g2x, v2[q] - u2[q], r[j][N - 1 - q]);
          }
          if (N & 1) r[j][H] = fma(g2x, m2, r[j][H]);
        }
      }
      if (active) {
#pragma unroll
        for (int i = 0; i < N; ++i) {
          double t[N], c[N], u2[HH], v2[HH], m2, rp[HH], rm[HH], u[HH], v[HH], m;
#pragma unroll
          for (int j = 0; j < N; ++j) { t[j] = a[j * S2 + i * S1]; c[j] = r[j][i]; }
          eo_dtd<PDEG>(t, u2, v2, m2);
          eo_split<N>(c, rp, rm);
#pragma unroll
          for (int q = 0; q < H; ++q) { rp[q] = fma(g4y, v2[q], rp[q]); rm[q] = fma(g4y, u2[q], rm[q]); }
          const double rc = (N & 1) ? fma(g2y, m2, c[H]) : 0.0;
          eo_mult<PDEG, NSM, true, false>(rp, rm, rc, u, v, m);
          eo_combine<N, false>(u, v, m, c);
#pragma unroll
          for (int j = 0; j < N; ++j) r[j][i] = c[j];
        }
#pragma unroll
        for (int j = 0; j < N; ++j) {
          eo_full<PDEG, NSM, true>(r[j], r[j]);
#pragma unroll
          for (int i = 0; i < N; ++i) b[j * S2 + i * S1] = r[j][i];
        }
      }
    }
    __syncthreads();
    // tile A is free: prefetch the next item's tile (overlaps P4 and the other resident block)
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
    // P4: z-lines (i1, i2 = k): Ns^T along z, in place in B
    if (active) {
      double xn[N], wn[N];
#pragma unroll
      for (int j = 0; j < N; ++j) xn[j] = B[k * S2 + beta + j * S3];
      // IDENT: the z-line (i1, i2 = k) of W in global memory: node (ix, iy, ez p + j), periodic wrap
      const bool wlive = IDENT && (v0 + beta) < P.nvec;
      const long long zstep = (long long)P.ndx * P.ndy * P.nvec;
      int iyw = ey * PDEG + k; if (iyw >= P.ndy) iyw -= P.ndy;
      const double* wrow = P.W + ((long long)iyw * P.ndx + (long long)ez * PDEG * P.ndx * P.ndy) * P.nvec + v0 + beta;
      const long long zwrap = wz ? (long long)P.ndz * zstep : 0;   // subtracted at j = N-1 in the last layer
      const double wk = (k == 0 || k == N - 1) ? 0.5 * P.idw : P.idw;
      auto load_w = [&](int i1, double (&w)[N]) {
        int ixw = ex * PDEG + i1; if (ixw >= P.ndx) ixw -= P.ndx;
        const double* q = wrow + (long long)ixw * P.nvec;
#pragma unroll
        for (int j = 0; j < N; ++j) w[j] = wlive ? __ldg(q + j * zstep - (j == N - 1 ? zwrap : 0)) : 0.0;
      };
      if (IDENT) load_w(0, wn);
FE_ZLOOP_PRAGMA
      for (int i = 0; i < N; ++i) {
        double* b = B + k * S2 + i * S1 + beta;
        double x[N], w[N];
#pragma unroll
        for (int j = 0; j < N; ++j) { x[j] = xn[j]; if (IDENT) w[j] = wn[j]; }
        if (i + 1 < N) {
#pragma unroll
          for (int j = 0; j < N; ++j) xn[j] = b[S1 + j * S3];
          if (IDENT) load_w(i + 1, wn);
        }
        eo_full<PDEG, NSM, true>(x, x);
        if (IDENT) {
          const double wi = (i == 0 || i == N - 1) ? 0.5 * wk : wk;
#pragma unroll
          for (int j = 0; j < N; ++j) x[j] = fma((j == 0 || j == N - 1) ? 0.5 * wi : wi, w[j], x[j]);
        }
        if (dlow) {
          const bool zl = (ey == 0 && k == 0) || (ex == 0 && i == 0);
#pragma unroll
          for (int j = 0; j < N; ++j)
            if (zl || (j == 0 && zlow)) x[j] = 0.0;
        }
#pragma unroll
        for (int j = 0; j < N; ++j) b[j * S3] = x[j];
      }
    }
    fence_async_smem();
    __syncthreads();
    if (special) plane_wrap_fixup<PDEG, BV, NT, true>(B, P, tid, ex, ey, ez, v0, wx, wy, wz);
    if (tid == 0) {
      tma_reduce_add_4d(&tmZ, B, v0, ex * PDEG, ey * PDEG, ez * PDEG);
      tma_commit();
    }
    item = *s_next;   // written before the barrier that ended P4
  }
  if (tid == 0) tma_wait_all0();
}

}  // namespace fe
