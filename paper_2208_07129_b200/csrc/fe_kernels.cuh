// Device code, part 1: shared declarations, constant tables, the general ("v1") fused kernel.
// One thread block = one FE cell x BV vectors; the whole of Alg. 2 / Alg. 4 (PAPER.md:209-247,
// 690-740) runs between one gather and one scatter with all intermediates in shared memory.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "fe_params.h"

namespace fe {

// 1D tables per degree p (functions of p only, so contexts can share them).
// c_N[p][q*n+i] = N1D, c_D[p][q*n+r] = D~1D, c_w[p][q] = Gauss weights.
// static: every translation unit that includes this header owns a private copy, filled by its upload function.
static __constant__ double c_N[KMAXN][KMAXN * KMAXN];
static __constant__ double c_D[KMAXN][KMAXN * KMAXN];
static __constant__ double c_w[KMAXN][KMAXN];

// y[q] = sum_i M[q][i] x[i] (TRANS = false) or sum_i M[i][q] x[i] (TRANS = true) along one line.
template <int N, bool TRANS, bool ADD>
__device__ __forceinline__ void line_contract(const double* __restrict__ M, const double* src, int sstride,
                                              double* dst, int dstride) {
  double x[N];
#pragma unroll
  for (int i = 0; i < N; ++i) x[i] = src[i * sstride];
#pragma unroll
  for (int q = 0; q < N; ++q) {
    double acc = ADD ? dst[q * dstride] : 0.0;
#pragma unroll
    for (int i = 0; i < N; ++i) acc = fma(TRANS ? M[i * N + q] : M[q * N + i], x[i], acc);
    dst[q * dstride] = acc;
  }
}

// All n^2 lines along direction DIR of a [n][n][n][bv] tile.
template <int N, int DIR, bool TRANS, bool ADD>
__device__ __forceinline__ void pass(const double* __restrict__ M, const double* src, double* dst, int bv,
                                     int tid, int nthreads) {
  const int nlines = N * N * bv;
  for (int t = tid; t < nlines; t += nthreads) {
    const int beta = t % bv, l = t / bv;
    const int a = l % N, b = l / N;
    int base, stride;
    if (DIR == 0) { base = (N * a + N * N * b) * bv; stride = bv; }
    else if (DIR == 1) { base = (a + N * N * b) * bv; stride = N * bv; }
    else { base = (a + N * b) * bv; stride = N * N * bv; }
    line_contract<N, TRANS, ADD>(M, src + base + beta, stride, dst + base + beta, stride);
  }
}

__device__ __forceinline__ long long global_node(const ApplyParams& P, int ix, int iy, int iz) {
  return (long long)ix + (long long)P.ndx * ((long long)iy + (long long)P.ndy * iz);
}

template <int PDEG>
__global__ void __launch_bounds__(256) fe_apply_general(const ApplyParams P) {
  constexpr int N = PDEG + 1, NN = N * N * N;
  extern __shared__ double smem[];
  const int bv = P.bv;
  double* T = smem;
  double* T0 = T + NN * bv;
  double* T1 = T0 + NN * bv;
  double* T2 = T1 + NN * bv;
  const int tid = threadIdx.x, nth = blockDim.x;
  const int vb = blockIdx.x % P.nvb;
  const int cell = blockIdx.x / P.nvb;
  const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
  const int v0 = vb * bv;
  const double* Nm = c_N[PDEG];
  const double* Dm = c_D[PDEG];

  // S2 gather (Q^(e), C): tile[i3][i2][i1][beta]  (Eq. 18)
  for (int t = tid; t < NN * bv; t += nth) {
    const int beta = t % bv, I = t / bv;
    const int i1 = I % N, i2 = (I / N) % N, i3 = I / (N * N);
    int ix = ex * PDEG + i1, iy = ey * PDEG + i2, iz = ez * PDEG + i3;
    bool live = (v0 + beta) < P.nvec;
    if (P.dirichlet) {
      if (ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz)) live = false;
    } else {
      if (ix >= P.ndx) ix -= P.ndx;
      if (iy >= P.ndy) iy -= P.ndy;
      if (iz >= P.ndz) iz -= P.ndz;
    }
    double xv = live ? P.W[global_node(P, ix, iy, iz) * P.nvec + v0 + beta] : 0.0;
    if (P.dscale && live) xv *= __ldg(P.dscale + global_node(P, ix, iy, iz));   // M^-1/2 at extraction
    T0[t] = xv;
  }
  __syncthreads();
  // S3 interpolate (Alg. 1)
  pass<N, 0, false, false>(Nm, T0, T1, bv, tid, nth); __syncthreads();
  pass<N, 1, false, false>(Nm, T1, T0, bv, tid, nth); __syncthreads();
  pass<N, 2, false, false>(Nm, T0, T, bv, tid, nth); __syncthreads();
  // S4 gradients (Alg. 2 l.2-4)
  pass<N, 0, false, false>(Dm, T, T0, bv, tid, nth);
  pass<N, 1, false, false>(Dm, T, T1, bv, tid, nth);
  pass<N, 2, false, false>(Dm, T, T2, bv, tid, nth);
  __syncthreads();
  // S5 quadrature-point scaling (Alg. 2 l.5-6; Eq. 22-23)
  for (int t = tid; t < NN * bv; t += nth) {
    const int Q = t / bv;
    const int q1 = Q % N, q2 = (Q / N) % N, q3 = Q / (N * N);
    double g[7];
    const double wq = c_w[PDEG][q1] * c_w[PDEG][q2] * c_w[PDEG][q3];
    if (P.geom_mode == 2) {
      const double* gp = P.geom + (size_t)cell * P.geom_stride + Q;
#pragma unroll
      for (int k = 0; k < 7; ++k) g[k] = __ldg(gp + k * NN) * wq;
    } else {
      if (P.geom_mode == 1) {
#pragma unroll
        for (int k = 0; k < 7; ++k) g[k] = __ldg(P.geom + (size_t)cell * 7 + k) * wq;
      } else {
#pragma unroll
        for (int k = 0; k < 7; ++k) g[k] = P.ug[k] * wq;
        if (P.kappa) g[6] *= __ldg(P.kappa + (size_t)cell * NN + Q);
      }
    }
    const double a = T0[t], b = T1[t], c = T2[t];
    T0[t] = g[0] * a + g[1] * b + g[2] * c;
    T1[t] = g[1] * a + g[3] * b + g[4] * c;
    T2[t] = g[2] * a + g[4] * b + g[5] * c;
    T[t] = g[6] * T[t];
  }
  __syncthreads();
  // S6 transposed gradients (Alg. 2 l.7-9)
  pass<N, 0, true, true>(Dm, T0, T, bv, tid, nth); __syncthreads();
  pass<N, 1, true, true>(Dm, T1, T, bv, tid, nth); __syncthreads();
  pass<N, 2, true, true>(Dm, T2, T, bv, tid, nth); __syncthreads();
  // S7 integrate (N^T)
  pass<N, 0, true, false>(Nm, T, T0, bv, tid, nth); __syncthreads();
  pass<N, 1, true, false>(Nm, T0, T1, bv, tid, nth); __syncthreads();
  pass<N, 2, true, false>(Nm, T1, T0, bv, tid, nth); __syncthreads();
  // S8 scatter-add (Q^(e)T, C^T)
  for (int t = tid; t < NN * bv; t += nth) {
    const int beta = t % bv, I = t / bv;
    const int i1 = I % N, i2 = (I / N) % N, i3 = I / (N * N);
    int ix = ex * PDEG + i1, iy = ey * PDEG + i2, iz = ez * PDEG + i3;
    bool live = (v0 + beta) < P.nvec;
    if (P.dirichlet) {
      if (ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz)) live = false;
    } else {
      if (ix >= P.ndx) ix -= P.ndx;
      if (iy >= P.ndy) iy -= P.ndy;
      if (iz >= P.ndz) iz -= P.ndz;
    }
    if (live) {
      const double dv = P.dscale ? __ldg(P.dscale + global_node(P, ix, iy, iz)) : 1.0;   // M^-1/2 at assembly
      atomicAdd(&P.Z[global_node(P, ix, iy, iz) * P.nvec + v0 + beta], P.alpha * (dv * T0[t]));
    }
  }
}

// ---- n_q != n_p Gauss points per direction (over-integration) ----------------
// Plain sum factorisation with RECTANGULAR 1D tables (N: n_q x n_p) and the collocation derivative on the n_q points
// (D = D~ N), n_q a run-time value: the general fallback of this operator variant, any geometry, any nvec.

// dst (+)= M src along direction `dir` of a (d0, d1, d2) x bv array; M is mo x mi (or its transpose, stored mi x mo)
__device__ __forceinline__ void contract_rt(const double* M, int ldm, bool trans, int mo, int mi, int dir, const double* src,
                                            double* dst, int d0, int d1, int d2, int bv, bool add, int tid, int nth) {
  const int e0 = dir == 0 ? mo : d0, e1 = dir == 1 ? mo : d1, e2 = dir == 2 ? mo : d2;
  const int total = e0 * e1 * e2 * bv;
  const int sstride = (dir == 0 ? 1 : (dir == 1 ? d0 : d0 * d1)) * bv;
  for (int t = tid; t < total; t += nth) {
    const int beta = t % bv, r = t / bv;
    const int o0 = r % e0, o1 = (r / e0) % e1, o2 = r / (e0 * e1);
    const int o = dir == 0 ? o0 : (dir == 1 ? o1 : o2);
    const int s0 = dir == 0 ? 0 : o0, s1 = dir == 1 ? 0 : o1, s2 = dir == 2 ? 0 : o2;
    const double* sp = src + (size_t)(s0 + d0 * (s1 + d1 * s2)) * bv + beta;
    double acc = add ? dst[t] : 0.0;
    for (int i = 0; i < mi; ++i) acc = fma(trans ? M[i * ldm + o] : M[o * ldm + i], sp[(size_t)i * sstride], acc);
    dst[t] = acc;
  }
}

template <int PDEG>
__global__ void __launch_bounds__(256) fe_apply_general_oi(const ApplyParams P, const OiParams O) {
  constexpr int N = PDEG + 1;
  const int nq = O.nq, nq3 = nq * nq * nq;
  extern __shared__ double smem[];
  const int bv = P.bv;
  double* B0 = smem;
  double* B1 = B0 + (size_t)nq3 * bv;
  double* B2 = B1 + (size_t)nq3 * bv;
  double* T = B2 + (size_t)nq3 * bv;
  double* sN = T + (size_t)nq3 * bv;      // [nq][N]
  double* sD = sN + nq * N;               // [nq][nq]
  const int tid = threadIdx.x, nth = blockDim.x;
  const int vb = blockIdx.x % P.nvb;
  const int cell = blockIdx.x / P.nvb;
  const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
  const int v0 = vb * bv;
  for (int t = tid; t < nq * N; t += nth) sN[t] = O.Nq[t];
  for (int t = tid; t < nq * nq; t += nth) sD[t] = O.Dq[t];
  // S2 gather into B0 as (N, N, N)
  for (int t = tid; t < N * N * N * bv; t += nth) {
    const int beta = t % bv, I = t / bv;
    const int i1 = I % N, i2 = (I / N) % N, i3 = I / (N * N);
    int ix = ex * PDEG + i1, iy = ey * PDEG + i2, iz = ez * PDEG + i3;
    bool live = (v0 + beta) < P.nvec;
    if (P.dirichlet) {
      if (ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz)) live = false;
    } else {
      if (ix >= P.ndx) ix -= P.ndx;
      if (iy >= P.ndy) iy -= P.ndy;
      if (iz >= P.ndz) iz -= P.ndz;
    }
    double xv = live ? P.W[global_node(P, ix, iy, iz) * P.nvec + v0 + beta] : 0.0;
    if (P.dscale && live) xv *= __ldg(P.dscale + global_node(P, ix, iy, iz));
    B0[t] = xv;
  }
  __syncthreads();
  // S3 interpolate to the n_q^3 points (Alg. 1 with rectangular N)
  contract_rt(sN, N, false, nq, N, 0, B0, B1, N, N, N, bv, false, tid, nth); __syncthreads();
  contract_rt(sN, N, false, nq, N, 1, B1, B0, nq, N, N, bv, false, tid, nth); __syncthreads();
  contract_rt(sN, N, false, nq, N, 2, B0, T, nq, nq, N, bv, false, tid, nth); __syncthreads();
  // S4 reference gradients by collocation on the quadrature points
  contract_rt(sD, nq, false, nq, nq, 0, T, B0, nq, nq, nq, bv, false, tid, nth);
  contract_rt(sD, nq, false, nq, nq, 1, T, B1, nq, nq, nq, bv, false, tid, nth);
  contract_rt(sD, nq, false, nq, nq, 2, T, B2, nq, nq, nq, bv, false, tid, nth);
  __syncthreads();
  // S5 quadrature-point scaling (Alg. 2 l.5-6; Eq. 22-23)
  for (int t = tid; t < nq3 * bv; t += nth) {
    const int Q = t / bv;
    const int q1 = Q % nq, q2 = (Q / nq) % nq, q3 = Q / (nq * nq);
    const double wq = __ldg(O.wq + q1) * __ldg(O.wq + q2) * __ldg(O.wq + q3);
    double g[7];
    if (P.geom_mode == 2) {
      const double* gp = O.geom + (size_t)cell * O.geom_stride + Q;
#pragma unroll
      for (int k = 0; k < 7; ++k) g[k] = __ldg(gp + (size_t)k * nq3) * wq;
    } else {
#pragma unroll
      for (int k = 0; k < 7; ++k) g[k] = (P.geom_mode == 1 ? __ldg(P.geom + (size_t)cell * 7 + k) : P.ug[k]) * wq;
      if (P.kappa) g[6] *= __ldg(P.kappa + (size_t)cell * nq3 + Q);
    }
    const double a = B0[t], b = B1[t], c = B2[t];
    B0[t] = g[0] * a + g[1] * b + g[2] * c;
    B1[t] = g[1] * a + g[3] * b + g[4] * c;
    B2[t] = g[2] * a + g[4] * b + g[5] * c;
    T[t] = g[6] * T[t];
  }
  __syncthreads();
  // S6 transposed gradients, accumulated on the mass term
  contract_rt(sD, nq, true, nq, nq, 0, B0, T, nq, nq, nq, bv, true, tid, nth); __syncthreads();
  contract_rt(sD, nq, true, nq, nq, 1, B1, T, nq, nq, nq, bv, true, tid, nth); __syncthreads();
  contract_rt(sD, nq, true, nq, nq, 2, B2, T, nq, nq, nq, bv, true, tid, nth); __syncthreads();
  // S7 integrate back to the nodes (N^T, rectangular)
  contract_rt(sN, N, true, N, nq, 2, T, B0, nq, nq, nq, bv, false, tid, nth); __syncthreads();
  contract_rt(sN, N, true, N, nq, 1, B0, B1, nq, nq, N, bv, false, tid, nth); __syncthreads();
  contract_rt(sN, N, true, N, nq, 0, B1, B0, nq, N, N, bv, false, tid, nth); __syncthreads();
  // S8 scatter-add
  for (int t = tid; t < N * N * N * bv; t += nth) {
    const int beta = t % bv, I = t / bv;
    const int i1 = I % N, i2 = (I / N) % N, i3 = I / (N * N);
    int ix = ex * PDEG + i1, iy = ey * PDEG + i2, iz = ez * PDEG + i3;
    bool live = (v0 + beta) < P.nvec;
    if (P.dirichlet) {
      if (ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz)) live = false;
    } else {
      if (ix >= P.ndx) ix -= P.ndx;
      if (iy >= P.ndy) iy -= P.ndy;
      if (iz >= P.ndz) iz -= P.ndz;
    }
    if (live) {
      const double dv = P.dscale ? __ldg(P.dscale + global_node(P, ix, iy, iz)) : 1.0;
      atomicAdd(&P.Z[global_node(P, ix, iy, iz) * P.nvec + v0 + beta], P.alpha * (dv * B0[t]));
    }
  }
}

}  // namespace fe
