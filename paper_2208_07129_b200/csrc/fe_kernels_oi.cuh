// Device code, part 9: the compile-time kernel of the n_q = n_p + 2 rule:
// even-odd line tasks on rectangular tables, cell tile by TMA on interior cells (loads / atomics on the others).
#pragma once
#include "fe_kernels.cuh"
#include "fe_kernels_tma.cuh"

namespace fe {

// Tables of the n_q = n_p + 2 rule, packed per degree at oi_offset(p) as even / odd halves (uploaded by
// fe_mf_set_quadrature; the values depend on p only): [Ne | No | De | Do], N (nq x n) centro-symmetric, D~ (nq x nq)
// centro-antisymmetric (SURVEY.md 8(c) reading 14), Me[o][i] = (M[o][i] + M[o][C-1-i]) / 2, Mo[o][i] = (M[o][i] - M[o][C-1-i]) / 2
// for o < ceil(R/2), i < ceil(C/2).  Constant-bank FMA operands like the other tables.
static __constant__ double c_oi[OiOffset<9>::value];

// The same with compile-time sizes (the paper's n_q = n_p + 2), LINE tasks and even-odd contractions: one thread
// contracts one line of one vector in registers (one tile read and one tile write per point and pass instead of n reads
// per output).  Array (D0, D1, D2) x bv -> the extent along DIR becomes MO.  The table at c_oi + MOFF is the [Me | Mo]
// pair of a matrix stored [MO][MI] (TRANS: [MI][MO], applied transposed); ANTI: centro-antisymmetric (D~), else
// centro-symmetric (N).  y_o = u + v, y_{MO-1-o} = +-(u - v) with u, v the even / odd half products.
template <int D0, int D1, int D2, int DIR, int MO, bool TRANS, bool ANTI, bool ADD, int MOFF, int bv>
__device__ __forceinline__ void contract_lines_impl(const double* src, double* dst, int tid);
// INPLACE: src == dst (square operator, !ADD): a thread reads its whole line before it writes, and no two lines overlap
template <int D0, int D1, int D2, int DIR, int MO, bool TRANS, bool ANTI, bool ADD, int MOFF, int bv, bool INPLACE = false>
__device__ __forceinline__ void contract_lines(const double* src, double* dst, int tid) {
  if (INPLACE) {
    contract_lines_impl<D0, D1, D2, DIR, MO, TRANS, ANTI, ADD, MOFF, bv>(src, dst, tid);
  } else {
    const double* __restrict__ s = src;
    double* __restrict__ d = dst;
    contract_lines_impl<D0, D1, D2, DIR, MO, TRANS, ANTI, ADD, MOFF, bv>(s, d, tid);
  }
}
template <int D0, int D1, int D2, int DIR, int MO, bool TRANS, bool ANTI, bool ADD, int MOFF, int bv>
__device__ __forceinline__ void contract_lines_impl(const double* src, double* dst, int tid) {
  constexpr int nth = 256;   // the block size, as a constant: the trip count of the line loop is then known (1 or 2), and
                             // the table values are not hoisted out of it into more uniform registers than exist
  constexpr int MI = DIR == 0 ? D0 : (DIR == 1 ? D1 : D2);
  constexpr int EA = DIR == 0 ? D1 : D0, EB = DIR == 2 ? D1 : D2;          // the two other extents, in index order
  constexpr int SS = DIR == 0 ? 1 : (DIR == 1 ? D0 : D0 * D1);              // source stride along DIR (in points)
  constexpr int E0 = DIR == 0 ? MO : D0, E1 = DIR == 1 ? MO : D1;            // destination extents
  constexpr int DS = DIR == 0 ? 1 : (DIR == 1 ? E0 : E0 * E1);
  constexpr int nlines = EA * EB * bv;
  constexpr int HI = (MI + 1) / 2, FI = MI / 2, HO = (MO + 1) / 2, FO = MO / 2;
  constexpr int HC = TRANS ? HO : HI;                                        // columns of the stored half tables
  constexpr int TE = MOFF, TO = MOFF + HI * HO;                              // Me, Mo
  // a transposed antisymmetric matrix has its even part in the stored odd half and vice versa
  constexpr int UE = (TRANS && ANTI) ? TO : TE, UO = (TRANS && ANTI) ? TE : TO;
#pragma unroll
  for (int t0 = 0; t0 < nlines; t0 += nth) {
    const int t = t0 + tid;
    if (t >= nlines) break;
    const int beta = t % bv, r = t / bv, a = r % EA, b = r / EA;
    // point index of the line start in source / destination
    const int sbase = DIR == 0 ? D0 * (a + D1 * b) : (DIR == 1 ? a + D0 * D1 * b : a + D0 * b);
    const int dbase = DIR == 0 ? E0 * (a + E1 * b) : (DIR == 1 ? a + E0 * E1 * b : a + E0 * b);
    double xe[HI], xo[FI > 0 ? FI : 1];
#pragma unroll
    for (int i = 0; i < FI; ++i) {
      const double p = src[(size_t)(sbase + i * SS) * bv + beta], q = src[(size_t)(sbase + (MI - 1 - i) * SS) * bv + beta];
      xe[i] = p + q;
      xo[i] = p - q;
    }
    if (MI & 1) xe[FI] = src[(size_t)(sbase + FI * SS) * bv + beta];
#pragma unroll
    for (int o = 0; o < FO; ++o) {
      double u = 0.0, v = 0.0;
#pragma unroll
      for (int i = 0; i < HI; ++i) u = fma(TRANS ? c_oi[UE + i * HC + o] : c_oi[UE + o * HC + i], xe[i], u);
#pragma unroll
      for (int i = 0; i < FI; ++i) v = fma(TRANS ? c_oi[UO + i * HC + o] : c_oi[UO + o * HC + i], xo[i], v);
      double* d0 = dst + (size_t)(dbase + o * DS) * bv + beta;
      double* d1 = dst + (size_t)(dbase + (MO - 1 - o) * DS) * bv + beta;
      const double y0 = u + v, y1 = ANTI ? v - u : u - v;
      *d0 = ADD ? *d0 + y0 : y0;
      *d1 = ADD ? *d1 + y1 : y1;
    }
    if (MO & 1) {   // middle output: the odd (symmetric matrix) or even (antisymmetric) half vanishes
      double y = 0.0;
      if (ANTI) {
#pragma unroll
        for (int i = 0; i < FI; ++i) y = fma(TRANS ? c_oi[UO + i * HC + FO] : c_oi[UO + FO * HC + i], xo[i], y);
      } else {
#pragma unroll
        for (int i = 0; i < HI; ++i) y = fma(TRANS ? c_oi[UE + i * HC + FO] : c_oi[UE + FO * HC + i], xe[i], y);
      }
      double* d0 = dst + (size_t)(dbase + FO * DS) * bv + beta;
      *d0 = ADD ? *d0 + y : y;
    }
  }
}

// The even-odd product of contract_lines on a line held in registers: y = M x (TRANS: M^T x), table pair at c_oi + MOFF.
template <int MI, int MO, bool TRANS, bool ANTI, int MOFF>
__device__ __forceinline__ void eo_line(const double (&x)[MI], double (&y)[MO]) {
  constexpr int HI = (MI + 1) / 2, FI = MI / 2, HO = (MO + 1) / 2, FO = MO / 2;
  constexpr int HC = TRANS ? HO : HI;
  constexpr int TE = MOFF, TO = MOFF + HI * HO;
  constexpr int UE = (TRANS && ANTI) ? TO : TE, UO = (TRANS && ANTI) ? TE : TO;
  double xe[HI], xo[FI > 0 ? FI : 1];
#pragma unroll
  for (int i = 0; i < FI; ++i) { xe[i] = x[i] + x[MI - 1 - i]; xo[i] = x[i] - x[MI - 1 - i]; }
  if (MI & 1) xe[FI] = x[FI];
#pragma unroll
  for (int o = 0; o < FO; ++o) {
    double u = 0.0, v = 0.0;
#pragma unroll
    for (int i = 0; i < HI; ++i) u = fma(TRANS ? c_oi[UE + i * HC + o] : c_oi[UE + o * HC + i], xe[i], u);
#pragma unroll
    for (int i = 0; i < FI; ++i) v = fma(TRANS ? c_oi[UO + i * HC + o] : c_oi[UO + o * HC + i], xo[i], v);
    y[o] = u + v;
    y[MO - 1 - o] = ANTI ? v - u : u - v;
  }
  if (MO & 1) {
    double m = 0.0;
    if (ANTI) {
#pragma unroll
      for (int i = 0; i < FI; ++i) m = fma(TRANS ? c_oi[UO + i * HC + FO] : c_oi[UO + FO * HC + i], xo[i], m);
    } else {
#pragma unroll
      for (int i = 0; i < HI; ++i) m = fma(TRANS ? c_oi[UE + i * HC + FO] : c_oi[UE + FO * HC + i], xe[i], m);
    }
    y[FO] = m;
  }
}

// z-lines, forward: T = N_z B (N -> NQ points) and, from the same registers, G2 = D~_z T (one tile read, two writes).
// z-lines, backward: R = D~_z^T G2 + T + G0 + G1 on the line, then N_z^T R (NQ -> N) written IN PLACE over the first N
// entries of the G2 line (a thread reads its whole line before it writes; lines of different threads are disjoint).
template <int N, int NQ, int ON, int OD, int bv, bool BACK>
__device__ __forceinline__ void z_lines(double* B0, double* B1, double* B2, double* T, int tid) {
  constexpr int nlines = NQ * NQ * bv, ZS = NQ * NQ;
#pragma unroll
  for (int t0 = 0; t0 < nlines; t0 += 256) {
    const int t = t0 + tid;
    if (t >= nlines) break;
    const int beta = t % bv, r = t / bv;       // r = a + NQ b: the line's first point
    if (!BACK) {
      double x[N], y[NQ], d[NQ];
#pragma unroll
      for (int i = 0; i < N; ++i) x[i] = B0[(size_t)(r + i * ZS) * bv + beta];
      eo_line<N, NQ, false, false, ON>(x, y);
#pragma unroll
      for (int o = 0; o < NQ; ++o) T[(size_t)(r + o * ZS) * bv + beta] = y[o];
      eo_line<NQ, NQ, false, true, OD>(y, d);
#pragma unroll
      for (int o = 0; o < NQ; ++o) B2[(size_t)(r + o * ZS) * bv + beta] = d[o];
    } else {
      double x[NQ], y[NQ], z[N];
#pragma unroll
      for (int i = 0; i < NQ; ++i) x[i] = B2[(size_t)(r + i * ZS) * bv + beta];
      eo_line<NQ, NQ, true, true, OD>(x, y);
#pragma unroll
      for (int i = 0; i < NQ; ++i) {
        const size_t k = (size_t)(r + i * ZS) * bv + beta;
        y[i] += (T[k] + B0[k]) + B1[k];
      }
      eo_line<NQ, N, true, false, ON>(y, z);
#pragma unroll
      for (int o = 0; o < N; ++o) B2[(size_t)(r + o * ZS) * bv + beta] = z[o];
    }
  }
}

template <int PDEG, int NQ, int bv, int MINB = 2>
__global__ void __launch_bounds__(256, MINB)
fe_apply_oi(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmZ, const ApplyParams P,
            const OiParams O, int use_tma) {
  constexpr int N = PDEG + 1, NQ3 = NQ * NQ * NQ;
  extern __shared__ __align__(128) unsigned char smem_oi[];
  FE_STATIC_SHARED uint64_t bar;
  double* B0 = reinterpret_cast<double*>(smem_oi);
  double* B1 = B0 + (size_t)NQ3 * bv;
  double* B2 = B1 + (size_t)NQ3 * bv;
  double* T = B2 + (size_t)NQ3 * bv;
  constexpr int ON = OiOffset<PDEG>::value, OD = ON + 2 * ((NQ + 1) / 2) * ((N + 1) / 2);   // [Ne | No] and [De | Do] in c_oi
  const int tid = threadIdx.x, nth = blockDim.x;
  const int vb = blockIdx.x % P.nvb;
  const int cell = blockIdx.x / P.nvb;
  const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
  const int v0 = vb * bv;
  // S2 gather: ONE 4-D tensor-map bulk copy per block (box (bv, n, n, n) = the layout of B0; the vector tail and the
  // nodes past the end of a periodic mesh are zero-filled by the TMA unit).  A cell that wraps around then fetches its
  // wrapped nodes with loads, a cell on the Dirichlet boundary zeroes its boundary nodes in the tile.  Contexts with the
  // M^-1/2 diagonal, and calls the TMA conditions exclude, gather with loads, branch-free and in two stages (all the
  // loads of a thread are issued before the first is consumed: with one load per dependent iteration the phase took
  // 30 % of the kernel, ncu)
  const bool special = P.dirichlet ? (ex == 0 || ex == P.ncx - 1 || ey == 0 || ey == P.ncy - 1 || ez == 0 || ez == P.ncz - 1)
                                   : (ex == P.ncx - 1 || ey == P.ncy - 1 || ez == P.ncz - 1);
  const bool tma = use_tma && !P.dscale;   // uniform over the block
  constexpr int TOT = N * N * N * bv, GI = (TOT + 255) / 256;
  if (tma) {
    if (tid == 0) {
      mbar_init(&bar, 1);
      mbar_init_fence();
      mbar_expect_tx(&bar, TOT * 8);
      tma_load_4d(B0, &tmW, &bar, v0, ex * PDEG, ey * PDEG, ez * PDEG);
    }
    __syncthreads();
    mbar_wait(&bar, 0);
    if (special) {
#pragma unroll
      for (int k = 0; k < GI; ++k) {
        const int t = k * 256 + tid;
        const int beta = t % bv, I = t / bv;
        const int i1 = I % N, i2 = (I / N) % N, i3 = I / (N * N);
        int ix = ex * PDEG + i1, iy = ey * PDEG + i2, iz = ez * PDEG + i3;
        const bool in = (k + 1) * 256 <= TOT || t < TOT;
        if (P.dirichlet) {
          const bool bnd = ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz);
          if (in && bnd) B0[t] = 0.0;
        } else {
          const bool wrapped = ix >= P.ndx || iy >= P.ndy || iz >= P.ndz;
          ix = ix >= P.ndx ? ix - P.ndx : ix;
          iy = iy >= P.ndy ? iy - P.ndy : iy;
          iz = iz >= P.ndz ? iz - P.ndz : iz;
          if (in && wrapped && (v0 + beta) < P.nvec) B0[t] = __ldg(P.W + global_node(P, ix, iy, iz) * P.nvec + v0 + beta);
        }
      }
    }
  } else
  {
    double xv[GI];
    long long node[GI];
    unsigned livemask = 0;
#pragma unroll
    for (int k = 0; k < GI; ++k) {
      const int t = k * 256 + tid;
      const int beta = t % bv, I = t / bv;
      const int i1 = I % N, i2 = (I / N) % N, i3 = I / (N * N);
      int ix = ex * PDEG + i1, iy = ey * PDEG + i2, iz = ez * PDEG + i3;
      bool live = ((k + 1) * 256 <= TOT || t < TOT) && (v0 + beta) < P.nvec;
      const bool bnd = ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz);
      live = live && !(P.dirichlet && bnd);
      ix = ix >= P.ndx ? ix - P.ndx : ix;   // periodic wrap (never taken on a Dirichlet mesh)
      iy = iy >= P.ndy ? iy - P.ndy : iy;
      iz = iz >= P.ndz ? iz - P.ndz : iz;
      node[k] = live ? global_node(P, ix, iy, iz) : 0;
      xv[k] = __ldg(P.W + node[k] * P.nvec + (live ? v0 + beta : 0));
      livemask |= (live ? 1u : 0u) << k;
    }
    if (P.dscale) {
      double dv[GI];
#pragma unroll
      for (int k = 0; k < GI; ++k) dv[k] = __ldg(P.dscale + node[k]);
#pragma unroll
      for (int k = 0; k < GI; ++k) xv[k] *= dv[k];
    }
#pragma unroll
    for (int k = 0; k < GI; ++k) {
      const int t = k * 256 + tid;
      if ((k + 1) * 256 <= TOT || t < TOT) B0[t] = ((livemask >> k) & 1u) ? xv[k] : 0.0;
    }
  }
  __syncthreads();
  contract_lines<N, N, N, 0, NQ, false, false, false, ON, bv>(B0, B1, tid); __syncthreads();
  contract_lines<NQ, N, N, 1, NQ, false, false, false, ON, bv>(B1, B0, tid); __syncthreads();
  z_lines<N, NQ, ON, OD, bv, false>(B0, B1, B2, T, tid); __syncthreads();   // N_z and D~_z chained in registers
  contract_lines<NQ, NQ, NQ, 0, NQ, false, true, false, OD, bv>(T, B0, tid);
  contract_lines<NQ, NQ, NQ, 1, NQ, false, true, false, OD, bv>(T, B1, tid);
  __syncthreads();
  // S5: one thread = one point for all the block's vectors (the 7 factors are loaded once); the factors of PF points are
  // loaded before the first is used
  constexpr int QI = (NQ3 + 255) / 256, PF = 3;
#pragma unroll
  for (int k0 = 0; k0 < QI; k0 += PF) {
    double g[PF][7];
#pragma unroll
    for (int j = 0; j < PF; ++j) {
      const int k = k0 + j;
      if (k >= QI) break;
      int Q = k * 256 + tid;
      if (!((k + 1) * 256 <= NQ3 || Q < NQ3)) Q = 0;
      if (P.geom_mode == 2) {
        const double* gp = O.geom + (size_t)cell * O.geom_stride + Q;
#pragma unroll
        for (int c = 0; c < 7; ++c) g[j][c] = __ldg(gp + (size_t)c * NQ3);
      } else {
#pragma unroll
        for (int c = 0; c < 7; ++c) g[j][c] = P.geom_mode == 1 ? __ldg(P.geom + (size_t)cell * 7 + c) : P.ug[c];
        if (P.kappa) g[j][6] *= __ldg(P.kappa + (size_t)cell * NQ3 + Q);
      }
    }
#pragma unroll
    for (int j = 0; j < PF; ++j) {
      const int k = k0 + j;
      if (k >= QI) break;
      const int Q = k * 256 + tid;
      if (!((k + 1) * 256 <= NQ3 || Q < NQ3)) break;
      const int q1 = Q % NQ, q2 = (Q / NQ) % NQ, q3 = Q / (NQ * NQ);
      const double wq = P.alpha * (__ldg(O.wq + q1) * __ldg(O.wq + q2) * __ldg(O.wq + q3));   // the result is linear in the factors
#pragma unroll
      for (int c = 0; c < 7; ++c) g[j][c] *= wq;
      for (int beta = 0; beta < bv; ++beta) {
        const int t = Q * bv + beta;
        const double a = B0[t], b = B1[t], c = B2[t];
        B0[t] = g[j][0] * a + g[j][1] * b + g[j][2] * c;
        B1[t] = g[j][1] * a + g[j][3] * b + g[j][4] * c;
        B2[t] = g[j][2] * a + g[j][4] * b + g[j][5] * c;
        T[t] = g[j][6] * T[t];
      }
    }
  }
  __syncthreads();
  // S6: D~^T_x and D~^T_y in place on their own tiles (no barrier between them), then the z-lines add the four terms
  // and go on to N^T_z in registers: 11 block barriers per cell instead of 14, no read-modify-write of T
  contract_lines<NQ, NQ, NQ, 0, NQ, true, true, false, OD, bv, true>(B0, B0, tid);
  contract_lines<NQ, NQ, NQ, 1, NQ, true, true, false, OD, bv, true>(B1, B1, tid); __syncthreads();
  z_lines<N, NQ, ON, OD, bv, true>(B0, B1, B2, T, tid); __syncthreads();
  contract_lines<NQ, NQ, N, 1, N, true, false, false, ON, bv>(B2, B1, tid); __syncthreads();
  contract_lines<NQ, N, N, 0, N, true, false, false, ON, bv>(B1, B0, tid); __syncthreads();
  // S8 scatter-add: ONE bulk tensor reduction (add.f64 in L2, clipped at the vector tail and at the end of the mesh)
  if (tma) {
    if (special) {   // wrapped nodes (clipped by the reduction) leave through atomics; Dirichlet boundary rows add 0
      for (int t = tid; t < TOT; t += nth) {
        const int beta = t % bv, I = t / bv;
        const int i1 = I % N, i2 = (I / N) % N, i3 = I / (N * N);
        int ix = ex * PDEG + i1, iy = ey * PDEG + i2, iz = ez * PDEG + i3;
        if (P.dirichlet) {
          if (ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz)) B0[t] = 0.0;
        } else {
          const bool wrapped = ix >= P.ndx || iy >= P.ndy || iz >= P.ndz;
          ix = ix >= P.ndx ? ix - P.ndx : ix;
          iy = iy >= P.ndy ? iy - P.ndy : iy;
          iz = iz >= P.ndz ? iz - P.ndz : iz;
          if (wrapped && (v0 + beta) < P.nvec) atomicAdd(&P.Z[global_node(P, ix, iy, iz) * P.nvec + v0 + beta], B0[t]);
        }
      }
    }
    fence_async_smem();
    __syncthreads();
    if (tid == 0) {
      tma_reduce_add_4d(&tmZ, B0, v0, ex * PDEG, ey * PDEG, ez * PDEG);
      tma_commit();
      tma_wait_all0();
    }
    return;
  }
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
      atomicAdd(&P.Z[global_node(P, ix, iy, iz) * P.nvec + v0 + beta], dv * B0[t]);
    }
  }
}

}  // namespace fe
