// Device code, part 2: the optimised fused kernels.
//
//  * even-odd decomposed 1D contractions (derived from the centro-symmetry
//    N[q][i] = N[n-1-q][n-1-i], D~[q][r] = -D~[n-1-q][n-1-r], not from Listing 2 -- DESIGN.md reading 14),
//    operands in registers, table halves as constant-bank immediates;
//  * sqrt(w)-rescaled tables: Ns = diag(sqrt w) N, Ds = diag(sqrt w) D~ diag(1/sqrt w), so the
//    quadrature-point step needs only J^-1 J^-T det J and sigma det J;
//  * "pencil" passes fused so that each shared-memory round trip carries as many contractions as the data
//    dependences allow (the D~ / scale / D~^T triple of one direction never leaves registers when the
//    metric is diagonal), 15 tile accesses per point instead of 24.
#pragma once
#include "fe_kernels.cuh"

namespace fe {

static __constant__ EoTab c_eo[KMAXN][5];

template <int PDEG, int KIND>
__device__ __forceinline__ void eo_apply(const double (&x)[PDEG + 1], double (&y)[PDEG + 1]) {
  constexpr int N = PDEG + 1, H = N / 2;
  constexpr bool ODD = (N & 1) != 0, ANTI = (KIND == EO_DS || KIND == EO_DST);
  const EoTab& t = c_eo[PDEG][KIND];
  double xp[H > 0 ? H : 1], xm[H > 0 ? H : 1];
#pragma unroll
  for (int i = 0; i < H; ++i) { xp[i] = x[i] + x[N - 1 - i]; xm[i] = x[i] - x[N - 1 - i]; }
#pragma unroll
  for (int q = 0; q < H; ++q) {
    double u = t.P[q * H] * xp[0];
#pragma unroll
    for (int i = 1; i < H; ++i) u = fma(t.P[q * H + i], xp[i], u);
    if (ODD) u = fma(t.Pm[q], x[H], u);
    double v = t.Mn[q * H] * xm[0];
#pragma unroll
    for (int i = 1; i < H; ++i) v = fma(t.Mn[q * H + i], xm[i], v);
    y[q] = u + v;
    y[N - 1 - q] = ANTI ? (v - u) : (u - v);
  }
  if (ODD) {
    double m;
    if (ANTI) {
      m = t.mid[0] * xm[0];
#pragma unroll
      for (int i = 1; i < H; ++i) m = fma(t.mid[i], xm[i], m);
    } else {
      m = t.midm * x[H];
#pragma unroll
      for (int i = 0; i < H; ++i) m = fma(t.mid[i], xp[i], m);
    }
    y[H] = m;
  }
}

// r += Ds^T (g * (Ds t)) : one direction of the stiffness term at the quadrature points (Alg. 2 l.2-9 restricted to
// a diagonal metric entry g that is constant along the line, so that Ds^T g Ds = 2g (Ds^T Ds / 2): ONE contraction
// with the host-precomputed 1D operator, as in fe_kernels_plane.cuh).
template <int PDEG>
__device__ __forceinline__ void kterm(const double (&t)[PDEG + 1], double (&r)[PDEG + 1], double g) {
  constexpr int N = PDEG + 1;
  double b[N];
  eo_apply<PDEG, EO_SH>(t, b);
  const double g2 = 2.0 * g;
#pragma unroll
  for (int i = 0; i < N; ++i) r[i] = fma(g2, b[i], r[i]);
}

// Shared-memory tile layout [i3][i2][i1][beta] with the x-line pitch padded by one node when n is even and
// a line is narrower than a 128-byte wavefront, so that the two lines of a half-warp fall in disjoint banks.
template <int PDEG, int BV>
struct Tile {
  static constexpr int N = PDEG + 1;
  static constexpr int XP = N * BV + ((N % 2 == 0 && BV < 16) ? BV : 0);
  static constexpr int SIZE = N * N * XP;
  // base offset and element stride of line l along direction DIR
  template <int DIR>
  static __device__ __forceinline__ void line(int l, int& base, int& stride) {
    const int a = l % N, b = l / N;
    if (DIR == 0) { base = (b * N + a) * XP; stride = BV; }          // a = i2, b = i3
    else if (DIR == 1) { base = b * N * XP + a * BV; stride = XP; }  // a = i1, b = i3
    else { base = b * XP + a * BV; stride = N * XP; }                // a = i1, b = i2
  }
};

template <int N>
__device__ __forceinline__ void lds_line(const double* s, int stride, double (&x)[N]) {
#pragma unroll
  for (int i = 0; i < N; ++i) x[i] = s[i * stride];
}
template <int N>
__device__ __forceinline__ void sts_line(double* s, int stride, const double (&x)[N]) {
#pragma unroll
  for (int i = 0; i < N; ++i) s[i * stride] = x[i];
}

// Fused apply for cells whose metric is diagonal and constant per cell (uniform Cartesian meshes: configs
// 1, 2, 4, 5).  Z += alpha * A * W.  One block = one cell x BV vectors; NT threads; 2 tiles of shared memory.
// CELLS (calls with 1-3 vectors, e.g. the single-vector point of config 4's sweep): the BV slots of a tile hold
// P.nvec vectors of BV / P.nvec consecutive cells of an x-row instead of BV vectors of one cell, so that the
// lanes stay busy and the shared-memory layout (slot innermost) stays conflict-free.
template <int PDEG, int BV, int NT, int MINB, bool CELLS = false>
__global__ void __launch_bounds__(NT, MINB) fe_apply_cart(const ApplyParams P) {
  using TL = Tile<PDEG, BV>;
  constexpr int N = PDEG + 1, NL = N * N, TASKS = NL * BV;
  extern __shared__ double smem[];
  double* A = smem;
  double* B = smem + TL::SIZE;
  const int tid = threadIdx.x;
  const int nvb = CELLS ? (P.ncx + (BV / P.nvec) - 1) / (BV / P.nvec) : P.nvb;   // CELLS: cell groups per x-row
  const int vb = blockIdx.x % nvb;
  const int cell = CELLS ? (blockIdx.x / nvb) * P.ncx : blockIdx.x / P.nvb;      // CELLS: first cell of the x-row
  const int ex0 = CELLS ? vb * (BV / P.nvec) : cell % P.ncx;
  const int ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
  const int v0 = CELLS ? 0 : vb * BV;
  const double gxx = P.ug[0], gyy = P.ug[3], gzz = P.ug[5], gm = P.ug[6];

  // phase 0: gather x-lines (S2) + Ns along x (S3, dim 1)
  for (int t = tid; t < TASKS; t += NT) {
    const int beta = t % BV, l = t / BV;
    const int i2 = l % N, i3 = l / N;
    int iy = ey * PDEG + i2, iz = ez * PDEG + i3;
    const int ex = CELLS ? ex0 + beta / P.nvec : ex0;     // slot -> (cell, vector)
    const int vv = CELLS ? beta % P.nvec : v0 + beta;
    bool live = CELLS ? (ex < P.ncx && beta < (BV / P.nvec) * P.nvec) : (vv < P.nvec);
    if (P.dirichlet) {
      if (iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz)) live = false;
    } else {
      if (iy >= P.ndy) iy -= P.ndy;
      if (iz >= P.ndz) iz -= P.ndz;
    }
    double x[N], y[N];
    const long long row = (long long)P.ndx * ((long long)iy + (long long)P.ndy * iz);
    const double* src = P.W + (row + (long long)ex * PDEG) * P.nvec + vv;
#pragma unroll
    for (int i = 0; i < N; ++i) {
      int ix = ex * PDEG + i;
      bool ok = live;
      long long off = (long long)i * P.nvec;
      if (P.dirichlet) { if (ix == 0 || ix == P.ndx - 1) ok = false; }
      else if (ix >= P.ndx) off -= (long long)P.ndx * P.nvec;
      x[i] = ok ? __ldg(src + off) : 0.0;
    }
    eo_apply<PDEG, EO_NS>(x, y);
    int base, stride; TL::template line<0>(l, base, stride);
    sts_line<N>(A + base + beta, stride, y);
  }
  __syncthreads();
  // phase 1: Ns along y, in place
  for (int t = tid; t < TASKS; t += NT) {
    const int beta = t % BV, l = t / BV;
    int base, stride; TL::template line<1>(l, base, stride);
    double x[N], y[N];
    lds_line<N>(A + base + beta, stride, x);
    eo_apply<PDEG, EO_NS>(x, y);
    sts_line<N>(A + base + beta, stride, y);
  }
  __syncthreads();
  // phase 2: Ns along z -> T (kept in A); R = gm*T + Ds^T gzz Ds T along z -> B   (S3 dim 3, S4-S6 z-part)
  for (int t = tid; t < TASKS; t += NT) {
    const int beta = t % BV, l = t / BV;
    int base, stride; TL::template line<2>(l, base, stride);
    double x[N], tq[N], r[N];
    lds_line<N>(A + base + beta, stride, x);
    eo_apply<PDEG, EO_NS>(x, tq);
    sts_line<N>(A + base + beta, stride, tq);
#pragma unroll
    for (int i = 0; i < N; ++i) r[i] = gm * tq[i];
    kterm<PDEG>(tq, r, gzz);
    sts_line<N>(B + base + beta, stride, r);
  }
  __syncthreads();
  // phase 3: R += Ds^T gxx Ds T along x
  for (int t = tid; t < TASKS; t += NT) {
    const int beta = t % BV, l = t / BV;
    int base, stride; TL::template line<0>(l, base, stride);
    double tq[N], r[N];
    lds_line<N>(A + base + beta, stride, tq);
    lds_line<N>(B + base + beta, stride, r);
    kterm<PDEG>(tq, r, gxx);
    sts_line<N>(B + base + beta, stride, r);
  }
  __syncthreads();
  // phase 4: R += Ds^T gyy Ds T along y, then Ns^T along y (S7), in place in B
  for (int t = tid; t < TASKS; t += NT) {
    const int beta = t % BV, l = t / BV;
    int base, stride; TL::template line<1>(l, base, stride);
    double tq[N], r[N], u[N];
    lds_line<N>(A + base + beta, stride, tq);
    lds_line<N>(B + base + beta, stride, r);
    kterm<PDEG>(tq, r, gyy);
    eo_apply<PDEG, EO_NST>(r, u);
    sts_line<N>(B + base + beta, stride, u);
  }
  __syncthreads();
  // phase 5: Ns^T along x, in place
  for (int t = tid; t < TASKS; t += NT) {
    const int beta = t % BV, l = t / BV;
    int base, stride; TL::template line<0>(l, base, stride);
    double x[N], y[N];
    lds_line<N>(B + base + beta, stride, x);
    eo_apply<PDEG, EO_NST>(x, y);
    sts_line<N>(B + base + beta, stride, y);
  }
  __syncthreads();
  // phase 6: Ns^T along z + scatter-add (S7 dim 3 fused with S8)
  for (int t = tid; t < TASKS; t += NT) {
    const int beta = t % BV, l = t / BV;
    const int i1 = l % N, i2 = l / N;
    int base, stride; TL::template line<2>(l, base, stride);
    double x[N], y[N];
    lds_line<N>(B + base + beta, stride, x);
    eo_apply<PDEG, EO_NST>(x, y);
    const int ex = CELLS ? ex0 + beta / P.nvec : ex0;
    const int vv = CELLS ? beta % P.nvec : v0 + beta;
    int ix = ex * PDEG + i1, iy = ey * PDEG + i2;
    bool live = CELLS ? (ex < P.ncx && beta < (BV / P.nvec) * P.nvec) : (vv < P.nvec);
    if (P.dirichlet) {
      if (ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1) live = false;
    } else {
      if (ix >= P.ndx) ix -= P.ndx;
      if (iy >= P.ndy) iy -= P.ndy;
    }
    if (live) {
      const long long plane = (long long)P.ndx * P.ndy;
      double* dst = P.Z + ((long long)ix + (long long)P.ndx * iy) * P.nvec + vv;
#pragma unroll
      for (int i = 0; i < N; ++i) {
        int iz = ez * PDEG + i;
        bool ok = true;
        if (P.dirichlet) { if (fe_z_masked(P, iz)) ok = false; }
        else if (iz >= P.ndz) iz -= P.ndz;
        if (ok) atomicAdd(dst + plane * iz * P.nvec, P.alpha * y[i]);
      }
    }
  }
}

}  // namespace fe
