// Device code, part 3: the production Cartesian kernel.  Same fused pass structure as fe_apply_cart
// (fe_kernels_eo.cuh) but each thread carries TWO vectors (a double2 per node):
//   * ptxas materialises every FP64 table entry with an LDC.64 (sm_100 DFMA takes no 64-bit constant-bank
//     operand), and a matrix entry is used once per line, so one vector per thread costs one LDC per DFMA
//     and saturates the issue slots (profiles/r1_v2_*: issue 67 %, FP64 pipe 45 %).  Two vectors per thread
//     halve the LDC and LDS/STS instruction counts per FP64 instruction (128-bit shared-memory accesses);
//   * D~s and D~s^T (and Ns, Ns^T) read the SAME half tables (the transpose of a centro-(anti)symmetric
//     matrix has the transposed half tables), so the D~/scale/D~^T triple loads 24 constants, not 49.
#pragma once
#include "fe_kernels_eo.cuh"

namespace fe {

struct v2 { double a, b; };
__device__ __forceinline__ v2 operator+(v2 x, v2 y) { return {x.a + y.a, x.b + y.b}; }
__device__ __forceinline__ v2 operator-(v2 x, v2 y) { return {x.a - y.a, x.b - y.b}; }
__device__ __forceinline__ v2 vmul(double c, v2 x) { return {c * x.a, c * x.b}; }
__device__ __forceinline__ v2 vfma(double c, v2 x, v2 y) { return {fma(c, x.a, y.a), fma(c, x.b, y.b)}; }

enum { MAT_NS = 0, MAT_DS = 1 };

// y = M x or M^T x from the half tables of M (c_eo[PDEG][EO_NS] or c_eo[PDEG][EO_DS]).
template <int PDEG, int MAT, bool TRANS, typename T>
__device__ __forceinline__ void eo2(const T (&x)[PDEG + 1], T (&y)[PDEG + 1]) {
  constexpr int N = PDEG + 1, H = N / 2;
  constexpr bool ODD = (N & 1) != 0, ANTI = (MAT == MAT_DS);
  const EoTab& t = c_eo[PDEG][MAT == MAT_NS ? EO_NS : EO_DS];
  T xp[H > 0 ? H : 1], xm[H > 0 ? H : 1];
#pragma unroll
  for (int i = 0; i < H; ++i) { xp[i] = x[i] + x[N - 1 - i]; xm[i] = x[i] - x[N - 1 - i]; }
#pragma unroll
  for (int q = 0; q < H; ++q) {
    // P_T[q][i] = P[i][q] (sym) | Mn[i][q] (anti);  Mn_T[q][i] = Mn[i][q] (sym) | P[i][q] (anti)
    T u = vmul(!TRANS ? t.P[q * H] : (ANTI ? t.Mn[q] : t.P[q]), xp[0]);
#pragma unroll
    for (int i = 1; i < H; ++i) u = vfma(!TRANS ? t.P[q * H + i] : (ANTI ? t.Mn[i * H + q] : t.P[i * H + q]), xp[i], u);
    if (ODD) u = vfma(!TRANS ? t.Pm[q] : t.mid[q], x[H], u);
    T v = vmul(!TRANS ? t.Mn[q * H] : (ANTI ? t.P[q] : t.Mn[q]), xm[0]);
#pragma unroll
    for (int i = 1; i < H; ++i) v = vfma(!TRANS ? t.Mn[q * H + i] : (ANTI ? t.P[i * H + q] : t.Mn[i * H + q]), xm[i], v);
    y[q] = u + v;
    y[N - 1 - q] = ANTI ? (v - u) : (u - v);
  }
  if (ODD) {
    T m;
    if (ANTI) {
      m = vmul(!TRANS ? t.mid[0] : t.Pm[0], xm[0]);
#pragma unroll
      for (int i = 1; i < H; ++i) m = vfma(!TRANS ? t.mid[i] : t.Pm[i], xm[i], m);
    } else {
      m = vmul(t.midm, x[H]);
#pragma unroll
      for (int i = 0; i < H; ++i) m = vfma(!TRANS ? t.mid[i] : t.Pm[i], xp[i], m);
    }
    y[H] = m;
  }
}

// r += Ds^T (g * (Ds t))
template <int PDEG, typename T>
__device__ __forceinline__ void kterm2(const T (&t)[PDEG + 1], T (&r)[PDEG + 1], double g) {
  constexpr int N = PDEG + 1;
  T a[N], b[N];
  eo2<PDEG, MAT_DS, false>(t, a);
#pragma unroll
  for (int i = 0; i < N; ++i) a[i] = vmul(g, a[i]);
  eo2<PDEG, MAT_DS, true>(a, b);
#pragma unroll
  for (int i = 0; i < N; ++i) r[i] = r[i] + b[i];
}

template <int N>
__device__ __forceinline__ void lds_line2(const double* s, int stride, v2 (&x)[N]) {
#pragma unroll
  for (int i = 0; i < N; ++i) { const double2 d = *reinterpret_cast<const double2*>(s + i * stride); x[i] = {d.x, d.y}; }
}
template <int N>
__device__ __forceinline__ void sts_line2(double* s, int stride, const v2 (&x)[N]) {
#pragma unroll
  for (int i = 0; i < N; ++i) *reinterpret_cast<double2*>(s + i * stride) = make_double2(x[i].a, x[i].b);
}

// Z += A*W with alpha folded into P.ug (the result is linear in the four metric constants).
// Requires: diagonal constant metric, nvec even, W/Z 16-byte aligned.
template <int PDEG, int BV, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) fe_apply_cart2(const ApplyParams P) {
  using TL = Tile<PDEG, BV>;
  constexpr int N = PDEG + 1, NL = N * N, TPL = BV / 2, TASKS = NL * TPL;
  extern __shared__ __align__(16) double smem[];
  double* A = smem;
  double* B = smem + TL::SIZE;
  const int tid = threadIdx.x;
  const int vb = blockIdx.x % P.nvb;
  const int cell = blockIdx.x / P.nvb;
  const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
  const int v0 = vb * BV;
  const double gxx = P.ug[0], gyy = P.ug[3], gzz = P.ug[5], gm = P.ug[6];
  const long long nvec = P.nvec;

  // phase 0: gather x-lines (S2) + Ns along x
  for (int t = tid; t < TASKS; t += NT) {
    const int b2 = (t % TPL) * 2, l = t / TPL;
    const int i2 = l % N, i3 = l / N;
    int iy = ey * PDEG + i2, iz = ez * PDEG + i3;
    bool live = (v0 + b2) < P.nvec;
    bool first_ok = true, last_ok = true;
    long long last_off = (long long)PDEG * nvec;
    if (P.dirichlet) {
      if (iy == 0 || iy == P.ndy - 1 || iz == 0 || iz == P.ndz - 1) live = false;
      first_ok = (ex != 0); last_ok = (ex != P.ncx - 1);
    } else {
      if (iy >= P.ndy) iy -= P.ndy;
      if (iz >= P.ndz) iz -= P.ndz;
      if (ex == P.ncx - 1) last_off -= (long long)P.ndx * nvec;
    }
    const long long row = (long long)P.ndx * ((long long)iy + (long long)P.ndy * iz);
    const double* src = P.W + (row + (long long)ex * PDEG) * nvec + v0 + b2;
    v2 x[N], y[N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
      const bool ok = live && (i == 0 ? first_ok : (i == N - 1 ? last_ok : true));
      const long long off = (i == N - 1) ? last_off : (long long)i * nvec;
      double2 d = make_double2(0.0, 0.0);
      if (ok) d = __ldg(reinterpret_cast<const double2*>(src + off));
      x[i] = {d.x, d.y};
    }
    eo2<PDEG, MAT_NS, false>(x, y);
    int base, stride; TL::template line<0>(l, base, stride);
    sts_line2<N>(A + base + b2, stride, y);
  }
  __syncthreads();
  // phase 1: Ns along y, in place
  for (int t = tid; t < TASKS; t += NT) {
    const int b2 = (t % TPL) * 2, l = t / TPL;
    int base, stride; TL::template line<1>(l, base, stride);
    v2 x[N], y[N];
    lds_line2<N>(A + base + b2, stride, x);
    eo2<PDEG, MAT_NS, false>(x, y);
    sts_line2<N>(A + base + b2, stride, y);
  }
  __syncthreads();
  // phase 2: Ns along z -> T (A); R = gm*T + Ds^T gzz Ds T along z -> B
  for (int t = tid; t < TASKS; t += NT) {
    const int b2 = (t % TPL) * 2, l = t / TPL;
    int base, stride; TL::template line<2>(l, base, stride);
    v2 x[N], tq[N], r[N];
    lds_line2<N>(A + base + b2, stride, x);
    eo2<PDEG, MAT_NS, false>(x, tq);
    sts_line2<N>(A + base + b2, stride, tq);
#pragma unroll
    for (int i = 0; i < N; ++i) r[i] = vmul(gm, tq[i]);
    kterm2<PDEG>(tq, r, gzz);
    sts_line2<N>(B + base + b2, stride, r);
  }
  __syncthreads();
  // phase 3: R += Ds^T gxx Ds T along x
  for (int t = tid; t < TASKS; t += NT) {
    const int b2 = (t % TPL) * 2, l = t / TPL;
    int base, stride; TL::template line<0>(l, base, stride);
    v2 tq[N], r[N];
    lds_line2<N>(A + base + b2, stride, tq);
    lds_line2<N>(B + base + b2, stride, r);
    kterm2<PDEG>(tq, r, gxx);
    sts_line2<N>(B + base + b2, stride, r);
  }
  __syncthreads();
  // phase 4: R += Ds^T gyy Ds T along y, then Ns^T along y, in place in B
  for (int t = tid; t < TASKS; t += NT) {
    const int b2 = (t % TPL) * 2, l = t / TPL;
    int base, stride; TL::template line<1>(l, base, stride);
    v2 tq[N], r[N], u[N];
    lds_line2<N>(A + base + b2, stride, tq);
    lds_line2<N>(B + base + b2, stride, r);
    kterm2<PDEG>(tq, r, gyy);
    eo2<PDEG, MAT_NS, true>(r, u);
    sts_line2<N>(B + base + b2, stride, u);
  }
  __syncthreads();
  // phase 5: Ns^T along x, in place
  for (int t = tid; t < TASKS; t += NT) {
    const int b2 = (t % TPL) * 2, l = t / TPL;
    int base, stride; TL::template line<0>(l, base, stride);
    v2 x[N], y[N];
    lds_line2<N>(B + base + b2, stride, x);
    eo2<PDEG, MAT_NS, true>(x, y);
    sts_line2<N>(B + base + b2, stride, y);
  }
  __syncthreads();
  // phase 6: Ns^T along z + scatter-add
  for (int t = tid; t < TASKS; t += NT) {
    const int b2 = (t % TPL) * 2, l = t / TPL;
    const int i1 = l % N, i2 = l / N;
    int base, stride; TL::template line<2>(l, base, stride);
    v2 x[N], y[N];
    lds_line2<N>(B + base + b2, stride, x);
    eo2<PDEG, MAT_NS, true>(x, y);
    int ix = ex * PDEG + i1, iy = ey * PDEG + i2;
    bool live = (v0 + b2) < P.nvec;
    bool first_ok = true, last_ok = true;
    const long long plane = (long long)P.ndx * P.ndy * nvec;
    long long last_off = (long long)PDEG * plane;
    if (P.dirichlet) {
      if (ix == 0 || ix == P.ndx - 1 || iy == 0 || iy == P.ndy - 1) live = false;
      first_ok = (ez != 0); last_ok = (ez != P.ncz - 1);
    } else {
      if (ix >= P.ndx) ix -= P.ndx;
      if (iy >= P.ndy) iy -= P.ndy;
      if (ez == P.ncz - 1) last_off -= (long long)P.ndz * plane;
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
  }
}

}  // namespace fe
