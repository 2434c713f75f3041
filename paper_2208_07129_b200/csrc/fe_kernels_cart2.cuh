// Device code, part 3: two vectors per thread (a double2 per node) -- the value type of the line kernels.
//   * two vectors per thread halve the shared-memory instruction count per FP64 instruction (128-bit LDS/STS)
//     and let one uniform-register table operand feed two DFMAs;
//   * D~s and D~s^T (and Ns, Ns^T) read the SAME half tables (the transpose of a centro-(anti)symmetric
//     matrix has the transposed half tables).
#pragma once
#include "fe_kernels_eo.cuh"

namespace fe {

struct v2 { double a, b; };
__device__ __forceinline__ v2 operator+(v2 x, v2 y) { return {x.a + y.a, x.b + y.b}; }
__device__ __forceinline__ v2 operator-(v2 x, v2 y) { return {x.a - y.a, x.b - y.b}; }
__device__ __forceinline__ v2 vmul(double c, v2 x) { return {c * x.a, c * x.b}; }
__device__ __forceinline__ v2 vfma(double c, v2 x, v2 y) { return {fma(c, x.a, y.a), fma(c, x.b, y.b)}; }

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

}  // namespace fe
