// Device code: the streaming kernels of S1 / S9 (axpby, scale, swap) and the synthetic-input generator.  Plain
// (non-template) kernels: included by exactly one translation unit (fe_tu_misc.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fe {

// S1 / S9 pre-pass: Z <- beta*Z + gamma*W  (Eq. B.1's bX + cY part)
__global__ void fe_axpby_kernel(double* __restrict__ Z, const double* __restrict__ W, double beta, double gamma,
                                size_t count) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const size_t n2 = count / 2;
  double2* Z2 = reinterpret_cast<double2*>(Z);
  const double2* W2 = reinterpret_cast<const double2*>(W);
  for (size_t k = i; k < n2; k += stride) {
    double2 z = Z2[k], w = W2[k];
    z.x = beta * z.x + gamma * w.x;
    z.y = beta * z.y + gamma * w.y;
    Z2[k] = z;
  }
  if (i == 0 && (count & 1)) Z[count - 1] = beta * Z[count - 1] + gamma * W[count - 1];
}

// The same for pointers that are only 8-byte aligned (a view of a larger allocation offset by an odd number of
// doubles); W may alias Z element by element (Z <- beta Z with gamma = 0)
__global__ void fe_axpby_scalar_kernel(double* Z, const double* W, double beta, double gamma, size_t count) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t k = i; k < count; k += stride) Z[k] = beta * Z[k] + gamma * W[k];
}

// Z <- gamma*W (beta == 0: Z is not read, so it may hold anything, e.g. NaN from a fresh allocation)
__global__ void fe_scale_copy_kernel(double* __restrict__ Z, const double* __restrict__ W, double gamma, size_t count) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t k = i; k < count; k += stride) Z[k] = gamma * W[k];
}

__global__ void fe_scale_kernel(double* Z, double beta, size_t count) {   // Z <- beta Z
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  double2* Z2 = reinterpret_cast<double2*>(Z);
  for (size_t k = i; k < count / 2; k += stride) { double2 z = Z2[k]; z.x *= beta; z.y *= beta; Z2[k] = z; }
  if (i == 0 && (count & 1)) Z[count - 1] *= beta;
}

// The end of the scaled Chebyshev recurrence (fe_cheb_filter): A <- sa * A, B <- sb * B (swap = 0) or
// A <- sa * B_old, B <- sb * A_old (swap = 1).  On a Dirichlet mesh (bnd = 1) the kernels never touch the boundary
// nodes, whose entries follow the scalar recurrence: there A still holds the input x0, and A <- qa x0, B <- qb x0.
__global__ void fe_scale2_kernel(double* __restrict__ A, double* __restrict__ B, double sa, double sb, int swap, size_t count,
                                 int bnd, double qa, double qb, int ndx, int ndy, int ndz, int nvec) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t k = i; k < count; k += stride) {
    const double a = A[k], b = B[k];
    if (bnd) {
      const size_t node = k / (size_t)nvec;
      const int ix = (int)(node % ndx), iy = (int)((node / ndx) % ndy), iz = (int)(node / ((size_t)ndx * ndy));
      if (ix == 0 || ix == ndx - 1 || iy == 0 || iy == ndy - 1 || iz == 0 || iz == ndz - 1) {
        A[k] = qa * a; B[k] = qb * a;
        continue;
      }
    }
    A[k] = sa * (swap ? b : a);
    B[k] = sb * (swap ? a : b);
  }
}

__global__ void fe_swap_kernel(double* __restrict__ A, double* __restrict__ B, size_t count) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t k = i; k < count; k += stride) { double a = A[k]; A[k] = B[k]; B[k] = a; }
}

// NEXT-4, the FP32 boundary payload: the plane that crosses a task boundary is recast as binary32
// (round to nearest even) on the sending side ...
__global__ void fe_halo_pack_f32_kernel(float* __restrict__ dst, const double* __restrict__ src, size_t count) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t k = i; k < count; k += stride) dst[k] = __double2float_rn(src[k]);
}
// ... and widened on the receiving side: dst <- src (add = 0: ghost values of U) or dst += src (add = 1: ghost rows of V)
__global__ void fe_halo_unpack_f32_kernel(double* __restrict__ dst, const float* __restrict__ src, size_t count, int add) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t k = i; k < count; k += stride) {
    const double v = (double)src[k];
    dst[k] = add ? dst[k] + v : v;
  }
}

// Input generator; not part of the operator.
__global__ void fe_fill_uniform_kernel(double* __restrict__ out, long long count, unsigned long long seed,
                                       long long offset) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long k = i; k < count; k += stride) {
    unsigned long long z = seed + (unsigned long long)(offset + k) * 0x9E3779B97F4A7C15ULL;
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    out[k] = 2.0 * ((double)(z >> 11) * 0x1.0p-53) - 1.0;
  }
}

}  // namespace fe
