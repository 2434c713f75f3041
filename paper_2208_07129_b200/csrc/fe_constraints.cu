// include/fe_constraints.h: the constraint matrices C, C^T of PAPER.md:288-302 (section 3.2.2) as two kernels over all sets.
// One thread block per (set, block of <= 32 vectors); a warp works on one slave (or master) row of the set's small
// dense product, its lanes on consecutive vectors, so that every multivector access is one contiguous row segment and
// every weight is a warp-wide broadcast.  Closed sets (no slave is a master) make the in-place update race-free:
// distribute reads master rows and writes slave rows only; the transpose adds into master rows (atomics: a master may
// serve several sets) and zeroes the slave rows of its own (set, vector block) after a block barrier.
#include <cuda_runtime.h>

#include <cstdint>
#include <new>
#include <string>
#include <vector>

#include "../../include/fe_constraints.h"
#include "../../include/fe_mf.h"

struct fe_constraints {
  long long ndof = 0;
  int nsets = 0;
  long long nmasters = 0, nslaves = 0;
  int device = 0;
  // device copies (four arrays per set, stored set after set, plus the offsets)
  long long *m_ptr = nullptr, *s_ptr = nullptr, *w_ptr = nullptr;   // [nsets+1] each
  long long *masters = nullptr, *slaves = nullptr;
  double *weights = nullptr, *inhomog = nullptr;
  std::string err;
};

namespace {

thread_local std::string g_create_error;

int fail(fe_constraints* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return code;
}

struct Guard {
  int prev = -1; bool ok = false;
  explicit Guard(int dev) { if (cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess) ok = true; }
  ~Guard() { if (prev >= 0) cudaSetDevice(prev); }
};

constexpr int kThreads = 256;
constexpr int kVecBlock = 32;

// [device-code-begin]  (tests/test_host_emulation.py compiles the lines up to the end marker for the host and runs them on threads)
struct SetArrays {
  const long long* m_ptr; const long long* s_ptr; const long long* w_ptr;
  const long long* masters; const long long* slaves;
  const double* weights; const double* inhomog;
};

// C: U[S_I] = W_I U[M_I] (+ b_I)
__global__ void fe_constraints_distribute_kernel(SetArrays A, double* U, int nvec, int homogeneous) {
  const long long set = blockIdx.x;
  const int v0 = blockIdx.y * kVecBlock;
  const int bw = min(kVecBlock, nvec - v0);
  const long long m0 = A.m_ptr[set], nm = A.m_ptr[set + 1] - m0;
  const long long s0 = A.s_ptr[set], ns = A.s_ptr[set + 1] - s0;
  const double* W = A.weights + A.w_ptr[set];
  for (long long pair = threadIdx.x; pair < ns * bw; pair += blockDim.x) {
    const long long s = pair / bw;
    const int beta = (int)(pair - s * bw);
    double acc = homogeneous ? 0.0 : A.inhomog[s0 + s];
    for (long long m = 0; m < nm; ++m)
      acc = fma(W[s * nm + m], U[A.masters[m0 + m] * (long long)nvec + v0 + beta], acc);
    U[A.slaves[s0 + s] * (long long)nvec + v0 + beta] = acc;
  }
}

// C^T: V[M_I] += W_I^T V[S_I];  V[S_I] = 0
__global__ void fe_constraints_transpose_kernel(SetArrays A, double* V, int nvec) {
  const long long set = blockIdx.x;
  const int v0 = blockIdx.y * kVecBlock;
  const int bw = min(kVecBlock, nvec - v0);
  const long long m0 = A.m_ptr[set], nm = A.m_ptr[set + 1] - m0;
  const long long s0 = A.s_ptr[set], ns = A.s_ptr[set + 1] - s0;
  const double* W = A.weights + A.w_ptr[set];
  for (long long pair = threadIdx.x; pair < nm * bw; pair += blockDim.x) {
    const long long m = pair / bw;
    const int beta = (int)(pair - m * bw);
    double acc = 0.0;
    for (long long s = 0; s < ns; ++s)
      acc = fma(W[s * nm + m], V[A.slaves[s0 + s] * (long long)nvec + v0 + beta], acc);
    atomicAdd(&V[A.masters[m0 + m] * (long long)nvec + v0 + beta], acc);
  }
  __syncthreads();   // every read of this block's slave entries is done (no other block touches them)
  for (long long pair = threadIdx.x; pair < ns * bw; pair += blockDim.x) {
    const long long s = pair / bw;
    const int beta = (int)(pair - s * bw);
    V[A.slaves[s0 + s] * (long long)nvec + v0 + beta] = 0.0;
  }
}

// [device-code-end]

template <typename T>
cudaError_t upload(T*& dst, const T* src, size_t count) {
  dst = nullptr;
  if (count == 0) return cudaSuccess;
  cudaError_t e = cudaMalloc(&dst, count * sizeof(T));
  if (e != cudaSuccess) return e;
  return cudaMemcpy(dst, src, count * sizeof(T), cudaMemcpyHostToDevice);
}

void release(fe_constraints* c) {
  cudaFree(c->m_ptr); cudaFree(c->s_ptr); cudaFree(c->w_ptr);
  cudaFree(c->masters); cudaFree(c->slaves); cudaFree(c->weights); cudaFree(c->inhomog);
}

SetArrays arrays(const fe_constraints* c) {
  return SetArrays{c->m_ptr, c->s_ptr, c->w_ptr, c->masters, c->slaves, c->weights, c->inhomog};
}

int check_call(fe_constraints* c, const double* X, int nvec) {
  if (!c) return FE_MF_EINVAL;
  if (!X) return fail(c, FE_MF_EINVAL, "null device pointer");
  if (nvec < 1) return fail(c, FE_MF_EINVAL, "nvec must be >= 1");
  if ((nvec + kVecBlock - 1) / kVecBlock > 65535) return fail(c, FE_MF_EINVAL, "nvec too large (more than 65535 blocks of 32 vectors)");
  return FE_MF_OK;
}

}  // namespace

static int create_impl(fe_constraints** out, long long ndof, int nsets, const long long* master_ptr,
                       const long long* masters, const long long* slave_ptr, const long long* slaves,
                       const double* weights, const double* inhomog, int cuda_device) {
  if (!out) return fail(nullptr, FE_MF_EINVAL, "out is NULL");
  *out = nullptr;
  if (ndof < 1 || nsets < 0) return fail(nullptr, FE_MF_EINVAL, "ndof must be > 0 and nsets >= 0");
  if (!master_ptr || !slave_ptr) return fail(nullptr, FE_MF_EINVAL, "master_ptr / slave_ptr is NULL");
  if (master_ptr[0] != 0 || slave_ptr[0] != 0) return fail(nullptr, FE_MF_EINVAL, "offset arrays must start at 0");
  for (int i = 0; i < nsets; ++i)
    if (master_ptr[i + 1] < master_ptr[i] || slave_ptr[i + 1] < slave_ptr[i])
      return fail(nullptr, FE_MF_EINVAL, "offset arrays must be non-decreasing");
  const long long nm_total = master_ptr[nsets], ns_total = slave_ptr[nsets];
  if ((nm_total > 0 && !masters) || (ns_total > 0 && !slaves)) return fail(nullptr, FE_MF_EINVAL, "masters / slaves is NULL");
  std::vector<long long> w_ptr((size_t)nsets + 1, 0);
  for (int i = 0; i < nsets; ++i)
    w_ptr[i + 1] = w_ptr[i] + (master_ptr[i + 1] - master_ptr[i]) * (slave_ptr[i + 1] - slave_ptr[i]);
  if (w_ptr[nsets] > 0 && !weights) return fail(nullptr, FE_MF_EINVAL, "weights is NULL");
  // closed sets (reading 19)
  {
    std::vector<unsigned char> is_slave((size_t)ndof, 0);
    for (long long k = 0; k < ns_total; ++k) {
      const long long s = slaves[k];
      if (s < 0 || s >= ndof) return fail(nullptr, FE_MF_EINVAL, "slave index out of range");
      if (is_slave[(size_t)s]) return fail(nullptr, FE_MF_EINVAL, "a slave belongs to two sets (or twice to one)");
      is_slave[(size_t)s] = 1;
    }
    for (long long k = 0; k < nm_total; ++k) {
      const long long m = masters[k];
      if (m < 0 || m >= ndof) return fail(nullptr, FE_MF_EINVAL, "master index out of range");
      if (is_slave[(size_t)m]) return fail(nullptr, FE_MF_EINVAL, "a slave is a master: the constraint sets are not closed");
    }
  }
  Guard g(cuda_device);
  if (!g.ok) return fail(nullptr, FE_MF_ECUDA, "cudaSetDevice failed (no CUDA device?): there is no CPU fallback");
  std::vector<double> zero_b;
  if (!inhomog && ns_total > 0) { zero_b.assign((size_t)ns_total, 0.0); inhomog = zero_b.data(); }
  fe_constraints* c = new (std::nothrow) fe_constraints;
  if (!c) return fail(nullptr, FE_MF_ENOMEM, "host allocation failed");
  c->ndof = ndof; c->nsets = nsets; c->nmasters = nm_total; c->nslaves = ns_total; c->device = cuda_device;
  cudaError_t e = upload(c->m_ptr, master_ptr, (size_t)nsets + 1);
  if (e == cudaSuccess) e = upload(c->s_ptr, slave_ptr, (size_t)nsets + 1);
  if (e == cudaSuccess) e = upload(c->w_ptr, w_ptr.data(), (size_t)nsets + 1);
  if (e == cudaSuccess) e = upload(c->masters, masters, (size_t)nm_total);
  if (e == cudaSuccess) e = upload(c->slaves, slaves, (size_t)ns_total);
  if (e == cudaSuccess) e = upload(c->weights, weights, (size_t)w_ptr[nsets]);
  if (e == cudaSuccess) e = upload(c->inhomog, inhomog, (size_t)ns_total);
  if (e != cudaSuccess) {
    const int code = e == cudaErrorMemoryAllocation ? FE_MF_ENOMEM : FE_MF_ECUDA;
    const std::string msg = std::string("device upload of the constraint sets: ") + cudaGetErrorString(e);
    release(c);
    delete c;
    return fail(nullptr, code, msg);
  }
  *out = c;
  return FE_MF_OK;
}

extern "C" int fe_constraints_create(fe_constraints** out, long long ndof, int nsets, const long long* master_ptr,
                                     const long long* masters, const long long* slave_ptr, const long long* slaves,
                                     const double* weights, const double* inhomog, int cuda_device) {
  try {
    return create_impl(out, ndof, nsets, master_ptr, masters, slave_ptr, slaves, weights, inhomog, cuda_device);
  } catch (const std::bad_alloc&) {
    if (out) *out = nullptr;
    return fail(nullptr, FE_MF_ENOMEM, "host allocation failed");
  } catch (...) {
    if (out) *out = nullptr;
    return fail(nullptr, FE_MF_EINVAL, "unexpected exception in fe_constraints_create");
  }
}

extern "C" int fe_constraints_distribute(fe_constraints* c, double* U_dev, int nvec, int homogeneous, void* cuda_stream) {
  if (int rc = check_call(c, U_dev, nvec)) return rc;
  if (c->nsets == 0) return FE_MF_OK;
  Guard g(c->device);
  if (!g.ok) return fail(c, FE_MF_ECUDA, "cudaSetDevice failed");
  const dim3 grid((unsigned)c->nsets, (unsigned)((nvec + kVecBlock - 1) / kVecBlock));
  fe_constraints_distribute_kernel<<<grid, kThreads, 0, (cudaStream_t)cuda_stream>>>(arrays(c), U_dev, nvec, homogeneous ? 1 : 0);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, FE_MF_ECUDA, std::string("fe_constraints_distribute: ") + cudaGetErrorString(e));
  return FE_MF_OK;
}

extern "C" int fe_constraints_distribute_transpose(fe_constraints* c, double* V_dev, int nvec, void* cuda_stream) {
  if (int rc = check_call(c, V_dev, nvec)) return rc;
  if (c->nsets == 0) return FE_MF_OK;
  Guard g(c->device);
  if (!g.ok) return fail(c, FE_MF_ECUDA, "cudaSetDevice failed");
  const dim3 grid((unsigned)c->nsets, (unsigned)((nvec + kVecBlock - 1) / kVecBlock));
  fe_constraints_transpose_kernel<<<grid, kThreads, 0, (cudaStream_t)cuda_stream>>>(arrays(c), V_dev, nvec);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, FE_MF_ECUDA, std::string("fe_constraints_distribute_transpose: ") + cudaGetErrorString(e));
  return FE_MF_OK;
}

extern "C" int fe_constraints_counts(const fe_constraints* c, int* nsets, long long* nmasters, long long* nslaves) {
  if (!c) return FE_MF_EINVAL;
  if (nsets) *nsets = c->nsets;
  if (nmasters) *nmasters = c->nmasters;
  if (nslaves) *nslaves = c->nslaves;
  return FE_MF_OK;
}

extern "C" const char* fe_constraints_last_error(const fe_constraints* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

extern "C" void fe_constraints_destroy(fe_constraints* c) {
  if (!c) return;
  {
    Guard g(c->device);
    release(c);
  }
  delete c;
}
