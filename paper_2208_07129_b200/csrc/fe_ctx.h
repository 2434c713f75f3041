// Host-side context of include/fe_mf.h and the launcher interface between the translation units of libfe_mf.so.
// fe_mf.cu (context, setup), fe_dispatch.cu (kernel selection, entry points) and one fe_tu_*.cu per kernel family;
// each kernel unit owns private copies of the constant-memory tables it reads and exports an upload function.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/fe_mf.h"
#include "fe_params.h"

struct fe_mf_ctx {
  int ncx, ncy, ncz, p, n, bc, geom;
  int zopen = 0;            // NEXT-4: bit 0 / 1 = the low / high z face is a cut plane of a decomposed mesh (fe_mf_create_slab)
  int ndx, ndy, ndz;
  long long ndof, ncells;
  double sigma;
  int device;
  int nsm = 148;
  int geom_mode;            // 0 uniform, 1 per-cell, 2 per-q-point
  double ug[7];
  double* geom_dev = nullptr;
  long long geom_stride = 7;   // doubles per cell in geom_dev
  // Control words of the persistent kernels (the dynamic item counter), zeroed on the stream before each launch.
  // kCtrlSlots slots of kCtrlWords words: slot 0 serves the caller's stream, slots 1 and 2 the two internal streams
  // of fe_mf_apply_host, so that launches on different streams never share a counter.
  static constexpr int kCtrlSlots = 3, kCtrlWords = 8;
  unsigned* ctrl = nullptr;
  int ctrl_slot = 0;
  // kappa at the quadrature points and the mass-scaled operator
  std::vector<double> verts;   // copy of vertices_host (empty: uniform box)
  double lo[3] = {0, 0, 0}, h[3] = {1, 1, 1};
  std::vector<double> detq;    // geom_mode 2: det J at the quadrature points [cell][n^3]
  double* dscale_dev = nullptr;   // diag(M)^-1/2 of the GLL-lumped mass matrix [ndof]
  std::vector<double> mass_diag;  // diag(M) [ndof] (host copy, filled with dscale_dev)
  bool mass_scaled = false;
  double* kappa_dev = nullptr;    // geom_mode 0: kappa at the quadrature points [cell][n^3] (set_kappa, or sigma everywhere
                                  // once mass scaling is on: the EIG kernels always read it)
  bool kappa_user = false;        // a caller-supplied kappa array is in force (any geometry mode)
  // n_q != n_p points per direction (0 = off): tables and per-point geometry of that rule
  int nq_oi = 0;
  double *oi_N = nullptr, *oi_D = nullptr, *oi_w = nullptr, *oi_geom = nullptr;
  long long oi_geom_stride = 0;
  std::vector<double> oi_detq;   // geom_mode 2: det J at the n_q^3 points [cell][nq^3]
  double detj0 = 1.0;             // geom_mode 0: det J of every cell
  int variant = 0;
  int last_launches = 0;
  // per-context (hence per-device) launcher state: the opted-in dynamic shared memory and the resident blocks per SM
  // of every kernel this context has launched, keyed by the kernel's address
  std::unordered_map<const void*, long long> kstate;
  // fe_mf_apply_host workspace
  double* ws_x = nullptr; double* ws_y = nullptr; size_t ws_elems = 0;
  cudaStream_t hs[3] = {nullptr, nullptr, nullptr};   // column-chunk path: two streams; slab path: H2D, kernels, D2H
  std::vector<cudaEvent_t> hev;                       // slab path: one "slab is on the device" and one "chunk is done" event per chunk
  std::string err;
};

namespace fe_host {

constexpr size_t kMaxSmem = 232448;  // 227 KB opt-in per block on sm_100

int fail(fe_mf_ctx* c, int code, const std::string& msg);

#define FE_CUDA(c, call)                                                                      \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess)                                                                    \
      return fe_host::fail((c), FE_MF_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
  } while (0)

struct DeviceGuard {
  int prev = -1; bool ok = false;
  explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess) ok = true; }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Opt a kernel in to `smem` bytes of dynamic shared memory once per context (i.e. per device).
template <typename Kern>
cudaError_t ensure_smem(fe_mf_ctx* c, Kern kern, size_t smem) {
  long long& have = c->kstate[(const void*)kern];
  if ((long long)smem > have) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    have = (long long)smem;
  }
  return cudaSuccess;
}

// Persistent kernels: grid = resident blocks (a multiple of the SM count), never more than the items.
template <typename Kern>
cudaError_t persistent_grid(fe_mf_ctx* c, Kern kern, int nt, size_t smem, long long nitems, long long& grid) {
  long long& bps = c->kstate[(const void*)kern];
  if (bps == 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int b = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, kern, nt, smem);
    if (e != cudaSuccess) return e;
    if (b < 1) return cudaErrorLaunchOutOfResources;
    bps = b;
  }
  grid = bps * c->nsm;
  if (grid > nitems) grid = nitems;
  return cudaSuccess;
}

inline int* item_counter(const fe_mf_ctx* c) { return reinterpret_cast<int*>(c->ctrl + c->ctrl_slot * fe_mf_ctx::kCtrlWords); }
inline cudaError_t reset_counter(const fe_mf_ctx* c, cudaStream_t st) {
  return cudaMemsetAsync(item_counter(c), 0, sizeof(unsigned) * fe_mf_ctx::kCtrlWords, st);
}

// ---- table uploads, one per kernel translation unit (current device)
cudaError_t upload_tables_misc(const fe::HostTables& t);
cudaError_t upload_tables_gen(const fe::HostTables& t);
cudaError_t upload_tables_plane(const fe::HostTables& t);
cudaError_t upload_tables_line16(const fe::HostTables& t);
cudaError_t upload_tables_line8(const fe::HostTables& t);
cudaError_t upload_tables_oi(const double* pack, size_t count, size_t offset_doubles);

// ---- launchers (each enqueues ONE kernel on st)
// fe_tu_misc.cu
cudaError_t launch_general(fe_mf_ctx* c, const fe::ApplyParams& P, cudaStream_t st);
cudaError_t launch_cart(fe_mf_ctx* c, const fe::ApplyParams& P, cudaStream_t st);
cudaError_t launch_cart_cells(fe_mf_ctx* c, const fe::ApplyParams& P, cudaStream_t st);
int general_bv(int p, int nvec);
cudaError_t launch_axpby(double* Z, const double* W, double beta, double gamma, size_t count, cudaStream_t st);
cudaError_t launch_scale_copy(double* Z, const double* W, double gamma, size_t count, cudaStream_t st);
cudaError_t launch_scale(double* Z, double beta, size_t count, cudaStream_t st);
cudaError_t launch_scale2(double* A, double* B, double sa, double sb, int swap, size_t count, int bnd, double qa, double qb,
                          int ndx, int ndy, int ndz, int nvec, cudaStream_t st);
cudaError_t launch_swap(double* A, double* B, size_t count, cudaStream_t st);
cudaError_t launch_fill_uniform(double* out, long long count, unsigned long long seed, long long offset, cudaStream_t st);
cudaError_t launch_halo_pack_f32(float* dst, const double* src, size_t count, cudaStream_t st);
cudaError_t launch_halo_unpack_f32(double* dst, const float* src, size_t count, int add, cudaStream_t st);
// fe_tu_gen.cu: full symmetric metric (per-q-point or per-cell geometry), TMA tiles
cudaError_t launch_gen(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap& tw, const CUtensorMap& tz, cudaStream_t st);
int gen_bv(const fe_mf_ctx* c, int nvec);
// fe_tu_plane.cu: uniform Cartesian cells, p = 6, one plane of one vector per thread
cudaError_t launch_plane(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap& tw, const CUtensorMap& tz, cudaStream_t st);
// fe_tu_line16.cu / fe_tu_line8.cu: uniform Cartesian cells, one line of two vectors per thread, 16 / 8 vectors per block
cudaError_t launch_line16(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap& tw, const CUtensorMap& tz, cudaStream_t st);
cudaError_t launch_line8(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap& tw, const CUtensorMap& tz, cudaStream_t st);
// fe_tu_oi.cu: n_q != n_p points per direction.  tw / tz may be NULL (no TMA)
cudaError_t launch_oi(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap* tw, const CUtensorMap* tz, cudaStream_t st);
int oi_bv(int nq, int nvec);
bool oi_compile_time_kernel(const fe_mf_ctx* c, int nvec);

// 8-vector (and 4-vector) blocks with an even number of nodes per direction: one pad node per x-row (see DenseTile)
constexpr int line_padx(int p, int bv) { return ((bv == 8 || bv == 4) && (p + 1) % 2 == 0 && p >= 3) ? 1 : 0; }

}  // namespace fe_host

#define FE_DISPATCH_P(CALL)                                           \
  switch (c->p) {                                                     \
    case 1: e = CALL(1); break; case 2: e = CALL(2); break;           \
    case 3: e = CALL(3); break; case 4: e = CALL(4); break;           \
    case 5: e = CALL(5); break; case 6: e = CALL(6); break;           \
    case 7: e = CALL(7); break; case 8: e = CALL(8); break;           \
  }
