// Included by fe_mf.cu: kernel selection and the stream-ordered entry points.
//
// Kernels:
//   kind 8  fe_apply_cart_plane  uniform Cartesian cells, p = 6: one n x n plane of one vector per thread
//   kind 9  fe_apply_cart_line   uniform Cartesian cells, any p: one line of two vectors per thread
//   kind 6  fe_apply_gen_tma     full symmetric metric (per-q-point or per-cell geometry)
//   kind 2  fe_apply_cart        Cartesian, odd nvec or unaligned pointers (LDG gather / RED scatter)
//   kind 3  fe_apply_cart<CELLS> Cartesian, 1-3 vectors: the tile slots hold several cells of an x-row
//   kind 1  fe_apply_general     anything else (nvec = 1, odd nvec with a full metric): plain contractions
// fe_mf_set_variant forces a kind for tests and experiments: 1 -> kind 1, 2 -> kind 2, 7 -> kind 6 on a Cartesian
// mesh, 8 -> plane, 10 -> line with 16-vector blocks, 11 -> line with 8-vector blocks, 19 -> plane kernel that
// also initialises Z (fe_init_ahead.cuh; measured neutral, off by default).

namespace {

constexpr size_t kMaxSmem = 232448;  // 227 KB opt-in per block on sm_100

// ---- kind 1: general fallback, 4 tiles of n^3*bv doubles; keep >= 2 blocks per SM resident
int general_bv(int p, int nvec) {
  const int nn = (p + 1) * (p + 1) * (p + 1);
  int bv = 32;
  while (bv > 1 && ((size_t)4 * nn * bv * 8 > kMaxSmem / 2 - 1024 || bv > nvec)) bv >>= 1;
  return bv;
}

template <int PDEG>
cudaError_t launch_general(const fe::ApplyParams& prm, long long ncells, cudaStream_t st) {
  constexpr int NN = (PDEG + 1) * (PDEG + 1) * (PDEG + 1);
  const size_t smem = (size_t)4 * NN * prm.bv * sizeof(double);
  static size_t configured = 0;
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(fe::fe_apply_general<PDEG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  fe::fe_apply_general<PDEG><<<(unsigned)(ncells * prm.nvb), 256, smem, st>>>(prm);
  return cudaGetLastError();
}

// ---- kind 11: n_q != n_p points per direction (over-integration): plain kernel with rectangular tables
bool make_tensor_map(CUtensorMap* tm, const fe_mf_ctx* c, const void* base, int nvec, int bv, int trim, int padx);
int oi_bv(int nq, int nvec, int variant = 0) {
  // the compile-time kernel is instantiated for 2 and 4 vectors per block; 2 wherever three such blocks fit an SM
  int bv = ((size_t)3 * ((size_t)4 * nq * nq * nq * 2 * 8 + 4096) <= kMaxSmem || variant == 21 || variant == 22) ? 2 : 4;
  while (bv > 1 && ((size_t)4 * nq * nq * nq * bv * 8 > kMaxSmem / 2 - 4096 || bv > nvec)) bv >>= 1;
  return bv;
}
template <int PDEG>
cudaError_t launch_general_oi(const fe_mf_ctx* c, const fe::ApplyParams& prm, cudaStream_t st) {
  const int nq = c->nq_oi;
  fe::OiParams O{nq, c->oi_N, c->oi_D, c->oi_w, c->oi_geom, c->oi_geom_stride};
  const size_t smem = ((size_t)4 * nq * nq * nq * prm.bv + (size_t)nq * (PDEG + 1) + (size_t)nq * nq) * sizeof(double);
  static size_t configured = 0;
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(fe::fe_apply_general_oi<PDEG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  if (nq == PDEG + 3 && (prm.bv == 2 || prm.bv == 4)) {   // the paper's n_q = n_p + 2: compile-time sizes, line tasks
    // 2-vector blocks, three or four per SM, where four tiles fit that often (n_q <= 10 / n_q <= 9): measured faster
    // than two 4-vector blocks (p = 6: 25.4 -> 27.2 with three); variants 21 / 22 force three / two for comparison
    constexpr size_t TB2 = (size_t)4 * (PDEG + 3) * (PDEG + 3) * (PDEG + 3) * 2 * 8 + 4096;
    constexpr int MB = 4 * TB2 <= kMaxSmem ? 4 : (3 * TB2 <= kMaxSmem ? 3 : 2);
    const int mb = prm.bv != 2 ? 2 : (c->variant == 22 ? 2 : (c->variant == 21 ? (MB >= 3 ? 3 : 2) : MB));
    auto kern = prm.bv == 4 ? fe::fe_apply_oi<PDEG, PDEG + 3, 4>
              : mb == 4 ? fe::fe_apply_oi<PDEG, PDEG + 3, 2, MB == 4 ? 4 : 2>
              : mb == 3 ? fe::fe_apply_oi<PDEG, PDEG + 3, 2, MB >= 3 ? 3 : 2> : fe::fe_apply_oi<PDEG, PDEG + 3, 2>;
    static size_t configured2[4] = {0, 0, 0, 0};
    size_t& conf = configured2[prm.bv == 4 ? 0 : mb - 1];
    if (smem > conf) {
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e != cudaSuccess) return e;
      conf = smem;
    }
    // interior cells take their tile through TMA (same conditions as the other TMA kernels); the rest of the cells, and
    // calls that do not meet them, gather with loads and scatter with atomics inside the same kernel
    CUtensorMap tw, tz;
    memset(&tw, 0, sizeof(tw)); memset(&tz, 0, sizeof(tz));
    const bool aligned = ((((uintptr_t)prm.W) | ((uintptr_t)prm.Z)) & 15) == 0;
    const int use_tma = !(prm.nvec & 1) && aligned && c->variant != 1 &&
                        make_tensor_map(&tw, c, prm.W, prm.nvec, prm.bv, 0, 0) && make_tensor_map(&tz, c, prm.Z, prm.nvec, prm.bv, 0, 0);
    kern<<<(unsigned)(c->ncells * prm.nvb), 256, smem, st>>>(tw, tz, prm, O, use_tma);
    return cudaGetLastError();
  }
  fe::fe_apply_general_oi<PDEG><<<(unsigned)(c->ncells * prm.nvb), 256, smem, st>>>(prm, O);
  return cudaGetLastError();
}

// ---- kind 2: even-odd Cartesian kernel, one vector per thread, 8 vectors per block
template <int PDEG>
struct CartCfg {
  static constexpr int BV = 8, N = PDEG + 1;
  static constexpr int TASKS = N * N * BV;
  static constexpr int NT = (PDEG >= 5) ? TASKS / 2 : (TASKS < 32 ? 32 : TASKS);
  static constexpr size_t SMEM = (size_t)2 * fe::Tile<PDEG, BV>::SIZE * sizeof(double);
  static constexpr int BY_SMEM = (int)((kMaxSmem - 1024) / (SMEM + 1024));
  static constexpr int BY_THREADS = 2048 / NT;
  static constexpr int MINB0 = BY_SMEM < BY_THREADS ? BY_SMEM : BY_THREADS;
  static constexpr int MINB = MINB0 > 4 ? 4 : (MINB0 < 1 ? 1 : MINB0);
};

template <int PDEG>
cudaError_t launch_cart(const fe::ApplyParams& prm, long long ncells, cudaStream_t st) {
  using C = CartCfg<PDEG>;
  static bool configured = false;
  auto kern = fe::fe_apply_cart<PDEG, C::BV, C::NT, C::MINB>;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  kern<<<(unsigned)(ncells * prm.nvb), C::NT, C::SMEM, st>>>(prm);
  return cudaGetLastError();
}

// kind 3: the same kernel with the 8 tile slots holding 1-3 vectors of 8 / nvec consecutive cells of an x-row
template <int PDEG>
cudaError_t launch_cart_cells(const fe::ApplyParams& prm, const fe_mf_ctx* c, cudaStream_t st) {
  using C = CartCfg<PDEG>;
  static bool configured = false;
  auto kern = fe::fe_apply_cart<PDEG, C::BV, C::NT, C::MINB, true>;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  const int cb = C::BV / prm.nvec;                      // cells per block
  const long long groups = (c->ncx + cb - 1) / cb;
  const long long grid = groups * c->ncy * c->ncz;
  if (grid > 2147483647LL) return cudaErrorInvalidValue;
  kern<<<(unsigned)grid, C::NT, C::SMEM, st>>>(prm);
  return cudaGetLastError();
}

// ---- tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
    (void)cudaGetLastError();
  }
  return fn;
}

// 4-D FP64 tensor map of a multivector [z][y][x][beta] with box (bv, n, n, n).
// Dirichlet meshes (Cartesian kernels): trim = 2 -> the map covers nodes 1 .. nd-2 in every direction, origin at
// node (1,1,1), so that boundary nodes are out of bounds (zero on load; box coordinates shift by -1); trim = 1 ->
// nodes 0 .. nd-2, origin unchanged (the last node is clipped on reduce).
bool make_tensor_map(CUtensorMap* tm, const fe_mf_ctx* c, const void* base, int nvec, int bv, int trim = 0, int padx = 0) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  if (trim && (c->ndx < 3 || c->ndy < 3 || c->ndz < 3)) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)nvec, (cuuint64_t)(c->ndx - trim), (cuuint64_t)(c->ndy - trim), (cuuint64_t)(c->ndz - trim)};
  const cuuint64_t strides[3] = {(cuuint64_t)nvec * 8, (cuuint64_t)nvec * 8 * c->ndx, (cuuint64_t)nvec * 8 * c->ndx * c->ndy};
  if (strides[2] >= ((cuuint64_t)1 << 40)) return false;
  if (trim == 2) base = (const char*)base + (strides[0] + strides[1] + strides[2]);
  const cuuint32_t box[4] = {(cuuint32_t)bv, (cuuint32_t)(c->n + padx), (cuuint32_t)c->n, (cuuint32_t)c->n};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// ---- persistent kernels: grid = resident blocks; the work counter is zeroed on the stream before each launch
template <typename Kern>
cudaError_t persistent_grid(Kern kern, int nt, size_t smem, int& blocks_per_sm, const fe_mf_ctx* c, long long nitems,
                            long long& grid) {
  if (blocks_per_sm == 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, kern, nt, smem);
    if (e != cudaSuccess) return e;
    if (blocks_per_sm < 1) return cudaErrorLaunchOutOfResources;
  }
  grid = (long long)blocks_per_sm * c->nsm;
  if (grid > nitems) grid = nitems;
  return cudaSuccess;
}

// ---- kind 6: full symmetric metric
template <int PDEG> struct GenCfg;
template <> struct GenCfg<1> { static constexpr int BV = 8, NT = 32, MINB = 4; };
template <> struct GenCfg<2> { static constexpr int BV = 8, NT = 64, MINB = 4; };
template <> struct GenCfg<3> { static constexpr int BV = 8, NT = 64, MINB = 4; };
template <> struct GenCfg<4> { static constexpr int BV = 8, NT = 128, MINB = 3; };
template <> struct GenCfg<5> { static constexpr int BV = 8, NT = 160, MINB = 2; };
template <> struct GenCfg<6> { static constexpr int BV = 8, NT = 128, MINB = 3; };
template <> struct GenCfg<7> { static constexpr int BV = 8, NT = 256, MINB = 1; };
template <> struct GenCfg<8> { static constexpr int BV = 4, NT = 192, MINB = 2; };
constexpr int kGenBv = 8;

template <int PDEG, bool MSC = false>
cudaError_t launch_gen(const fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap& tw, const CUtensorMap& tz,
                       cudaStream_t st) {
  using C = GenCfg<PDEG>;
  constexpr int NN = (PDEG + 1) * (PDEG + 1) * (PDEG + 1);
  constexpr size_t SMEM = (size_t)3 * fe::DenseTile<PDEG, C::BV>::PITCH + ((size_t)7 * NN * 8 + 15) / 16 * 16 + 64;
  static int bps = 0;
  auto kern = fe::fe_apply_gen_tma<PDEG, C::BV, C::NT, C::MINB, MSC>;
  const long long nitems = c->ncells * prm.nvb;
  long long grid = 0;
  cudaError_t e = persistent_grid(kern, C::NT, SMEM, bps, c, nitems, grid);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->ctrl, 0, 16, st);
  if (e != cudaSuccess) return e;
  kern<<<(unsigned)grid, C::NT, SMEM, st>>>(tw, tz, prm, (int)nitems);
  return cudaGetLastError();
}

// ---- kind 8: plane kernel (one thread = one n x n plane of one vector), 16 vectors per block
template <int PDEG> struct PlaneCfg;
template <> struct PlaneCfg<6> { static constexpr int BV = 16, NT = 128, MINB = 2; };
template <> struct PlaneCfg<7> { static constexpr int BV = 16, NT = 128, MINB = 1; };   // spills; kept for comparison
bool plane_ok(int p) { return p == 6 || p == 7; }

template <int PDEG, int IM, bool IDENT = false, bool EIG = false>
cudaError_t launch_plane_im(fe_mf_ctx* c, const fe::ApplyParams& prm, fe::InitParams init, const CUtensorMap& tw,
                            const CUtensorMap& tz, cudaStream_t st) {
  using C = PlaneCfg<PDEG>;
  constexpr size_t SMEM = (size_t)2 * fe::DenseTile<PDEG, C::BV>::PITCH + 64 + fe::InitAhead<C::NT, IM>::STAGE_BYTES;
  static int bps = 0;
  auto kern = fe::fe_apply_cart_plane<PDEG, C::BV, C::NT, C::MINB, IM, IDENT, EIG>;
  long long grid = 0;
  int nitems = (int)(c->ncells * prm.nvb);
  cudaError_t e = persistent_grid(kern, C::NT, SMEM, bps, c, nitems, grid);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->ctrl, 0, IM == 0 ? 16 : c->ctrl_bytes, st);
  if (e != cudaSuccess) return e;
  if (IM == 0) {
    kern<<<(unsigned)grid, C::NT, SMEM, st>>>(tw, tz, prm, init, nitems);
    return cudaGetLastError();
  }
  // the blocks wait for one another's initialisation: they must all be resident (cooperative launch)
  init.slice_ctr = c->ctrl + 4;
  init.done = c->ctrl + 4 + c->ncz;
  void* args[] = {(void*)&tw, (void*)&tz, (void*)&prm, (void*)&init, (void*)&nitems};
  return cudaLaunchCooperativeKernel((const void*)kern, dim3((unsigned)grid), dim3(C::NT), args, SMEM, st);
}
template <int PDEG>
cudaError_t launch_plane(fe_mf_ctx* c, const fe::ApplyParams& prm, const fe::InitParams& init, const CUtensorMap& tw,
                         const CUtensorMap& tz, cudaStream_t st) {
  if (prm.kappa) {   // eigenproblem operator (EIG): never combined with the fused initialisation
    if (init.mode != fe::INIT_NONE) return cudaErrorInvalidValue;
    return prm.idw != 0.0 ? launch_plane_im<PDEG, 0, true, true>(c, prm, init, tw, tz, st)
                          : launch_plane_im<PDEG, 0, false, true>(c, prm, init, tw, tz, st);
  }
  if (init.mode == fe::INIT_NONE && prm.idw != 0.0) return launch_plane_im<PDEG, 0, true>(c, prm, init, tw, tz, st);
  if (init.mode == fe::INIT_NONE) return launch_plane_im<PDEG, 0>(c, prm, init, tw, tz, st);
  if (init.mode == fe::INIT_ZERO) return launch_plane_im<PDEG, 1>(c, prm, init, tw, tz, st);
  return launch_plane_im<PDEG, 2>(c, prm, init, tw, tz, st);
}

// ---- kind 9: line kernel (one thread = one line of two vectors)
template <int CFG> struct LineCfg;
template <> struct LineCfg<1> { static constexpr int BV = 16, NT = 32, MINB = 4; };
template <> struct LineCfg<2> { static constexpr int BV = 16, NT = 96, MINB = 4; };
template <> struct LineCfg<3> { static constexpr int BV = 16, NT = 128, MINB = 4; };
template <> struct LineCfg<4> { static constexpr int BV = 16, NT = 112, MINB = 4; };
template <> struct LineCfg<5> { static constexpr int BV = 16, NT = 160, MINB = 3; };
template <> struct LineCfg<6> { static constexpr int BV = 16, NT = 256, MINB = 2; };
template <> struct LineCfg<7> { static constexpr int BV = 16, NT = 256, MINB = 1; };
template <> struct LineCfg<8> { static constexpr int BV = 8, NT = 192, MINB = 2; };
// 8 vectors per block: calls with <= 8 vectors (no lanes wasted on the vector tail) and, for p = 7, always
// (three 8-vector blocks per SM beat one 16-vector block: 105 vs 99.6 GDoF*vec/s)
template <> struct LineCfg<101> { static constexpr int BV = 8, NT = 32, MINB = 4; };
template <> struct LineCfg<102> { static constexpr int BV = 8, NT = 64, MINB = 4; };
template <> struct LineCfg<103> { static constexpr int BV = 8, NT = 64, MINB = 4; };
template <> struct LineCfg<104> { static constexpr int BV = 8, NT = 128, MINB = 4; };
template <> struct LineCfg<105> { static constexpr int BV = 8, NT = 160, MINB = 4; };
template <> struct LineCfg<106> { static constexpr int BV = 8, NT = 128, MINB = 5; };
template <> struct LineCfg<107> { static constexpr int BV = 8, NT = 128, MINB = 3; };
int line_bv(const fe_mf_ctx* c, int nvec) {
  if (c->p == 8 || c->variant == 11 || nvec <= 8) return 8;
  if (c->p == 7 && c->variant != 10) return 8;
  return 16;
}

// 8-vector blocks with an even number of nodes per direction: one pad node per x-row (see DenseTile)
constexpr int line_padx(int p, int bv) { return ((bv == 8 || bv == 4) && (p + 1) % 2 == 0 && p >= 3) ? 1 : 0; }

template <int PDEG, int CFG, bool IDENT = false, bool EIG = false>
cudaError_t launch_line_id(const fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap& tw, const CUtensorMap& tz,
                        cudaStream_t st) {
  using C = LineCfg<CFG>;
  constexpr int PADX = line_padx(PDEG, C::BV);
  constexpr size_t SMEM = (size_t)2 * fe::DenseTile<PDEG, C::BV, PADX>::PITCH + 64;
  static int bps = 0;
  auto kern = fe::fe_apply_cart_line<PDEG, C::BV, C::NT, C::MINB, PADX, IDENT, EIG>;
  const long long nitems = c->ncells * prm.nvb;
  long long grid = 0;
  cudaError_t e = persistent_grid(kern, C::NT, SMEM, bps, c, nitems, grid);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->ctrl, 0, 16, st);
  if (e != cudaSuccess) return e;
  kern<<<(unsigned)grid, C::NT, SMEM, st>>>(tw, tz, prm, (int)nitems);
  return cudaGetLastError();
}

template <int PDEG, int CFG>
cudaError_t launch_line(const fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap& tw, const CUtensorMap& tz,
                        cudaStream_t st) {
  if (prm.kappa)
    return prm.idw != 0.0 ? launch_line_id<PDEG, CFG, true, true>(c, prm, tw, tz, st)
                          : launch_line_id<PDEG, CFG, false, true>(c, prm, tw, tz, st);
  return prm.idw != 0.0 ? launch_line_id<PDEG, CFG, true>(c, prm, tw, tz, st) : launch_line_id<PDEG, CFG, false>(c, prm, tw, tz, st);
}

// ---- kind 10: Kronecker kernel (uniform box, constant kappa): three tiles.  Variant 12 only: measured on the B200 it
// is no faster than the plane / line kernels (p = 6: 146 vs 144, p = 7: 121 vs 129 GDoF*vec/s; one vector per thread
// with twice the warps: 134 / 114) -- 25 % fewer FP64 instructions, but the same 10 tile accesses per point as the
// plane kernel and three short phases per item
template <int PDEG> struct KronCfg;
template <> struct KronCfg<1> { static constexpr int BV = 8, NT = 32, MINB = 4, VPT = 2; };
template <> struct KronCfg<2> { static constexpr int BV = 8, NT = 64, MINB = 4, VPT = 2; };
template <> struct KronCfg<3> { static constexpr int BV = 8, NT = 64, MINB = 4, VPT = 2; };
template <> struct KronCfg<4> { static constexpr int BV = 8, NT = 128, MINB = 4, VPT = 2; };
template <> struct KronCfg<5> { static constexpr int BV = 8, NT = 160, MINB = 4, VPT = 2; };
template <> struct KronCfg<6> { static constexpr int BV = 8, NT = 224, MINB = 2, VPT = 2; };
// p = 7, 8: the y-pass holds two lines and three products of two vectors (~150-160 registers): 4-vector blocks keep
// three / two blocks per SM resident without spills
template <> struct KronCfg<7> { static constexpr int BV = 4, NT = 128, MINB = 3, VPT = 2; };
template <> struct KronCfg<8> { static constexpr int BV = 4, NT = 192, MINB = 2, VPT = 2; };
int kron_bv(int p) { return p >= 7 ? 4 : 8; }

template <int PDEG, bool IDENT>
cudaError_t launch_kron_id(const fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap& tw, const CUtensorMap& tz,
                           cudaStream_t st) {
  using C = KronCfg<PDEG>;
  constexpr int BV = C::BV, PADX = line_padx(PDEG, BV);
  constexpr size_t SMEM = (size_t)3 * fe::DenseTile<PDEG, BV, PADX>::PITCH + 64;
  static int bps = 0;
  auto kern = fe::fe_apply_cart_kron<PDEG, BV, C::NT, C::MINB, PADX, IDENT, C::VPT>;
  const long long nitems = c->ncells * prm.nvb;
  long long grid = 0;
  cudaError_t e = persistent_grid(kern, C::NT, SMEM, bps, c, nitems, grid);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->ctrl, 0, 16, st);
  if (e != cudaSuccess) return e;
  kern<<<(unsigned)grid, C::NT, SMEM, st>>>(tw, tz, prm, (int)nitems);
  return cudaGetLastError();
}
template <int PDEG>
cudaError_t launch_kron(const fe_mf_ctx* c, const fe::ApplyParams& prm, const CUtensorMap& tw, const CUtensorMap& tz,
                        cudaStream_t st) {
  return prm.idw != 0.0 ? launch_kron_id<PDEG, true>(c, prm, tw, tz, st) : launch_kron_id<PDEG, false>(c, prm, tw, tz, st);
}

// ---- which kernel serves (ctx, nvec, pointers)
int pick_kernel(const fe_mf_ctx* c, int nvec, const void* W, const void* Z) {
  if (c->nq_oi) return 11;   // n_q != n_p: only the plain kernel with rectangular tables
  if (c->variant == 1) return 1;
  // NEXT-1 operator: a uniform box with mass scaling runs on the Cartesian TMA kernels instantiated with EIG (kappa per
  // point, M^-1/2 inside the interpolation tables); kappa without mass scaling on such a context only on the general
  // kernel; every other mesh on the full-metric kernels (kinds 6, 1), which read d = diag(M)^-1/2 from memory
  const bool msc = c->mass_scaled;
  const bool eig = msc && c->geom_mode == 0;
  if (c->kappa_dev && !msc) return 1;
  const bool diag = (!msc || eig) && (c->geom_mode == 0) && c->ug[1] == 0.0 && c->ug[2] == 0.0 && c->ug[4] == 0.0;
  const bool aligned = ((((uintptr_t)W) | ((uintptr_t)Z)) & 15) == 0;
  const bool tma_ok = !(nvec & 1) && aligned && encode_tiled_fn() &&
                      (unsigned long long)nvec * 8ULL * c->ndx * c->ndy < (1ULL << 40) &&
                      c->ncells * ((nvec + 7) / 8) < (1LL << 31);
  const bool trim_ok = (c->bc != FE_BC_DIRICHLET) || (c->ndx >= 3 && c->ndy >= 3 && c->ndz >= 3);
  if (eig) {   // kinds 8 / 9 or the general kernel (which then reads d and kappa from memory)
    if (!tma_ok || !trim_ok || nvec < 4 || c->variant == 2 || c->variant == 7) return 1;
  } else {
    if ((!diag || c->variant == 7) && tma_ok) return 6;
    if (!diag) return 1;
    if (nvec < 4) return 3;
    if (!tma_ok || c->variant == 2) return 2;
    if (!trim_ok) return 2;
  }
  if (c->variant == 12 && !eig) return 10;
  if (c->variant == 10 || c->variant == 11) return 9;
  if ((c->variant == 8 || c->variant == 19) && plane_ok(c->p)) return 8;
  // plane kernel: 16 vectors per block; worth it when the last block of vectors is mostly full
  const int tail = nvec % 16;
  if (c->p == 6 && nvec >= 12 && (tail == 0 || tail >= 12)) return 8;
  return 9;
}
int kernel_bv(const fe_mf_ctx* c, int kind, int nvec) {
  switch (kind) {
    case 1: return general_bv(c->p, nvec);
    case 2: return 8;
    case 3: return nvec;
    case 6: return c->p == 8 ? 4 : kGenBv;
    case 8: return 16;
    case 10: return kron_bv(c->p);
    case 11: return oi_bv(c->nq_oi, nvec, c->variant);
    default: return line_bv(c, nvec);
  }
}

fe::ApplyParams make_params(const fe_mf_ctx* c, const double* W, double* Z, double alpha, int nvec, int bv) {
  fe::ApplyParams P;
  P.W = W; P.Z = Z; P.geom = c->geom_dev;
  for (int k = 0; k < 7; ++k) P.ug[k] = c->ug[k];
  P.alpha = alpha;
  P.ncx = c->ncx; P.ncy = c->ncy; P.ncz = c->ncz;
  P.ndx = c->ndx; P.ndy = c->ndy; P.ndz = c->ndz;
  P.nvec = nvec; P.bv = bv; P.nvb = (nvec + bv - 1) / bv;
  P.dirichlet = (c->bc == FE_BC_DIRICHLET) ? 1 : 0;
  P.geom_mode = c->geom_mode;
  P.nsm = c->nsm;
  P.geom_stride = c->geom_stride;
  P.item_ctr = reinterpret_cast<int*>(c->ctrl);
  P.idw = 0.0;
  P.dscale = c->mass_scaled ? c->dscale_dev : nullptr;
  P.kappa = c->kappa_dev;
  if (P.kappa) P.ug[6] = c->detj0;   // mass factor = det J * kappa_Q
  return P;
}

// Can this kernel kind initialise Z itself?  (plane kernel, cooperative launch, 32-bit chunk sizes; opt-in)
bool kind_fuses_init(const fe_mf_ctx* c, int kind, int nvec) {
  const long long chunk2 = (long long)(c->p + 1) * c->ndx * c->ndy * nvec / 2;   // double2 elements of the largest chunk
  return kind == 8 && c->coop && c->variant == 19 && chunk2 < (1LL << 31) && !c->kappa_dev;
}

// Can this kernel add a multiple of W (identity term, partition-of-unity weights) in the same pass?  The Cartesian
// plane and line kernels, at every node they write: all nodes on periodic meshes, the interior nodes on Dirichlet
// meshes (the boundary nodes never enter a tile: callers treat them separately).
bool kind_adds_identity(const fe_mf_ctx* c, int kind) { return (kind == 8 && c->p == 6) || kind == 9 || kind == 10; }

#define FE_DISPATCH_P(CALL)                                           \
  switch (c->p) {                                                     \
    case 1: e = CALL(1); break; case 2: e = CALL(2); break;           \
    case 3: e = CALL(3); break; case 4: e = CALL(4); break;           \
    case 5: e = CALL(5); break; case 6: e = CALL(6); break;           \
    case 7: e = CALL(7); break; case 8: e = CALL(8); break;           \
  }

// Z += alpha * A * W  (Z already initialised), or with init.mode != INIT_NONE (only if kind_fuses_init):
// Z <- beta Z + gamma W + alpha A W in ONE launch.  Counts launches into c->last_launches.
// idw != 0 (only if kind_adds_identity): Z += alpha A W + idw W in one launch.
int launch_accumulate(fe_mf_ctx* c, double alpha, const double* W, double* Z, int nvec, cudaStream_t st,
                      fe::InitParams init = fe::InitParams{fe::INIT_NONE, 0.0, 0.0, nullptr, nullptr}, double idw = 0.0) {
  const int kind = pick_kernel(c, nvec, W, Z);
  const int bv = kernel_bv(c, kind, nvec);
  fe::ApplyParams P = make_params(c, W, Z, alpha, nvec, bv);
  P.idw = idw;
  if (c->ncells * (long long)P.nvb > 2147483647LL) return fail(c, FE_MF_EINVAL, "grid too large");
  cudaError_t e = cudaErrorInvalidValue;
  CUtensorMap tw, tz;
  if (kind == 6 || kind == 8 || kind == 9 || kind == 10) {
    // Cartesian kernels on Dirichlet meshes: boundary nodes are out of bounds of the maps (see make_tensor_map)
    const bool trim = (kind != 6) && (c->bc == FE_BC_DIRICHLET);
    const int padx = (kind == 9 || kind == 10) ? line_padx(c->p, bv) : 0;
    if (!make_tensor_map(&tw, c, W, nvec, bv, trim ? 2 : 0, padx) || !make_tensor_map(&tz, c, Z, nvec, bv, trim ? 1 : 0, padx))
      return fail(c, FE_MF_ECUDA, "cuTensorMapEncodeTiled failed");
  }
  if (kind == 8 || kind == 9 || kind == 10 || kind == 2 || kind == 3)
    for (int k = 0; k < 7; ++k) P.ug[k] *= alpha;   // Cartesian kernels: the result is linear in the metric constants
  if ((kind == 8 || kind == 9) && c->mass_scaled) {
    // EIG kernels: diag(M)^-1/2 = (det J)^-1/2 kron diag(w~)^-1/2; the tables carry the second factor (both sides)
    for (int k = 0; k < 7; ++k) P.ug[k] /= c->detj0;
    P.dscale = nullptr;
  }
  if (kind == 11) {
#define FE_CALL(p_) launch_general_oi<p_>(c, P, st)
    FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  } else if (kind == 6 && P.dscale) {
#define FE_CALL(p_) launch_gen<p_, true>(c, P, tw, tz, st)
    FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  } else if (kind == 6) {
#define FE_CALL(p_) launch_gen<p_>(c, P, tw, tz, st)
    FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  } else if (kind == 10) {
#define FE_CALL(p_) launch_kron<p_>(c, P, tw, tz, st)
    FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  } else if (kind == 8) {
    e = (c->p == 6) ? launch_plane<6>(c, P, init, tw, tz, st) : launch_plane<7>(c, P, init, tw, tz, st);
  } else if (kind == 9) {
    if (bv == 16) {
#define FE_CALL(p_) launch_line<p_, p_>(c, P, tw, tz, st)
      FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
    } else if (c->p == 8) {
      e = launch_line<8, 8>(c, P, tw, tz, st);
    } else {
#define FE_CALL(p_) launch_line<p_, 100 + p_>(c, P, tw, tz, st)
      switch (c->p) {
        case 1: e = FE_CALL(1); break; case 2: e = FE_CALL(2); break; case 3: e = FE_CALL(3); break;
        case 4: e = FE_CALL(4); break; case 5: e = FE_CALL(5); break; case 6: e = FE_CALL(6); break;
        case 7: e = FE_CALL(7); break;
      }
#undef FE_CALL
    }
  } else if (kind == 3) {
    P.alpha = 1.0;
#define FE_CALL(p_) launch_cart_cells<p_>(P, c, st)
    FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  } else if (kind == 2) {
    P.alpha = 1.0;
#define FE_CALL(p_) launch_cart<p_>(P, c->ncells, st)
    FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  } else {
#define FE_CALL(p_) launch_general<p_>(P, c->ncells, st)
    FE_DISPATCH_P(FE_CALL)
#undef FE_CALL
  }
  if (e != cudaSuccess) return fail(c, FE_MF_ECUDA, std::string("apply kernel launch: ") + cudaGetErrorString(e));
  c->last_launches += 1;
  return FE_MF_OK;
}

int stream_grid(size_t count) {
  size_t b = (count + 255) / 256;
  if (b > 148 * 16) b = 148 * 16;
  if (b < 1) b = 1;
  return (int)b;
}

// Z <- beta*Z + gamma*W, stream-ordered (S1 / the axpby half of S9).
int launch_init(fe_mf_ctx* c, double* Z, const double* W, double beta, double gamma, size_t count, cudaStream_t st) {
  if (beta == 0.0 && gamma == 0.0) {
    FE_CUDA(c, cudaMemsetAsync(Z, 0, count * sizeof(double), st));   // a driver memset: not counted as a kernel launch
    return FE_MF_OK;
  }
  if (beta == 0.0) fe::fe_scale_copy_kernel<<<stream_grid(count), 256, 0, st>>>(Z, W, gamma, count);
  else fe::fe_axpby_kernel<<<stream_grid(count / 2 + 1), 256, 0, st>>>(Z, W, beta, gamma, count);
  FE_CUDA(c, cudaGetLastError());
  c->last_launches += 1;
  return FE_MF_OK;
}

int check_io(fe_mf_ctx* c, const double* W, const double* Z, int nvec) {
  if (!c) return FE_MF_EINVAL;
  if (!W || !Z) return fail(c, FE_MF_EINVAL, "null device pointer");
  if (nvec < 1) return fail(c, FE_MF_EINVAL, "nvec must be >= 1");
  const size_t bytes = (size_t)c->ndof * nvec * sizeof(double);
  const char* a = (const char*)W; const char* b = (const char*)Z;
  if (a < b + bytes && b < a + bytes) return fail(c, FE_MF_EINVAL, "input and output alias");
  return FE_MF_OK;
}

}  // namespace

extern "C" int fe_mf_apply_axpby(fe_mf_ctx* ctx, double alpha, const double* W_dev, double beta, double gamma,
                                 double* Z_dev, int nvec, void* cuda_stream) {
  int rc = check_io(ctx, W_dev, Z_dev, nvec);
  if (rc) return rc;
  DeviceGuard guard(ctx->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  ctx->last_launches = 0;
  const size_t count = (size_t)ctx->ndof * nvec;
  const int kind = pick_kernel(ctx, nvec, W_dev, Z_dev);
  if (kind_fuses_init(ctx, kind, nvec)) {   // S1 folded into the apply kernel (fe_init_ahead.cuh): one launch
    fe::InitParams init{beta == 0.0 ? (gamma == 0.0 ? fe::INIT_ZERO : fe::INIT_SCALE) : fe::INIT_AXPBY, beta, gamma, nullptr, nullptr};
    return launch_accumulate(ctx, alpha, W_dev, Z_dev, nvec, st, init);
  }
  if (kind_adds_identity(ctx, kind) && gamma != 0.0 && ctx->bc == FE_BC_PERIODIC) {
    // the kernel adds gamma W itself (IDENT): the separate pass only has to scale Z (or zero it)
    if (beta == 0.0) {
      FE_CUDA(ctx, cudaMemsetAsync(Z_dev, 0, count * sizeof(double), st));
    } else if (beta != 1.0) {
      fe::fe_scale_kernel<<<stream_grid(count / 2 + 1), 256, 0, st>>>(Z_dev, beta, count);
      FE_CUDA(ctx, cudaGetLastError());
      ctx->last_launches += 1;
    }
    return launch_accumulate(ctx, alpha, W_dev, Z_dev, nvec, st, fe::InitParams{fe::INIT_NONE, 0.0, 0.0, nullptr, nullptr}, gamma);
  }
  rc = launch_init(ctx, Z_dev, W_dev, beta, gamma, count, st);
  if (rc) return rc;
  return launch_accumulate(ctx, alpha, W_dev, Z_dev, nvec, st);
}

extern "C" int fe_mf_accumulate(fe_mf_ctx* ctx, double alpha, const double* W_dev, double* Z_dev, int nvec,
                                void* cuda_stream) {
  int rc = check_io(ctx, W_dev, Z_dev, nvec);
  if (rc) return rc;
  DeviceGuard guard(ctx->device);
  ctx->last_launches = 0;
  return launch_accumulate(ctx, alpha, W_dev, Z_dev, nvec, (cudaStream_t)cuda_stream);
}

extern "C" int fe_mf_apply(fe_mf_ctx* ctx, const double* X_dev, double* Y_dev, int nvec, void* cuda_stream) {
  return fe_mf_apply_axpby(ctx, 1.0, X_dev, 0.0, 0.0, Y_dev, nvec, cuda_stream);
}

extern "C" int fe_cheb_filter(fe_mf_ctx* ctx, double* X_dev, double* Y_dev, int nvec, int m, double a, double b,
                              double a0, void* cuda_stream) {
  int rc = check_io(ctx, X_dev, Y_dev, nvec);
  if (rc) return rc;
  if (m < 1) return fail(ctx, FE_MF_EINVAL, "m must be >= 1");
  if (!(b > a)) return fail(ctx, FE_MF_EINVAL, "need b > a (inverted or empty damping interval)");
  if (!(a0 < a)) return fail(ctx, FE_MF_EINVAL, "need a0 < a");
  DeviceGuard guard(ctx->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t count = (size_t)ctx->ndof * nvec;
  int launches = 0;
  // Alg. 6 lines 2-9 (garbled lines per DESIGN.md reading 10)
  const double e = (b - a) / 2.0;
  const double c = (b + a) / 2.0;
  double sigma = e / (a0 - c);
  const double sigma1 = sigma;
  const double gamma = 2.0 / sigma1;
  double alpha1 = sigma1 / e;
  double alpha2 = -c;
  double* X = X_dev; double* Y = Y_dev;
  if (m <= 200 && c != 0.0 && kind_adds_identity(ctx, pick_kernel(ctx, nvec, X_dev, Y_dev))) {
    // The same recurrence, X_1 = a_0 (A - cI) X_0, X_{k+1} = a_k (A - cI) X_k + b_k X_{k-1}  (a_0 = sigma_1/e,
    // a_k = 2 sigma_2/e, b_k = -sigma sigma_2), in the scaled variables X_k = s_k U_k with s_0 = s_1 = 1,
    // s_{k+1} = b_k s_{k-1}:   U_{k+1} = U_{k-1} + (a_k s_k / s_{k+1}) (A - cI) U_k.
    // Every step is then ONE accumulate launch into the buffer of U_{k-1} (the plane kernel adds the -cI part with
    // partition-of-unity weights): no axpby pass.  s_m and s_{m-1} are applied once at the end.  (|s_k| shrinks
    // like |b|^(k/2); m <= 200 keeps it far from underflow.)  Dirichlet meshes: the kernels neither read nor write
    // the boundary nodes, whose entries obey the scalar recurrence with A = 0 (q_k); X_dev keeps the input there
    // until the final kernel writes q_m x0 and q_{m-1} x0.
    const fe::InitParams none{fe::INIT_NONE, 0.0, 0.0, nullptr, nullptr};
    FE_CUDA(ctx, cudaMemsetAsync(Y, 0, count * sizeof(double), st));
    ctx->last_launches = 0;
    rc = launch_accumulate(ctx, alpha1, X, Y, nvec, st, none, -c * alpha1);
    if (rc) return rc;
    launches += ctx->last_launches;
    double s_prev = 1.0, s_cur = 1.0;
    double q_prev = 1.0, q_cur = -c * alpha1;   // the same recurrence at a boundary node of a Dirichlet mesh: (A X) = 0 there
    double* Uprev = X; double* Ucur = Y;
    for (int d = 2; d <= m; ++d) {
      const double sigma2 = 1.0 / (gamma - sigma);
      alpha1 = 2.0 * sigma2 / e;
      alpha2 = -sigma * sigma2;
      const double s_next = alpha2 * s_prev;
      const double al = alpha1 * s_cur / s_next;
      const double q_next = -c * alpha1 * q_cur + alpha2 * q_prev;
      q_prev = q_cur; q_cur = q_next;
      ctx->last_launches = 0;
      rc = launch_accumulate(ctx, al, Ucur, Uprev, nvec, st, none, -c * al);
      if (rc) return rc;
      launches += ctx->last_launches;
      double* t = Uprev; Uprev = Ucur; Ucur = t;
      s_prev = s_cur; s_cur = s_next;
      sigma = sigma2;
    }
    // Y_dev <- s_m U_m, X_dev <- s_{m-1} U_{m-1}
    const int swap = (Ucur != Y_dev) ? 1 : 0;
    const int bnd = (ctx->bc == FE_BC_DIRICHLET) ? 1 : 0;
    if (swap || bnd || s_cur != 1.0 || s_prev != 1.0) {
      fe::fe_scale2_kernel<<<stream_grid(count), 256, 0, st>>>(X_dev, Y_dev, s_prev, s_cur, swap, count, bnd, q_prev, q_cur,
                                                               ctx->ndx, ctx->ndy, ctx->ndz, nvec);
      FE_CUDA(ctx, cudaGetLastError());
      launches += 1;
    }
    ctx->last_launches = launches;
    return FE_MF_OK;
  }
  // line 10: Y <- alpha1 A X + alpha1 alpha2 X
  rc = fe_mf_apply_axpby(ctx, alpha1, X, 0.0, alpha1 * alpha2, Y, nvec, cuda_stream);
  if (rc) return rc;
  launches += ctx->last_launches;
  for (int d = 2; d <= m; ++d) {
    const double sigma2 = 1.0 / (gamma - sigma);
    alpha1 = 2.0 * sigma2 / e;
    alpha2 = -sigma * sigma2;
    // line 15: X <- alpha1 A Y + alpha2 X - c alpha1 Y ; line 16: swap
    rc = fe_mf_apply_axpby(ctx, alpha1, Y, alpha2, -(c * alpha1), X, nvec, cuda_stream);
    if (rc) return rc;
    launches += ctx->last_launches;
    double* t = X; X = Y; Y = t;
    sigma = sigma2;
  }
  if (Y != Y_dev) {  // m even: the result sits in the caller's X buffer; exchange contents
    fe::fe_swap_kernel<<<stream_grid(count), 256, 0, st>>>(X_dev, Y_dev, count);
    FE_CUDA(ctx, cudaGetLastError());
    launches += 1;
  }
  ctx->last_launches = launches;
  return FE_MF_OK;
}

extern "C" int fe_mf_apply_host(fe_mf_ctx* ctx, const double* X_host, double* Y_host, int nvec) {
  if (!ctx) return FE_MF_EINVAL;
  if (!X_host || !Y_host) return fail(ctx, FE_MF_EINVAL, "null host pointer");
  if (nvec < 1) return fail(ctx, FE_MF_EINVAL, "nvec must be >= 1");
  DeviceGuard guard(ctx->device);
  // column chunks: copies of chunk k+1 / k-1 overlap the kernels of chunk k on two streams
  // (at least 16 columns = 128-byte rows per chunk: strided host copies with 64-byte rows ran at half the rate;
  // measured on config 2: 1 chunk 42 ms, 2 chunks of 16 columns 30 ms, 4 chunks of 8 columns 43 ms)
  int cw = (nvec + 3) / 4;
  if (cw < 16) cw = 16;
  cw = (cw + 3) / 4 * 4;
  if (cw > nvec) cw = nvec;
  const int nchunks = (nvec + cw - 1) / cw;
  const size_t per = (size_t)ctx->ndof * cw;
  const int nbuf = nchunks > 1 ? 2 : 1;
  if (ctx->ws_elems < per * nbuf) {
    if (ctx->ws_x) cudaFree(ctx->ws_x);
    if (ctx->ws_y) cudaFree(ctx->ws_y);
    ctx->ws_x = ctx->ws_y = nullptr; ctx->ws_elems = 0;
    if (cudaMalloc(&ctx->ws_x, per * nbuf * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&ctx->ws_y, per * nbuf * sizeof(double)) != cudaSuccess) {
      if (ctx->ws_x) cudaFree(ctx->ws_x);
      ctx->ws_x = nullptr; (void)cudaGetLastError();
      return fail(ctx, FE_MF_ENOMEM, "device workspace allocation failed");
    }
    ctx->ws_elems = per * nbuf;
  }
  for (int i = 0; i < 2; ++i)
    if (!ctx->hs[i]) FE_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->hs[i], cudaStreamNonBlocking));
  int launches = 0;
  for (int k = 0; k < nchunks; ++k) {
    const int c0 = k * cw, w = (c0 + cw <= nvec) ? cw : (nvec - c0);
    cudaStream_t st = ctx->hs[k & 1];
    double* dx = ctx->ws_x + (size_t)(k % nbuf) * per;
    double* dy = ctx->ws_y + (size_t)(k % nbuf) * per;
    FE_CUDA(ctx, cudaMemcpy2DAsync(dx, (size_t)w * 8, X_host + c0, (size_t)nvec * 8, (size_t)w * 8, (size_t)ctx->ndof,
                                   cudaMemcpyHostToDevice, st));
    int rc = fe_mf_apply(ctx, dx, dy, w, st);
    if (rc) return rc;
    launches += ctx->last_launches;
    FE_CUDA(ctx, cudaMemcpy2DAsync(Y_host + c0, (size_t)nvec * 8, dy, (size_t)w * 8, (size_t)w * 8, (size_t)ctx->ndof,
                                   cudaMemcpyDeviceToHost, st));
  }
  FE_CUDA(ctx, cudaStreamSynchronize(ctx->hs[0]));
  FE_CUDA(ctx, cudaStreamSynchronize(ctx->hs[1]));
  ctx->last_launches = launches;
  return FE_MF_OK;
}

extern "C" int fe_fill_uniform(double* out_dev, long long count, unsigned long long seed, long long offset,
                               void* cuda_stream) {
  if (!out_dev || count < 0) return FE_MF_EINVAL;
  if (count == 0) return FE_MF_OK;
  fe::fe_fill_uniform_kernel<<<stream_grid((size_t)count), 256, 0, (cudaStream_t)cuda_stream>>>(out_dev, count, seed, offset);
  return cudaGetLastError() == cudaSuccess ? FE_MF_OK : FE_MF_ECUDA;
}

extern "C" int fe_mf_batch_width(const fe_mf_ctx* ctx, int nvec) {
  if (!ctx || nvec < 1) return -1;
  const int kind = pick_kernel(ctx, nvec, nullptr, nullptr);
  return kernel_bv(ctx, kind, nvec);
}

extern "C" const char* fe_mf_kernel_name(const fe_mf_ctx* ctx, int nvec) {
  if (!ctx || nvec < 1) return "";
  switch (pick_kernel(ctx, nvec, nullptr, nullptr)) {
    case 1: return "fe_apply_general";
    case 2: return "fe_apply_cart";
    case 3: return "fe_apply_cart<CELLS>";
    case 6: return "fe_apply_gen_tma";
    case 8: return "fe_apply_cart_plane";
    case 10: return "fe_apply_cart_kron";
    case 11: return (ctx->nq_oi == ctx->p + 3 && oi_bv(ctx->nq_oi, nvec) >= 2) ? "fe_apply_oi" : "fe_apply_general_oi";
    default: return "fe_apply_cart_line";
  }
}

extern "C" int fe_mf_last_launch_count(const fe_mf_ctx* ctx) { return ctx ? ctx->last_launches : -1; }

extern "C" int fe_mf_set_variant(fe_mf_ctx* ctx, int variant) {
  if (!ctx) return FE_MF_EINVAL;
  const bool known = variant == 0 || variant == 1 || variant == 2 || variant == 7 || variant == 8 || variant == 10 ||
                     variant == 11 || variant == 12 || variant == 19 || variant == 21 || variant == 22;
  if (!known) return fail(ctx, FE_MF_EINVAL, "unknown kernel variant");
  ctx->variant = variant;
  return FE_MF_OK;
}
