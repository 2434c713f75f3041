// Plain structs shared by the host code and every kernel translation unit: kernel parameters, the layouts of the
// constant-memory tables and the host image of one degree's tables.  No CUDA code.
#pragma once
#include <cstddef>

namespace fe {

constexpr int KMAXN = 9;   // p <= 8

struct ApplyParams {
  const double* __restrict__ W;   // input multivector  [ndof][nvec]
  double* __restrict__ Z;         // output multivector [ndof][nvec], pre-initialised; Z += alpha*A*W
  const double* __restrict__ geom;  // per-q-point: [cell][7][n^3]; per-cell: [cell][7]; or nullptr (uniform); no w_Q factor
  double ug[7];                   // uniform Cartesian: G00,G01,G02,G11,G12,G22 (x det J), sigma*det J
  double alpha;
  int ncx, ncy, ncz;
  int ndx, ndy, ndz;
  int nvec;
  int bv;                         // vectors per block
  int nvb;                        // ceil(nvec / bv)
  int dirichlet;                  // 1: boundary nodes read as 0 / not written
  int zopen;                      // z-slab of a decomposed mesh: bit 0 / bit 1 = the low / high z face is
                                  // a CUT plane, not a boundary: no Dirichlet mask there and no periodic wrap in z (a periodic
                                  // slab has both bits set and ndz = ncz p + 1: its top plane is the ghost plane)
  int geom_mode;                  // 0 uniform (ug), 1 per-cell constants, 2 per-q-point
  int nsm;                        // SM count (persistent kernels)
  long long geom_stride;          // doubles per cell in geom (per-q-point: 7 n^3 rounded up to even; per-cell: 7)
  int* item_ctr;                  // persistent kernels: work counter (0 at launch); item = gridDim.x + atomicAdd after the first
  int item0, item_count;          // persistent kernels: the launch processes items item0 .. item0 + item_count - 1 of the
                                  // ncells * nvb items (cell-major: a range of cell layers); item_count = 0: all of them
  double idw;                     // Cartesian kernels with IDENT: Z += alpha A W + idw W
  const double* dscale;           // nullptr, or d = diag(M)^-1/2 [ndof] of the GLL-lumped mass matrix: Z += alpha d.(A (d.W))
                                  // (Eq. B.1; full-metric kernels only)
  const double* kappa;            // nullptr, or kappa at the quadrature points [cell][n^3] of a uniform box (geom_mode 0):
                                  // the mass factor is ug[6] * kappa_Q, ug[6] then holding det J without sigma
                                  // (general kernel, and the Cartesian kernels instantiated with EIG)
};

#if defined(__CUDACC__) || defined(FE_HOST_EMULATION)   // FE_HOST_EMULATION: tests/host/shim (device code on host threads)
// the z planes that the Dirichlet constraint masks (the physical boundary; a cut plane of a slab is not one)
__host__ __device__ inline bool fe_z_masked(const ApplyParams& P, int iz) {
  return (iz == 0 && !(P.zopen & 1)) || (iz == P.ndz - 1 && !(P.zopen & 2));
}
#endif

// The 4-D FP64 tensor map of a multivector [z][y][x][beta] with box (bv, n + padx, n, n), as plain numbers (host code
// hands them to cuTensorMapEncodeTiled: fe_dispatch.cu make_tensor_map).
// Dirichlet meshes (Cartesian kernels): trim = 2 -> the map covers nodes 1 .. nd-2 in every direction, origin at
// node (1,1,1), so that boundary nodes are out of bounds (zero on load; box coordinates shift by -1); trim = 1 ->
// nodes 0 .. nd-2, origin unchanged (the last node is clipped on reduce).  A cut plane of a slab (zopen, NEXT-4) is not
// a boundary: nothing is dropped there.
struct TensorMapDesc {
  unsigned long long base_offset;   // bytes from the multivector's first element to the map's origin
  unsigned long long dims[4];       // elements: beta, x, y, z
  unsigned long long strides[3];    // bytes: x, y, z
  unsigned box[4];
};
inline bool tensor_map_desc(TensorMapDesc& d, int ndx, int ndy, int ndz, int n, int zopen, int nvec, int bv, int trim, int padx) {
  if (trim && (ndx < 3 || ndy < 3 || ndz < 3)) return false;
  const int lo = (trim == 2) ? 1 : 0, hi = trim ? 1 : 0;   // nodes dropped at the low / high end of each direction
  const int loz = (zopen & 1) ? 0 : lo, hiz = (zopen & 2) ? 0 : hi;
  d.dims[0] = (unsigned long long)nvec;
  d.dims[1] = (unsigned long long)(ndx - lo - hi);
  d.dims[2] = (unsigned long long)(ndy - lo - hi);
  d.dims[3] = (unsigned long long)(ndz - loz - hiz);
  d.strides[0] = (unsigned long long)nvec * 8;
  d.strides[1] = (unsigned long long)nvec * 8 * ndx;
  d.strides[2] = (unsigned long long)nvec * 8 * ndx * ndy;
  if (d.strides[2] >= (1ULL << 40)) return false;
  d.base_offset = lo * d.strides[0] + lo * d.strides[1] + loz * d.strides[2];
  d.box[0] = (unsigned)bv; d.box[1] = (unsigned)(n + padx); d.box[2] = (unsigned)n; d.box[3] = (unsigned)n;
  return true;
}

// n_q != n_p Gauss points per direction
struct OiParams {
  int nq;                     // Gauss points per direction
  const double* Nq;           // [nq][n]   N[q][i] = l_i(xq_q)
  const double* Dq;           // [nq][nq]  D~[q][r] = l~_r'(xq_q)
  const double* wq;           // [nq]
  const double* geom;         // geom_mode 2: [cell][7][nq^3] (no w factor), else unused
  long long geom_stride;
};

// Half tables of one n x n matrix M with M[n-1-q][n-1-i] = s M[q][i] (s = +1 "sym", -1 "anti"); h = n/2.
//   P[q][i]  = (M[q][i] + M[q][n-1-i])/2   multiplies x+_i = x_i + x_{n-1-i}
//   Mn[q][i] = (M[q][i] - M[q][n-1-i])/2   multiplies x-_i = x_i - x_{n-1-i}
//   Pm[q]    = M[q][m]                      multiplies the middle entry (n odd)
//   mid[i]   = M[m][i] (i < h), midm = M[m][m]: the middle row (n odd)
// y_q = u + v, y_{n-1-q} = s (u - v) with u = P x+ + Pm x_m, v = Mn x-.
struct EoTab {
  double P[16];
  double Mn[16];
  double Pm[4];
  double mid[4];
  double midm;
  double pad[3];
};
enum { EO_NS = 0, EO_NST = 1, EO_DS = 2, EO_DST = 3, EO_SH = 4 };   // EO_SH: Ds^T Ds / 2 (symmetric type)

// The same with the halved middle column / row that the chained even/odd operators need (fe_kernels_plane.cuh)
struct EoTab2 {
  double P[16], Mn[16];
  double Pm[4], mid[4];
  double Pmh[4], midh[4];   // Pm / 2, mid / 2
  double midm, midmh;       // M[mid][mid] and half of it
  double pad[2];
};
enum { MAT_NS = 0, MAT_DS = 1, MAT_SH = 2, MAT_NSS = 3, MAT_COUNT = 4 };   // Ns, Ds, Ds^T Ds / 2 (symmetric type, like Ns),
                                                                           // Ns diag(w~)^-1/2 (mass-scaled interpolation, EIG)

// Host image of the tables of one degree p, uploaded into the constant memory of every kernel translation unit
// (each unit owns a private copy of the symbols it uses: the library is built without relocatable device code)
struct HostTables {
  int p;
  double N[KMAXN * KMAXN], D[KMAXN * KMAXN], w[KMAXN];
  EoTab eo[5];
  EoTab2 eo2[MAT_COUNT];
};

// Tables of the n_q = n_p + 2 rule, packed per degree at oi_offset(p) as even / odd halves: [Ne | No | De | Do]
constexpr int oi_size(int p) { return 2 * ((p + 4) / 2) * ((p + 2) / 2) + 2 * ((p + 4) / 2) * ((p + 4) / 2); }
template <int P_> struct OiOffset { static constexpr int value = OiOffset<P_ - 1>::value + oi_size(P_ - 1); };
template <> struct OiOffset<1> { static constexpr int value = 0; };
inline int oi_offset(int p) {
  int off = 0;
  for (int k = 1; k < p; ++k) off += oi_size(k);
  return off;
}

}  // namespace fe
