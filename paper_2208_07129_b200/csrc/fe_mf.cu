// C-ABI of include/fe_mf.h: context, host-side setup, kernel dispatch.  sm_100a only.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "fe_ctx.h"
#include "fe_tables.h"
#include "fe_eo_tables.h"
#include "fe_oi_tables.h"

static thread_local std::string g_create_err = "";

namespace fe_host {
int fail(fe_mf_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_err = msg;
  return code;
}
}  // namespace fe_host

using fe_host::fail;
using fe_host::DeviceGuard;
using fe_host::make_eo_tables;

namespace {

void cell_vertices(const fe_mf_ctx* c, const double* verts, const double lo[3], const double h[3], int ex, int ey,
                   int ez, double v[8][3]) {
  for (int k = 0; k < 8; ++k) {
    int vx = ex + (k & 1), vy = ey + ((k >> 1) & 1), vz = ez + ((k >> 2) & 1);
    if (verts) {
      const double* s = verts + 3 * ((size_t)vx + (size_t)(c->ncx + 1) * ((size_t)vy + (size_t)(c->ncy + 1) * vz));
      v[k][0] = s[0]; v[k][1] = s[1]; v[k][2] = s[2];
    } else {
      v[k][0] = lo[0] + h[0] * vx; v[k][1] = lo[1] + h[1] * vy; v[k][2] = lo[2] + h[2] * vz;
    }
  }
}

}  // namespace

static int create_impl(fe_mf_ctx** out, int ncx, int ncy, int ncz, int p, double sigma, int bc, int geom,
                       const double box_lo[3], const double box_hi[3], const double* vertices_host,
                       int cuda_device, int zopen) {
  if (!out) return fail(nullptr, FE_MF_EINVAL, "out is NULL");
  *out = nullptr;
  if (ncx < 1 || ncy < 1 || ncz < 1) return fail(nullptr, FE_MF_EINVAL, "cells per direction must be >= 1");
  if (p < 1 || p > 8) return fail(nullptr, FE_MF_EINVAL, "p must be in 1..8");
  if (bc != FE_BC_PERIODIC && bc != FE_BC_DIRICHLET) return fail(nullptr, FE_MF_EINVAL, "unknown bc");
  if (geom != FE_GEOM_AFFINE && geom != FE_GEOM_QPOINT) return fail(nullptr, FE_MF_EINVAL, "unknown geom");
  if (zopen < 0 || zopen > 3 || (bc == FE_BC_PERIODIC && zopen != 0 && zopen != 3))
    return fail(nullptr, FE_MF_EINVAL, "z_open must be 0..3; a periodic slab is cut at both z faces (3)");
  if (bc == FE_BC_PERIODIC && (ncx < 2 || ncy < 2 || (ncz < 2 && !zopen)))
    return fail(nullptr, FE_MF_EINVAL, "periodic needs >= 2 cells per direction");
  if (!vertices_host) {
    if (!box_lo || !box_hi) return fail(nullptr, FE_MF_EINVAL, "box_lo/box_hi are NULL");
    for (int d = 0; d < 3; ++d)
      if (!(box_hi[d] > box_lo[d])) return fail(nullptr, FE_MF_EINVAL, "box_hi must exceed box_lo");
  }
  if ((long long)ncx * p + 1 > 2000000 || (long long)ncy * p + 1 > 2000000 || (long long)ncz * p + 1 > 2000000)
    return fail(nullptr, FE_MF_EINVAL, "mesh too large");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev)
    return fail(nullptr, FE_MF_ECUDA, "no such CUDA device (this library has no CPU fallback)");
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return fail(nullptr, FE_MF_ECUDA, "cudaGetDeviceProperties failed");
  if (prop.major != 10) return fail(nullptr, FE_MF_EUNSUPPORTED, "device is not sm_100 (Blackwell B200)");

  fe_mf_ctx* c = new (std::nothrow) fe_mf_ctx();
  if (!c) return fail(nullptr, FE_MF_ENOMEM, "out of host memory");
  c->ncx = ncx; c->ncy = ncy; c->ncz = ncz; c->p = p; c->n = p + 1; c->bc = bc; c->geom = geom;
  const int add = (bc == FE_BC_DIRICHLET) ? 1 : 0;
  c->zopen = zopen;
  c->ndx = ncx * p + add; c->ndy = ncy * p + add; c->ndz = ncz * p + (zopen ? 1 : add);   // a slab carries its top (ghost) plane
  c->ndof = (long long)c->ndx * c->ndy * c->ndz;
  c->ncells = (long long)ncx * ncy * ncz;
  c->sigma = sigma; c->device = cuda_device; c->nsm = prop.multiProcessorCount;

  DeviceGuard guard(cuda_device);
  if (!guard.ok) { delete c; return fail(nullptr, FE_MF_ECUDA, "cudaSetDevice failed"); }

  const fe::Tables1D tab = fe::make_tables(p);
  const int n = p + 1, nn = n * n * n;
  cudaError_t e;
  {
    // the tables are functions of p only: every context of degree p uploads the same values into slot p of the
    // constant-memory arrays of each kernel translation unit (of the current device)
    fe::HostTables ht;
    std::memset(&ht, 0, sizeof(ht));
    ht.p = p;
    std::memcpy(ht.N, tab.N, sizeof(double) * n * n);
    std::memcpy(ht.D, tab.Dt, sizeof(double) * n * n);
    std::memcpy(ht.w, tab.w, sizeof(double) * n);
    make_eo_tables(tab, ht.eo, ht.eo2);
    e = fe_host::upload_tables_misc(ht);
    if (e == cudaSuccess) e = fe_host::upload_tables_gen(ht);
    if (e == cudaSuccess) e = fe_host::upload_tables_plane(ht);
    if (e == cudaSuccess) e = fe_host::upload_tables_line16(ht);
    if (e == cudaSuccess) e = fe_host::upload_tables_line8(ht);
  }
  if (e != cudaSuccess) { delete c; return fail(nullptr, FE_MF_ECUDA, std::string("table upload: ") + cudaGetErrorString(e)); }

  double lo[3] = {0, 0, 0}, h[3] = {1, 1, 1};
  if (!vertices_host) {
    const int nc[3] = {ncx, ncy, ncz};
    for (int d = 0; d < 3; ++d) { lo[d] = box_lo[d]; h[d] = (box_hi[d] - box_lo[d]) / nc[d]; }
  }
  for (int d = 0; d < 3; ++d) { c->lo[d] = lo[d]; c->h[d] = h[d]; }
  if (vertices_host) {
    try { c->verts.assign(vertices_host, vertices_host + 3 * (size_t)(ncx + 1) * (ncy + 1) * (ncz + 1)); }
    catch (...) { delete c; return fail(nullptr, FE_MF_ENOMEM, "out of host memory (vertices)"); }
  }
  const double centre[3] = {0.0, 0.0, 0.0};
  if (!vertices_host && geom == FE_GEOM_AFFINE) {
    c->geom_mode = 0;
    double v[8][3], J[3][3];
    cell_vertices(c, nullptr, lo, h, 0, 0, 0, v);
    fe::trilinear_jacobian(v, centre, J);
    if (!fe::metric_from_jacobian(J, c->ug)) { delete c; return fail(nullptr, FE_MF_EINVAL, "non-positive det J"); }
    c->detj0 = c->ug[6];
    c->ug[6] *= sigma;
    e = cudaMalloc(&c->geom_dev, 7 * sizeof(double));   // the general TMA kernel reads the uniform metric from memory
    if (e == cudaSuccess) e = cudaMemcpy(c->geom_dev, c->ug, 7 * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { if (c->geom_dev) cudaFree(c->geom_dev); delete c; return fail(nullptr, FE_MF_ECUDA, std::string("geometry upload: ") + cudaGetErrorString(e)); }
  } else {
    const bool perq = (geom == FE_GEOM_QPOINT);
    c->geom_mode = perq ? 2 : 1;
    const size_t per_cell = perq ? (((size_t)7 * nn + 1) & ~(size_t)1) : 7;   // even: 16-byte bulk copies
    c->geom_stride = (long long)per_cell;
    std::vector<double> G;
    try { G.resize(per_cell * (size_t)c->ncells); if (perq) c->detq.resize((size_t)nn * c->ncells); }
    catch (...) { delete c; return fail(nullptr, FE_MF_ENOMEM, "out of host memory (geometry)"); }
    bool bad = false;
    for (int ez = 0; ez < ncz; ++ez)
      for (int ey = 0; ey < ncy; ++ey)
        for (int ex = 0; ex < ncx; ++ex) {
          double v[8][3], J[3][3], m[7];
          cell_vertices(c, vertices_host, lo, h, ex, ey, ez, v);
          const size_t cell = (size_t)ex + (size_t)ncx * ((size_t)ey + (size_t)ncy * ez);
          double* g = G.data() + cell * per_cell;
          if (!perq) {
            fe::trilinear_jacobian(v, centre, J);
            if (!fe::metric_from_jacobian(J, m)) { bad = true; continue; }
            for (int k = 0; k < 6; ++k) g[k] = m[k];
            g[6] = sigma * m[6];
          } else {
            for (int q3 = 0; q3 < n; ++q3)
              for (int q2 = 0; q2 < n; ++q2)
                for (int q1 = 0; q1 < n; ++q1) {
                  const double xi[3] = {tab.xq[q1], tab.xq[q2], tab.xq[q3]};
                  fe::trilinear_jacobian(v, xi, J);
                  if (!fe::metric_from_jacobian(J, m)) { bad = true; continue; }
                  const int Q = q1 + n * (q2 + n * q3);
                  for (int k = 0; k < 6; ++k) g[(size_t)k * nn + Q] = m[k];
                  g[(size_t)6 * nn + Q] = sigma * m[6];
                  c->detq[cell * nn + Q] = m[6];
                }
          }
        }
    if (bad) { delete c; return fail(nullptr, FE_MF_EINVAL, "non-positive det J at a quadrature point"); }
    e = cudaMalloc(&c->geom_dev, G.size() * sizeof(double));
    if (e != cudaSuccess) { delete c; return fail(nullptr, FE_MF_ENOMEM, std::string("geometry cudaMalloc: ") + cudaGetErrorString(e)); }
    e = cudaMemcpy(c->geom_dev, G.data(), G.size() * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(c->geom_dev); delete c; return fail(nullptr, FE_MF_ECUDA, std::string("geometry upload: ") + cudaGetErrorString(e)); }
  }
  if (cudaMalloc(&c->ctrl, sizeof(unsigned) * fe_mf_ctx::kCtrlSlots * fe_mf_ctx::kCtrlWords) != cudaSuccess) {
    cudaFree(c->geom_dev); delete c;
    return fail(nullptr, FE_MF_ENOMEM, "cudaMalloc (control words) failed");
  }
  *out = c;
  return FE_MF_OK;
}

extern "C" int fe_mf_create(fe_mf_ctx** out, int ncx, int ncy, int ncz, int p, double sigma, int bc, int geom,
                            const double box_lo[3], const double box_hi[3], const double* vertices_host,
                            int cuda_device) {
  return create_impl(out, ncx, ncy, ncz, p, sigma, bc, geom, box_lo, box_hi, vertices_host, cuda_device, 0);
}

extern "C" int fe_mf_create_slab(fe_mf_ctx** out, int ncx, int ncy, int ncz, int p, double sigma, int bc, int geom,
                                 const double box_lo[3], const double box_hi[3], const double* vertices_host,
                                 int z_open, int cuda_device) {
  return create_impl(out, ncx, ncy, ncz, p, sigma, bc, geom, box_lo, box_hi, vertices_host, cuda_device, z_open);
}

extern "C" long long fe_mf_ndofs(const fe_mf_ctx* ctx) { return ctx ? ctx->ndof : -1; }

extern "C" int fe_mf_shape(const fe_mf_ctx* ctx, int nd[3], int* bc, int* cuda_device) {
  if (!ctx) return FE_MF_EINVAL;
  if (nd) { nd[0] = ctx->ndx; nd[1] = ctx->ndy; nd[2] = ctx->ndz; }
  if (bc) *bc = ctx->bc;
  if (cuda_device) *cuda_device = ctx->device;
  return FE_MF_OK;
}

extern "C" const char* fe_mf_last_error(const fe_mf_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

extern "C" void fe_mf_destroy(fe_mf_ctx* ctx) {
  if (!ctx) return;
  DeviceGuard guard(ctx->device);
  if (ctx->geom_dev) cudaFree(ctx->geom_dev);
  if (ctx->ctrl) cudaFree(ctx->ctrl);
  if (ctx->dscale_dev) cudaFree(ctx->dscale_dev);
  if (ctx->kappa_dev) cudaFree(ctx->kappa_dev);
  { double* b[] = {ctx->oi_N, ctx->oi_D, ctx->oi_w, ctx->oi_geom}; for (double* q : b) if (q) cudaFree(q); }
  if (ctx->ws_x) cudaFree(ctx->ws_x);
  if (ctx->ws_y) cudaFree(ctx->ws_y);
  for (cudaStream_t s_ : ctx->hs) if (s_) cudaStreamDestroy(s_);
  for (cudaEvent_t ev : ctx->hev) if (ev) cudaEventDestroy(ev);
  delete ctx;
}

// ---- kappa(x) at the quadrature points, GLL-lumped mass scaling ---------------------------

extern "C" int fe_mf_set_kappa(fe_mf_ctx* ctx, const double* kappa_host) {
  if (!ctx) return FE_MF_EINVAL;
  if (ctx->geom_mode == 1)
    return fail(ctx, FE_MF_EINVAL, "fe_mf_set_kappa needs a uniform box or a context created with FE_GEOM_QPOINT");
  DeviceGuard guard(ctx->device);
  if (!guard.ok) return fail(ctx, FE_MF_ECUDA, "cudaSetDevice failed");
  const int nqe = ctx->nq_oi ? ctx->nq_oi : ctx->n;   // points per direction of the current rule
  const size_t nn = (size_t)nqe * nqe * nqe, total = nn * (size_t)ctx->ncells;
  if (ctx->geom_mode == 0) {   // uniform box: the raw kappa array, read by the EIG kernels and the general kernel
    FE_CUDA(ctx, cudaDeviceSynchronize());
    ctx->kappa_user = kappa_host != nullptr;
    if (!kappa_host && !ctx->mass_scaled) {
      if (ctx->kappa_dev) cudaFree(ctx->kappa_dev);
      ctx->kappa_dev = nullptr;
      return FE_MF_OK;
    }
    if (!ctx->kappa_dev && cudaMalloc(&ctx->kappa_dev, total * sizeof(double)) != cudaSuccess) {
      ctx->kappa_dev = nullptr;
      return fail(ctx, FE_MF_ENOMEM, "cudaMalloc (kappa) failed");
    }
    if (kappa_host) {
      FE_CUDA(ctx, cudaMemcpy(ctx->kappa_dev, kappa_host, total * sizeof(double), cudaMemcpyHostToDevice));
    } else {
      std::vector<double> k0;
      try { k0.assign(total, ctx->sigma); } catch (...) { return fail(ctx, FE_MF_ENOMEM, "out of host memory (kappa)"); }
      FE_CUDA(ctx, cudaMemcpy(ctx->kappa_dev, k0.data(), total * sizeof(double), cudaMemcpyHostToDevice));
    }
    return FE_MF_OK;
  }
  std::vector<double> g;
  try { g.resize(total); } catch (...) { return fail(ctx, FE_MF_ENOMEM, "out of host memory (kappa)"); }
  // G_QQ = kappa_Q det J; the weight w_Q lives in the sqrt(w)-scaled 1D tables
  const std::vector<double>& det = ctx->nq_oi ? ctx->oi_detq : ctx->detq;
  for (size_t i = 0; i < total; ++i) g[i] = (kappa_host ? kappa_host[i] : ctx->sigma) * det[i];
  FE_CUDA(ctx, cudaDeviceSynchronize());
  double* gdst = ctx->nq_oi ? ctx->oi_geom : ctx->geom_dev;
  const size_t gstride = (size_t)(ctx->nq_oi ? ctx->oi_geom_stride : ctx->geom_stride);
  FE_CUDA(ctx, cudaMemcpy2D(gdst + 6 * nn, gstride * sizeof(double), g.data(), nn * sizeof(double),
                            nn * sizeof(double), (size_t)ctx->ncells, cudaMemcpyHostToDevice));
  ctx->kappa_user = kappa_host != nullptr;
  return FE_MF_OK;
}

// ---- n_q != n_p Gauss points per direction ------------------------------------------------------

extern "C" int fe_mf_set_quadrature(fe_mf_ctx* ctx, int nq) {
  if (!ctx) return FE_MF_EINVAL;
  if (nq < ctx->n || nq > 12) return fail(ctx, FE_MF_EINVAL, "need p + 1 <= nq <= 12");
  DeviceGuard guard(ctx->device);
  if (!guard.ok) return fail(ctx, FE_MF_ECUDA, "cudaSetDevice failed");
  FE_CUDA(ctx, cudaDeviceSynchronize());
  // A kappa array belongs to the points of one rule: back to the constant sigma.  On a per-q-point context the
  // caller's kappa sits inside the default rule's factors (slot 6 of geom_dev): rewrite them BEFORE the rule changes,
  // otherwise the old kappa would silently come back with nq = p + 1.
  if (ctx->geom_mode == 2 && ctx->kappa_user && !ctx->nq_oi) {
    const int rc = fe_mf_set_kappa(ctx, nullptr);
    if (rc != FE_MF_OK) return rc;
  }
  { double** b[] = {&ctx->oi_N, &ctx->oi_D, &ctx->oi_w, &ctx->oi_geom}; for (double** q : b) if (*q) { cudaFree(*q); *q = nullptr; } }
  ctx->oi_detq.clear();
  ctx->nq_oi = (nq == ctx->n) ? 0 : nq;
  ctx->kappa_user = false;
  if (ctx->geom_mode == 0) {
    if (ctx->kappa_dev) { cudaFree(ctx->kappa_dev); ctx->kappa_dev = nullptr; }
    if (ctx->mass_scaled && !ctx->nq_oi) { const int rc = fe_mf_set_kappa(ctx, nullptr); if (rc != FE_MF_OK) return rc; }
  }
  if (!ctx->nq_oi) return FE_MF_OK;
  const int n = ctx->n;
  // tables of the nq-point rule (fe_oi_tables.h): N[q][i] = l_i(xq_q) on the GLL nodes, D~ on the quadrature points
  fe_host::OiTables oit;
  try { fe_host::make_oi_tables(ctx->p, nq, oit); }
  catch (...) { ctx->nq_oi = 0; return fail(ctx, FE_MF_ENOMEM, "out of host memory (quadrature tables)"); }
  const std::vector<double>&hN = oit.N, &hD = oit.D, &hw = oit.w;
  const long double* xq = oit.xq;
  auto upload = [&](double** dst, const std::vector<double>& src) {
    if (cudaMalloc(dst, src.size() * sizeof(double)) != cudaSuccess) { *dst = nullptr; return false; }
    return cudaMemcpy(*dst, src.data(), src.size() * sizeof(double), cudaMemcpyHostToDevice) == cudaSuccess;
  };
  if (!upload(&ctx->oi_N, hN) || !upload(&ctx->oi_D, hD) || !upload(&ctx->oi_w, hw)) {
    ctx->nq_oi = 0;
    return fail(ctx, FE_MF_ENOMEM, "table upload failed (quadrature)");
  }
  if (nq == ctx->p + 3)   // the compile-time kernel of n_q = n_p + 2 reads its tables (even / odd halves) from constant memory
    FE_CUDA(ctx, fe_host::upload_tables_oi(oit.pack.data(), oit.pack.size(), (size_t)fe::oi_offset(ctx->p)));
  if (ctx->geom_mode == 2) {   // per-point metric at the nq^3 points (Eq. 7c evaluated at every point of the rule)
    const size_t nn = (size_t)nq * nq * nq;
    ctx->oi_geom_stride = (long long)(7 * nn);
    std::vector<double> G;
    try { G.resize(7 * nn * (size_t)ctx->ncells); ctx->oi_detq.resize(nn * (size_t)ctx->ncells); }
    catch (...) { ctx->nq_oi = 0; return fail(ctx, FE_MF_ENOMEM, "out of host memory (geometry)"); }
    const double* verts = ctx->verts.empty() ? nullptr : ctx->verts.data();
    for (int ez = 0; ez < ctx->ncz; ++ez)
      for (int ey = 0; ey < ctx->ncy; ++ey)
        for (int ex = 0; ex < ctx->ncx; ++ex) {
          double v[8][3], J[3][3], m[7];
          cell_vertices(ctx, verts, ctx->lo, ctx->h, ex, ey, ez, v);
          const size_t cell = (size_t)ex + (size_t)ctx->ncx * ((size_t)ey + (size_t)ctx->ncy * ez);
          double* g = G.data() + cell * 7 * nn;
          for (int q3 = 0; q3 < nq; ++q3)
            for (int q2 = 0; q2 < nq; ++q2)
              for (int q1 = 0; q1 < nq; ++q1) {
                const double x3[3] = {(double)xq[q1], (double)xq[q2], (double)xq[q3]};
                fe::trilinear_jacobian(v, x3, J);
                if (!fe::metric_from_jacobian(J, m)) { ctx->nq_oi = 0; return fail(ctx, FE_MF_EINVAL, "non-positive det J at a quadrature point"); }
                const size_t Q = (size_t)q1 + (size_t)nq * (q2 + (size_t)nq * q3);
                for (int k = 0; k < 6; ++k) g[(size_t)k * nn + Q] = m[k];
                g[6 * nn + Q] = ctx->sigma * m[6];
                ctx->oi_detq[cell * nn + Q] = m[6];
              }
        }
    if (!upload(&ctx->oi_geom, G)) { ctx->nq_oi = 0; return fail(ctx, FE_MF_ENOMEM, "geometry upload failed (quadrature)"); }
  }
  return FE_MF_OK;
}

namespace {

// diag(M) by the (p+1)-point Gauss-Lobatto-Legendre rule on the nodes:
// M_ii = sum over cells containing node i of det J(xi_i) w_i1 w_i2 w_i3, w = 2 / (p (p+1) P_p(xi)^2)
int build_mass_diagonal(fe_mf_ctx* c) {
  const int p = c->p, n = c->n;
  long double xl[fe::MAXN], wl[fe::MAXN];
  fe::gll_nodes(p, xl);
  for (int i = 0; i < n; ++i) {
    long double pn, pm;
    fe::legendre(p, xl[i], pn, pm);
    wl[i] = 2.0L / ((long double)p * (p + 1) * pn * pn);
  }
  double w[fe::MAXN], x[fe::MAXN];
  for (int i = 0; i < n; ++i) { w[i] = (double)(0.5L * (wl[i] + wl[n - 1 - i])); x[i] = (double)xl[i]; }
  try { c->mass_diag.assign((size_t)c->ndof, 0.0); } catch (...) { return fail(c, FE_MF_ENOMEM, "out of host memory (mass diagonal)"); }
  const double* verts = c->verts.empty() ? nullptr : c->verts.data();
  for (int ez = 0; ez < c->ncz; ++ez)
    for (int ey = 0; ey < c->ncy; ++ey)
      for (int ex = 0; ex < c->ncx; ++ex) {
        double v[8][3], J[3][3], m[7];
        cell_vertices(c, verts, c->lo, c->h, ex, ey, ez, v);
        for (int i3 = 0; i3 < n; ++i3)
          for (int i2 = 0; i2 < n; ++i2)
            for (int i1 = 0; i1 < n; ++i1) {
              const double xi[3] = {x[i1], x[i2], x[i3]};
              fe::trilinear_jacobian(v, xi, J);
              if (!fe::metric_from_jacobian(J, m)) return fail(c, FE_MF_EINVAL, "non-positive det J at a node");
              int ix = ex * p + i1, iy = ey * p + i2, iz = ez * p + i3;
              if (ix >= c->ndx) ix -= c->ndx;
              if (iy >= c->ndy) iy -= c->ndy;
              if (iz >= c->ndz) iz -= c->ndz;
              c->mass_diag[(size_t)ix + (size_t)c->ndx * ((size_t)iy + (size_t)c->ndy * iz)] += m[6] * (w[i1] * w[i2] * w[i3]);
            }
      }
  std::vector<double> d;
  try { d.resize((size_t)c->ndof); } catch (...) { return fail(c, FE_MF_ENOMEM, "out of host memory (mass diagonal)"); }
  for (size_t i = 0; i < d.size(); ++i) d[i] = 1.0 / std::sqrt(c->mass_diag[i]);
  if (cudaMalloc(&c->dscale_dev, d.size() * sizeof(double)) != cudaSuccess) {
    c->dscale_dev = nullptr; c->mass_diag.clear();
    return fail(c, FE_MF_ENOMEM, "cudaMalloc (mass scaling) failed");
  }
  FE_CUDA(c, cudaMemcpy(c->dscale_dev, d.data(), d.size() * sizeof(double), cudaMemcpyHostToDevice));
  return FE_MF_OK;
}

}  // namespace

extern "C" int fe_mf_set_mass_scaling(fe_mf_ctx* ctx, int on) {
  if (!ctx) return FE_MF_EINVAL;
  if (ctx->zopen) return fail(ctx, FE_MF_EUNSUPPORTED, "mass scaling on a slab context: diag(M) at a cut plane needs the neighbour's cells");
  DeviceGuard guard(ctx->device);
  if (!guard.ok) return fail(ctx, FE_MF_ECUDA, "cudaSetDevice failed");
  FE_CUDA(ctx, cudaDeviceSynchronize());
  if (on && !ctx->dscale_dev) {
    const int rc = build_mass_diagonal(ctx);
    if (rc != FE_MF_OK) return rc;
  }
  ctx->mass_scaled = on != 0;
  if (ctx->geom_mode == 0) {
    // the EIG kernels read kappa per point: constant sigma becomes an array while the scaling is on
    if (on && !ctx->kappa_dev && !ctx->nq_oi) return fe_mf_set_kappa(ctx, nullptr);
    if (!on && ctx->kappa_dev && !ctx->kappa_user) { cudaFree(ctx->kappa_dev); ctx->kappa_dev = nullptr; }
  }
  return FE_MF_OK;
}

extern "C" int fe_mf_mass_diagonal(fe_mf_ctx* ctx, double* out_host) {
  if (!ctx) return FE_MF_EINVAL;
  if (ctx->zopen) return fail(ctx, FE_MF_EUNSUPPORTED, "mass diagonal of a slab context: a cut plane needs the neighbour's cells");
  if (!out_host) return fail(ctx, FE_MF_EINVAL, "out_host is NULL");
  DeviceGuard guard(ctx->device);
  if (!guard.ok) return fail(ctx, FE_MF_ECUDA, "cudaSetDevice failed");
  if (!ctx->dscale_dev) {
    const int rc = build_mass_diagonal(ctx);
    if (rc != FE_MF_OK) return rc;
  }
  std::memcpy(out_host, ctx->mass_diag.data(), sizeof(double) * (size_t)ctx->ndof);
  return FE_MF_OK;
}

