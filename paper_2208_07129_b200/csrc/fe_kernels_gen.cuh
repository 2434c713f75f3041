// Device code, part 5: persistent TMA kernel for a full symmetric metric (per-q-point geometry of config 3,
// or one sheared metric per cell).  Same ingredients as fe_apply_cart_tma (even-odd, sqrt(w)-scaled tables,
// two vectors per thread, TMA gather + TMA f64 reduce, persistent blocks) but the three reference gradients
// couple at every quadrature point (Alg. 2 line 5; Eq. 8), so three tiles are live:
//
//   ph0 x : A <- Ns_x A            ph1 y : A <- Ns_y A
//   ph2 z : T = Ns_z A -> A ; T2 = Ds_z T -> C
//   ph3 x : T0 = Ds_x T -> B
//   ph4 y : T1 = Ds_y T (registers); S = G (T0,T1,T2), Sm = g T at each point;
//           R = Sm + Ds_y^T S1 -> A ; S0 -> B ; S2 -> C
//   ph5 x : R += Ds_x^T S0 -> A    (B free: prefetch the next item's tile into B)
//   ph6 z : R += Ds_z^T S2 ; A <- Ns_z^T R
//   ph7 y : A <- Ns_y^T A          ph8 x : A <- Ns_x^T A ; TMA reduce-add A -> Z
//
// 25 thread tile accesses per point + 2 by the TMA unit.  The tile roles rotate (A,B,C) <- (B,C,A) per item.
// The cell's geometric factors (7 n^3 doubles, or 7 constants) are staged in shared memory by one bulk copy
// (cp.async.bulk, mbarrier-tracked) issued one item ahead, so that ph4 never waits on global memory.
#pragma once
#include "fe_kernels_tma.cuh"

namespace fe {

// d at the N nodes of x-line l = i2 + N i3 of cell (ex,ey,ez), periodic indices wrapped
template <int PDEG>
__device__ __forceinline__ void load_dscale(const ApplyParams& P, int ex, int ey, int ez, int l, double* dn) {
  constexpr int N = PDEG + 1;
  int iy = ey * PDEG + l % N, iz = ez * PDEG + l / N;
  if (iy >= P.ndy) iy -= P.ndy;
  if (iz >= P.ndz) iz -= P.ndz;
  const double* src = P.dscale + (long long)P.ndx * ((long long)iy + (long long)P.ndy * iz);
  const int x0 = ex * PDEG;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    int ix = x0 + i;
    if (ix >= P.ndx) ix -= P.ndx;
    dn[i] = __ldg(src + ix);
  }
}

// MSC: the mass-scaled operator Z += alpha d.(A (d.W)), d = diag(M)^-1/2 of the GLL-lumped mass matrix
// (PAPER.md:925-929), applied where the paper applies it -- at extraction and assembly: ph0 scales
// the x-lines it reads, ph8 the x-lines it writes; d is read through L2 (one value per node, shared by all vectors).
template <int PDEG, int BV, int NT, int MINB, bool MSC>
__global__ void __launch_bounds__(NT, MINB)
fe_apply_gen_tma(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmZ,
                 const __grid_constant__ ApplyParams P, int nitems) {
  using TL = DenseTile<PDEG, BV>;
  constexpr int N = PDEG + 1, NN = N * N * N, NL = N * N, TPL = BV / 2, TASKS = NL * TPL;
  constexpr int ROUNDS = (TASKS + NT - 1) / NT;
  constexpr bool ROTATE = (NT % 32 == 0) && (NT >= 128);
  constexpr int NW = NT / 32;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* A = reinterpret_cast<double*>(smem_raw);
  double* B = reinterpret_cast<double*>(smem_raw + TL::PITCH);
  double* C = reinterpret_cast<double*>(smem_raw + 2 * TL::PITCH);
  constexpr int GBYTES = ((7 * NN * 8) + 15) / 16 * 16;
  double* GS = reinterpret_cast<double*>(smem_raw + 3 * TL::PITCH);
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 3 * TL::PITCH + GBYTES);
  uint64_t* gbar = bar + 1;
  int* s_next = reinterpret_cast<int*>(bar + 2);
  const bool perq = (P.geom_mode == 2);
  const int tid = threadIdx.x;
  const long long nvec = P.nvec;
  const bool dirichlet = P.dirichlet != 0;
  const double alpha = P.alpha;

  if (tid == 0) {
    mbar_init(bar, 1);
    mbar_init(gbar, 1);
    mbar_init_fence();
  }
  __syncthreads();

  int item = blockIdx.x;
  if (tid == 0 && item < nitems) {
    const int vb = (item + P.item0) % P.nvb, cell = (item + P.item0) / P.nvb;
    const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
    mbar_expect_tx(bar, TL::BYTES);
    tma_load_4d(A, &tmW, bar, vb * BV, ex * PDEG, ey * PDEG, ez * PDEG);
    if (perq) {
      mbar_expect_tx(gbar, GBYTES);
      bulk_load(GS, P.geom + (size_t)cell * P.geom_stride, GBYTES, gbar);
    }
  }
  uint32_t parity = 0, gparity = 0;
  int rot = (blockIdx.x / P.nsm) & 3;
  // items are handed out dynamically after the first one (co-resident blocks do not run at the same speed)
  for (; item < nitems; rot = (rot + 1) & 3) {
    unsigned nxt_raw = 0;
    if (tid == 0) nxt_raw = item_counter_next(P.item_ctr);
    const int rot_tid = ROTATE ? ((((tid >> 5) + NW - rot) % NW) << 5) + (tid & 31) : tid;
    const int vb = (item + P.item0) % P.nvb, cell = (item + P.item0) / P.nvb;
    const int ex = cell % P.ncx, ey = (cell / P.ncx) % P.ncy, ez = cell / (P.ncx * P.ncy);
    const int v0 = vb * BV;
    const bool wx = !dirichlet && ex == P.ncx - 1, wy = !dirichlet && ey == P.ncy - 1, wz = !dirichlet && !P.zopen && ez == P.ncz - 1;
    const bool special = dirichlet ? (ex == 0 || ex == P.ncx - 1 || ey == 0 || ey == P.ncy - 1 || ez == 0 || ez == P.ncz - 1)
                                   : (wx || wy || wz);
    if (!perq && tid < 7) GS[tid] = __ldg(P.geom + (P.geom_mode == 1 ? (size_t)cell * 7 : 0) + tid);   // visible after the barriers below
    // MSC: the first round's d values are requested before the waits that precede their use (L2 latency)
    const int t_first = (ROUNDS > 1 || !ROTATE) ? tid : rot_tid;
    double dpre[N];
    if (MSC && t_first < TASKS) load_dscale<PDEG>(P, ex, ey, ez, t_first / TPL, dpre);
    mbar_wait(bar, parity);
    parity ^= 1u;

    // ph0: Ns along x, in place; Dirichlet masking / periodic wrap patching
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 x[N], y[N];
      lds_line2<N>(A + base + b2, stride, x);
      if (special) {
        const int i2 = l % N, i3 = l / N;
        if (dirichlet) {
          const int iy = ey * PDEG + i2, iz = ez * PDEG + i3;
          if (iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz)) {
#pragma unroll
            for (int i = 0; i < N; ++i) x[i] = {0.0, 0.0};
          }
          if (ex == 0) x[0] = {0.0, 0.0};
          if (ex == P.ncx - 1) x[N - 1] = {0.0, 0.0};
        } else if ((v0 + b2) < P.nvec) {
          int iy = ey * PDEG + i2, iz = ez * PDEG + i3;
          const bool line_wrapped = (iy >= P.ndy) || (iz >= P.ndz);
          if (iy >= P.ndy) iy -= P.ndy;
          if (iz >= P.ndz) iz -= P.ndz;
          const long long row = (long long)P.ndx * ((long long)iy + (long long)P.ndy * iz);
          const double* src = P.W + (row + (long long)ex * PDEG) * nvec + v0 + b2;
          if (line_wrapped) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
              long long off = (long long)i * nvec;
              if (wx && i == N - 1) off -= (long long)P.ndx * nvec;
              const double2 d = __ldg(reinterpret_cast<const double2*>(src + off));
              x[i] = {d.x, d.y};
            }
          } else if (wx) {
            const double2 d = __ldg(reinterpret_cast<const double2*>(src + (long long)(PDEG - P.ndx) * nvec));
            x[N - 1] = {d.x, d.y};
          }
        }
      }
      if (MSC) {
        double dn[N];
        if (r_ == 0) {
#pragma unroll
          for (int i = 0; i < N; ++i) dn[i] = dpre[i];
        } else {
          load_dscale<PDEG>(P, ex, ey, ez, l, dn);
        }
#pragma unroll
        for (int i = 0; i < N; ++i) x[i] = vmul(dn[i], x[i]);
      }
      eo2<PDEG, MAT_NS, false>(x, y);
      sts_line2<N>(A + base + b2, stride, y);
    }
    __syncthreads();
    // ph1: Ns along y, in place
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<1>(l, base, stride);
      v2 x[N], y[N];
      lds_line2<N>(A + base + b2, stride, x);
      eo2<PDEG, MAT_NS, false>(x, y);
      sts_line2<N>(A + base + b2, stride, y);
    }
    if (tid == 0) tma_wait_read0();   // the previous item's reduction has finished reading what is now tile C
    __syncthreads();
    // ph2: T = alpha * Ns_z A -> A ; T2 = Ds_z T -> C
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<2>(l, base, stride);
      v2 x[N], tq[N], d[N];
      lds_line2<N>(A + base + b2, stride, x);
      eo2<PDEG, MAT_NS, false>(x, tq);
      if (alpha != 1.0) {
#pragma unroll
        for (int i = 0; i < N; ++i) tq[i] = vmul(alpha, tq[i]);
      }
      sts_line2<N>(A + base + b2, stride, tq);
      eo2<PDEG, MAT_DS, false>(tq, d);
      sts_line2<N>(C + base + b2, stride, d);
    }
    __syncthreads();
    // ph3: T0 = Ds_x T -> B
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 tq[N], d[N];
      lds_line2<N>(A + base + b2, stride, tq);
      eo2<PDEG, MAT_DS, false>(tq, d);
      sts_line2<N>(B + base + b2, stride, d);
    }
    __syncthreads();
    if (perq) { mbar_wait(gbar, gparity); gparity ^= 1u; }
    // ph4: T1 = Ds_y T; quadrature-point scaling with the symmetric metric (Alg. 2 l.5-6; Eq. 8, 22-23);
    //      R = Sm + Ds_y^T S1 -> A ; S0 -> B ; S2 -> C
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      const int i1 = l % N, i3 = l / N;
      int base, stride; TL::template line<1>(l, base, stride);
      v2 tq[N], t1[N], r[N];
      lds_line2<N>(A + base + b2, stride, tq);
      eo2<PDEG, MAT_DS, false>(tq, t1);
      // staged geometry: [7][n^3] (per q-point) or [7] (per cell / uniform); no w_Q factor (sqrt(w) tables)
      const double* gp = perq ? GS + (i1 + N * N * i3) : GS;
      const int gstep = perq ? NN : 1;       // stride between the 7 factors
      const int qstep = perq ? N : 0;        // stride between points along the y-line
#pragma unroll
      for (int i = 0; i < N; ++i) {
        const double* g = gp + i * qstep;
        const double g00 = g[0], g01 = g[gstep], g02 = g[2 * gstep], g11 = g[3 * gstep],
                     g12 = g[4 * gstep], g22 = g[5 * gstep], gm = g[6 * gstep];
        const double2 a0 = *reinterpret_cast<const double2*>(B + base + b2 + i * stride);
        const double2 a2 = *reinterpret_cast<const double2*>(C + base + b2 + i * stride);
        const v2 t0 = {a0.x, a0.y}, t2 = {a2.x, a2.y}, t1i = t1[i];
        const v2 s0 = vfma(g02, t2, vfma(g01, t1i, vmul(g00, t0)));
        const v2 s1 = vfma(g12, t2, vfma(g11, t1i, vmul(g01, t0)));
        const v2 s2 = vfma(g22, t2, vfma(g12, t1i, vmul(g02, t0)));
        *reinterpret_cast<double2*>(B + base + b2 + i * stride) = make_double2(s0.a, s0.b);
        *reinterpret_cast<double2*>(C + base + b2 + i * stride) = make_double2(s2.a, s2.b);
        t1[i] = s1;
        tq[i] = vmul(gm, tq[i]);
      }
      eo2<PDEG, MAT_DS, true>(t1, r);
#pragma unroll
      for (int i = 0; i < N; ++i) r[i] = r[i] + tq[i];
      sts_line2<N>(A + base + b2, stride, r);
    }
    __syncthreads();
    // the staged geometry is consumed: fetch the next item's
    if (tid == 0) *s_next = (int)(gridDim.x + nxt_raw);
    if (tid == 0 && perq) {
      const int nxt = (int)(gridDim.x + nxt_raw);
      if (nxt < nitems) {
        mbar_expect_tx(gbar, GBYTES);
        bulk_load(GS, P.geom + (size_t)((nxt + P.item0) / P.nvb) * P.geom_stride, GBYTES, gbar);
      }
    }
    // ph5: R += Ds_x^T S0 -> A
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 s[N], r[N], d[N];
      lds_line2<N>(B + base + b2, stride, s);
      lds_line2<N>(A + base + b2, stride, r);
      eo2<PDEG, MAT_DS, true>(s, d);
#pragma unroll
      for (int i = 0; i < N; ++i) r[i] = r[i] + d[i];
      sts_line2<N>(A + base + b2, stride, r);
    }
    __syncthreads();
    // tile B is free: prefetch the next item's tile into it (it becomes tile A of the next item)
    if (tid == 0) {
      const int nxt = (int)(gridDim.x + nxt_raw);
      if (nxt < nitems) {
        const int nvb_ = (nxt + P.item0) % P.nvb, ncell = (nxt + P.item0) / P.nvb;
        const int nex = ncell % P.ncx, ney = (ncell / P.ncx) % P.ncy, nez = ncell / (P.ncx * P.ncy);
        mbar_expect_tx(bar, TL::BYTES);
        tma_load_4d(B, &tmW, bar, nvb_ * BV, nex * PDEG, ney * PDEG, nez * PDEG);
      }
    }
    // ph6: R += Ds_z^T S2 ; A <- Ns_z^T R
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<2>(l, base, stride);
      v2 s[N], r[N], d[N];
      lds_line2<N>(C + base + b2, stride, s);
      lds_line2<N>(A + base + b2, stride, r);
      eo2<PDEG, MAT_DS, true>(s, d);
#pragma unroll
      for (int i = 0; i < N; ++i) r[i] = r[i] + d[i];
      eo2<PDEG, MAT_NS, true>(r, d);
      sts_line2<N>(A + base + b2, stride, d);
    }
    __syncthreads();
    // ph7: Ns^T along y, in place
    if (MSC && t_first < TASKS) load_dscale<PDEG>(P, ex, ey, ez, t_first / TPL, dpre);   // for ph8
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<1>(l, base, stride);
      v2 x[N], y[N];
      lds_line2<N>(A + base + b2, stride, x);
      eo2<PDEG, MAT_NS, true>(x, y);
      sts_line2<N>(A + base + b2, stride, y);
    }
    __syncthreads();
    // ph8: Ns^T along x, in place; Dirichlet rows zeroed; wrap-around elements scattered by RED
    FE_FOR_TASKS(t) {
      const int b2 = (t % TPL) * 2, l = t / TPL;
      int base, stride; TL::template line<0>(l, base, stride);
      v2 x[N], y[N];
      double dn[N];
      if (MSC) {
        if (r_ == 0) {
#pragma unroll
          for (int i = 0; i < N; ++i) dn[i] = dpre[i];
        } else {
          load_dscale<PDEG>(P, ex, ey, ez, l, dn);
        }
      }
      lds_line2<N>(A + base + b2, stride, x);
      eo2<PDEG, MAT_NS, true>(x, y);
      if (MSC) {
#pragma unroll
        for (int i = 0; i < N; ++i) y[i] = vmul(dn[i], y[i]);
      }
      if (special) {
        const int i2 = l % N, i3 = l / N;
        int iy = ey * PDEG + i2, iz = ez * PDEG + i3;
        if (dirichlet) {
          if (iy == 0 || iy == P.ndy - 1 || fe_z_masked(P, iz)) {
#pragma unroll
            for (int i = 0; i < N; ++i) y[i] = {0.0, 0.0};
          }
          if (ex == 0) y[0] = {0.0, 0.0};
          if (ex == P.ncx - 1) y[N - 1] = {0.0, 0.0};
        } else if ((v0 + b2) < P.nvec) {
          const bool line_wrapped = (iy >= P.ndy) || (iz >= P.ndz);
          if (iy >= P.ndy) iy -= P.ndy;
          if (iz >= P.ndz) iz -= P.ndz;
          const long long row = (long long)P.ndx * ((long long)iy + (long long)P.ndy * iz);
          double* dst = P.Z + (row + (long long)ex * PDEG) * nvec + v0 + b2;
          if (line_wrapped) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
              long long off = (long long)i * nvec;
              if (wx && i == N - 1) off -= (long long)P.ndx * nvec;
              atomicAdd(dst + off, y[i].a); atomicAdd(dst + off + 1, y[i].b);
            }
          } else if (wx) {
            const long long off = (long long)(PDEG - P.ndx) * nvec;
            atomicAdd(dst + off, y[N - 1].a); atomicAdd(dst + off + 1, y[N - 1].b);
          }
        }
      }
      sts_line2<N>(A + base + b2, stride, y);
    }
    fence_async_smem();
    __syncthreads();
    if (tid == 0) {
      tma_reduce_add_4d(&tmZ, A, v0, ex * PDEG, ey * PDEG, ez * PDEG);
      tma_commit();
    }
    { double* t_ = A; A = B; B = C; C = t_; }   // (A,B,C) <- (B,C,A)
    item = *s_next;   // written during ph5, several barriers ago
  }
  if (tid == 0) tma_wait_all0();
}

}  // namespace fe
