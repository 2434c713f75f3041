// Device code, part 8: "init-ahead" -- S1 (Z <- 0 or Z <- beta Z + gamma W) folded into
// the persistent apply kernels instead of a separate streaming pass.
//
// The output is initialised chunk by chunk (chunk c = the node planes of cell layer c, contiguous in memory)
// a little AHEAD of the layer the blocks are accumulating into, by the blocks themselves, a few slices per
// item, so that the HBM-bound initialisation overlaps the FP64-bound cell work:
//   * a slice is NT consecutive double2 elements of a chunk; chunks 0 .. LOOK-1 are split statically over the
//     blocks at kernel start; the slices of chunk L+LOOK are handed out dynamically (one atomicAdd per item on
//     slice_ctr[c]) to the items of layer L, k = ceil(slices / items per layer) at a time -- like the items
//     themselves, because co-resident blocks do not run at the same speed;
//   * a block adds the number of slices it finished to done[c] with release semantics once it has moved on to
//     the next chunk (one release per block and chunk); chunk c is complete when done[c] = slices(c);
//   * before a block reduces into layer L it makes sure (acquire) that chunks L and L+1 are complete.
// No block waits for a block that waits for it (a chunk is handed out entirely to items that START before any
// item that needs it finishes), but all blocks must be co-resident: the kernels are launched cooperatively.
// The control words are zeroed on the stream before every launch.
#pragma once
#include "fe_kernels_tma.cuh"

namespace fe {

enum { INIT_NONE = -1, INIT_ZERO = 0, INIT_SCALE = 1, INIT_AXPBY = 2 };

struct InitParams {
  int mode;                          // INIT_*
  double beta, gamma;                // Z <- beta Z + gamma W
  unsigned* slice_ctr;               // [ncz] next slice of chunk c to hand out (0 at launch)
  unsigned* done;                    // [ncz] warp-slices of chunk c completed (0 at launch)
};

// IM: 0 = no initialisation (everything compiles out), 1 = zero fill (stores only), 2 = scale / axpby: the old Z
// and W slices are STAGED through shared memory by bulk copies (no registers, no load latency on the threads):
// after each block barrier of the cell pipeline ("slot") the threads combine the sub-batch that landed in one
// buffer and store it, and thread 0 starts the copies of the next sub-batch into the other buffer (all threads
// finished reading that one before the barrier).  Slice and element counts are 32-bit (the host falls back to a
// separate pass when a chunk has 2^31 or more double2 elements).
template <int NT, int IM>
struct InitAhead {
  static constexpr int KB = 4;       // IM = 2, start-up only: slices per register batch
  static constexpr int SB = 3;       // IM = 2: slices per staged sub-batch
  static constexpr int STAGE_BYTES = (IM == 2) ? 2 * 2 * SB * NT * 16 + 16 : 0;   // two buffers x (Z, W) + two mbarriers
  static constexpr int NW = NT / 32;
  double2* stage = nullptr; uint64_t* fbar = nullptr;
  int cur = 0; uint32_t par0 = 0, par1 = 0;
  // per buffer: chunk, slices (0 = empty), valid elements of the last slice, where its first slice goes in Z
  int bc0 = 0, bc1 = 0; unsigned bn0 = 0, bn1 = 0, vl0 = 0, vl1 = 0; double2* gz0 = nullptr; double2* gz1 = nullptr;
  const InitParams& I;
  const int tid, last;               // last chunk index
  unsigned len_reg = 0, len_last = 0;   // double2 elements per regular / last chunk
  unsigned ns_reg = 0, ns_last = 0;     // slices per regular / last chunk
  int k_reg = 0, k_last = 0;            // slices handed to one item
  double2* Z2 = nullptr; const double2* W2 = nullptr;
  int ready = -1;                    // chunks <= ready are known to be complete
  // the current hand-out: slices [s_cur, s_end) of chunk c_cur
  int c_cur = -1; unsigned s_cur = 0, s_end = 0;
  double2 zr[IM == 2 ? KB : 1], wr[IM == 2 ? KB : 1];
  int pend = 0;

  __device__ __forceinline__ InitAhead(const InitParams& i_, const ApplyParams& P, int pdeg, int tid_, int layer_items)
      : I(i_), tid(tid_), last(P.ncz - 1) {
    if (IM != 0) {
      const long long plane2 = (long long)P.ndx * P.ndy * P.nvec / 2;
      len_reg = (unsigned)(pdeg * plane2);
      len_last = (unsigned)((P.ndz - last * pdeg) * plane2);
      ns_reg = (len_reg + NT - 1) / NT;
      ns_last = (len_last + NT - 1) / NT;
      k_reg = (int)((ns_reg + layer_items - 1) / layer_items);
      k_last = (int)((ns_last + layer_items - 1) / layer_items);
      Z2 = reinterpret_cast<double2*>(P.Z);
      W2 = reinterpret_cast<const double2*>(P.W);
    }
  }
  __device__ __forceinline__ unsigned nslices(int c) const { return c == last ? ns_last : ns_reg; }
  __device__ __forceinline__ unsigned len(int c) const { return c == last ? len_last : len_reg; }
  __device__ __forceinline__ int per_item(int c) const { return c == last ? k_last : k_reg; }
  __device__ __forceinline__ long long begin(int c) const { return (long long)c * len_reg; }

  // Publication.  A release makes the issuing warp wait until earlier stores are visible, so it is done rarely:
  // a block adds up the slices it finished per chunk (acc_*), and thread 0 publishes the total once the block has
  // moved on to another chunk, right after a block barrier (which orders every warp's stores before the release).
  int acc_c = -1; unsigned acc_cnt = 0;   // being accumulated
  int pub_c = -1; unsigned pub_cnt = 0;   // complete, to be published at the next publish_point()
  __device__ __forceinline__ void note(int c, unsigned cnt) {
    if (c != acc_c) {
      if (acc_cnt) { pub_c = acc_c; pub_cnt = acc_cnt; }   // (at most one chunk is pending: a block meets chunks in order)
      acc_c = c; acc_cnt = 0;
    }
    acc_cnt += cnt;
  }
  // call by all threads right AFTER a block barrier
  __device__ __forceinline__ void publish_point() {
    if (IM == 0 || pub_cnt == 0) return;
    if (tid == 0)
      asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(I.done + pub_c), "r"(pub_cnt) : "memory");
    pub_cnt = 0;
  }
  __device__ __forceinline__ void finish() {   // kernel end, all threads
    if (IM == 0) return;
    __syncthreads();
    publish_point();
    note(-2, 0u);
    publish_point();
  }
  __device__ __forceinline__ void zero_slices(int c, unsigned s0, unsigned s1, unsigned step) {
    if (s0 >= s1) return;
    const unsigned n = len(c);
    unsigned e = s0 * NT + tid;
    double2* z = Z2 + begin(c) + e;
    const unsigned de = step * NT;
    const double2 zero = make_double2(0.0, 0.0);
#pragma unroll 2
    for (unsigned s = s0; s < s1; s += step, e += de, z += de)
      if (e < n) *z = zero;
  }
  // loads of up to KB slices s0, s0+step, ... (< s1) of chunk c; they stay in flight until finish_loads()
  __device__ __forceinline__ void start_loads(int c, unsigned s0, unsigned s1, unsigned step) {
    const unsigned n = len(c);
    const double2* z = Z2 + begin(c);
    const double2* w = W2 + begin(c);
    pend = 0;
#pragma unroll
    for (int k = 0; k < KB; ++k) {
      const unsigned s = s0 + (unsigned)k * step;
      if (s >= s1) break;
      const unsigned e = s * NT + tid;
      if (e < n) {
        if (I.mode == INIT_AXPBY) zr[k] = z[e];
        asm volatile("ld.global.nc.v2.f64 {%0, %1}, [%2];" : "=d"(wr[k].x), "=d"(wr[k].y) : "l"(w + e));
      }
      pend = k + 1;
    }
  }
  __device__ __forceinline__ void finish_loads(int c, unsigned s0, unsigned step) {
    const unsigned n = len(c);
    double2* z = Z2 + begin(c);
#pragma unroll
    for (int k = 0; k < KB; ++k) {
      if (k >= pend) break;
      const unsigned e = (s0 + (unsigned)k * step) * NT + tid;
      if (e < n) {
        double2 r;
        if (I.mode == INIT_AXPBY) { r.x = fma(I.beta, zr[k].x, I.gamma * wr[k].x); r.y = fma(I.beta, zr[k].y, I.gamma * wr[k].y); }
        else { r.x = I.gamma * wr[k].x; r.y = I.gamma * wr[k].y; }
        z[e] = r;
      }
    }
  }
  // kernel start: chunks 0 .. look-1, slices b, b+G, ... of each (synchronous)
  __device__ __forceinline__ void startup(int look) {
    if (IM == 0) return;
    for (int c = 0; c < look && c <= last; ++c) {
      const unsigned ns = nslices(c);
      unsigned cnt = 0;
      if (IM == 1) {
        zero_slices(c, blockIdx.x, ns, gridDim.x);
        for (unsigned s = blockIdx.x; s < ns; s += gridDim.x) ++cnt;
      } else {
        for (unsigned s = blockIdx.x; s < ns; s += KB * gridDim.x) {
          start_loads(c, s, ns, gridDim.x);
          finish_loads(c, s, gridDim.x);
          cnt += pend;
        }
      }
      __syncthreads();   // every warp's stores precede thread 0's release
      if (tid == 0 && cnt)
        asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(I.done + c), "r"(cnt) : "memory");
    }
  }
  // tid 0, at the top of an item of layer L: reserve this item's slices of chunk c = L + look
  __device__ __forceinline__ unsigned grab(int c) const {
    if (IM == 0 || c > last) return 0u;
    unsigned r;
    asm volatile("atom.global.add.u32 %0, [%1], %2;" : "=r"(r) : "l"(I.slice_ctr + c), "r"((unsigned)per_item(c)) : "memory");
    return r;
  }
  // thread 0, as soon as a reservation is known (most of an item before its slices are staged): pull them into L2,
  // so that the staging copies, which are issued only one slot ahead, do not wait for DRAM
  __device__ __forceinline__ void prefetch_l2(int c, unsigned s0) const {
    if (IM != 2 || c > last) return;
    const unsigned ns = nslices(c);
    if (s0 >= ns) return;
    const unsigned s1 = s0 + per_item(c) < ns ? s0 + per_item(c) : ns;
    const unsigned n = len(c), e0 = s0 * NT, e1 = s1 * NT < n ? s1 * NT : n;
    const uint32_t bytes = (e1 - e0) * 16u;
    if (I.mode == INIT_AXPBY)
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(Z2 + begin(c) + e0), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(W2 + begin(c) + e0), "r"(bytes) : "memory");
  }
  // all threads, once the reservation has been broadcast (s0 = first slice); right after a block barrier.
  // IM = 2: the sub-batch in flight belongs to the previous hand-out and is finished first, so that a block never
  // has more than one chunk waiting for publication.
  __device__ __forceinline__ void accept(int c, unsigned s0) {
    if (IM == 0) return;
    if (IM == 2) { slot_process(); while (busy()) { slot_issue(); __syncthreads(); slot_process(); } }
    note(c > last ? -2 : c, 0u);   // the block has moved on: what it did for the previous chunk becomes publishable
    if (c > last) { c_cur = -1; s_cur = s_end = 0; return; }
    const unsigned ns = nslices(c);
    c_cur = c; s_cur = s0 < ns ? s0 : ns;
    s_end = s0 + per_item(c) < ns ? s0 + per_item(c) : ns;
  }
  // IM = 1: all accepted slices now (stores only)
  __device__ __forceinline__ void batch_begin() {
    if (IM != 1 || s_cur >= s_end) return;
    zero_slices(c_cur, s_cur, s_end, 1u);
    note(c_cur, s_end - s_cur);
    s_cur = s_end;
  }
  // IM = 2: shared-memory staging.  init_stage() once (thread 0 initialises the mbarriers; a block barrier follows).
  __device__ __forceinline__ void init_stage(unsigned char* smem) {
    if (IM != 2) return;
    stage = reinterpret_cast<double2*>(smem);
    fbar = reinterpret_cast<uint64_t*>(smem + 2 * 2 * SB * NT * 16);
    if (tid == 0) { mbar_init(fbar, 1); mbar_init(fbar + 1, 1); }
  }
  __device__ __forceinline__ double2* zbuf(int b) const { return stage + (size_t)b * 2 * SB * NT; }
  __device__ __forceinline__ double2* wbuf(int b) const { return zbuf(b) + SB * NT; }
  // all threads, right AFTER a block barrier: combine + store the sub-batch that landed in buffer `cur`, start the
  // copies of the next one into the other buffer, swap
  __device__ __forceinline__ void slot() { slot_process(); slot_issue(); }
  __device__ __forceinline__ void slot_process() {
    if (IM != 2) return;
    const unsigned bn = cur ? bn1 : bn0;
    if (bn == 0) return;
    mbar_wait(fbar + cur, cur ? par1 : par0);
    if (cur) par1 ^= 1u; else par0 ^= 1u;
    double2* z = (cur ? gz1 : gz0) + tid;                       // this thread's element of the first slice, in Z
    const double2* zs = zbuf(cur) + tid; const double2* ws = wbuf(cur) + tid;
    const unsigned vl = cur ? vl1 : vl0;                         // valid elements of the LAST slice (others are full)
    const double be = I.beta, ga = I.gamma;
    const bool axpby = (I.mode == INIT_AXPBY);
#pragma unroll
    for (int k = 0; k < SB; ++k) {
      if ((unsigned)k >= bn) break;
      if ((unsigned)k + 1 == bn && (unsigned)tid >= vl) break;
      const double2 w = ws[k * NT];
      double2 r;
      if (axpby) { const double2 o = zs[k * NT]; r.x = fma(be, o.x, ga * w.x); r.y = fma(be, o.y, ga * w.y); }
      else { r.x = ga * w.x; r.y = ga * w.y; }
      z[k * NT] = r;
    }
    note(cur ? bc1 : bc0, bn);
    if (cur) bn1 = 0; else bn0 = 0;
  }
  __device__ __forceinline__ void slot_issue() {
    if (IM != 2) return;
    const int nb = cur ^ 1;
    if (s_cur < s_end) {
      const unsigned cnt = (s_end - s_cur < (unsigned)SB) ? s_end - s_cur : (unsigned)SB;
      const unsigned n = len(c_cur), e0 = s_cur * NT;
      const unsigned e1 = (e0 + cnt * NT < n) ? e0 + cnt * NT : n;
      double2* zg = Z2 + begin(c_cur) + e0;
      if (tid == 0) {
        const uint32_t bytes = (e1 - e0) * 16u;
        fence_async_smem();
        mbar_expect_tx(fbar + nb, I.mode == INIT_AXPBY ? 2u * bytes : bytes);
        if (I.mode == INIT_AXPBY) bulk_load(zbuf(nb), zg, bytes, fbar + nb);
        bulk_load(wbuf(nb), W2 + begin(c_cur) + e0, bytes, fbar + nb);
      }
      const unsigned vl = e1 - e0 - (cnt - 1) * NT;
      if (nb) { bc1 = c_cur; gz1 = zg; vl1 = vl; bn1 = cnt; } else { bc0 = c_cur; gz0 = zg; vl0 = vl; bn0 = cnt; }
      s_cur += cnt;
    }
    cur = nb;
  }
  __device__ __forceinline__ bool busy() const { return IM == 2 && (s_cur < s_end || bn0 || bn1); }
  // whatever the slots of an item did not cover (rare), and at kernel end the sub-batches still in flight
  __device__ __forceinline__ void drain() {
    if (IM != 2) return;
    while (busy()) { __syncthreads(); slot(); }
  }
  // acquire: chunks c-1 and c are complete (called by all threads; the caller has a block barrier after it)
  __device__ __forceinline__ void wait_ready(int c) {
    if (IM == 0) return;
    if (c > last) c = last;
    if (c <= ready) return;
    if (tid == 0) {
      // (the first wait of a block also covers chunk 0: the periodic wrap of the last layer adds into it)
      for (int cc = (ready < 0 ? 0 : c - 1); cc <= c; ++cc) {
        const unsigned target = nslices(cc);
        unsigned v;
        do {
          asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(I.done + cc) : "memory");
          if (v < target) __nanosleep(100);
        } while (v < target);
      }
      asm volatile("fence.proxy.async;" ::: "memory");
    }
    ready = c;
  }
};

}  // namespace fe
