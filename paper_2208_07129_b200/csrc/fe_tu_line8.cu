// Kernel translation unit: the Cartesian line kernel with 8 vectors per block (fe_kernels_line.cuh): calls with <= 8
// vectors (no lanes wasted on the vector tail), p = 7 always (three 8-vector blocks per SM beat one 16-vector block:
// 105 vs 99.6 GDoF*vec/s) and p = 8.
#include "fe_ctx.h"
#include "fe_kernels_line.cuh"

namespace fe_host {

cudaError_t upload_tables_line8(const fe::HostTables& t) {
  return cudaMemcpyToSymbol(fe::c_eo2, t.eo2, sizeof(t.eo2), sizeof(fe::EoTab2) * fe::MAT_COUNT * t.p);
}

template <int CFG> struct LineCfg;
template <> struct LineCfg<101> { static constexpr int BV = 8, NT = 32, MINB = 4; };
template <> struct LineCfg<102> { static constexpr int BV = 8, NT = 64, MINB = 4; };
template <> struct LineCfg<103> { static constexpr int BV = 8, NT = 64, MINB = 4; };
template <> struct LineCfg<104> { static constexpr int BV = 8, NT = 128, MINB = 4; };
template <> struct LineCfg<105> { static constexpr int BV = 8, NT = 160, MINB = 4; };
template <> struct LineCfg<106> { static constexpr int BV = 8, NT = 128, MINB = 5; };
template <> struct LineCfg<107> { static constexpr int BV = 8, NT = 128, MINB = 3; };
template <> struct LineCfg<108> { static constexpr int BV = 8, NT = 192, MINB = 2; };

#include "fe_line_launch.inl"

cudaError_t launch_line8(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap& tw, const CUtensorMap& tz, cudaStream_t st) {
  switch (c->p) {
    case 1: return launch_line_p<1, 101>(c, P, tw, tz, st);
    case 2: return launch_line_p<2, 102>(c, P, tw, tz, st);
    case 3: return launch_line_p<3, 103>(c, P, tw, tz, st);
    case 4: return launch_line_p<4, 104>(c, P, tw, tz, st);
    case 5: return launch_line_p<5, 105>(c, P, tw, tz, st);
    case 6: return launch_line_p<6, 106>(c, P, tw, tz, st);
    case 7: return launch_line_p<7, 107>(c, P, tw, tz, st);
    case 8: return launch_line_p<8, 108>(c, P, tw, tz, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace fe_host
