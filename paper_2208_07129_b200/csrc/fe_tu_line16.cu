// Kernel translation unit: the Cartesian line kernel with 16 vectors per block (fe_kernels_line.cuh), p = 1..7.
#include "fe_ctx.h"
#include "fe_kernels_line.cuh"

namespace fe_host {

cudaError_t upload_tables_line16(const fe::HostTables& t) {
  return cudaMemcpyToSymbol(fe::c_eo2, t.eo2, sizeof(t.eo2), sizeof(fe::EoTab2) * fe::MAT_COUNT * t.p);
}

template <int CFG> struct LineCfg;
template <> struct LineCfg<1> { static constexpr int BV = 16, NT = 32, MINB = 4; };
template <> struct LineCfg<2> { static constexpr int BV = 16, NT = 96, MINB = 4; };
template <> struct LineCfg<3> { static constexpr int BV = 16, NT = 128, MINB = 4; };
template <> struct LineCfg<4> { static constexpr int BV = 16, NT = 112, MINB = 4; };
template <> struct LineCfg<5> { static constexpr int BV = 16, NT = 160, MINB = 3; };
template <> struct LineCfg<6> { static constexpr int BV = 16, NT = 256, MINB = 2; };
template <> struct LineCfg<7> { static constexpr int BV = 16, NT = 256, MINB = 1; };

#include "fe_line_launch.inl"

cudaError_t launch_line16(fe_mf_ctx* c, const fe::ApplyParams& P, const CUtensorMap& tw, const CUtensorMap& tz, cudaStream_t st) {
  switch (c->p) {
    case 1: return launch_line_p<1, 1>(c, P, tw, tz, st);
    case 2: return launch_line_p<2, 2>(c, P, tw, tz, st);
    case 3: return launch_line_p<3, 3>(c, P, tw, tz, st);
    case 4: return launch_line_p<4, 4>(c, P, tw, tz, st);
    case 5: return launch_line_p<5, 5>(c, P, tw, tz, st);
    case 6: return launch_line_p<6, 6>(c, P, tw, tz, st);
    case 7: return launch_line_p<7, 7>(c, P, tw, tz, st);
  }
  return cudaErrorInvalidValue;   // p = 8 has no 16-vector configuration (three tiles would not fit twice)
}

}  // namespace fe_host
