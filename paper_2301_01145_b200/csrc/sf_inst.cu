// sf_inst.cu -- explicit kernel instantiations.  Compiled once per (SF_INST_KIND, SF_INST_T) pair
// by the build script so that the ten translation units build in parallel:
//   SF_INST_KIND 0: X passes (S1, S5);  1 / 2 / 3: strided pass MODE 0 / 1 / 2 (S2, S4, S3)
#define SF_LAUNCH_IMPL
#include "sf_launch.cuh"

#ifndef SF_INST_KIND
#error "define SF_INST_KIND (0..3) and SF_INST_T (float|double)"
#endif

namespace sf {
#if SF_INST_KIND == 0
template <> cudaError_t launch_xfwd<SF_INST_T>(int L, const XParams<SF_INST_T>& p, int ncomp, cudaStream_t st)
{
    return launch_x_any<SF_INST_T, false>(L, p, ncomp, st);
}
template <> cudaError_t launch_xinv<SF_INST_T>(int L, const XParams<SF_INST_T>& p, int ncomp, cudaStream_t st)
{
    return launch_x_any<SF_INST_T, true>(L, p, ncomp, st);
}
#else
template <>
cudaError_t launch_spass_m<SF_INST_T, SF_INST_KIND - 1>(int L, const SParams<SF_INST_T>& p, int nb, int nz, int nbuf,
                                                         cudaStream_t st)
{
    return launch_s_any<SF_INST_T, SF_INST_KIND - 1>(L, p, nb, nz, nbuf, st);
}
#endif
} // namespace sf
