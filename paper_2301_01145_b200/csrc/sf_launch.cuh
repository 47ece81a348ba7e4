// sf_launch.cuh -- host-side launchers: pick the kernel instantiation for a transform length and
// launch it.  Declarations only need the parameter structs; the definitions live in the
// sf_inst_*.cu translation units (one per precision and kernel family, so they build in parallel).
#pragma once
#include "sf_spass.cuh"
#include "sf_xpass.cuh"

namespace sf {

constexpr int kThreads = 256;

// S1 / S5: L = complex length of the packed row (half the real transform length); ncomp fields
template <typename T> cudaError_t launch_xfwd(int L, const XParams<T>& p, int ncomp, cudaStream_t st);
template <typename T> cudaError_t launch_xinv(int L, const XParams<T>& p, int ncomp, cudaStream_t st);
// S2 / S3 / S4: mode 0 forward, 1 backward, 2 fused; nb batches, nz independent fields on gridDim.z,
// nbuf shared-memory tiles per CTA (1 solve, 2 gradient, 3 curl)
template <typename T, int MODE> cudaError_t launch_spass_m(int L, const SParams<T>& p, int nb, int nz, int nbuf, cudaStream_t st);
template <typename T> inline cudaError_t launch_spass(int L, int mode, const SParams<T>& p, int nb, int nz, int nbuf, cudaStream_t st)
{
    switch (mode) {
    case 0: return launch_spass_m<T, 0>(L, p, nb, nz, nbuf, st);
    case 1: return launch_spass_m<T, 1>(L, p, nb, nz, nbuf, st);
    default: return launch_spass_m<T, 2>(L, p, nb, nz, nbuf, st);
    }
}
// columns per tile of the strided kernels for this length
template <typename T> inline int spass_tile_columns(int L)
{
    const int e = 2 * (int)sizeof(T), t = 65536 / (L * e);
    return t >= 16 ? 16 : (t >= 8 ? 8 : 4);
}
// shared memory one CTA of the strided kernel needs
template <typename T> inline size_t spass_smem_bytes(int L, int nbuf)
{
    return (size_t)nbuf * L * spass_tile_columns<T>(L) * 2 * sizeof(T);
}
inline bool length_built(int L) { return L >= 4 && L <= 2048 && (L & (L - 1)) == 0; }

#ifdef SF_LAUNCH_IMPL
template <typename K> static cudaError_t set_smem(K kernel, size_t bytes)
{
    if (bytes > 48 * 1024) return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    return cudaSuccess;
}

template <typename T, int L, bool INV> static cudaError_t launch_x_one(const XParams<T>& p, int ncomp, cudaStream_t st)
{
    constexpr int ROWS = x_rows<T, L>();
    constexpr int LP = x_lp<T, L>();
    const size_t smem = (size_t)2 * ROWS * LP * sizeof(SF_CX);
    const long long rows = (long long)p.ny * p.nz;
    dim3 grid((unsigned)((rows + ROWS - 1) / ROWS), (unsigned)ncomp);
    // fp32 rows of 512 and more complex points: three or fewer CTAs fit per SM, so give each 512 threads
    constexpr int NT = (sizeof(T) == 4 && L >= 512) ? 512 : kThreads;
    auto kernel = INV ? xinv_kernel<T, L, NT> : xfwd_kernel<T, L, NT>;
    cudaError_t e = set_smem(kernel, smem);
    if (e != cudaSuccess) return e;
    kernel<<<grid, NT, smem, st>>>(p);
    return cudaGetLastError();
}

template <typename T, bool INV> static cudaError_t launch_x_any(int L, const XParams<T>& p, int ncomp, cudaStream_t st)
{
    switch (L) {
#define SF_CASE(LL) case LL: return launch_x_one<T, LL, INV>(p, ncomp, st);
        SF_CASE(4) SF_CASE(8) SF_CASE(16) SF_CASE(32) SF_CASE(64) SF_CASE(128) SF_CASE(256) SF_CASE(512)
        SF_CASE(1024) SF_CASE(2048)
#undef SF_CASE
    default: return cudaErrorInvalidValue;
    }
}

template <typename T, int L, int MODE, int NT> static cudaError_t launch_s_nt(const SParams<T>& p, int nb, int nz, size_t smem, cudaStream_t st)
{
    constexpr int TX = s_tx<T, L>();
    dim3 grid((unsigned)((p.nx + TX - 1) / TX), (unsigned)nb, (unsigned)nz);
    auto kernel = spass_kernel<T, L, TX, NT, MODE>;
    cudaError_t e = set_smem(kernel, smem);
    if (e != cudaSuccess) return e;
    kernel<<<grid, NT, smem, st>>>(p);
    return cudaGetLastError();
}

template <typename T, int L, int MODE> static cudaError_t launch_s_one(const SParams<T>& p, int nb, int nz, int nbuf, cudaStream_t st)
{
    constexpr int TX = s_tx<T, L>();
    const size_t smem = (size_t)nbuf * L * TX * sizeof(SF_CX);
    if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
    // The fused pass with two or three tiles (gradient, curl, divergence) of a long transform fills most
    // of an SM's shared memory: when only one or two CTAs fit, give each more threads so that the SM
    // still holds 1024 (cfg 5: 192 KB per CTA, one CTA of 1024 threads instead of 256).
    if constexpr (MODE == 2 && L >= 256) {
        if (smem > 113 * 1024) {
            constexpr int NTB = (sizeof(T) == 4) ? 1024 : 512;    // 64 / 128 registers per thread
            return launch_s_nt<T, L, MODE, NTB>(p, nb, nz, smem, st);
        }
        if (smem > 75 * 1024) return launch_s_nt<T, L, MODE, 512>(p, nb, nz, smem, st);
    }
    return launch_s_nt<T, L, MODE, kThreads>(p, nb, nz, smem, st);
}

template <typename T, int MODE> static cudaError_t launch_s_any(int L, const SParams<T>& p, int nb, int nz, int nbuf, cudaStream_t st)
{
    switch (L) {
#define SF_CASE(LL) case LL: return launch_s_one<T, LL, MODE>(p, nb, nz, nbuf, st);
        SF_CASE(4) SF_CASE(8) SF_CASE(16) SF_CASE(32) SF_CASE(64) SF_CASE(128) SF_CASE(256) SF_CASE(512)
        SF_CASE(1024) SF_CASE(2048)
#undef SF_CASE
    default: return cudaErrorInvalidValue;
    }
}
#endif

} // namespace sf
