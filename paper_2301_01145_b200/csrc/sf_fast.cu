// sf_fast.cu -- the one translation unit of kernel generation 2 (sf_fast.cuh): constant tables,
// shared-memory opt-in and the persistent-grid launchers.
#include "sf_fast.cuh"
#include "sf_fastper.cuh"
#include "sf_fast512.cuh"
#include "sf_fast2p.cuh"
#include "sf_fast64.cuh"
#include "sf_tcprobe.cuh"
#include "sf_fastx64.cuh"
#include "sf_fastr2r64.cuh"
#include "sf_fastper64.cuh"
#include "sf_fastxw.cuh"
#include "sf_fastxw64.cuh"
#include "sf_fastx5w.cuh"

#include <cmath>
#include <cstdlib>
#include <mutex>
#include <vector>

namespace sf2 {

namespace {
std::mutex g_mu;
int g_ready_dev = -1;
int g_sms = 0;
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;
} // namespace

cudaError_t fast_init()
{
    std::lock_guard<std::mutex> lk(g_mu);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (g_ready_dev == dev) return cudaSuccess;
    std::vector<float2> tw(1024);
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int j = 0; j < 1024; ++j) {
        const long double a = 2.0L * pi * (long double)j / 1024.0L;
        tw[j] = make_float2((float)cosl(a), (float)(-sinl(a)));
    }
    if ((e = cudaMemcpyToSymbol(c_tw1024, tw.data(), sizeof(float2) * 1024)) != cudaSuccess) return e;
    {
        std::vector<float2> tm(1024);
        for (int j = 0; j < 1024; ++j) {
            const long double a = 2.0L * pi * (long double)j / 1024.0L;
            tm[j] = make_float2((float)(cosl(a) - 1.0L), (float)(-sinl(a)));
        }
        if ((e = cudaMemcpyToSymbol(c_tw1024m1, tm.data(), sizeof(float2) * 1024)) != cudaSuccess) return e;
    }
    {
        std::vector<float2> tp(768), tx(544, make_float2(0.f, 0.f));
        for (int a = 0; a < 16; ++a)
            for (int b = 0; b < 16; ++b) {
                tp[a * 16 + b] = tw[4 * a * b];
                tp[256 + a * 16 + b] = make_float2(1.f, 0.f);
                tp[256 + (16 + a) * 16 + b] = tw[2 * (a + 16 * b)];
            }
        for (int a = 0; a < 8; ++a)
            for (int b = 0; b < 16; ++b) {
                tx[a * 16 + b] = tw[8 * a * b];
                tx[128 + (a * 16 + b) * 2] = make_float2(1.f, 0.f);
                tx[128 + (a * 16 + b) * 2 + 1] = tw[4 * (a + 8 * b)];
                if (b < 9) {
                    tx[384 + (a * 10 + b) * 2] = tw[2 * (2 * a + 16 * b)];
                    tx[384 + (a * 10 + b) * 2 + 1] = tw[2 * (2 * a + 1 + 16 * b)];
                }
            }
        if ((e = cudaMemcpyToSymbol(g_tab_pad, tp.data(), sizeof(float2) * 768)) != cudaSuccess) return e;
        if ((e = cudaMemcpyToSymbol(g_tab_x, tx.data(), sizeof(float2) * 544)) != cudaSuccess) return e;
        // the same factors for the warp-autonomous X passes (sf_fastxw.cuh), residue w fastest
        std::vector<float2> txw(kXwTab, make_float2(0.f, 0.f));
        for (int q = 0; q < 16; ++q)
            for (int h = 0; h < 2; ++h)
                for (int w = 0; w < 8; ++w) {
                    txw[q * 16 + h * 8 + w] = tw[(4 * (2 * q + h) * w) & 1023];
                    txw[256 + q * 16 + h * 8 + w] = tw[(4 * q * (2 * w + h)) & 1023];
                }
        for (int m = 0; m < 8; ++m)
            for (int i = 0; i < 16; ++i) txw[512 + m * 16 + i] = tw[2 * (i + 16 * m)];
        if ((e = cudaMemcpyToSymbol(g_tab_xw, txw.data(), sizeof(float2) * kXwTab)) != cudaSuccess) return e;
        // and for the rows of 512 (sf_fastx5w.cuh)
        std::vector<float2> tx5(kX5wTab);
        for (int q = 0; q < 16; ++q)
            for (int h = 0; h < 2; ++h)
                for (int o = 0; o < 16; ++o) {
                    tx5[q * 32 + h * 16 + o] = tw[(2 * (2 * q + h) * o) & 1023];
                    tx5[512 + q * 32 + h * 16 + o] = tw[(2 * q * (2 * o + h)) & 1023];
                }
        for (int m = 0; m < 8; ++m)
            for (int i = 0; i < 32; ++i) tx5[1024 + m * 32 + i] = tw[i + 32 * m];
        if ((e = cudaMemcpyToSymbol(g_tab_x5w, tx5.data(), sizeof(float2) * kX5wTab)) != cudaSuccess) return e;
    }
    if ((e = cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_pad_kernel<FMODE_FWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FastCfg<FMODE_FWD>::kSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_pad_kernel<FMODE_INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FastCfg<FMODE_INV>::kSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_pad_kernel<FMODE_FUSED>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FastCfg<FMODE_FUSED>::kSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_xper_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXpSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_xper_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXpSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_per_kernel<FMODE_FWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPerSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_per_kernel<FMODE_INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPerSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_per_kernel<FMODE_FUSED>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPerSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_per_kernel<FMODE_FUSED, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPerSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_x_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_x_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_xw_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXwSmemFwd)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_xw_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXwSmemInv)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_x5w_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kX5wSmemFwd)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_x5w_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kX5wSmemInv)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_xpw_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXpwSmemFwd)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_xpw_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXpwSmemInv)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast5_kernel<F5_FWD, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kSmem5 / 2))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast5_kernel<F5_INV, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem5NoSlot)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast5_kernel<F5_FUSED, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kSmem5 / 2))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast5_kernel<F5_CURL, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kSmem5 / 2))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_x5_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kX5Smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_x5_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kX5Smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_fused2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem2)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_fused2h_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem2)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_inv2h_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemInv2)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast_fwd2h_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem2)) != cudaSuccess) return e;
    {
        std::vector<double2> td(1024);
        for (int j = 0; j < 1024; ++j) {
            const long double a = 2.0L * pi * (long double)j / 1024.0L;
            td[j] = make_double2((double)cosl(a), (double)(-sinl(a)));
        }
        if ((e = cudaMemcpyToSymbol(c_tw1024d, td.data(), sizeof(double2) * 1024)) != cudaSuccess) return e;
    }
    if ((e = cudaFuncSetAttribute(fast64_kernel<FMODE_FWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem64)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast64_kernel<FMODE_INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem64NoSlot)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(fast64_kernel<FMODE_FUSED>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem64)) != cudaSuccess) return e;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if ((e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres)) != cudaSuccess) return e;
    if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
    g_encode = (EncodeTiledFn)fn;
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return e;   // the symbol uploads above have landed
    g_ready_dev = dev;
    return cudaSuccess;
}

static_assert(sizeof(CUtensorMap) == sizeof(TileMap), "TileMap must be able to hold a CUtensorMap");

cudaError_t fast_make_map(TileMap* out, const void* base, const unsigned long long dims[4],
                          const unsigned long long strides_bytes[3], const unsigned box[4])
{
    if (!g_encode) return cudaErrorNotReady;
    cuuint64_t gd[4] = { dims[0], dims[1], dims[2], dims[3] };
    cuuint64_t gs[3] = { strides_bytes[0], strides_bytes[1], strides_bytes[2] };
    cuuint32_t bx[4] = { box[0], box[1], box[2], box[3] };
    cuuint32_t es[4] = { 1, 1, 1, 1 };
    // 8-byte elements (one complex fp32 number); the data are moved, not interpreted
    CUresult r = g_encode(reinterpret_cast<CUtensorMap*>(out), CU_TENSOR_MAP_DATA_TYPE_UINT64, 4, const_cast<void*>(base), gd, gs, bx,
                          es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

namespace {
__global__ void green_tiles_kernel(float* tiles, const float* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                                   int rows, int kTile, long long total)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int pen = (int)(i % kTile);
        const int fp = (int)((i / kTile) % rows);
        const long long t = i / ((long long)kTile * rows);
        const long long nfull = (long long)(Pb / 2 + 1) * nct;
        int fb, kx;
        if (t < nfull) {
            fb = (int)(t / nct);
            kx = (int)(t % nct) * kTile + pen;
        } else {
            const int kb = min((int)(t - nfull) * kTile + pen, Pb - 1);
            fb = min(kb, Pb - kb);
            kx = nyq_col;
        }
        tiles[i] = green[kx + fb * g_pb + fp * g_pp];
    }
}
} // namespace

cudaError_t fast_green_tiles_rows(float* tiles, const float* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                                  int rows, cudaStream_t st)
{
    return fast_green_tiles_rows_w(tiles, green, g_pb, g_pp, Pb, nct, nyq_col, rows, kTile, st);
}
cudaError_t fast_green_tiles_rows_w(float* tiles, const float* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                                    int rows, int width, cudaStream_t st)
{
    const long long total = (long long)fast_green_tiles_elems_rows_w(Pb, nct, nyq_col, rows, width);
    green_tiles_kernel<<<148 * 8, 256, 0, st>>>(tiles, green, g_pb, g_pp, Pb, nct, nyq_col, rows, width, total);
    return cudaGetLastError();
}
cudaError_t fast_green_tiles(float* tiles, const float* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                             cudaStream_t st)
{
    return fast_green_tiles_rows(tiles, green, g_pb, g_pp, Pb, nct, nyq_col, kGreenRows, st);
}

cudaError_t launch_fast_pad(int mode, const FastParams& p, const TileMap& in_map, cudaStream_t st)
{
    const CUtensorMap& tm = reinterpret_cast<const CUtensorMap&>(in_map);
    if (p.nct <= 0 || (1 << p.nct_shift) != p.nct) return cudaErrorInvalidValue;
    // the kernels index with 32-bit element offsets
    if ((long long)p.nb * p.in_bs + 256 * p.in_ps >= (1ll << 31) || (long long)p.nb * p.out_bs + 512 * p.out_ps >= (1ll << 31))
        return cudaErrorInvalidValue;
    const int ntiles = fast_ntiles(p.nb, p.nct, p.nyq_col);
    int grid = 2 * g_sms;
    if (grid > ntiles) grid = ntiles;
    if (grid <= 0) return cudaErrorInvalidValue;
    switch (mode) {
    case FMODE_FWD:
        // both halves of a pencil's padded transform per thread (sf_fast2p.cuh); SF_PAD_1H=1: one half per thread (sf_fast.cuh)
        if (!getenv("SF_PAD_1H")) fast_fwd2h_kernel<<<grid, kT2, kSmem2, st>>>(p, tm);
        else fast_pad_kernel<FMODE_FWD><<<grid, kThreads, FastCfg<FMODE_FWD>::kSmem, st>>>(p, tm);
        break;
    case FMODE_INV:
        if (!getenv("SF_PAD_1H")) fast_inv2h_kernel<<<grid, kT2, kSmemInv2, st>>>(p);
        else fast_pad_kernel<FMODE_INV><<<grid, kThreads, FastCfg<FMODE_INV>::kSmem, st>>>(p, tm);
        break;
    case FMODE_FUSED:
        // both halves of a pencil's padded transform per thread (sf_fast2p.cuh); SF_FUSED_2P=1: one half of two pencils
        // per thread (needs an even number of batches); SF_FUSED_1P=1: one half of one pencil per thread (sf_fast.cuh)
        if (getenv("SF_FUSED_1P")) fast_pad_kernel<FMODE_FUSED><<<grid, kThreads, FastCfg<FMODE_FUSED>::kSmem, st>>>(p, tm);
        else if (getenv("SF_FUSED_2P") && (p.nb & 1) == 0) fast_fused2_kernel<<<grid, kT2, kSmem2, st>>>(p, tm);
        else fast_fused2h_kernel<<<grid, kT2, kSmem2, st>>>(p, tm);
        break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_fast5(int mode, const Fast5Params& p, const TileMap& in_map, cudaStream_t st)
{
    const CUtensorMap& tm = reinterpret_cast<const CUtensorMap&>(in_map);
    if (p.nct <= 0 || (1 << p.nct_shift) != p.nct || p.nb <= 0) return cudaErrorInvalidValue;
    // row, batch and column offsets are formed in 32 bits before they are widened
    if ((long long)p.nb * p.in_bs + 1024 * p.in_ps >= (1ll << 31) || (long long)p.nb * p.out_bs + 1024 * p.out_ps >= (1ll << 31))
        return cudaErrorInvalidValue;
    if (mode == F5_CURL && (p.ncomp != 3 || !p.kap_x || !p.kap_b || !p.kap_p || 3 * p.out_cs >= (1ll << 31))) return cudaErrorInvalidValue;
    if ((mode == F5_CURL || mode == F5_FUSED) && !p.green_tiles) return cudaErrorInvalidValue;
    // INV: 16-pencil tiles, one CTA per SM; FWD / FUSED / CURL: 8-pencil tiles, two CTAs per SM (p.nct counts those)
    const bool half = (mode != F5_INV);
    const int pen = half ? 8 : 16;
    const long long ntiles = ((long long)p.nb * p.nct + (p.nyq_col >= 0 ? (p.nb + pen - 1) / pen : 0)) * (mode == F5_FUSED ? p.ncomp : 1);
    if (ntiles + 4ll * g_sms >= (1ll << 31)) return cudaErrorInvalidValue;
    int grid = half ? 2 * g_sms : g_sms;
    if (grid > ntiles) grid = (int)ntiles;
    if (grid <= 0) return cudaErrorInvalidValue;
    switch (mode) {
    case F5_FWD: fast5_kernel<F5_FWD, 8><<<grid, kT5 / 2, kSmem5 / 2, st>>>(p, tm); break;   // (measured: 2.08 -> 1.98 ms on cfg 5)
    case F5_INV: fast5_kernel<F5_INV, 16><<<grid, kT5, kSmem5NoSlot, st>>>(p, tm); break;      // (8-pencil tiles: 2.13 -> 2.21 ms)
    // the multiplying passes work on 8-pencil tiles: two 512-thread CTAs per SM
    case F5_FUSED: fast5_kernel<F5_FUSED, 8><<<grid, kT5 / 2, kSmem5 / 2, st>>>(p, tm); break;
    case F5_CURL: fast5_kernel<F5_CURL, 8><<<grid, kT5 / 2, kSmem5 / 2, st>>>(p, tm); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t fast64_green_tiles(double* tiles, const double* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                               cudaStream_t st)
{
    const long long total = (long long)fast64_green_tiles_elems(Pb, nct, nyq_col);
    green_tiles64_kernel<<<148 * 8, 256, 0, st>>>(tiles, green, g_pb, g_pp, Pb, nct, nyq_col, total);
    return cudaGetLastError();
}

cudaError_t launch_fast64(int mode, const Fast64Params& p, const TileMap& in_map, cudaStream_t st)
{
    const CUtensorMap& tm = reinterpret_cast<const CUtensorMap&>(in_map);
    if (p.nct <= 0 || (1 << p.nct_shift) != p.nct || p.nb <= 0) return cudaErrorInvalidValue;
    // the kernels index with 32-bit element offsets
    if ((long long)p.nb * p.in_bs + 512 * p.in_ps >= (1ll << 31) || (long long)p.nb * p.out_bs + 512 * p.out_ps >= (1ll << 31))
        return cudaErrorInvalidValue;
    if (mode == FMODE_FUSED && !p.green_tiles) return cudaErrorInvalidValue;
    const int ntiles = p.nb * p.nct + (p.nyq_col >= 0 ? (p.nb + kTile64 - 1) / kTile64 : 0);
    int grid = 2 * g_sms;
    if (grid > ntiles) grid = ntiles;
    switch (mode) {
    case FMODE_FWD: fast64_kernel<FMODE_FWD><<<grid, kT64, kSmem64, st>>>(p, tm); break;
    case FMODE_INV: fast64_kernel<FMODE_INV><<<grid, kT64, kSmem64NoSlot, st>>>(p, tm); break;
    case FMODE_FUSED: fast64_kernel<FMODE_FUSED><<<grid, kT64, kSmem64, st>>>(p, tm); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

namespace {
template <int KIND, int MODE> cudaError_t launch_r64(const FastR64Params& p, const CUtensorMap& tm, int grid, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(fast_r2r64_kernel<KIND, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemR64);
    if (e != cudaSuccess) return e;
    fast_r2r64_kernel<KIND, MODE><<<grid, kT64, kSmemR64, st>>>(p, tm);
    return cudaGetLastError();
}
} // namespace

cudaError_t launch_fast_r2r64(int kind, int mode, const FastR64Params& p, const TileMap& in_map, cudaStream_t st)
{
    const CUtensorMap& tm = reinterpret_cast<const CUtensorMap&>(in_map);
    if (p.nb <= 0 || p.nct <= 0 || (kind == R2RK_DST1 && p.n != 255) || (kind == R2RK_DCT && p.n != 256)) return cudaErrorInvalidValue;
    if (kind == R2RK_DST1 && mode == RMODE_INV) return cudaErrorInvalidValue;   // DST-I is its own inverse: use RMODE_FWD
    if (mode == RMODE_FUSED && (!p.lam_x || !p.lam_b || !p.lam_p)) return cudaErrorInvalidValue;
    const long long ntiles = (long long)p.nb * p.nct;
    if (ntiles + 4ll * g_sms >= (1ll << 31)) return cudaErrorInvalidValue;
    int grid = 2 * g_sms;
    if (grid > ntiles) grid = (int)ntiles;
    if (kind == R2RK_DST1) {
        if (mode == RMODE_FWD) return launch_r64<R2RK_DST1, RMODE_FWD>(p, tm, grid, st);
        return launch_r64<R2RK_DST1, RMODE_FUSED>(p, tm, grid, st);
    }
    if (mode == RMODE_FWD) return launch_r64<R2RK_DCT, RMODE_FWD>(p, tm, grid, st);
    if (mode == RMODE_INV) return launch_r64<R2RK_DCT, RMODE_INV>(p, tm, grid, st);
    if (mode == RMODE_FUSED) return launch_r64<R2RK_DCT, RMODE_FUSED>(p, tm, grid, st);
    return cudaErrorInvalidValue;
}

cudaError_t launch_fast_per(int mode, const FastPerParams& p, cudaStream_t st)
{
    if (p.nyq_col >= 0 && !p.nyq) return cudaErrorInvalidValue;
    if (p.nct <= 0 || p.nb <= 0) return cudaErrorInvalidValue;
    if ((long long)p.nb * p.in_bs + 256 * p.in_ps >= (1ll << 31) || (long long)p.nb * p.out_bs + 256 * p.out_ps >= (1ll << 31))
        return cudaErrorInvalidValue;
    if (p.grad && ((long long)p.nb * p.out_bs + 256 * p.out_ps + 3 * p.out_cs >= (1ll << 31) || mode != FMODE_FUSED)) return cudaErrorInvalidValue;
    const int ntiles = p.nb * p.nct + (p.nyq_col >= 0 ? (p.nb + kPerTile - 1) / kPerTile : 0);
    int grid = 2 * g_sms;
    if (grid > ntiles) grid = ntiles;
    switch (mode) {
    case FMODE_FWD: fast_per_kernel<FMODE_FWD><<<grid, kThreads, kPerSmem, st>>>(p); break;
    case FMODE_INV: fast_per_kernel<FMODE_INV><<<grid, kThreads, kPerSmem, st>>>(p); break;
    case FMODE_FUSED:
        if (p.grad) {
            // one CTA per SM (96 registers per thread)
            if (grid > g_sms) grid = g_sms;
            fast_per_kernel<FMODE_FUSED, true><<<grid, kThreads, kPerSmem, st>>>(p);
        } else {
            fast_per_kernel<FMODE_FUSED><<<grid, kThreads, kPerSmem, st>>>(p);
        }
        break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_fast_per64(int mode, const FastPer64Params& p, cudaStream_t st)
{
    if (p.nyq_col >= 0 && !p.nyq) return cudaErrorInvalidValue;
    if (p.nct <= 0 || p.nb <= 0) return cudaErrorInvalidValue;
    if (p.grad && mode != FMODE_FUSED) return cudaErrorInvalidValue;
    if (mode == FMODE_FUSED && (!p.lam_x || !p.lam_b || !p.lam_p || (p.grad && (!p.kap_x || !p.kap_b || !p.kap_p)))) return cudaErrorInvalidValue;
    const long long ntiles = (long long)p.nb * p.nct + (p.nyq_col >= 0 ? (p.nb + kPer64Tile - 1) / kPer64Tile : 0);
    if (ntiles + 4ll * g_sms >= (1ll << 31)) return cudaErrorInvalidValue;
    int grid = 2 * g_sms;
    if (grid > ntiles) grid = (int)ntiles;
    cudaError_t e = cudaSuccess;
    switch (mode) {
    case FMODE_FWD:
        if ((e = cudaFuncSetAttribute(fast_per64_kernel<FMODE_FWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPer64Smem)) != cudaSuccess) return e;
        fast_per64_kernel<FMODE_FWD><<<grid, kT64, kPer64Smem, st>>>(p);
        break;
    case FMODE_INV:
        if ((e = cudaFuncSetAttribute(fast_per64_kernel<FMODE_INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPer64Smem)) != cudaSuccess) return e;
        fast_per64_kernel<FMODE_INV><<<grid, kT64, kPer64Smem, st>>>(p);
        break;
    case FMODE_FUSED:
        if (p.grad) {
            if ((e = cudaFuncSetAttribute(fast_per64_kernel<FMODE_FUSED, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPer64Smem)) != cudaSuccess) return e;
            fast_per64_kernel<FMODE_FUSED, true><<<grid, kT64, kPer64Smem, st>>>(p);
        } else {
            if ((e = cudaFuncSetAttribute(fast_per64_kernel<FMODE_FUSED>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPer64Smem)) != cudaSuccess) return e;
            fast_per64_kernel<FMODE_FUSED><<<grid, kT64, kPer64Smem, st>>>(p);
        }
        break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_fast_xper(bool inv, const FastXPerParams& p, cudaStream_t st)
{
    if (p.nrows <= 0 || p.nrows % kXpRows || !p.nyq) return cudaErrorInvalidValue;
    int grid = 2 * g_sms;
    // one pipeline per warp (sf_fastxw.cuh; its bulk copies want 16-byte aligned spectrum rows); SF_X_CTA=1 selects
    // the kernel with one pipeline per CTA
    const bool cta_kernel = (getenv("SF_X_CTA") != nullptr);
    if (!cta_kernel && p.spec_pitch % 2 == 0 && (reinterpret_cast<unsigned long long>(p.spec) & 15ull) == 0ull &&
        (reinterpret_cast<unsigned long long>(inv ? (const void*)p.real_out : (const void*)p.real_in) & 15ull) == 0ull) {
        const int need = (p.nrows / 4 + kXwWarps - 1) / kXwWarps;
        if (grid > need) grid = need;
        if (inv) fast_xpw_kernel<true><<<grid, kXwThreads, kXpwSmemInv, st>>>(p);
        else fast_xpw_kernel<false><<<grid, kXwThreads, kXpwSmemFwd, st>>>(p);
        return cudaGetLastError();
    }
    if (grid > p.nrows / kXpRows) grid = p.nrows / kXpRows;
    if (inv) fast_xper_kernel<true><<<grid, kXpThreads, kXpSmem, st>>>(p);
    else fast_xper_kernel<false><<<grid, kXpThreads, kXpSmem, st>>>(p);
    return cudaGetLastError();
}

namespace {
template <int MODE, bool INV> cudaError_t launch_xgw(const sf::XParams<double>& p, int ncomp, cudaStream_t st)
{
    constexpr size_t sm = xw64_smem<MODE, INV>();
    const long long npairs = ((long long)p.ny * p.nz + 1) / 2;
    long long gx = 2ll * g_sms;
    if (gx > (npairs + kXw64Warps - 1) / kXw64Warps) gx = (npairs + kXw64Warps - 1) / kXw64Warps;
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(fast_xgw_kernel<MODE, INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)) != cudaSuccess) return e;
    fast_xgw_kernel<MODE, INV><<<dim3((unsigned)gx, (unsigned)ncomp), kXw64Threads, sm, st>>>(p);
    return cudaGetLastError();
}
template <int MODE> cudaError_t launch_xg_mode(bool inv, const sf::XParams<double>& p, int ncomp, cudaStream_t st)
{
    // one pipeline per warp (sf_fastxw64.cuh); SF_X_CTA=1 selects the kernel with one pipeline per CTA
    const bool cta_kernel = (getenv("SF_X_CTA") != nullptr);
    if (!cta_kernel) return inv ? launch_xgw<MODE, true>(p, ncomp, st) : launch_xgw<MODE, false>(p, ncomp, st);
    const long long ntiles = ((long long)p.ny * p.nz + kXgRows - 1) / kXgRows;
    long long gx = 4ll * g_sms;
    if (gx > ntiles) gx = ntiles;
    const dim3 grid((unsigned)gx, (unsigned)ncomp);
    cudaError_t e;
    if (inv) {
        constexpr size_t sm = xg_smem<MODE, true>();
        if ((e = cudaFuncSetAttribute(fast_xg_kernel<MODE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)) != cudaSuccess) return e;
        fast_xg_kernel<MODE, true><<<grid, kXgThreads, sm, st>>>(p);
    } else {
        constexpr size_t sm = xg_smem<MODE, false>();
        if ((e = cudaFuncSetAttribute(fast_xg_kernel<MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)) != cudaSuccess) return e;
        fast_xg_kernel<MODE, false><<<grid, kXgThreads, sm, st>>>(p);
    }
    return cudaGetLastError();
}
} // namespace

cudaError_t launch_fast_xg(bool inv, const sf::XParams<double>& p, int ncomp, cudaStream_t st)
{
    if (p.nyq_side || p.dfield1 || p.ny <= 0 || p.nz <= 0 || ncomp <= 0 || g_sms <= 0) return cudaErrorInvalidValue;
    switch (p.mode) {
    case sf::X_ZEROPAD: return p.n == 256 ? launch_xg_mode<sf::X_ZEROPAD>(inv, p, ncomp, st) : cudaErrorInvalidValue;
    case sf::X_DST1: return p.n == 255 ? launch_xg_mode<sf::X_DST1>(inv, p, ncomp, st) : cudaErrorInvalidValue;
    case sf::X_DCT2: return (p.n == 256 && p.ptw) ? launch_xg_mode<sf::X_DCT2>(inv, p, ncomp, st) : cudaErrorInvalidValue;
    default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_fast_xp64(bool inv, const sf::XParams<double>& p, int ncomp, cudaStream_t st)
{
    if (p.mode != sf::X_PERIODIC || p.n != 256 || p.nyq_side_yz || p.dfield1 || p.has_faces || p.ny <= 0 || p.nz <= 0 || ncomp <= 0 || g_sms <= 0)
        return cudaErrorInvalidValue;
    // one pipeline per warp (sf_fastxw64.cuh); SF_X_CTA=1 selects the kernel with one pipeline per CTA
    const bool cta_kernel = (getenv("SF_X_CTA") != nullptr);
    if (!cta_kernel) {
        const long long nquads = ((long long)p.ny * p.nz + 3) / 4;
        long long gw = 2ll * g_sms;
        if (gw > (nquads + kXw64Warps - 1) / kXw64Warps) gw = (nquads + kXw64Warps - 1) / kXw64Warps;
        const dim3 gridw((unsigned)gw, (unsigned)ncomp);
        cudaError_t ew;
        if (inv) {
            if ((ew = cudaFuncSetAttribute(fast_xpw64_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXpw64Smem)) != cudaSuccess) return ew;
            fast_xpw64_kernel<true><<<gridw, kXw64Threads, kXpw64Smem, st>>>(p);
        } else {
            if ((ew = cudaFuncSetAttribute(fast_xpw64_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXpw64Smem)) != cudaSuccess) return ew;
            fast_xpw64_kernel<false><<<gridw, kXw64Threads, kXpw64Smem, st>>>(p);
        }
        return cudaGetLastError();
    }
    const long long ntiles = ((long long)p.ny * p.nz + kXp64Rows - 1) / kXp64Rows;
    long long gx = 4ll * g_sms;
    if (gx > ntiles) gx = ntiles;
    const dim3 grid((unsigned)gx, (unsigned)ncomp);
    cudaError_t e;
    if (inv) {
        if ((e = cudaFuncSetAttribute(fast_xp64_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXp64Smem)) != cudaSuccess) return e;
        fast_xp64_kernel<true><<<grid, kXp64Threads, kXp64Smem, st>>>(p);
    } else {
        if ((e = cudaFuncSetAttribute(fast_xp64_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXp64Smem)) != cudaSuccess) return e;
        fast_xp64_kernel<false><<<grid, kXp64Threads, kXp64Smem, st>>>(p);
    }
    return cudaGetLastError();
}

cudaError_t launch_fast_x5(bool inv, const FastXParams& p, cudaStream_t st)
{
    if (p.nrows <= 0 || p.nrows % kX5Rows || p.spec_pitch < kX5SpPitch || p.nyq) return cudaErrorInvalidValue;
    int grid = 2 * g_sms;
    // one pipeline per warp (sf_fastx5w.cuh; its bulk copies want 16-byte aligned spectrum rows); SF_X_CTA=1 selects
    // the kernel with one pipeline per CTA
    const bool cta_kernel = (getenv("SF_X_CTA") != nullptr);
    if (!cta_kernel && p.spec_pitch % 2 == 0 && (reinterpret_cast<unsigned long long>(p.spec) & 15ull) == 0ull) {
        const int need = (p.nrows + kX5wWarps - 1) / kX5wWarps;
        if (grid > need) grid = need;
        if (inv) fast_x5w_kernel<true><<<grid, kX5wThreads, kX5wSmemInv, st>>>(p);
        else fast_x5w_kernel<false><<<grid, kX5wThreads, kX5wSmemFwd, st>>>(p);
        return cudaGetLastError();
    }
    if (grid > p.nrows / kX5Rows) grid = p.nrows / kX5Rows;
    if (inv) fast_x5_kernel<true><<<grid, kX5Threads, kX5Smem, st>>>(p);
    else fast_x5_kernel<false><<<grid, kX5Threads, kX5Smem, st>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_fast_x(bool inv, const FastXParams& p, cudaStream_t st)
{
    if (p.nrows <= 0 || p.nrows % kXRows) return cudaErrorInvalidValue;
    int grid = 2 * g_sms;
    // one pipeline per warp (sf_fastxw.cuh); SF_X_CTA=1 selects the kernel with one pipeline per CTA
    const bool cta_kernel = (getenv("SF_X_CTA") != nullptr);
    if (!cta_kernel) {
        const int nwarps = xw_warps(inv);
        const int need = (p.nrows / 2 + nwarps - 1) / nwarps;
        if (grid > need) grid = need;
        if (inv) fast_xw_kernel<true><<<grid, 32 * nwarps, kXwSmemInv, st>>>(p);
        else fast_xw_kernel<false><<<grid, 32 * nwarps, kXwSmemFwd, st>>>(p);
        return cudaGetLastError();
    }
    if (grid > p.nrows / kXRows) grid = p.nrows / kXRows;
    if (inv) fast_x_kernel<true><<<grid, kXThreads, kXSmem, st>>>(p);
    else fast_x_kernel<false><<<grid, kXThreads, kXSmem, st>>>(p);
    return cudaGetLastError();
}

} // namespace sf2
