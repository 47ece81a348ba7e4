// sf_tcprobe.cuh -- the measurement behind "no tensor cores" (BASELINE.json north_star:
// "Tensor cores are used only if a DFT-as-matmul stage demonstrably wins on ncu").
//
// The candidate stage is the second radix-16 stage of the register-resident 256-point transform of sf_fast.cuh
// (the N-D transform is a succession of 1-D pencil transforms; this is one half of one of them):
// every thread has written its 16 twiddled first-stage values to the exchange buffer and needs the 16-point DFT
// of the 16 values the buffer now holds for it.  Two implementations of exactly that stage, in one kernel body so
// that everything around it is identical:
//   variant 0  ALU: 16 shared-memory stores, barrier, 16 loads, radix-16 butterflies on packed fp32x2
//              (dft16 of sf_fast.cuh: 84 packed instructions) -- what the product kernels do;
//   variant 1  tensor cores, 3 x TF32: the values are split into a TF32 high part and the remainder (hi = x with the
//              low 13 mantissa bits cleared, lo = x - hi, exact), both written to shared memory in the canonical
//              K-major no-swizzle UMMA layout as a 512 x 32 real matrix X (row = (q, lane) = the consuming thread,
//              column = (o', re / im)); one thread issues tcgen05.mma kind::tf32, M = 128, N = 32, K = 8:
//              D = X_hi W_hi + X_lo W_hi + X_hi W_lo with W the 32 x 32 real form of the 16-point DFT matrix
//              (12 instructions per 128 rows), accumulators in tensor memory, tcgen05.commit on an mbarrier, and
//              every thread fetches its 32 results with one tcgen05.ld (32x32b.x32);
//   variant 2  tensor cores, 1 x TF32 (hi only; 1e-3 accuracy -- an upper bound on what the tensor path can gain).
// The stage is applied `reps` times to the same registers (scaled by 1/4 each time to keep the magnitudes), so that
// the launch measures the stage and nothing else.  One CTA of 512 threads per tile of 16 x 2 x 16 sequences, as in
// fast_pad_kernel; variants 1 / 2 need the exchange data twice (hi and lo): 128 KB, one CTA per SM.
#pragma once
#include "sf_fast.cuh"

#include <cmath>
#include <vector>

namespace sf2 {

namespace {

constexpr int kPT = 512;                      // threads per CTA
constexpr int kARows = 512, kAK = 32;         // X: 512 rows (16 q x 32 lanes), 32 reals per row
constexpr size_t kABytes = (size_t)kARows * kAK * 4;   // 64 KB per copy
constexpr size_t kBBytes = 32 * 32 * 4;                // 4 KB per copy
constexpr size_t kProbeSmemAlu = (size_t)16 * 16 * 32 * sizeof(C);
constexpr size_t kProbeSmemTc = 2 * kABytes + 2 * kBBytes + 1024;

// canonical K-major no-swizzle layout (units: bytes): 8 rows x 16 bytes = one 128-byte core matrix; the core
// matrices of one 8-row group are consecutive along K (LBO = 128), the groups follow each other (SBO = 8 * 128)
__host__ __device__ constexpr uint32_t canon_off(int row, int k)   // k = real column index
{
    return (uint32_t)((row >> 3) * (8 * 128) + (row & 7) * 16 + (k >> 2) * 128 + (k & 3) * 4);
}
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr)
{
    // start address >> 4 [0,14), LBO >> 4 [16,30), SBO >> 4 [32,46), version 1 [46,48), no swizzle
    return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46);
}
// kind::tf32, D fp32, A / B TF32 K-major, N = 32, M = 128
constexpr uint32_t kIdesc = (1u << 4) | (2u << 7) | (2u << 10) | ((32u >> 3) << 17) | ((128u >> 4) << 24);

__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(kIdesc),
                 "r"(accumulate)
                 : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld32f(uint32_t addr, float (&v)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]), "=f"(v[8]), "=f"(v[9]),
                   "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15]), "=f"(v[16]), "=f"(v[17]), "=f"(v[18]),
                   "=f"(v[19]), "=f"(v[20]), "=f"(v[21]), "=f"(v[22]), "=f"(v[23]), "=f"(v[24]), "=f"(v[25]), "=f"(v[26]), "=f"(v[27]),
                   "=f"(v[28]), "=f"(v[29]), "=f"(v[30]), "=f"(v[31])
                 : "r"(addr)
                 : "memory");
}

// VARIANT 0: in / out [tile][16][512] complex, element r of thread tid at ((tile * 16 + r) * 512 + tid); the stage maps
// the 16 values of a thread (its q-th value goes to thread q of the same lane) to the DFT over the source thread index.
template <int VARIANT> __global__ void __launch_bounds__(kPT, VARIANT == 0 ? 2 : 1) probe_kernel(const C* in, C* out, int ntiles, int reps, const float* wmat)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int o = tid >> 5;
    __shared__ __align__(8) uint64_t bar;
    __shared__ uint32_t s_tmem;
    unsigned char* a_hi = smem_raw;
    unsigned char* a_lo = smem_raw + kABytes;
    unsigned char* b_hi = smem_raw + 2 * kABytes;
    unsigned char* b_lo = b_hi + kBBytes;
    uint32_t tbase = 0;
    if (VARIANT != 0) {
        // W (real 32 x 32 form of the DFT matrix, row n = output column, K contiguous) in the canonical layout, hi and lo
        for (int i = tid; i < 32 * 32; i += kPT) {
            const int n = i >> 5, k = i & 31;
            const float w = wmat[n * 32 + k];
            const float hi = __uint_as_float(__float_as_uint(w) & 0xffffe000u);
            *reinterpret_cast<float*>(b_hi + canon_off(n, k)) = hi;
            *reinterpret_cast<float*>(b_lo + canon_off(n, k)) = w - hi;
        }
        if (tid == 0) {
            mbar_init(&bar, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        if (tid < 32) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(128u) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tbase = s_tmem;
    }
    uint32_t parity = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        C v[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = in[((size_t)tile * 16 + r) * kPT + tid];
        for (int rep = 0; rep < reps; ++rep) {
            if constexpr (VARIANT == 0) {
                C* xbuf = reinterpret_cast<C*>(smem_raw);
                // value q of thread o -> slot (q, o); thread o then reads slots (o, o'), o' < 16
#pragma unroll
                for (int q = 0; q < 16; ++q) xbuf[(q * 16 + o) * 32 + lane] = v[q];
                __syncthreads();
#pragma unroll
                for (int i = 0; i < 16; ++i) v[i] = xbuf[(o * 16 + i) * 32 + lane];
                __syncthreads();
                dft16<false>(v);
                // natural order, scaled
                C u[16];
#pragma unroll
                for (int k = 0; k < 16; ++k) u[k] = cscale(v[brev4(k)], 0.25f);
#pragma unroll
                for (int k = 0; k < 16; ++k) v[k] = u[k];
            } else {
                // X[row = (q, lane)][k = 2 o + c] = value q of thread o: hi and lo parts, 8 bytes each
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    const float hx = __uint_as_float(__float_as_uint(v[q].x) & 0xffffe000u);
                    const float hy = __uint_as_float(__float_as_uint(v[q].y) & 0xffffe000u);
                    const uint32_t off = canon_off(q * 32 + lane, 2 * o);
                    *reinterpret_cast<float2*>(a_hi + off) = make_float2(hx, hy);
                    if (VARIANT == 1) *reinterpret_cast<float2*>(a_lo + off) = make_float2(v[q].x - hx, v[q].y - hy);
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> tensor-core reads
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncthreads();
                if (tid == 0) {
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t ah = smem_u32(a_hi), al = smem_u32(a_lo), bh = smem_u32(b_hi), bl = smem_u32(b_lo);
#pragma unroll
                    for (int mb = 0; mb < 4; ++mb) {              // 128 rows each: q = 4 mb .. 4 mb + 3
                        const uint32_t d = tbase + (uint32_t)mb * 32;
                        const uint32_t arow = (uint32_t)mb * 16 * 1024;   // 16 groups of 8 rows
                        uint32_t acc = 0;
#pragma unroll
                        for (int ks = 0; ks < 4; ++ks) {          // K = 8 reals = two 16-byte chunks = 256 bytes along K
                            umma_tf32(d, umma_desc(ah + arow + ks * 256), umma_desc(bh + ks * 256), acc);
                            acc = 1;
                            if (VARIANT == 1) {
                                umma_tf32(d, umma_desc(al + arow + ks * 256), umma_desc(bh + ks * 256), 1);
                                umma_tf32(d, umma_desc(ah + arow + ks * 256), umma_desc(bl + ks * 256), 1);
                            }
                        }
                    }
                    umma_commit(&bar);
                }
                mbar_wait(&bar, parity);
                parity ^= 1;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                // thread (o, lane) owns row (o mod 4) * 32 + lane of block o / 4: TMEM lane quadrant o mod 4 = warp mod 4
                float d[32];
                tmem_ld32f(tbase + ((uint32_t)(o & 3) << 21) + (uint32_t)(o >> 2) * 32, d);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int k = 0; k < 16; ++k) v[k] = make_float2(0.25f * d[2 * k], 0.25f * d[2 * k + 1]);
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncthreads();   // the accumulators and the operand buffers are free again
            }
        }
#pragma unroll
        for (int r = 0; r < 16; ++r) out[((size_t)tile * 16 + r) * kPT + tid] = v[r];
    }
    if (VARIANT != 0) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tbase), "r"(128u) : "memory");
    }
}

} // namespace

// run `reps` stage applications on `ntiles` tiles (in / out: device, ntiles * 16 * 512 complex fp32 each); *ms = device
// time of the second of two launches (CUDA events).  variant as described at the top of this file.
cudaError_t probe_dft16_stage(int variant, int reps, int ntiles, const void* in, void* out, float* ms, cudaStream_t st)
{
    if (variant < 0 || variant > 2 || reps < 1 || ntiles < 1 || !in || !out) return cudaErrorInvalidValue;
    cudaError_t e;
    int dev = 0, sms = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    // real 32 x 32 form of the forward 16-point DFT, row n = 2 k2 + c' (output), column k = 2 o' + c (input)
    std::vector<float> w(32 * 32);
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int k2 = 0; k2 < 16; ++k2)
        for (int op = 0; op < 16; ++op) {
            const long double a = -2.0L * pi * (long double)((k2 * op) & 15) / 16.0L;
            const float wr = (float)cosl(a), wi = (float)sinl(a);
            w[(2 * k2 + 0) * 32 + 2 * op + 0] = wr;
            w[(2 * k2 + 0) * 32 + 2 * op + 1] = -wi;
            w[(2 * k2 + 1) * 32 + 2 * op + 0] = wi;
            w[(2 * k2 + 1) * 32 + 2 * op + 1] = wr;
        }
    float* dw = nullptr;
    if ((e = cudaMalloc(&dw, w.size() * sizeof(float))) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(dw, w.data(), w.size() * sizeof(float), cudaMemcpyHostToDevice, st)) != cudaSuccess) { cudaFree(dw); return e; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const size_t smem = variant == 0 ? kProbeSmemAlu : kProbeSmemTc;
    int grid = (variant == 0 ? 2 : 1) * sms;
    if (grid > ntiles) grid = ntiles;
    for (int pass = 0; pass < 2 && e == cudaSuccess; ++pass) {
        if (pass == 1) cudaEventRecord(e0, st);
        switch (variant) {
        case 0:
            cudaFuncSetAttribute(probe_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            probe_kernel<0><<<grid, kPT, smem, st>>>((const C*)in, (C*)out, ntiles, reps, dw);
            break;
        case 1:
            cudaFuncSetAttribute(probe_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            probe_kernel<1><<<grid, kPT, smem, st>>>((const C*)in, (C*)out, ntiles, reps, dw);
            break;
        default:
            cudaFuncSetAttribute(probe_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            probe_kernel<2><<<grid, kPT, smem, st>>>((const C*)in, (C*)out, ntiles, reps, dw);
            break;
        }
        e = cudaGetLastError();
        if (pass == 1) cudaEventRecord(e1, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess && ms) cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(dw);
    return e;
}

} // namespace sf2
