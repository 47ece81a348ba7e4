// sf_fast.cuh -- kernel generation 2 for the fp32 hot sizes: register-resident radix-16 FFTs on
// packed fp32x2 arithmetic, tiles streamed through shared memory by the bulk-copy engine.
//
// Same steps as sf_spass.cuh (S2 Y forward, S3 Z forward x multiplier x Z backward, S4 Y backward;
// PAPER.md:89-97 pencils, :103-109 four-step solve, :181 / :213 padded and pruned Hockney-Eastwood
// transforms), specialised to complex pencils of length 256 that are zero-padded to 512
// (unbounded, PAD) or transformed as they are (periodic).
//
// Mapping.  A CTA of 256 threads owns a tile of 16 neighbouring pencils (16 complex columns = one
// 128-byte run per row).  Lane bits 0..3 = pencil, lane bit 4 and the warp index = o in 0..15:
// thread (o, pencil) holds the 16 elements n = o + 16 r of its pencil in registers.  A 256-point
// transform is
//     radix-16 DFT over r (registers)  ->  twiddle w256^(q o)  ->  ONE shared-memory exchange
//     (q, o) -> (o, o')  ->  radix-16 DFT over o' (registers)
// and leaves X[o + 16 k2] in thread (o, pencil): input and output distributions are the same, so
// forward, multiply and backward chain without any reordering.  Consecutive transforms alternate
// the orientation of the exchange buffer, which makes every location be rewritten by the thread
// that read it last: one __syncthreads per transform.
// Complex numbers live in aligned register pairs and all arithmetic is FADD2 / FMUL2 / FFMA2
// (one issue slot per complex add, two per complex multiply, +-i free as an operand swizzle).
//
// Zero padding never exists: the 512-point transform of (x, 0) is two 256-point transforms, of x
// (even outputs) and of x w512^n (odd outputs); the truncated backward transform is the mirror,
// x_j = IDFT256(E)_j + conj(w512^j) IDFT256(O)_j for j < 256.
//
// Tiles arrive by cp.async.bulk (one 128-byte row per copy, completion on an mbarrier) into a
// two-deep ring, issued one tile ahead by warp 0; results go from registers to global memory as
// 128-byte runs.  Two CTAs share an SM so that one computes while the other waits at its barrier.
#pragma once
#include "sf_fast_api.h"
#include <cuda.h>
#include <stdint.h>

namespace sf2 {

constexpr int kThreads = 256;
constexpr int kL = 256;              // transform length
constexpr int kTileElems = kL * kTile;

// exp(-2 pi i j / 1024), j < 1024 (this header is compiled into one translation unit: sf_fast.cu)
__constant__ float2 c_tw1024[1024];

// ------------------------------------------------------------------------------------ complex, packed
__device__ __forceinline__ C cadd(C a, C b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ C csub(C a, C b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
// a * w
__device__ __forceinline__ C cmul(C a, C w)
{
    const C t = __fmul2_rn(make_float2(a.y, a.x), make_float2(w.y, w.y));
    return __ffma2_rn(a, make_float2(w.x, w.x), make_float2(-t.x, t.y));
}
// a * conj(w)
__device__ __forceinline__ C cmulc(C a, C w)
{
    const C t = __fmul2_rn(make_float2(a.y, a.x), make_float2(w.y, w.y));
    return __ffma2_rn(a, make_float2(w.x, w.x), make_float2(t.x, -t.y));
}
template <bool CONJ> __device__ __forceinline__ C cmul_sel(C a, C w) { return CONJ ? cmulc(a, w) : cmul(a, w); }
__device__ __forceinline__ C cscale(C a, float s) { return __fmul2_rn(a, make_float2(s, s)); }
__device__ __forceinline__ C cmuli(C a) { return make_float2(-a.y, a.x); }
__device__ __forceinline__ C cmulmi(C a) { return make_float2(a.y, -a.x); }

// ------------------------------------------------------------------------------------ radix-16
__host__ __device__ constexpr double cos16(int i)
{
    constexpr double c[16] = { 1.0, 0.92387953251128675613, 0.70710678118654752440, 0.38268343236508977173,
                               0.0, -0.38268343236508977173, -0.70710678118654752440, -0.92387953251128675613,
                               -1.0, -0.92387953251128675613, -0.70710678118654752440, -0.38268343236508977173,
                               0.0, 0.38268343236508977173, 0.70710678118654752440, 0.92387953251128675613 };
    return c[i & 15];
}
__host__ __device__ constexpr double sin16(int i) { return cos16(i - 4); }

// d * exp(-/+ 2 pi i I16 / 16)   (forward: minus)
template <int I16, bool INV> __device__ __forceinline__ C mul_w16(C d)
{
    if constexpr (I16 == 0) {
        return d;
    } else if constexpr (I16 == 4) {
        return INV ? cmuli(d) : cmulmi(d);
    } else {
        constexpr float c = (float)cos16(I16);
        constexpr float s = (float)(INV ? sin16(I16) : -sin16(I16));
        return cmul(d, make_float2(c, s));
    }
}

__host__ __device__ constexpr int brev4(int q) { return ((q & 1) << 3) | ((q & 2) << 1) | ((q & 4) >> 1) | ((q & 8) >> 3); }

// radix-2 decimation-in-frequency recursion on v[0], v[S], ...: result q of the length-R DFT ends
// at v[bitrev_R(q) * S]
template <int R, int S, bool INV> struct dft_rec {
    template <int I> static __device__ __forceinline__ void level(C* v)
    {
        if constexpr (I < R / 2) {
            const C a = v[I * S], b = v[(I + R / 2) * S];
            v[I * S] = cadd(a, b);
            v[(I + R / 2) * S] = mul_w16<I * (16 / R), INV>(csub(a, b));
            level<I + 1>(v);
        }
    }
    static __device__ __forceinline__ void run(C* v)
    {
        level<0>(v);
        dft_rec<R / 2, S, INV>::run(v);
        dft_rec<R / 2, S, INV>::run(v + (R / 2) * S);
    }
};
template <int S, bool INV> struct dft_rec<1, S, INV> {
    static __device__ __forceinline__ void run(C*) {}
};
// v[0..16) natural order in; DFT output q at v[brev4(q)]
template <bool INV> __device__ __forceinline__ void dft16(C (&v)[16]) { dft_rec<16, 1, INV>::run(v); }

// ------------------------------------------------------------------------------------ 256-point transform
// Exchange buffer: 16 x 16 slots of kTile complex.  Orientation A: slot (a, b) at (a*16 + b)*kTile;
// thread o writes (q, o), reads (o, o').  Orientation B is the transpose.  `ea` / `eb` are the
// thread's two base offsets (o*16 + pencil with stride 256, o*256 + pencil with stride 16).
struct Xchg {
    C* base;
    int ea, eb;
};

// first half: radix-16 over r, twiddle, write.  v[r] = x[o + 16 r] in; nothing valid out.
template <bool INV, bool ORIENT_B> __device__ __forceinline__ void fft256_a(C (&v)[16], int o, const Xchg& x)
{
    dft16<INV>(v);
#pragma unroll
    for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul_sel<INV>(v[brev4(q)], c_tw1024[4 * q * o]);
    C* w = x.base + (ORIENT_B ? x.eb : x.ea);
    constexpr int ws = (ORIENT_B ? 16 : 256);
#pragma unroll
    for (int q = 0; q < 16; ++q) w[q * ws] = v[brev4(q)];
}
// second half (after a barrier): read, radix-16 over o'.  X[o + 16 k2] at v[brev4(k2)] out.
template <bool INV, bool ORIENT_B> __device__ __forceinline__ void fft256_b(C (&v)[16], const Xchg& x)
{
    const C* r = x.base + (ORIENT_B ? x.ea : x.eb);
    constexpr int rs = (ORIENT_B ? 256 : 16);
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = r[i * rs];
    dft16<INV>(v);
}

// ------------------------------------------------------------------------------------ async copies
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "WAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@p bra DONE_%=;\n\t"
                 "bra WAIT_%=;\n\t"
                 "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one TMA box of a rank-4 tensor map global -> shared (dense, no swizzle), completion counted in
// bytes on the mbarrier
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
                     smem_u32(dst)),
                 "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
                 : "memory");
}

// ------------------------------------------------------------------------------------ tiles
// tile -> (batch, first column) and per-pencil geometry
struct TileGeom {
    bool full;      // 16 neighbouring columns of one batch (bulk-copyable); else 16 batches of one column
    int b, col;     // first batch / first column
};
__device__ __forceinline__ int batch_order(const FastParams& p, int bi)
{
    if (!p.pair_batches) return bi;
    if (bi == 0) return 0;
    if (bi == 1) return p.nb / 2;
    const int j = bi >> 1;
    return (bi & 1) ? p.nb - j : j;
}
__device__ __forceinline__ TileGeom tile_geom(const FastParams& p, int t)
{
    TileGeom g;
    const int nfull = p.nb * p.nct;
    if (t < nfull) {
        g.full = true;
        g.b = batch_order(p, t / p.nct);
        g.col = (t % p.nct) * kTile;
    } else {
        g.full = false;
        g.b = (t - nfull) * kTile;
        g.col = p.nyq_col;
    }
    return g;
}

// ------------------------------------------------------------------------------------ the kernel
// PAD: pencils of 256 stored rows, transform length 512 (zero-padded / truncated).
//   FMODE_FWD   : in rows n < 256        -> out rows k < 512            (S2)
//   FMODE_INV   : in rows k < 512        -> out rows j < 256            (S4)
//   FMODE_FUSED : in rows n < 256 -> x Green -> out rows j < 256        (S3; in == out allowed)
// `tm` describes `in` as a rank-4 tensor whose box is one tile image [256 rows][16 columns]:
//   FWD   dims (column, row, batch, 1)         box {16, 256, 1, 1}   coordinates {col, 0, b, 0}
//   FUSED dims (column, batch, row, 1)         box {16, 1, 256, 1}   coordinates {col, b, 0, 0}
//   INV   dims (column, parity, row/2, batch)  box {16, 1, 256, 1}   coordinates {col, half, 0, b}
template <int MODE>
__global__ void __launch_bounds__(kThreads, 2) fast_pad_kernel(const FastParams p, const __grid_constant__ CUtensorMap tm)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* ring0 = reinterpret_cast<C*>(smem_raw);
    C* ring1 = ring0 + kTileElems;
    C* xbuf = ring1 + kTileElems;
    __shared__ __align__(8) uint64_t bars[2];

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int pen = lane & 15;
    const int o = ((tid >> 5) << 1) | (lane >> 4);
    Xchg xc;
    xc.base = xbuf;
    xc.ea = o * 16 + pen;
    xc.eb = o * 256 + pen;

    if (tid == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int ntiles = fast_ntiles(p.nb, p.nct, p.nyq_col);
    const int ips = (int)p.in_ps, ops = (int)p.out_ps;
    uint32_t ph0 = 0, ph1 = 0;   // parity to wait for on bars[0] / bars[1]

    // A "unit" is one 256-row tile image: FWD / FUSED: one per tile; INV: two per tile (even rows, odd rows).
    // issue the TMA load of unit (tile t, half hf) into ring[slot]: one thread, one instruction
    auto issue = [&](int t, int hf, int slot) {
        if (tid != 0 || t >= ntiles) return;
        const TileGeom g = tile_geom(p, t);
        if (!g.full) return;   // gathered synchronously by the consumer
        uint64_t* bar = &bars[slot];
        mbar_expect_tx(bar, kTileElems * (uint32_t)sizeof(C));
        C* dst = slot ? ring1 : ring0;
        if (MODE == FMODE_FWD) tma_load_4d(dst, &tm, g.col, 0, g.b, 0, bar);
        else if (MODE == FMODE_FUSED) tma_load_4d(dst, &tm, g.col, g.b, 0, 0, bar);
        else tma_load_4d(dst, &tm, g.col, hf, 0, g.b, bar);
    };
    // make unit (t, hf) readable in ring[slot]
    auto acquire = [&](const TileGeom& g, int hf, int slot) {
        if (g.full) {
            if (slot) { mbar_wait(&bars[1], ph1); ph1 ^= 1; }
            else { mbar_wait(&bars[0], ph0); ph0 ^= 1; }
        } else {
            C* dst = slot ? ring1 : ring0;
            const int rs = (MODE == FMODE_INV) ? 2 * ips : ips;
            for (int idx = tid; idx < kTileElems; idx += kThreads) {
                const int pp = idx & 15, row = idx >> 4;
                C v = make_float2(0.f, 0.f);
                if (g.b + pp < p.nb)
                    v = p.in[(long long)(g.b + pp) * p.in_bs + g.col + (MODE == FMODE_INV ? hf * ips : 0) + row * rs];
                dst[idx] = v;
            }
            __syncthreads();
        }
    };

    int t = blockIdx.x;
    if (MODE == FMODE_INV) { issue(t, 0, 0); issue(t, 1, 1); }
    else issue(t, 0, 0);

    int it = 0;
    for (; t < ntiles; t += gridDim.x, ++it) {
        const TileGeom g = tile_geom(p, t);
        const int tn = t + gridDim.x;
        // this thread's pencil: output pointer, validity
        const bool pvalid = g.full || (g.b + pen < p.nb);
        const long long ob = g.full ? ((long long)g.b * p.out_bs + g.col + pen) : ((long long)(g.b + pen) * p.out_bs + g.col);
        C* outp = p.out + ob;

        C v[16];
        if constexpr (MODE == FMODE_FWD) {
            const int slot = it & 1;
            issue(tn, 0, slot ^ 1);
            acquire(g, 0, slot);
            const C* xs = (slot ? ring1 : ring0) + o * kTile + pen;
            // even outputs: rows 2 (o + 16 k2)
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = xs[r * 16 * kTile];
            fft256_a<false, false>(v, o, xc);
            __syncthreads();
            fft256_b<false, false>(v, xc);
            if (pvalid) {
                C* q = outp + 2 * o * ops;
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) q[k2 * 32 * ops] = v[brev4(k2)];
            }
            // odd outputs: rows 2 (o + 16 k2) + 1
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = cmul(xs[r * 16 * kTile], c_tw1024[2 * (o + 16 * r)]);
            fft256_a<false, true>(v, o, xc);
            __syncthreads();
            fft256_b<false, true>(v, xc);
            if (pvalid) {
                C* q = outp + (2 * o + 1) * ops;
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) q[k2 * 32 * ops] = v[brev4(k2)];
            }
        } else if constexpr (MODE == FMODE_INV) {
            C e[16];
            acquire(g, 0, 0);
            {
                const C* xs = ring0 + o * kTile + pen;
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) v[k2] = xs[k2 * 16 * kTile];
            }
            fft256_a<true, false>(v, o, xc);
            __syncthreads();
            issue(tn, 0, 0);
            fft256_b<true, false>(v, xc);
#pragma unroll
            for (int r = 0; r < 16; ++r) e[r] = v[brev4(r)];
            acquire(g, 1, 1);
            {
                const C* xs = ring1 + o * kTile + pen;
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) v[k2] = xs[k2 * 16 * kTile];
            }
            fft256_a<true, true>(v, o, xc);
            __syncthreads();
            issue(tn, 1, 1);
            fft256_b<true, true>(v, xc);
            if (pvalid) {
                C* q = outp + o * ops;
#pragma unroll
                for (int r = 0; r < 16; ++r) q[r * 16 * ops] = cadd(e[r], cmulc(v[brev4(r)], c_tw1024[2 * (o + 16 * r)]));
            }
        } else {
            // fused: forward (padded), multiply by the Green's spectrum, backward (truncated)
            const int slot = it & 1;
            issue(tn, 0, slot ^ 1);
            acquire(g, 0, slot);
            const C* xs = (slot ? ring1 : ring0) + o * kTile + pen;
            // table pointer of this thread's pencil: row fb = min(kb, Pb - kb), column kx
            const int kb = g.full ? g.b : min(g.b + pen, p.nb - 1);
            const int kx = g.full ? g.col + pen : g.col;
            const float* gp = p.green + (long long)min(kb, p.Pb - kb) * p.g_pb + kx;
            const int gpp = (int)p.g_pp;
            float gm[16];
            C e[16];
            // ---- even half of the spectrum: kp = 2 (o + 16 k2), folded to min(kp, 512 - kp)
            {
                const float* glo = gp + 2 * o * gpp;               // kp = 2 o + 32 k2        (k2 < 8)
                const float* ghi = gp + (2 * kL - 2 * o) * gpp;    // 512 - kp, kp = 2 o + 32 k2 (k2 >= 8)
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) gm[k2] = __ldg(k2 < 8 ? glo + k2 * 32 * gpp : ghi - k2 * 32 * gpp);
            }
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = xs[r * 16 * kTile];
            fft256_a<false, false>(v, o, xc);
            __syncthreads();
            fft256_b<false, false>(v, xc);
            {
                C u[16];
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) u[k2] = cscale(v[brev4(k2)], gm[k2]);
                fft256_a<true, true>(u, o, xc);
                __syncthreads();
                fft256_b<true, true>(u, xc);
#pragma unroll
                for (int r = 0; r < 16; ++r) e[r] = u[brev4(r)];
            }
            // ---- odd half: kp = 2 (o + 16 k2) + 1
            {
                const float* glo = gp + (2 * o + 1) * gpp;
                const float* ghi = gp + (2 * kL - 2 * o - 1) * gpp;
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) gm[k2] = __ldg(k2 < 8 ? glo + k2 * 32 * gpp : ghi - k2 * 32 * gpp);
            }
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = cmul(xs[r * 16 * kTile], c_tw1024[2 * (o + 16 * r)]);
            fft256_a<false, false>(v, o, xc);
            __syncthreads();
            fft256_b<false, false>(v, xc);
            {
                C u[16];
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) u[k2] = cscale(v[brev4(k2)], gm[k2]);
                fft256_a<true, true>(u, o, xc);
                __syncthreads();
                fft256_b<true, true>(u, xc);
                if (pvalid) {
                    C* q = outp + o * ops;
#pragma unroll
                    for (int r = 0; r < 16; ++r) q[r * 16 * ops] = cadd(e[r], cmulc(u[brev4(r)], c_tw1024[2 * (o + 16 * r)]));
                }
            }
        }
    }
}

} // namespace sf2
