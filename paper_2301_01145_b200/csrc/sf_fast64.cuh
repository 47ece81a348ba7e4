// sf_fast64.cuh -- kernel generation 2 in double precision: the strided passes S2 (Y forward), S3 (Z forward x
// Green x Z backward, fused) and S4 (Y backward) of unbounded plans with 256-long y / z pencils zero-padded to 512
// (PAPER.md:89-97 pencils, :103-109 four-step solve, :181 / :213 padded and pruned Hockney-Eastwood transforms;
// BASELINE.json configs[3] in fp64).
//
// The register-resident design of sf_fast.cuh with 16-byte elements.  A tile is 8 neighbouring pencils (8 complex
// doubles = one 128-byte run per row, as 16 pencils are in fp32).  A CTA has 256 threads: half-warp = residue o of
// the 256-point transform (16 of them), its 16 lanes = 8 pencils x 2 halves h of the padded problem (the 512-point
// transform of (x, 0) is two 256-point transforms, of x and of x w512^n; the truncated backward transform is the
// mirror).  A thread holds the 16 elements n = o + 16 r of its pencil: 64 registers of data, <= 128 in all, two CTAs
// per SM.  A 256-point transform is radix-16 in registers, twiddle, ONE exchange through shared memory (16-byte
// accesses, orientation alternating between consecutive transforms so that one barrier per transform suffices),
// radix-16 in registers; double-precision arithmetic is plain DADD / DMUL / DFMA.  Tiles of the forward and fused
// passes arrive by TMA (the tensor map addresses the array as 8-byte words, a tile row is 16 of them) in a 32 KB
// slot that is refilled as soon as the tile sits in registers; the backward pass loads straight into registers.
// Persistent CTAs, dynamic tile queue.  The Nyquist column (257 = 32 x 8 + 1) is handled 8 batches at a time with
// gathered 16-byte accesses (1 % of the tiles).
#pragma once
#include "sf_fast.cuh"

namespace sf2 {

constexpr int kT64 = 256;
constexpr int kTile64 = 8;                      // pencils per tile
constexpr int kXchg64Elems = 16 * 16 * 16;      // complex doubles
constexpr int kSlot64Elems = kL * kTile64;
constexpr size_t kSmem64 = ((size_t)kXchg64Elems + kSlot64Elems) * sizeof(D);
constexpr size_t kSmem64NoSlot = (size_t)kXchg64Elems * sizeof(D);

// exp(-2 pi i j / 1024) in double precision
__constant__ double2 c_tw1024d[1024];

template <bool INV, bool ORIENT_B> __device__ __forceinline__ void fft256d_a(D (&v)[16], const D* tw256, D* x, int ea, int eb)
{
    dft16<INV>(v);
#pragma unroll
    for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul_sel<INV>(v[brev4(q)], tw256[q]);   // w256^(q o)
    D* w = x + (ORIENT_B ? eb : ea);
    constexpr int ws = (ORIENT_B ? 16 : 256);
#pragma unroll
    for (int q = 0; q < 16; ++q) w[q * ws] = v[brev4(q)];
}
template <bool INV, bool ORIENT_B> __device__ __forceinline__ void fft256d_b(D (&v)[16], const D* x, int ea, int eb)
{
    const D* r = x + (ORIENT_B ? ea : eb);
    constexpr int rs = (ORIENT_B ? 256 : 16);
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = r[i * rs];
    dft16<INV>(v);
}

// 1 / d for the spectral multipliers: hardware seed (rcp.approx.ftz.f64, ~20 bits) and two Newton steps, 1 - 2 ulp; about half
// the instructions of the correctly rounded __drcp_rn (no special-case branch: d is a finite, normal sum of eigenvalues,
// or zero at the zero mode, whose multiplier is replaced afterwards)
__device__ __forceinline__ double fast_rcp(double d)
{
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
    double e = fma(-d, x, 1.0);
    x = fma(x, e, x);
    e = fma(-d, x, 1.0);
    return fma(x, e, x);
}
__device__ __forceinline__ D ldg_d(const D* p)
{
    const double2 t = __ldg(reinterpret_cast<const double2*>(p));
    return t;
}

struct Geom64 { bool full; int b, col; };
__device__ __forceinline__ Geom64 tile_geom64(const Fast64Params& p, int t)
{
    Geom64 g;
    const int nnyq = (p.nyq_col >= 0) ? (p.nb + kTile64 - 1) / kTile64 : 0;
    if (t < nnyq) {               // the gathered tiles first: they are the slow ones
        g.full = false;
        g.b = t * kTile64;
        g.col = p.nyq_col;
    } else {
        const int tf = t - nnyq;
        int bi = tf >> p.nct_shift;
        if (p.reverse_batches) bi = p.nb - 1 - bi;
        else if (p.pair_batches) {   // 0, P/2, 1, P-1, 2, P-2, ...: mirror batches share their Green's chunk
            if (bi == 1) bi = p.nb / 2;
            else if (bi > 1) bi = (bi & 1) ? p.nb - (bi >> 1) : (bi >> 1);
        }
        g.full = true;
        g.b = bi;
        g.col = (tf & (p.nct - 1)) * kTile64;
    }
    return g;
}
__device__ __forceinline__ int green_tile_index64(const Fast64Params& p, const Geom64& g)
{
    if (g.full) return (min(g.b, p.Pb - g.b) << p.nct_shift) + (g.col / kTile64);
    return ((p.Pb / 2 + 1) << p.nct_shift) + (g.b / kTile64);
}

// MODE as in sf_fast.cuh: FMODE_FWD in rows n < 256 -> out rows k < 512; FMODE_INV in rows k < 512 -> out rows
// j < 256; FMODE_FUSED in rows n < 256 -> x Green -> out rows j < 256 (in place allowed).
// `tm` describes `in` as 8-byte words: FWD dims (2 column, row, batch, 1), box {16, 256, 1, 1}, coordinates
// {2 col, 0, b, 0}; FUSED dims (2 column, batch, row, 1), box {16, 1, 256, 1}, coordinates {2 col, b, 0, 0}.
template <int MODE>
__global__ void __launch_bounds__(kT64, 2) fast64_kernel(const Fast64Params p, const __grid_constant__ CUtensorMap tm)
{
    constexpr bool kTma = (MODE != FMODE_INV);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    D* xbuf = reinterpret_cast<D*>(smem_raw);
    D* slot = xbuf + kXchg64Elems;
    __shared__ __align__(8) uint64_t bar;
    __shared__ __align__(16) D s_t256[256];   // [o][q] = w256^(q o)
    __shared__ __align__(16) D s_t512[512];   // [h][o][r] = h ? w512^(o + 16 r) : 1
    __shared__ int s_tile[2];

    const int tid = threadIdx.x;
    const int l16 = tid & 15;
    const int pen = l16 & 7;
    const int h = l16 >> 3;
    const int o = tid >> 4;
    const int ea = o * 16 + l16;
    const int eb = o * 256 + l16;
    const D* t256 = s_t256 + o * 16;
    const D* t512 = s_t512 + (h * 16 + o) * 16;

    const int nnyq = (p.nyq_col >= 0) ? (p.nb + kTile64 - 1) / kTile64 : 0;
    const int ntiles = (p.nb << p.nct_shift) + nnyq;
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;
    uint32_t parity = 0;

    auto issue = [&](int t) {
        if (!kTma || tid != 0 || t >= ntiles) return;
        const Geom64 g = tile_geom64(p, t);
        if (!g.full) return;
        mbar_expect_tx(&bar, kSlot64Elems * (uint32_t)sizeof(D));
        if (MODE == FMODE_FWD) tma_load_4d(slot, &tm, 2 * g.col, 0, g.b, 0, &bar);
        else tma_load_4d(slot, &tm, 2 * g.col, g.b, 0, 0, &bar);
    };
    auto advance = [&](int it) {
        if (tid != 0) return;
        issue(s_tile[(it + 1) & 1]);
        s_tile[it & 1] = atomicAdd(p.sched, 1) + 2 * (int)gridDim.x;
    };
    // v[r] = x[o + 16 r] of this thread's pencil (FWD / FUSED)
    auto load_x = [&](const Geom64& g, D (&v)[16]) {
        if (g.full) {
            mbar_wait(&bar, parity);
            parity ^= 1;
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = slot[(o + 16 * r) * kTile64 + pen];
        } else {
            const D* inp = p.in + (min(g.b + pen, p.nb - 1) * ibs + g.col + o * ips);
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = ldg_d(inp + r * 16 * ips);
        }
    };

    auto tile = [&](int t, int it, auto orient_tag) {
        constexpr bool OB = decltype(orient_tag)::value;
        const Geom64 g = tile_geom64(p, t);
        const bool pvalid = g.full || (g.b + pen < p.nb);
        D* outp = p.out + (g.full ? (g.b * obs + g.col + pen) : ((g.b + pen) * obs + g.col));
        D v[16];
        if constexpr (MODE == FMODE_FWD) {
            load_x(g, v);
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], t512[r]);   // h = 1: x w512^n -> odd outputs
            fft256d_a<false, OB>(v, t256, xbuf, ea, eb);
            __syncthreads();
            advance(it);
            fft256d_b<false, OB>(v, xbuf, ea, eb);
            if (pvalid) {
                D* q = outp + (2 * o + h) * ops;   // row 2 (o + 16 k2) + h
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) q[k2 * 32 * ops] = v[brev4(k2)];
            }
        } else {
            if constexpr (MODE == FMODE_FUSED) {
                load_x(g, v);
#pragma unroll
                for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], t512[r]);
                fft256d_a<false, OB>(v, t256, xbuf, ea, eb);
                __syncthreads();
                advance(it);
                // Green's factors of the spectral rows kp = 2 (o + 16 k2) + h, folded to min(kp, 512 - kp); requested
                // here so that they arrive while the second half of the transform runs
                double gm[16];
                {
                    const double* gt = p.green_tiles + ((size_t)green_tile_index64(p, g) * (kGreenRows * kTile64) + pen);
                    const double* glo = gt + (2 * o + h) * kTile64;
                    const double* ghi = gt + (2 * kL - 2 * o - h) * kTile64;
#pragma unroll
                    for (int k2 = 0; k2 < 16; ++k2) gm[k2] = __ldg(k2 < 8 ? glo + k2 * 32 * kTile64 : ghi - k2 * 32 * kTile64);
                }
                fft256d_b<false, OB>(v, xbuf, ea, eb);
                D u[16];
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) u[k2] = cscale(v[brev4(k2)], gm[k2]);
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) v[k2] = u[k2];
                fft256d_a<true, !OB>(v, t256, xbuf, ea, eb);
                __syncthreads();
                fft256d_b<true, !OB>(v, xbuf, ea, eb);
            } else {
                // rows 2 k + h, k = o + 16 k2: h = 0 even spectrum, h = 1 odd spectrum
                const D* inp = p.in + ((g.full ? (g.b * ibs + g.col + pen) : (min(g.b + pen, p.nb - 1) * ibs + g.col)) + (2 * o + h) * ips);
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) v[k2] = ldg_d(inp + k2 * 32 * ips);
                fft256d_a<true, OB>(v, t256, xbuf, ea, eb);
                __syncthreads();
                advance(it);
                fft256d_b<true, OB>(v, xbuf, ea, eb);
            }
            // x_j = e_j + conj(w512^j) o_j, j = o + 16 r: h = 0 holds e, h = 1 holds o; the two lanes swap half of
            // their values: h = 0 finishes r < 8, h = 1 finishes r >= 8
            D* q = outp + (o + 128 * h) * ops;
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const D tl = cmulc(v[brev4(r)], t512[r]), th = cmulc(v[brev4(r + 8)], t512[r + 8]);   // (h = 0: times one)
                const D send = h ? tl : th;
                const D keep = h ? th : tl;
                D recv;
                recv.x = __shfl_xor_sync(0xffffffffu, send.x, 8);
                recv.y = __shfl_xor_sync(0xffffffffu, send.y, 8);
                const D x = cadd(keep, recv);
                if (pvalid) q[r * 16 * ops] = x;
            }
        }
    };

    if (tid == 0) {
        if (kTma) {
            mbar_init(&bar, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        s_tile[0] = (int)blockIdx.x;
        s_tile[1] = (int)(blockIdx.x + gridDim.x);
        issue(s_tile[0]);
    }
    s_t256[tid] = c_tw1024d[(4 * (tid & 15) * (tid >> 4)) & 1023];
    s_t512[tid] = make_double2(1.0, 0.0);
    s_t512[256 + tid] = c_tw1024d[2 * ((tid >> 4) + 16 * (tid & 15))];
    __syncthreads();
    if constexpr (MODE == FMODE_FUSED) {
        for (int it = 0;; ++it) {
            const int t = s_tile[it & 1];
            if (t >= ntiles) break;
            tile(t, it, std::false_type());
        }
    } else {
        for (int it = 0;; it += 2) {
            int t = s_tile[0];
            if (t >= ntiles) break;
            tile(t, it, std::false_type());
            t = s_tile[1];
            if (t >= ntiles) break;
            tile(t, it + 1, std::true_type());
        }
    }
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(p.sched + 1, 1) == (int)gridDim.x - 1) {
            p.sched[0] = 0;
            p.sched[1] = 0;
            __threadfence();
        }
    }
}

// re-lay the compact table green[fp][fb][kx] tile-major: chunk [kGreenRows fp][8 pencils] per tile, full tiles
// (fb, column tile) first, then the Nyquist-column tiles (8 batches each)
__global__ void green_tiles64_kernel(double* tiles, const double* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                                     long long total)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int pen = (int)(i % kTile64);
        const int fp = (int)((i / kTile64) % kGreenRows);
        const long long t = i / ((long long)kTile64 * kGreenRows);
        const long long nfull = (long long)(Pb / 2 + 1) * nct;
        int fb, kx;
        if (t < nfull) {
            fb = (int)(t / nct);
            kx = (int)(t % nct) * kTile64 + pen;
        } else {
            const int kb = min((int)(t - nfull) * kTile64 + pen, Pb - 1);
            fb = min(kb, Pb - kb);
            kx = nyq_col;
        }
        tiles[i] = green[kx + fb * g_pb + fp * g_pp];
    }
}

} // namespace sf2
