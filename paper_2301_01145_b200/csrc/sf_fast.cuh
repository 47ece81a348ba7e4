// sf_fast.cuh -- kernel generation 2 for the fp32 hot sizes: register-resident radix-16 FFTs on
// packed fp32x2 arithmetic, tiles streamed through shared memory by the bulk-copy engine.
//
// Same steps as sf_spass.cuh (S2 Y forward, S3 Z forward x multiplier x Z backward, S4 Y backward;
// PAPER.md:89-97 pencils, :103-109 four-step solve, :181 / :213 padded and pruned Hockney-Eastwood
// transforms), specialised to complex pencils of length 256 that are zero-padded to 512
// (unbounded plans).
//
// Mapping.  A CTA of 512 threads owns a tile of 16 neighbouring pencils (16 complex columns = one
// 128-byte run per row).  Warp index = o in 0..15 (warp-uniform, so every twiddle factor is a
// uniform-register or broadcast shared-memory operand); lane bits 0..3 = pencil; lane bit 4 = h
// selects which HALF of the padded problem the thread works on (below).  Thread (o, pencil, h) holds the 16 elements
// n = o + 16 r of its pencil in registers.  A 256-point transform is
//     radix-16 DFT over r (registers)  ->  twiddle w256^(q o)  ->  ONE shared-memory exchange
//     (q, o) -> (o, o')  ->  radix-16 DFT over o' (registers)
// and leaves X[o + 16 k2] in thread (o, pencil): input and output distributions are the same, so
// forward, multiply and backward chain without any reordering.  Consecutive transforms alternate
// the orientation of the exchange buffer, which makes every location be rewritten by the thread
// that read it last: one __syncthreads per transform.
// Complex numbers live in aligned register pairs and all arithmetic is FADD2 / FMUL2 / FFMA2
// (one instruction per complex add, two per complex multiply, +-i free as an operand swizzle; on
// this part a packed instruction costs two issue cycles, like the two scalar ones it replaces, so
// the gain is in instruction count and register moves -- profiles/r01_b.md).
//
// Zero padding never exists: the 512-point transform of (x, 0) is two 256-point transforms, of x
// (even outputs, h = 0) and of x w512^n (odd outputs, h = 1); the truncated backward transform is
// the mirror, x_j = IDFT256(E)_j + conj(w512^j) IDFT256(O)_j for j < 256.  The two halves run side
// by side in the two half-warps and meet in one warp shuffle at the end.
//
// Tiles of the forward and fused passes arrive by TMA (cp.async.bulk.tensor, one instruction per
// tile, completion on an mbarrier) in a shared-memory slot that is refilled for the next tile as
// soon as the current one sits in registers; the backward pass (tile image twice as large) loads
// straight into registers; results go from registers to global memory as 128-byte runs.
// Persistent CTAs, two per SM (64 registers per thread): the two CTAs are independent barrier
// domains, so one does arithmetic while the other exchanges, loads or stores.
#pragma once
#include "sf_trig.cuh"
#include "sf_fast_api.h"
#include <cuda.h>
#include <stdint.h>
#include <type_traits>

namespace sf2 {

constexpr int kThreads = 512;
constexpr int kL = 256;              // transform length
constexpr int kTileElems = kL * kTile;

// exp(-2 pi i j / 1024), j < 1024 (this header is compiled into one translation unit: sf_fast.cu)
__constant__ float2 c_tw1024[1024];
// (Re - 1, Im) of the same: 1 + h (w - 1) selects between w and one with one packed multiply-add
__constant__ float2 c_tw1024m1[1024];
// the per-kernel twiddle tables, laid out as the kernels keep them in shared memory (filled once by
// fast_init; a CTA copies them with coalesced 16-byte loads):
//   strided passes: [0, 256) tw256[o][q] = w256^(q o); [256, 768) tw512[h][o][r] = h ? w512^(o + 16 r) : 1
//   X passes:       [0, 128) tw128[w][q] = w128^(q w); [128, 384) twin[w][j][h] = h ? w256^(w + 8 j) : 1;
//                   [384, 544) twsp[w][m][h] = w512^(2 w + h + 16 m), m < 10  (h innermost: the two
//                   halves of a lane pair read one 16-byte word)
__device__ float2 g_tab_pad[768];
__device__ float2 g_tab_x[544];

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
// a * s + b
__device__ __forceinline__ C cfma(C a, float s, C b) { return __ffma2_rn(a, make_float2(s, s), b); }
__device__ __forceinline__ C cmuli(C a) { return make_float2(-a.y, a.x); }
__device__ __forceinline__ C cmulmi(C a) { return make_float2(a.y, -a.x); }

// ------------------------------------------------------------------------------------ radix-16
using sftrig::cos16;   // cos / sin of 2 pi i / 16 (sf_trig.cuh)
using sftrig::sin16;

// the same complex helpers for double precision (sf_fast64.cuh): plain DADD / DMUL / DFMA
typedef double2 D;
__device__ __forceinline__ D cadd(D a, D b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ D csub(D a, D b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ D cmul(D a, D w) { return make_double2(fma(a.x, w.x, -a.y * w.y), fma(a.x, w.y, a.y * w.x)); }
__device__ __forceinline__ D cmulc(D a, D w) { return make_double2(fma(a.x, w.x, a.y * w.y), fma(a.y, w.x, -a.x * w.y)); }
template <bool CONJ> __device__ __forceinline__ D cmul_sel(D a, D w) { return CONJ ? cmulc(a, w) : cmul(a, w); }
__device__ __forceinline__ D cscale(D a, double s) { return make_double2(a.x * s, a.y * s); }
__device__ __forceinline__ D cmuli(D a) { return make_double2(-a.y, a.x); }
__device__ __forceinline__ D cmulmi(D a) { return make_double2(a.y, -a.x); }
__device__ __forceinline__ C mk_c(C, double x, double y) { return make_float2((float)x, (float)y); }
__device__ __forceinline__ D mk_c(D, double x, double y) { return make_double2(x, y); }

// d * exp(-/+ 2 pi i I16 / 16)   (forward: minus)
template <int I16, bool INV, typename CT> __device__ __forceinline__ CT mul_w16(CT d)
{
    if constexpr (I16 == 0) {
        return d;
    } else if constexpr (I16 == 4) {
        return INV ? cmuli(d) : cmulmi(d);
    } else {
        constexpr double c = cos16(I16);
        constexpr double s = (INV ? sin16(I16) : -sin16(I16));
        return cmul(d, mk_c(CT(), c, s));
    }
}

__host__ __device__ constexpr int brev4(int q) { return ((q & 1) << 3) | ((q & 2) << 1) | ((q & 4) >> 1) | ((q & 8) >> 3); }

// radix-2 decimation-in-frequency recursion on v[0], v[S], ...: result q of the length-R DFT ends
// at v[bitrev_R(q) * S]
template <int R, int S, bool INV> struct dft_rec {
    template <int I, typename CT> static __device__ __forceinline__ void level(CT* v)
    {
        if constexpr (I < R / 2) {
            const CT a = v[I * S], b = v[(I + R / 2) * S];
            v[I * S] = cadd(a, b);
            v[(I + R / 2) * S] = mul_w16<I * (16 / R), INV>(csub(a, b));
            level<I + 1>(v);
        }
    }
    template <typename CT> static __device__ __forceinline__ void run(CT* v)
    {
        level<0>(v);
        dft_rec<R / 2, S, INV>::run(v);
        dft_rec<R / 2, S, INV>::run(v + (R / 2) * S);
    }
};
template <int S, bool INV> struct dft_rec<1, S, INV> {
    template <typename CT> static __device__ __forceinline__ void run(CT*) {}
};
// v[0..16) natural order in; DFT output q at v[brev4(q)]
template <bool INV, typename CT> __device__ __forceinline__ void dft16(CT (&v)[16]) { dft_rec<16, 1, INV>::run(v); }

// ------------------------------------------------------------------------------------ 256-point transform
// Exchange buffer: 16 x 16 slots of 32 complex (one per lane).  Orientation A: slot (a, b) at
// (a*16 + b)*32; thread o writes (q, o), reads (o, o').  Orientation B is the transpose.  `ea` /
// `eb` are the thread's two base offsets (o*32 + lane with stride 512, o*512 + lane with stride 32).
struct Xchg {
    C* base;
    int ea, eb;
};

// first half: radix-16 over r, twiddle, write.  v[r] = x[o + 16 r] in; nothing valid out.
// Twiddles come from a per-warp row of a shared-memory table: base register + immediate, no
// address arithmetic, and a latency the other warps cover.
// (TWC: from the constant bank through uniform registers instead -- ptxas does that for the fused
// and backward kernels, where it is cheaper than the shared-memory reads)
template <bool INV, bool ORIENT_B, bool TWC> __device__ __forceinline__ void fft256_a(C (&v)[16], const C* tw256, int o, const Xchg& x)
{
    dft16<INV>(v);
#pragma unroll
    for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul_sel<INV>(v[brev4(q)], TWC ? c_tw1024[4 * q * o] : tw256[q]);   // w256^(q o)
    C* w = x.base + (ORIENT_B ? x.eb : x.ea);
    constexpr int ws = (ORIENT_B ? 32 : 512);
#pragma unroll
    for (int q = 0; q < 16; ++q) w[q * ws] = v[brev4(q)];
}
// second half (after a barrier): read, radix-16 over o'.  X[o + 16 k2] at v[brev4(k2)] out.
template <bool INV, bool ORIENT_B> __device__ __forceinline__ void fft256_b(C (&v)[16], const Xchg& x)
{
    const C* r = x.base + (ORIENT_B ? x.ea : x.eb);
    constexpr int rs = (ORIENT_B ? 512 : 32);
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

// one contiguous run global -> shared, completion counted in bytes on the mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// one contiguous run shared -> global (bulk async-group completion)
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
// pull one 128-byte line towards the L2 (no register, no dependency); used where a pass loads its tiles straight into
// registers and a tile is large (sf_fast512.cuh S4: 1024 rows; measured: -4 %; no gain for the 256- / 512-row tiles)
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// all bulk stores of this thread have finished READING shared memory
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// generic-proxy writes to shared memory become visible to the async proxy (bulk stores)
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ------------------------------------------------------------------------------------ tiles
// tile -> (batch, first column) and per-pencil geometry
struct TileGeom {
    bool full;      // 16 neighbouring columns of one batch (bulk-copyable); else 16 batches of one column
    int b, col;     // first batch / first column
};
__device__ __forceinline__ int batch_order(const FastParams& p, int bi)
{
    if (p.reverse_batches) return p.nb - 1 - bi;   // consume the producer's most recent output first: it is still in L2
    if (!p.pair_batches) return bi;
    if (bi == 0) return 0;
    if (bi == 1) return p.nb / 2;
    const int j = bi >> 1;
    return (bi & 1) ? p.nb - j : j;
}
// chunk of the tile-major Green's table that belongs to a tile: full tiles (fb, column tile) first,
// then the Nyquist-column tiles (16 batches each)
__device__ __forceinline__ int green_tile_index(const FastParams& p, const TileGeom& g)
{
    if (g.full) return (min(g.b, p.Pb - g.b) << p.nct_shift) + (g.col >> 4);
    return ((p.Pb / 2 + 1) << p.nct_shift) + (g.b >> 4);
}
__device__ __forceinline__ TileGeom tile_geom(const FastParams& p, int t)
{
    // The few Nyquist-column tiles are gathered and cost about three full tiles each.  nyq_first puts
    // them at the head of the dynamic tile queue, where the CTAs that take one simply take fewer full
    // tiles afterwards; measured, that shortens the fused pass (225 -> 201 us) and lengthens the other
    // two, which keep them at the tail.
    TileGeom g;
    const int nfull = p.nb << p.nct_shift;   // nct is a power of two: no integer division per tile
    const int nnyq = (p.nyq_col >= 0) ? (p.nb + kTile - 1) / kTile : 0;
    const int tf = p.nyq_first ? t - nnyq : t;          // index among the full tiles
    const int tn = p.nyq_first ? t : t - nfull;         // index among the Nyquist tiles
    if (tf >= 0 && tf < nfull) {
        g.full = true;
        g.b = batch_order(p, tf >> p.nct_shift);
        g.col = (tf & (p.nct - 1)) * kTile;
    } else {
        g.full = false;
        g.b = tn * kTile;
        g.col = p.nyq_col;
    }
    return g;
}

// ------------------------------------------------------------------------------------ the kernel
// PAD: pencils of 256 stored rows, transform length 512 (zero-padded / truncated).
//   FMODE_FWD   : in rows n < 256        -> out rows k < 512            (S2)
//   FMODE_INV   : in rows k < 512        -> out rows j < 256            (S4)
//   FMODE_FUSED : in rows n < 256 -> x Green -> out rows j < 256        (S3; in == out allowed)
// `tm` describes `in` as a rank-4 tensor whose box is one tile image, rows of 16 columns:
//   FWD   dims (column, row, batch, 1)         box {16, 256, 1, 1}   coordinates {col, 0, b, 0}
//   FUSED dims (column, batch, row, 1)         box {16, 1, 256, 1}   coordinates {col, b, 0, 0}
// (INV reads its rows straight into registers and ignores `tm`.)
template <int MODE> struct FastCfg {
    // FWD / FUSED stage the next tile in one shared-memory slot by TMA while the current one is
    // being transformed; INV (tile image twice as large) loads straight into registers.
    static constexpr bool kTma = (MODE != FMODE_INV);
    static constexpr int kSlotElems = kTma ? kL * kTile : 0;
    static constexpr int kXchgElems = 16 * 16 * 32;
    static constexpr size_t kSmem = ((size_t)kSlotElems + kXchgElems) * sizeof(C);
};

template <int MODE>
__global__ void __launch_bounds__(kThreads, 2) fast_pad_kernel(const FastParams p, const __grid_constant__ CUtensorMap tm)
{
    typedef FastCfg<MODE> Cfg;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* xbuf = reinterpret_cast<C*>(smem_raw);
    C* slot = xbuf + Cfg::kXchgElems;
    __shared__ __align__(8) uint64_t bar;

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int pen = lane & 15;
    const int h = lane >> 4;
    const int o = (int)__reduce_max_sync(0xffffffffu, (unsigned)(tid >> 5));   // warp-uniform: REDUX lands in a uniform register
    Xchg xc;
    xc.base = xbuf;
    xc.ea = o * 32 + lane;
    xc.eb = o * 512 + lane;

    // twiddle tables: s_tw256[o][q] = w256^(q o);  s_tw512[h][o][r] = w512^(o + 16 r) for h = 1, 1 for h = 0
    __shared__ __align__(16) C s_tab[768];
    const C* t256 = s_tab + o * 16;
    const C* t512 = s_tab + 256 + (h * 16 + o) * 16;

    const int ntiles = fast_ntiles(p.nb, p.nct, p.nyq_col);
    // element offsets fit 32 bits: an eligible plan's work arrays hold < 2^31 complex numbers (checked by the launcher)
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;
    uint32_t parity = 0;   // phase of `bar` the next full tile completes
    // dynamic tile scheduling: a CTA's first two tiles are blockIdx.x and blockIdx.x + gridDim.x (no atomic in
    // the prologue), the rest come from p.sched[0] (+ 2 gridDim.x), the next unclaimed tile.  s_tile[it & 1] is the tile of
    // this CTA's iteration `it`; thread 0 claims the tile of iteration it + 2 once iteration it has
    // read its index (after its first barrier), so the index is always known one tile ahead for the
    // TMA prefetch and the atomic's latency is off the critical path.
    __shared__ int s_tile[2];

    // issue the TMA load of this CTA's iteration `i` into the slot: one thread, one instruction.
    // Tiles that are not 16 neighbouring columns (the Nyquist column) are loaded by their consumer.
    auto issue = [&](int t) {
        if (!Cfg::kTma || tid != 0 || t >= ntiles) return;
        const TileGeom g = tile_geom(p, t);
        if (!g.full) return;
        mbar_expect_tx(&bar, Cfg::kSlotElems * (uint32_t)sizeof(C));
        if (MODE == FMODE_FWD) tma_load_4d(slot, &tm, g.col, 0, g.b, 0, &bar);
        else tma_load_4d(slot, &tm, g.col, g.b, 0, 0, &bar);
    };
    // v[r] = x[o + 16 r] of this thread's pencil (FWD / FUSED), then mark the slot reusable
    auto load_x = [&](const TileGeom& g, C (&v)[16]) {
        if (g.full) {
            mbar_wait(&bar, parity);
            parity ^= 1;
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = slot[(o + 16 * r) * kTile + pen];
        } else if (p.nyq_in) {
            // Nyquist column from its side array [row][batch]: the 16 batches are contiguous
            const C* inp = p.nyq_in + (o * p.nb + g.b + pen);
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = __ldg(inp + r * 16 * p.nb);
        } else {
            const C* inp = p.in + (min(g.b + pen, p.nb - 1) * ibs + g.col + o * ips);
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = __ldg(inp + r * 16 * ips);
        }
    };
    // staging of a Nyquist tile image in the exchange buffer for a transposing copy: element
    // (row, pencil) at row * 16 + ((pencil + row) & 15) -- conflict-free both along pencils and along rows
    auto stage = [&](int row, int pencil) -> C& { return xbuf[row * kTile + ((pencil + row) & 15)]; };

    // after the first barrier of iteration `it` (every thread has its tile index and its elements of
    // the slot): prefetch the next tile, claim the one after
    auto advance = [&](int it) {
        if (tid != 0) return;
        issue(s_tile[(it + 1) & 1]);
        s_tile[it & 1] = atomicAdd(p.sched, 1) + 2 * (int)gridDim.x;
    };

    // one tile; ORIENT = orientation of the exchange buffer its first transform starts with
    auto tile = [&](int t, int it, auto orient_tag) {
        constexpr bool OB = decltype(orient_tag)::value;
        const TileGeom g = tile_geom(p, t);
        // this thread's pencil: output pointer, validity
        const bool pvalid = g.full || (g.b + pen < p.nb);
        const bool side = !g.full && p.nyq_in != nullptr;   // Nyquist tile served by the side arrays
        const int ob = g.full ? (g.b * obs + g.col + pen) : ((g.b + pen) * obs + g.col);
        C* outp = side ? p.nyq_out + (g.b + pen) : p.out + ob;
        const int ost = side ? p.nb : ops;                  // row stride of the output
        (void)ost;
        C v[16];

        if constexpr (MODE == FMODE_FWD) {
            load_x(g, v);
            // h = 0: x -> even outputs;  h = 1: x w512^n -> odd outputs
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], t512[r]);
            fft256_a<false, OB, MODE != FMODE_FWD>(v, t256, o, xc);
            __syncthreads();
            advance(it);
            fft256_b<false, OB>(v, xc);
            if (side) {
                // the consumer (S3) wants this column as [pencil of S2 = z][ky]: transpose through the
                // exchange buffer and write 512 contiguous ky per z
                __syncthreads();   // every thread is done reading the exchange buffer
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) stage(2 * (o + 16 * k2) + h, pen) = v[brev4(k2)];
                __syncthreads();
                for (int idx = tid; idx < 2 * kL * kTile; idx += kThreads) {
                    const int pp = idx >> 9, ky = idx & (2 * kL - 1);
                    if (g.b + pp < p.nb) p.nyq_out[(g.b + pp) * (2 * kL) + ky] = stage(ky, pp);
                }
                __syncthreads();   // before the next tile's exchange
            } else if (pvalid) {
                C* q = outp + (2 * o + h) * ops;   // row 2 (o + 16 k2) + h
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) q[k2 * 32 * ops] = v[brev4(k2)];
            }
        } else {
            if constexpr (MODE == FMODE_FUSED) {
                float gm[16];
                // the tile's chunk of the tile-major table [257 fp][16 pencils]; the thread's spectral
                // indices kp = 2 (o + 16 k2) + h fold to fp = min(kp, 512 - kp): every offset is an immediate
                const float* gt = p.green_tiles + (green_tile_index(p, g) * (kGreenRows * kTile) + pen);
                const float* glo = gt + (2 * o + h) * kTile;              // kp            (k2 < 8)
                const float* ghi = gt + (2 * kL - 2 * o - h) * kTile;     // 512 - kp      (k2 >= 8)
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) gm[k2] = __ldg(k2 < 8 ? glo + k2 * 32 * kTile : ghi - k2 * 32 * kTile);
                load_x(g, v);
#pragma unroll
                for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], t512[r]);
                fft256_a<false, OB, MODE != FMODE_FWD>(v, t256, o, xc);
                __syncthreads();
                advance(it);
                fft256_b<false, OB>(v, xc);
                C u[16];
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) u[k2] = cscale(v[brev4(k2)], gm[k2]);
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) v[k2] = u[k2];
                fft256_a<true, !OB, MODE != FMODE_FWD>(v, t256, o, xc);
                __syncthreads();
                fft256_b<true, !OB>(v, xc);
            } else {
                // rows 2 k + h, k = o + 16 k2: h = 0 even spectrum E, h = 1 odd spectrum O; each half-warp
                // reads one 128-byte run per row (16 batches of one column for the Nyquist tiles)
                if (side) {
                    // the producer (S3) left this column as [pencil of S4 = z][ky]: read 512 contiguous ky
                    // per z and transpose through the exchange buffer (which the previous tile's second half may
                    // still be reading when this is not the CTA's first tile)
                    if (it > 0) __syncthreads();
                    for (int idx = tid; idx < 2 * kL * kTile; idx += kThreads) {
                        const int pp = idx >> 9, ky = idx & (2 * kL - 1);
                        stage(ky, pp) = (g.b + pp < p.nb) ? __ldg(p.nyq_in + (g.b + pp) * (2 * kL) + ky) : make_float2(0.f, 0.f);
                    }
                    __syncthreads();
#pragma unroll
                    for (int k2 = 0; k2 < 16; ++k2) v[k2] = stage(2 * (o + 16 * k2) + h, pen);
                    __syncthreads();   // before the exchange overwrites the staging
                } else {
                    const C* inp = p.in + ((g.full ? (g.b * ibs + g.col + pen) : (min(g.b + pen, p.nb - 1) * ibs + g.col)) + (2 * o + h) * ips);
#pragma unroll
                    for (int k2 = 0; k2 < 16; ++k2) v[k2] = __ldg(inp + k2 * 32 * ips);
                }
                fft256_a<true, OB, MODE != FMODE_FWD>(v, t256, o, xc);
                __syncthreads();
                advance(it);
                fft256_b<true, OB>(v, xc);
            }
            // x_j = e_j + conj(w512^j) o_j, j = o + 16 r: h = 0 holds e, h = 1 holds o.  The half-warps
            // swap half of their values: h = 0 finishes r < 8, h = 1 finishes r >= 8.
            C* q = outp + (o + 128 * h) * ost;
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                // h = 1: t_lo = conj(w) o_r (sent), t_hi = conj(w) o_{r+8} (kept);  h = 0: e_{r+8} sent, e_r kept
                // (the table row of h = 0 is all ones)
                const C tl = cmulc(v[brev4(r)], t512[r]), th = cmulc(v[brev4(r + 8)], t512[r + 8]);
                const C send = h ? tl : th;
                const C keep = h ? th : tl;
                C recv;
                recv.x = __shfl_xor_sync(0xffffffffu, send.x, 16);
                recv.y = __shfl_xor_sync(0xffffffffu, send.y, 16);
                const C x = cadd(keep, recv);
                if (pvalid) q[r * 16 * ost] = x;
            }
        }
    };

    // prologue: thread 0 arms the barrier and starts the first tile's TMA load while the others copy the tables
    if (tid == 0) {
        if (Cfg::kTma) {
            mbar_init(&bar, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        s_tile[0] = (int)blockIdx.x;
        s_tile[1] = (int)(blockIdx.x + gridDim.x);
        issue(s_tile[0]);
    }
    if (tid < 384) reinterpret_cast<float4*>(s_tab)[tid] = reinterpret_cast<const float4*>(g_tab_pad)[tid];
    __syncthreads();
    if constexpr (MODE == FMODE_FUSED) {
        // two transforms per tile: the orientation is back where it started
        for (int it = 0;; ++it) {
            const int t = s_tile[it & 1];
            if (t >= ntiles) break;
            tile(t, it, std::false_type());
        }
    } else {
        // one transform per tile: orientations alternate
        for (int it = 0;; it += 2) {
            int t = s_tile[0];
            if (t >= ntiles) break;
            tile(t, it, std::false_type());
            t = s_tile[1];
            if (t >= ntiles) break;
            tile(t, it + 1, std::true_type());
        }
    }
    // the last CTA to finish re-arms the counter for the next launch
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(p.sched + 1, 1) == (int)gridDim.x - 1) {
            p.sched[0] = 0;
            p.sched[1] = 0;
            __threadfence();
        }
    }
}

} // namespace sf2

namespace sf2 {

// ==================================================================================== X passes
// S1 (X forward) and S5 (X backward) for rows of 256 reals zero-padded to 512 (PAPER.md:87 real
// transform / half spectrum; PAPER.md:181 padding).  Rows are contiguous in memory, so a tile of 16
// rows is staged through shared memory by bulk copies (one per row) and transposed there: lane =
// 2 * row + h, warp = w in 0..7.
//   forward: the padded real row of length 512 is packed as z[n] = x[2n] + i x[2n+1], n < 256,
//   non-zero for n < 128.  Z = DFT256(z) is two 128-point transforms, of z (even outputs, h = 0)
//   and of z w256^n (odd outputs, h = 1); then the real-transform split
//       X[k] = ( (Z[k] + conj Z[256-k]) - i w512^k (Z[k] - conj Z[256-k]) ) / 2,   k = 0..256
//   is done pairwise in place in the staged rows, which leave by one bulk store per row.
//   backward: the exact mirror (merge, two truncated inverse transforms, unpack).
// A 128-point transform is radix-16 over r (n = w + 8 r), twiddle w128^(q w), one exchange,
// two radix-8 over o' for q = w and q = w + 8: thread w ends with the outputs k = w + 8 j.
constexpr int kXThreads = 256;
constexpr int kXRows = 16;
constexpr int kXN = 256;                 // stored reals per row
constexpr int kXInPitch = kXN + 4;       // floats per staged real row: 1040 B = 16 (mod 128): lanes hit distinct banks
constexpr int kXSpPitch = kXN + 2;       // complex per staged spectrum row: 2064 B = 16 (mod 128), multiple of 16
constexpr size_t kXSmem = (size_t)kXRows * kXInPitch * sizeof(float) + (size_t)16 * 8 * 32 * sizeof(C) + (size_t)kXRows * kXSpPitch * sizeof(C);

__host__ __device__ constexpr int brev3(int q) { return ((q & 1) << 2) | (q & 2) | ((q & 4) >> 2); }
template <bool INV, typename CT> __device__ __forceinline__ void dft8(CT (&v)[8]) { dft_rec<8, 1, INV>::run(v); }

// v[r] = a[w + 8 r] in; writes the twiddled radix-16 outputs into the exchange buffer
template <bool INV> __device__ __forceinline__ void fft128_a(C (&v)[16], const C* tw128, C* xw)
{
    dft16<INV>(v);
#pragma unroll
    for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul_sel<INV>(v[brev4(q)], tw128[q]);   // w128^(q w), row w of the table
#pragma unroll
    for (int q = 0; q < 16; ++q) xw[q * 8 * 32] = v[brev4(q)];
}
// after a barrier: A[w + 16 k2] at a[brev3(k2)], A[w + 8 + 16 k2] at b[brev3(k2)]
template <bool INV> __device__ __forceinline__ void fft128_b(C (&a)[8], C (&b)[8], const C* xr)
{
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = xr[i * 32]; b[i] = xr[(64 + i) * 32]; }
    dft8<INV>(a);
    dft8<INV>(b);
}


template <bool INV> __global__ void __launch_bounds__(kXThreads, 2) fast_x_kernel(const FastXParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* rbuf = reinterpret_cast<float*>(smem_raw);                               // [16][kXInPitch] reals
    C* xbuf = reinterpret_cast<C*>(smem_raw + (size_t)kXRows * kXInPitch * sizeof(float));   // exchange [16 q][8 o][32 lanes]
    C* sbuf = xbuf + 16 * 8 * 32;                                                   // [16][kXSpPitch] complex
    __shared__ __align__(8) uint64_t bar;

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    // lane = 2 * row + h: the 16 lanes of a half-warp (8 rows x 2 halves) then touch 16 different
    // 8-byte bank pairs of the staged rows, whose pitches are 16 (mod 128) bytes
    const int pen = lane >> 1;
    const int h = lane & 1;
    const int w = (int)__reduce_max_sync(0xffffffffu, (unsigned)(tid >> 5));
    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (!INV && tid < kXRows) sbuf[tid * kXSpPitch + kXN + 1] = make_float2(0.f, 0.f);   // pad column 257 leaves as zero
    // twiddle tables (base register + immediate addressing, no selects):
    //   s_tw128[w][q] = w128^(q w);  s_twin[h][w][j] = w256^(w + 8 j) for h = 1, 1 for h = 0;
    //   s_twsp[h][w][m] = w512^(2 w + h + 16 m)
    __shared__ __align__(16) C s_tab[544];
    for (int idx = tid; idx < 272; idx += kXThreads) reinterpret_cast<float4*>(s_tab)[idx] = reinterpret_cast<const float4*>(g_tab_x)[idx];
    const C* t128 = s_tab + w * 16;
    const C* tin = s_tab + 128 + w * 32 + h;   // twin[w][j][h]: index 2 j
    const C* tsp = s_tab + 384 + w * 20 + h;   // twsp[w][m][h]: index 2 m
    __syncthreads();

    const int ntiles = p.nrows / kXRows;
    const int nit = (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    uint32_t parity = 0;
    C* xw = xbuf + w * 32 + lane;          // slot (q, w)
    const C* xr = xbuf + w * 8 * 32 + lane; // slots (w, o'), (w + 8, o')
    C* srow = sbuf + pen * kXSpPitch;      // this thread's staged spectrum row

    // bulk loads of iteration i: one row per lane of warp 0
    auto issue = [&](int i) {
        if (tid >= kXRows || i >= nit) return;
        const long long tl = (long long)blockIdx.x + (long long)i * gridDim.x;
        const long long row = (p.reverse ? ntiles - 1 - tl : tl) * kXRows + tid;
        if (tid == 0) mbar_expect_tx(&bar, INV ? kXRows * kXSpPitch * (uint32_t)sizeof(C) : kXRows * kXN * (uint32_t)sizeof(float));
        __syncwarp(0xffffu);
        if (INV) bulk_g2s(sbuf + tid * kXSpPitch, p.spec + row * p.spec_pitch, kXSpPitch * (uint32_t)sizeof(C), &bar);
        else bulk_g2s(rbuf + tid * kXInPitch, p.real_in + row * kXN, kXN * (uint32_t)sizeof(float), &bar);
    };

    // S5: the Nyquist coefficient of this thread's row of iteration i, for the thread that merges the pair (0, 256)
    auto load_nyq = [&](int i) -> C {
        if (!INV || !p.nyq || w != 0 || h != 0 || i >= nit) return make_float2(0.f, 0.f);
        const long long tl = (long long)blockIdx.x + (long long)i * gridDim.x;
        const int row = (int)((p.reverse ? ntiles - 1 - tl : tl) * kXRows) + pen;
        return __ldg(p.nyq + (row % p.n1) * p.n2 + row / p.n1);
    };
    C xnyq_next = load_nyq(0);
    issue(0);
    for (int i = 0; i < nit; ++i) {
        const long long tl0 = (long long)blockIdx.x + (long long)i * gridDim.x;
        const long long row0 = (p.reverse ? ntiles - 1 - tl0 : tl0) * kXRows;
        C v[16];
        if constexpr (!INV) {
            // ---------------------------------------------------------------- S1
            mbar_wait(&bar, parity);
            parity ^= 1;
#pragma unroll
            for (int r = 0; r < 16; ++r)
                v[r] = cmul(*reinterpret_cast<const C*>(rbuf + pen * kXInPitch + 2 * (w + 8 * r)), tin[2 * r]);   // h = 1: z w256^n
            fft128_a<false>(v, t128, xw);
            if (tid < kXRows) bulk_wait_read();   // the previous tile's stores have left sbuf
            __syncthreads();
            issue(i + 1);                         // rbuf is in registers everywhere
            C a[8], b[8];
            fft128_b<false>(a, b, xr);
            // Z[2 k' + h], k' = w + 16 k2 (a) and w + 8 + 16 k2 (b), natural order into the staged row
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                srow[2 * (w + 16 * k2) + h] = a[brev3(k2)];
                srow[2 * (w + 8 + 16 * k2) + h] = b[brev3(k2)];
            }
            __syncthreads();
            // split in place: the 16 threads of a row own the pairs (k, 256 - k), k = idx + 16 m
            const int idx = 2 * w + h;
            {
                C zk[9], zm[9];
#pragma unroll
                for (int m = 0; m < 9; ++m) {
                    const int k = idx + 16 * m;
                    if (m < 8 || idx == 0) { zk[m] = srow[k]; zm[m] = srow[(kXN - k) & (kXN - 1)]; }
                }
#pragma unroll
                for (int m = 0; m < 9; ++m) {
                    const int k = idx + 16 * m;
                    if (m < 8 || idx == 0) {
                        const C e = cadd(zk[m], make_float2(zm[m].x, -zm[m].y));
                        const C d = csub(zk[m], make_float2(zm[m].x, -zm[m].y));
                        const C wd = cmul(d, tsp[2 * m]);   // w512^k d
                        // X[k] = (e - i wd) / 2,  X[256 - k] = (conj e - i conj wd) / 2
                        srow[k] = cscale(cadd(e, make_float2(wd.y, -wd.x)), 0.5f);
                        srow[kXN - k] = cscale(make_float2(e.x - wd.y, -e.y - wd.x), 0.5f);
                    }
                }
            }
            fence_async_smem();
            __syncthreads();
            if (tid < kXRows) {
                bulk_s2g(p.spec + (row0 + tid) * p.spec_pitch, sbuf + tid * kXSpPitch, kXSpPitch * (uint32_t)sizeof(C));
                bulk_commit();
                // the Nyquist coefficient X[256] of row (z, y) also goes to the side array [y][z] that the
                // strided passes read it from in 128-byte runs
                if (p.nyq) {
                    const int row = (int)(row0 + tid);
                    p.nyq[(row % p.n1) * p.n2 + row / p.n1] = sbuf[tid * kXSpPitch + kXN];
                }
            }
        } else {
            // ---------------------------------------------------------------- S5
            // X[256] of this thread's row comes from the side array [y][z] (only the owner of the pair
            // (0, 256) needs it); it was requested one tile ahead
            const C xnyq = xnyq_next;
            mbar_wait(&bar, parity);
            parity ^= 1;
            // merge in place: Z[k] = e + i conj(w512^k) d, Z[256 - k] = conj e + i conj(conj(w512^k) d)
            const int idx = 2 * w + h;
            {
                C xk[9], xm[9];
#pragma unroll
                for (int m = 0; m < 9; ++m) {
                    const int k = idx + 16 * m;
                    if (m < 8 || idx == 0) { xk[m] = srow[k]; xm[m] = srow[kXN - k]; }
                    if (m == 0 && idx == 0 && p.nyq) xm[0] = xnyq;
                }
#pragma unroll
                for (int m = 0; m < 9; ++m) {
                    const int k = idx + 16 * m;
                    if (m < 8 || idx == 0) {
                        const C e = cadd(xk[m], make_float2(xm[m].x, -xm[m].y));
                        const C d = csub(xk[m], make_float2(xm[m].x, -xm[m].y));
                        const C wd = cmulc(d, tsp[2 * m]);   // conj(w512^k) d
                        srow[k] = cadd(e, make_float2(-wd.y, wd.x));
                        if (k > 0) srow[kXN - k] = make_float2(e.x + wd.y, wd.x - e.y);
                    }
                }
            }
            __syncthreads();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = srow[2 * (w + 8 * j) + h];   // Z[2 k' + h], k' = w + 8 j
            fft128_a<true>(v, t128, xw);
            if (tid < kXRows) bulk_wait_read();   // the previous tile's stores have left rbuf
            fence_async_smem();                   // the merged values in sbuf are overwritten by the next bulk load
            __syncthreads();
            issue(i + 1);                         // sbuf is in registers everywhere
            xnyq_next = load_nyq(i + 1);
            C a[8], b[8];
            fft128_b<true>(a, b, xr);
            // z[n] = z0[n] + conj(w256^n) z1[n], n = w + 16 k2 (a) / w + 8 + 16 k2 (b): h = 0 holds z0,
            // h = 1 holds z1; h = 0 finishes the a set, h = 1 the b set
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                // (the table row of h = 0 is all ones)
                const C ta = cmulc(a[brev3(k2)], tin[4 * k2]), tb = cmulc(b[brev3(k2)], tin[4 * k2 + 2]);
                const C send = h ? ta : tb;
                const C keep = h ? tb : ta;
                C recv;
                recv.x = __shfl_xor_sync(0xffffffffu, send.x, 1);
                recv.y = __shfl_xor_sync(0xffffffffu, send.y, 1);
                const C z = cadd(keep, recv);
                const int n = w + 8 * h + 16 * k2;
                *reinterpret_cast<C*>(rbuf + pen * kXInPitch + 2 * n) = z;   // (x[2n], x[2n+1])
            }
            fence_async_smem();
            __syncthreads();
            if (tid < kXRows) {
                bulk_s2g(p.real_out + (row0 + tid) * kXN, rbuf + tid * kXInPitch, kXN * (uint32_t)sizeof(float));
                bulk_commit();
            }
        }
    }
    if (tid < kXRows) bulk_wait_read();
}

} // namespace sf2
