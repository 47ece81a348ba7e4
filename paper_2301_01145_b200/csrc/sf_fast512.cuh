// sf_fast512.cuh -- kernel generation 2 for fp32 unbounded plans with 512-long y / z pencils that are
// zero-padded to 1024 (BASELINE.json configs[4]: 512^3 -> 1024^3, three components, curl): the strided
// passes S2 (Y forward), S3 (Z forward x Green x [curl] x Z backward, fused) and S4 (Y backward)
// (PAPER.md:89-97 pencils, :103-109 four-step solve, :119 component-wise vector solve, :141 spectral curl,
// :181 / :213 padded and pruned Hockney-Eastwood transforms).
//
// Same ideas as sf_fast.cuh, one size up.  The 1024-point transform of (x, 0) is two 512-point transforms
// (h = 0: x -> even outputs; h = 1: x w1024^n -> odd outputs) that run side by side in the two half-warps.
// A residue w in 0..31 of the 512-point transform owns 2 PEN consecutive threads = PEN neighbouring pencils x the two
// halves h; thread (w, pencil, h) holds the 16 elements n = w + 32 r of its sequence.  A 512-point transform is
//     radix-16 over r (registers) -> twiddle w512^(q w) -> ONE shared-memory exchange ->
//     radix-32 over the 32 values o of slot row q0 = w mod 16, done as a radix-2 step that keeps the
//     output parity p = w div 16 (16 sums or twiddled differences) and a radix-16 over the rest (registers)
// and leaves X[w + 32 j] in thread w: input and output distributions agree, so forward, multiply and
// backward chain without reordering.  PEN = 16 (S4): one CTA of 1024 threads per SM, warp = residue (warp-uniform
// twiddles), 128 KB exchange buffer, the tile loaded straight into registers.  PEN = 8 (S2, S3): two CTAs of 512
// threads per SM (64 KB exchange buffer + 32 KB TMA slot each) -- two barrier domains, one transforms while the
// other waits; measured on cfg 5: S2 2.08 -> 1.98 ms, S3 (a chain of six transforms per tile) 7.14 -> 6.39 ms.
//
// Vector plans: sf_curl needs psi_hat of all three components at every spectral point, 393 KB per tile --
// more than the registers or the shared memory of an SM hold next to the exchange buffer.  The two spectra
// that have to wait are parked in TENSOR MEMORY (tcgen05.st / tcgen05.ld, shape 32x32b: each thread parks and
// fetches its own registers, which is exactly the access TMEM gives a warp; 2 x 32 of the 512 columns per
// warp, 8 warps per lane quadrant = all 256 KB).  Components are transformed forward in the order z, y, x:
//     psi_hat_z -> TMEM A;   psi_hat_y -> TMEM B,  u_hat_x = kappa_y A - kappa_z psi_hat_y -> backward -> u_x;
//     psi_hat_x:  u_hat_z = kappa_x B - kappa_y psi_hat_x -> TMEM A (over psi_hat_z, chunk by chunk),
//                 u_hat_y = kappa_z psi_hat_x - kappa_x A -> backward -> u_y;   TMEM A -> backward -> u_z
// (the common factor i is applied at the store).  Three forward and three backward transforms per tile, every
// component read once and every velocity component written once.
#pragma once
#include "sf_trig.cuh"
#include "sf_fast.cuh"

namespace sf2 {

constexpr int kT5 = 1024;            // threads per CTA
constexpr int kL5 = 512;             // transform length (stored rows per pencil)
static_assert(kGreenRows5 == kL5 + 1, "folded spectral indices 0 .. 512");
constexpr int kXchg5Elems = 16 * 32 * 32;                 // 128 KB
constexpr int kSlot5Elems = kL5 * kTile;                  // 64 KB
constexpr size_t kSmem5 = ((size_t)kXchg5Elems + kSlot5Elems) * sizeof(C);
constexpr size_t kSmem5NoSlot = (size_t)kXchg5Elems * sizeof(C);

using sftrig::cos32;   // cos / sin of 2 pi i / 32 (sf_trig.cuh)
using sftrig::sin32;
// d * exp(-/+ 2 pi i I32 / 32)   (forward: minus)
template <int I32, bool INV> __device__ __forceinline__ C mul_w32(C d)
{
    if constexpr (I32 == 0) {
        return d;
    } else if constexpr (I32 == 8) {
        return INV ? cmuli(d) : cmulmi(d);
    } else {
        constexpr float c = (float)cos32(I32);
        constexpr float s = (float)(INV ? sin32(I32) : -sin32(I32));
        return cmul(d, make_float2(c, s));
    }
}

// first half: radix-16 over r, twiddle w512^(q w) (row w of a shared-memory table), write slots (q, w)
template <bool INV, int LW = 32, typename TW> __device__ __forceinline__ void fft512_a(C (&v)[16], TW&& tw, C* xw)
{
    dft16<INV>(v);
#pragma unroll
    for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul_sel<INV>(v[brev4(q)], tw(q));
#pragma unroll
    for (int q = 0; q < 16; ++q) xw[q * (32 * LW)] = v[brev4(q)];
}
// second half (after a barrier): slots (q0, o), o < 32, radix-2 keeping parity p, radix-16.
// X[w + 32 j] at v[brev4(j)] out.
template <bool INV, int P, int LW> __device__ __forceinline__ void fft512_b_p(C (&v)[16], const C* xr)
{
    auto step = [&](auto tag) {
        constexpr int o2 = decltype(tag)::value;
        const C a = xr[o2 * LW], b = xr[(o2 + 16) * LW];
        if constexpr (P == 0) v[o2] = cadd(a, b);
        else v[o2] = mul_w32<o2, INV>(csub(a, b));
    };
    step(std::integral_constant<int, 0>()); step(std::integral_constant<int, 1>());
    step(std::integral_constant<int, 2>()); step(std::integral_constant<int, 3>());
    step(std::integral_constant<int, 4>()); step(std::integral_constant<int, 5>());
    step(std::integral_constant<int, 6>()); step(std::integral_constant<int, 7>());
    step(std::integral_constant<int, 8>()); step(std::integral_constant<int, 9>());
    step(std::integral_constant<int, 10>()); step(std::integral_constant<int, 11>());
    step(std::integral_constant<int, 12>()); step(std::integral_constant<int, 13>());
    step(std::integral_constant<int, 14>()); step(std::integral_constant<int, 15>());
    dft16<INV>(v);
}
template <bool INV, int LW = 32> __device__ __forceinline__ void fft512_b(C (&v)[16], const C* xr, int p)
{
    if (p) fft512_b_p<INV, 1, LW>(v, xr);     // p is warp-uniform: no divergence
    else fft512_b_p<INV, 0, LW>(v, xr);
}

// ------------------------------------------------------------------------------------ tensor memory as a parking lot
// 32x32b shape: lane i of the warp reads / writes TMEM lane (32 (warp mod 4) + i), consecutive 32-bit columns
__device__ __forceinline__ void tmem_alloc_cols(uint32_t* smem_dst, uint32_t cols)   // cols: a power of two >= 32
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_dst)), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_free_cols(uint32_t base, uint32_t cols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(cols) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t addr, const C (&v)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(addr),
                 "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y), "f"(v[3].x), "f"(v[3].y),
                 "f"(v[4].x), "f"(v[4].y), "f"(v[5].x), "f"(v[5].y), "f"(v[6].x), "f"(v[6].y), "f"(v[7].x), "f"(v[7].y)
                 : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t addr, C (&v)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y), "=f"(v[3].x), "=f"(v[3].y),
                   "=f"(v[4].x), "=f"(v[4].y), "=f"(v[5].x), "=f"(v[5].y), "=f"(v[6].x), "=f"(v[6].y), "=f"(v[7].x), "=f"(v[7].y)
                 : "r"(addr)
                 : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t addr, const C (&v)[4])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(addr),
                 "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y), "f"(v[3].x), "f"(v[3].y)
                 : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t addr, C (&v)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y), "=f"(v[3].x), "=f"(v[3].y)
                 : "r"(addr)
                 : "memory");
}
__device__ __forceinline__ void tmem_st4(uint32_t addr, const C (&v)[2])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y) : "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t addr, C (&v)[2])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y) : "r"(addr) : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t addr, const C (&v)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
                 "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(addr),
                 "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y), "f"(v[3].x), "f"(v[3].y),
                 "f"(v[4].x), "f"(v[4].y), "f"(v[5].x), "f"(v[5].y), "f"(v[6].x), "f"(v[6].y), "f"(v[7].x), "f"(v[7].y),
                 "f"(v[8].x), "f"(v[8].y), "f"(v[9].x), "f"(v[9].y), "f"(v[10].x), "f"(v[10].y), "f"(v[11].x), "f"(v[11].y),
                 "f"(v[12].x), "f"(v[12].y), "f"(v[13].x), "f"(v[13].y), "f"(v[14].x), "f"(v[14].y), "f"(v[15].x), "f"(v[15].y)
                 : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t addr, C (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y), "=f"(v[3].x), "=f"(v[3].y),
                   "=f"(v[4].x), "=f"(v[4].y), "=f"(v[5].x), "=f"(v[5].y), "=f"(v[6].x), "=f"(v[6].y), "=f"(v[7].x), "=f"(v[7].y),
                   "=f"(v[8].x), "=f"(v[8].y), "=f"(v[9].x), "=f"(v[9].y), "=f"(v[10].x), "=f"(v[10].y), "=f"(v[11].x), "=f"(v[11].y),
                   "=f"(v[12].x), "=f"(v[12].y), "=f"(v[13].x), "=f"(v[13].y), "=f"(v[14].x), "=f"(v[14].y), "=f"(v[15].x), "=f"(v[15].y)
                 : "r"(addr)
                 : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ------------------------------------------------------------------------------------ tiles
// chunk of the tile-major Green's table that belongs to a tile (as green_tile_index of sf_fast.cuh)
template <int PEN> __device__ __forceinline__ int green_tile_index5(const Fast5Params& p, bool full, int b, int col)
{
    if (full) return (min(b, p.Pb - b) << p.nct_shift) + (col / PEN);
    return ((p.Pb / 2 + 1) << p.nct_shift) + (b / PEN);
}

// MODE F5_FWD   : in rows n < 512 -> out rows k < 1024                       (S2; components are more batches)
//      F5_INV   : in rows k < 1024 -> out rows j < 512                       (S4; likewise)
//      F5_FUSED : in rows n < 512 -> x Green -> out rows j < 512, per component (S3 of sf_solve)
//      F5_CURL  : three components in, u = curl psi out                      (S3 of sf_curl)
// `tm` describes `in` as a rank-4 tensor; a tile image is fetched by two boxes of 256 rows:
//   FWD            dims (column, row, batch, 1)          box {16, 256, 1, 1}   coordinates {col, 0 | 256, b, 0}
//   FUSED / CURL   dims (column, batch, row, component)  box {16, 1, 256, 1}   coordinates {col, b, 0 | 256, c}
// The Nyquist column (column nyq_col of every batch) is handled 16 batches at a time with gathered 8-byte accesses.
// PEN = pencils per tile: 16 (one CTA of 1024 threads per SM; FWD / INV) or 8 (two CTAs of 512 threads per SM: two
// independent barrier domains, one transforms while the other waits at a barrier; FUSED / CURL, where a tile is a
// chain of two to six transforms).  A residue w owns LW = 2 PEN consecutive threads.
template <int MODE, int PEN>
__global__ void __launch_bounds__(64 * PEN, 16 / PEN) fast5_kernel(const Fast5Params p, const __grid_constant__ CUtensorMap tm)
{
    constexpr int LW = 2 * PEN;            // threads per residue: PEN pencils x 2 halves
    constexpr int NT = 64 * PEN;           // threads per CTA
    constexpr bool kTma = (MODE != F5_INV);
    constexpr bool kMul = (MODE == F5_FUSED || MODE == F5_CURL);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* xbuf = reinterpret_cast<C*>(smem_raw);
    C* slot = xbuf + 16 * 32 * LW;
    __shared__ __align__(8) uint64_t bar;
    // Twiddle factors: w512^(q w) between the two halves of a transform and w1024^(w + 32 r) of the odd half
    // (h = 1; the even half multiplies by one).  Both are warp-uniform and live in shared-memory tables (base
    // register + immediate).  (kTwc: from the constant bank instead -- tried for CURL to get under the 196 KB
    // shared-memory carve-out; the constants then occupy registers and the kernel spills 416 bytes per thread.)
    constexpr bool kTwc = false;
    __shared__ float s_kapp[MODE == F5_CURL ? 1024 : 1];
    // CURL: per-thread values of the current tile that are needed between the transforms only (kappa_x, kappa_y,
    // output offset): parked here, because the 64 registers of a 1024-thread CTA cannot hold them across the
    // transforms and a spill to local memory misses the (28 KB) L1
    constexpr bool kPark = (MODE == F5_CURL && PEN == 16);   // (PEN = 8: the shared memory of two CTAs has no room for it)
    __shared__ float s_qx[kPark ? NT : 1], s_qy[kPark ? NT : 1];
    __shared__ unsigned s_oo[kPark ? NT : 1];
    // (rows of 17 entries: with PEN = 8 a warp holds two residues w, whose rows must not start on the same bank)
    constexpr int kTwRow = 17;
    __shared__ __align__(16) C s_tw512[kTwc ? 1 : 32 * kTwRow];    // [w][q] = w512^(q w)
    // (PEN = 8: only the h = 1 half of the second table is kept, the even half selects one: shared memory for two CTAs)
    constexpr bool kHalfTab = (PEN == 8);
    __shared__ __align__(16) C s_tw1024[kTwc ? 1 : (kHalfTab ? 1 : 2) * 32 * kTwRow];   // [h][w][r] = h ? w1024^(w + 32 r) : 1
    __shared__ int s_tile[2];
    __shared__ uint32_t s_tmem;

    const int tid = threadIdx.x;
    const int lane = tid % LW;
    const int pen = lane % PEN;
    const int h = lane / PEN;
    // PEN = 16: the residue is the warp index (warp-uniform: REDUX puts it in a uniform register)
    const int w = (PEN == 16) ? (int)__reduce_max_sync(0xffffffffu, (unsigned)(tid >> 5)) : tid / LW;
    const int q0 = w & 15, par = w >> 4;            // (PEN = 8: the two residues of a warp share their parity)
    C* xw = xbuf + (w * LW + lane);                 // slot (q, w) at ((q * 32 + w) * LW + lane)
    const C* xr = xbuf + (q0 * 32 * LW + lane);     // slot (q0, o) at stride LW
    const C* t512 = s_tw512 + w * kTwRow;
    const C* t1024 = s_tw1024 + ((kHalfTab ? 0 : h * 32) + w) * kTwRow;
    const float hf = (float)h;
    auto tw512 = [&](int q) -> C { return kTwc ? c_tw1024[(2 * q * w) & 1023] : t512[q]; };
    // 1 + h (w1024^(w + 32 r) - 1): one packed multiply-add on the table of (Re w - 1, Im w)
    auto tw1024 = [&](int r) -> C {
        if (!kTwc && kHalfTab) { const C t = t1024[r]; return h ? t : make_float2(1.f, 0.f); }
        if (!kTwc) return t1024[r];
        const C m = c_tw1024m1[w + 32 * r];
        return __ffma2_rn(make_float2(hf, hf), m, make_float2(1.f, 0.f));
    };

    const int ncomp_tiles = (MODE == F5_FUSED) ? p.ncomp : 1;     // FUSED: components are independent tile sets
    const int nfull = p.nb << p.nct_shift;
    const int nnyq = (p.nyq_col >= 0) ? (p.nb + PEN - 1) / PEN : 0;
    const int ntile1 = nfull + nnyq;
    const int ntiles = ntile1 * ncomp_tiles;
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;
    uint32_t parity = 0;

    struct Geom { bool full; int b, col, comp; };
    auto geom = [&](int t) {
        Geom g;
        g.comp = 0;
        if (MODE == F5_FUSED) { g.comp = t / ntile1; t -= g.comp * ntile1; }
        if (t < nnyq) {               // Nyquist-column tiles first: they are the slow ones
            g.full = false;
            g.b = t * PEN;
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
            g.col = (tf & (p.nct - 1)) * PEN;
        }
        return g;
    };
    // TMA load of (tile t, component c) into the slot: one thread, two boxes of 256 rows
    auto issue = [&](int t, int c) {
        if (!kTma || tid != 0 || t >= ntiles) return;
        const Geom g = geom(t);
        if (!g.full) return;
        mbar_expect_tx(&bar, (uint32_t)(kL5 * PEN * sizeof(C)));
        if (MODE == F5_FWD) {
            tma_load_4d(slot, &tm, g.col, 0, g.b, 0, &bar);
            tma_load_4d(slot + 256 * PEN, &tm, g.col, 256, g.b, 0, &bar);
        } else {
            const int cc = (MODE == F5_CURL) ? c : g.comp;
            tma_load_4d(slot, &tm, g.col, g.b, 0, cc, &bar);
            tma_load_4d(slot + 256 * PEN, &tm, g.col, g.b, 256, cc, &bar);
        }
    };
    // v[r] = x[w + 32 r] of this thread's pencil (FWD / FUSED / CURL)
    // (stashed: a Nyquist tile's elements were put into the slot by this very thread, see the curl)
    auto load_x = [&](const Geom& g, int c, C (&v)[16], bool stashed = false) {
        if (g.full || stashed) {
            if (g.full) {
                mbar_wait(&bar, parity);
                parity ^= 1;
            }
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = slot[(w + 32 * r) * PEN + pen];
        } else {
            const C* inp = p.in + ((size_t)c * p.in_cs + (size_t)min(g.b + pen, p.nb - 1) * ibs + g.col + (size_t)w * ips);
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = __ldg(inp + (size_t)r * 32 * ips);
        }
    };
    // Every transform starts with a barrier: the exchange buffer may still be read by the previous one (and, at the
    // start of a tile, every thread has read its tile index and its elements of the slot); `after_barrier` runs
    // right behind it (prefetch of the next image into the slot, claim of the tile after next).
    // forward transform of this thread's half: v[r] = x[w + 32 r] in, X_h[w + 32 j] at v[brev4(j)] out.
    auto forward = [&](C (&v)[16], auto&& after_barrier) {
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], tw1024(r));
        __syncthreads();
        after_barrier();
        fft512_a<false, LW>(v, tw512, xw);
        __syncthreads();
        fft512_b<false, LW>(v, xr, par);
    };
    // backward transform (u natural order in: u[j] = U_h[w + 32 j]) and recombination of the halves:
    // x_j = e_j + conj(w1024^j) o_j, j = w + 32 r.  Thread h = 0 ends with rows w + 32 r (r < 8) in out[r],
    // thread h = 1 with rows w + 256 + 32 r.
    auto backward = [&](C (&u)[16], C (&out)[8], auto&& after_barrier) {
        __syncthreads();
        after_barrier();
        fft512_a<true, LW>(u, tw512, xw);
        __syncthreads();
        fft512_b<true, LW>(u, xr, par);
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const C tl = cmulc(u[brev4(r)], tw1024(r)), th = cmulc(u[brev4(r + 8)], tw1024(r + 8));
            const C send = h ? tl : th;
            const C keep = h ? th : tl;
            C recv;
            recv.x = __shfl_xor_sync(0xffffffffu, send.x, PEN);
            recv.y = __shfl_xor_sync(0xffffffffu, send.y, PEN);
            out[r] = cadd(keep, recv);
        }
    };
    auto nothing = []() {};
    // u[j] = G X_h[w + 32 j]: Green's factors of this thread's 16 spectral rows kp = 2 (w + 32 j) + h, folded to
    // min(kp, 1024 - kp), fetched when they are used (the registers cannot hold them across the transform)
    auto mul_green = [&](const Geom& g, const C (&v)[16], C (&u)[16]) {
        const float* glo = p.green_tiles + ((size_t)green_tile_index5<PEN>(p, g.full, g.b, g.col) * (kGreenRows5 * PEN) + pen + (2 * w + h) * PEN);
        const float* ghi = glo + (2 * kL5 - 4 * w - 2 * h) * PEN;   // 1024 - kp     (j >= 8)
#pragma unroll
        for (int j = 0; j < 16; ++j) u[j] = cscale(v[brev4(j)], __ldg(j < 8 ? glo + j * 64 * PEN : ghi - j * 64 * PEN));
    };

    // ---------------------------------------------------------------- prologue
    if (tid == 0) {
        if (kTma) {
            mbar_init(&bar, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        s_tile[0] = (int)blockIdx.x;
        s_tile[1] = (int)(blockIdx.x + gridDim.x);
        issue(s_tile[0], MODE == F5_CURL ? 2 : 0);
    }
    if (MODE == F5_CURL)
        for (int i = tid; i < 1024; i += NT) s_kapp[i] = __ldg(p.kap_p + i);
    if (!kTwc) {
        if (tid < 512) s_tw512[(tid >> 4) * kTwRow + (tid & 15)] = c_tw1024[(2 * (tid & 15) * (tid >> 4)) & 1023];
        for (int i = tid; i < (kHalfTab ? 1 : 2) * 512; i += NT) {
            const int r = i & 15, ww = (i >> 4) & 31, hh = kHalfTab ? 1 : (i >> 9);
            s_tw1024[(i >> 4) * kTwRow + r] = hh ? c_tw1024[ww + 32 * r] : make_float2(1.f, 0.f);
        }
    }
    uint32_t tbase = 0;
    if (MODE == F5_CURL) {
        if (tid < 32) tmem_alloc_cols(&s_tmem, (uint32_t)(NT / 2));   // 64 columns per warp, four warps (lane quadrants) side by side
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    __syncthreads();
    if (MODE == F5_CURL) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tbase = s_tmem + ((uint32_t)((tid >> 5) & 3) << 21);    // lane field (bits 16..31) = 32 (warp mod 4)
    }
    const uint32_t t_A = tbase + (uint32_t)(tid >> 7) * 64;   // this warp's 2 x 32 columns: 16 complex numbers per thread each
    const uint32_t t_B = t_A + 32;
    (void)t_A; (void)t_B;

    // ---------------------------------------------------------------- tiles
    for (int it = 0;; ++it) {
        const int t = (int)__reduce_max_sync(0xffffffffu, (unsigned)s_tile[it & 1]);   // warp-uniform: tile geometry in uniform registers
        if (t >= ntiles) break;
        const Geom g = geom(t);
        const bool pvalid = g.full || (g.b + pen < p.nb);
        // after the first barrier of the tile every thread has its tile index (and the slot's first image):
        // prefetch what comes next, claim the tile after next
        auto advance = [&]() {
            if (tid != 0) return;
            if (MODE == F5_CURL) issue(t, 1);
            else issue(s_tile[(it + 1) & 1], 0);   // (FUSED: the component is part of the tile index)
            s_tile[it & 1] = atomicAdd(p.sched, 1) + 2 * (int)gridDim.x;
        };
        C v[16];
        if constexpr (MODE == F5_FWD) {
            load_x(g, 0, v);
            forward(v, advance);
            if (pvalid) {
                C* q = p.out + ((size_t)(g.full ? g.b : g.b + pen) * obs + g.col + (g.full ? pen : 0) + (size_t)(2 * w + h) * ops);
#pragma unroll
                for (int j = 0; j < 16; ++j) q[(size_t)j * 64 * ops] = v[brev4(j)];    // row 2 (w + 32 j) + h
            }
        } else if constexpr (MODE == F5_INV) {
            // rows 2 k + h, k = w + 32 j
            {   // the next tile's 1024 rows (one 128-byte line each) are asked into the L2 now
                const int tn = s_tile[(it + 1) & 1];
                if (tn < ntiles) {
                    const Geom gn = geom(tn);
                    if (gn.full) prefetch_l2(p.in + ((size_t)gn.b * ibs + gn.col + (size_t)tid * ips));
                }
            }
            const C* inp = p.in + ((size_t)(g.full ? g.b : min(g.b + pen, p.nb - 1)) * ibs + g.col + (g.full ? pen : 0) + (size_t)(2 * w + h) * ips);
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = __ldg(inp + (size_t)j * 64 * ips);
            C o8[8];
            backward(v, o8, advance);
            if (pvalid) {
                C* q = p.out + ((size_t)(g.full ? g.b : g.b + pen) * obs + g.col + (g.full ? pen : 0) + (size_t)(w + 256 * h) * ops);
#pragma unroll
                for (int r = 0; r < 8; ++r) q[(size_t)r * 32 * ops] = o8[r];
            }
        } else if constexpr (MODE == F5_FUSED) {
            load_x(g, g.comp, v);
            forward(v, advance);
            C u[16];
            mul_green(g, v, u);
            C o8[8];
            backward(u, o8, nothing);
            if (pvalid) {
                C* q = p.out + ((size_t)g.comp * p.out_cs + (size_t)(g.full ? g.b : g.b + pen) * obs + g.col + (g.full ? pen : 0) + (size_t)(w + 256 * h) * ops);
#pragma unroll
                for (int r = 0; r < 8; ++r) q[(size_t)r * 32 * ops] = o8[r];
            }
        } else {
            // ---------------------------------------------------------------- curl
            // (two copies of the tile body: the full tiles' one carries no per-lane geometry)
            auto curl_tile = [&](auto full_tag) {
            constexpr bool FULL = decltype(full_tag)::value;
            Geom gg = g;
            gg.full = FULL;
            const int kx = FULL ? g.col + pen : g.col;
            const int kb = FULL ? g.b : min(g.b + pen, p.nb - 1);
            const float qx_r = __ldg(p.kap_x + kx), qy_r = __ldg(p.kap_b + kb);
            if (kPark) { s_qx[tid] = qx_r; s_qy[tid] = qy_r; }
            // element offsets of the outputs fit 32 bits (checked by the launcher)
            const unsigned oo_r = (unsigned)((FULL ? g.b : g.b + pen) * obs + g.col + (FULL ? pen : 0) + (w + 256 * h) * ops);
            if (kPark) s_oo[tid] = oo_r;
            const float* kz = s_kapp + (2 * w + h);    // kappa_z of spectral row 2 (w + 32 j) + h at kz[64 j]
            auto store = [&](int c, const C (&o8)[8]) {
                if (!FULL && !pvalid) return;
                C* q = p.out + ((kPark ? s_oo[tid] : oo_r) + (unsigned)c * (unsigned)p.out_cs);
#pragma unroll
                for (int r = 0; r < 8; ++r) q[(size_t)r * 32 * ops] = cmuli(o8[r]);   // the factor i of i kappa x psi_hat
            };
            C u[16], o8[8];
            {
                // component z: psi_hat_z -> TMEM A
                load_x(gg, 2, v);
                forward(v, advance);
                mul_green(gg, v, u);
                tmem_st32(t_A, u);
            }
            {
                // component y: psi_hat_y -> TMEM B;  u_hat_x = kappa_y psi_hat_z - kappa_z psi_hat_y
                load_x(gg, 1, v);
                forward(v, [&]() { if (tid == 0) issue(t, 0); });
                mul_green(gg, v, u);
                tmem_st32(t_B, u);
                tmem_wait_st();
                const float qy = kPark ? s_qy[tid] : qy_r;
#pragma unroll
                for (int c4 = 0; c4 < 4; ++c4) {
                    C pa[4];
                    tmem_ld8(t_A + 8 * c4, pa);
                    tmem_wait_ld();
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int j = 4 * c4 + i;
                        u[j] = cfma(pa[i], qy, cscale(u[j], -kz[64 * j]));
                    }
                }
                backward(u, o8, nothing);
                // u_x goes where psi_x sits (the pass works in place): psi_x must have left global memory first.
                // Full tiles: its TMA image has landed in the slot (the wait does not consume the phase); Nyquist
                // tiles: every thread fetches its own elements now and keeps them in the (otherwise unused) slot.
                if (FULL) {
                    mbar_wait(&bar, parity);
                } else {
                    load_x(gg, 0, u);
#pragma unroll
                    for (int r = 0; r < 16; ++r) slot[(w + 32 * r) * PEN + pen] = u[r];
                }
                store(0, o8);
            }
            {
                // component x: u_hat_z = kappa_x psi_hat_y - kappa_y psi_hat_x -> TMEM A (over psi_hat_z);
                //              u_hat_y = kappa_z psi_hat_x - kappa_x psi_hat_z
                load_x(gg, 0, v, true);
                forward(v, [&]() { if (tid == 0) issue(s_tile[(it + 1) & 1], 2); });
                mul_green(gg, v, u);
                const float qx = kPark ? s_qx[tid] : qx_r, qy = kPark ? s_qy[tid] : qy_r;
#pragma unroll
                for (int c2 = 0; c2 < 8; ++c2) {
                    C pa[2], pb[2];
                    tmem_ld4(t_A + 4 * c2, pa);
                    tmem_ld4(t_B + 4 * c2, pb);
                    tmem_wait_ld();
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        const int j = 2 * c2 + i;
                        pb[i] = cfma(pb[i], qx, cscale(u[j], -qy));
                        u[j] = cfma(pa[i], -qx, cscale(u[j], kz[64 * j]));
                    }
                    tmem_st4(t_A + 4 * c2, pb);
                }
                backward(u, o8, nothing);
                store(1, o8);
                tmem_wait_st();
                tmem_ld32(t_A, u);
                tmem_wait_ld();
                backward(u, o8, nothing);
                store(2, o8);
            }
            };
            if (g.full) curl_tile(std::true_type());
            else curl_tile(std::false_type());
        }
    }
    if (MODE == F5_CURL) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid < 32) tmem_free_cols(s_tmem, (uint32_t)(NT / 2));
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

// ==================================================================================== X passes, rows of 512 reals
// S1 (X forward) and S5 (X backward) for rows of 512 reals zero-padded to 1024 (PAPER.md:87 real transform / half
// spectrum; PAPER.md:181 padding): fast_x_kernel of sf_fast.cuh one size up.  The padded real row is packed as
// z[n] = x[2n] + i x[2n+1], n < 512, non-zero for n < 256; Z = DFT512(z) is two 256-point transforms, of z (even
// outputs, h = 0) and of z w512^n (odd outputs, h = 1); then the real-transform split
//     X[k] = ( (Z[k] + conj Z[512-k]) - i w1024^k (Z[k] - conj Z[512-k]) ) / 2,   k = 0..512
// pairwise in place in the staged rows.  A CTA of 256 threads owns 8 contiguous rows (two CTAs per SM): a
// half-warp = one residue o of the 256-point transform (radix 16 x 16, one exchange), its 16 lanes = 8 rows x 2
// halves.  Rows arrive and leave by bulk copies (one per row), the next tile's rows while this one is transformed.
constexpr int kX5Threads = 256;
constexpr int kX5Rows = 8;
constexpr int kX5N = 512;                  // stored reals per row
constexpr int kX5InPitch = kX5N + 4;       // floats per staged real row: 2064 B = 16 (mod 128)
constexpr int kX5SpPitch = kX5N + 2;       // complex per staged spectrum row: 4112 B = 16 (mod 128), multiple of 16
constexpr int kX5XchgElems = 16 * 16 * 16;
constexpr size_t kX5Smem = (size_t)kX5Rows * kX5InPitch * sizeof(float) + (size_t)kX5XchgElems * sizeof(C) + (size_t)kX5Rows * kX5SpPitch * sizeof(C);

template <bool INV> __global__ void __launch_bounds__(kX5Threads, 2) fast_x5_kernel(const FastXParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* rbuf = reinterpret_cast<float*>(smem_raw);                                          // [8][kX5InPitch] reals
    C* xbuf = reinterpret_cast<C*>(smem_raw + (size_t)kX5Rows * kX5InPitch * sizeof(float));   // exchange [16][16][16 lanes]
    C* sbuf = xbuf + kX5XchgElems;                                                             // [8][kX5SpPitch] complex
    __shared__ __align__(8) uint64_t bar;
    // s_t256[o][q] = w256^(q o);  s_tin[o][r] = w512^(o + 16 r);  s_tsp[k] = w1024^k, k <= 256
    __shared__ __align__(16) C s_t256[256];
    __shared__ __align__(16) C s_tin[256];
    __shared__ __align__(16) C s_tsp[264];

    const int tid = threadIdx.x;
    const int l16 = tid & 15;
    const int row = l16 >> 1;
    const int h = l16 & 1;
    const int o = tid >> 4;
    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (!INV && tid < kX5Rows) sbuf[tid * kX5SpPitch + kX5N + 1] = make_float2(0.f, 0.f);   // pad column 513 leaves as zero
    s_t256[tid] = c_tw1024[(4 * (tid & 15) * (tid >> 4)) & 1023];
    s_tin[tid] = c_tw1024[2 * ((tid >> 4) + 16 * (tid & 15))];
    s_tsp[tid] = c_tw1024[tid];
    if (tid < 8) s_tsp[256 + tid] = c_tw1024[256 + tid];
    const C* t256 = s_t256 + o * 16;
    const C* tin = s_tin + o * 16;
    __syncthreads();

    const int ntiles = p.nrows / kX5Rows;
    const int nit = (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    uint32_t parity = 0;
    C* xw = xbuf + o * 16 + l16;           // slot (q, o) at stride 256
    const C* xr = xbuf + o * 256 + l16;    // slot (o, o') at stride 16
    C* srow = sbuf + row * kX5SpPitch;     // this thread's staged spectrum row
    float* rrow = rbuf + row * kX5InPitch;
    const int idx = 2 * o + h;             // the 32 threads of a row own the pairs (k, 512 - k), k = idx + 32 m

    // bulk loads of iteration i: one row per lane of the first quarter-warp
    auto issue = [&](int i) {
        if (tid >= kX5Rows || i >= nit) return;
        const long long tl = (long long)blockIdx.x + (long long)i * gridDim.x;
        const long long r0 = (p.reverse ? ntiles - 1 - tl : tl) * kX5Rows + tid;
        if (tid == 0) mbar_expect_tx(&bar, INV ? kX5Rows * kX5SpPitch * (uint32_t)sizeof(C) : kX5Rows * kX5N * (uint32_t)sizeof(float));
        __syncwarp(0xffu);
        if (INV) bulk_g2s(sbuf + tid * kX5SpPitch, p.spec + r0 * p.spec_pitch, kX5SpPitch * (uint32_t)sizeof(C), &bar);
        else bulk_g2s(rbuf + tid * kX5InPitch, p.real_in + r0 * kX5N, kX5N * (uint32_t)sizeof(float), &bar);
    };

    issue(0);
    for (int i = 0; i < nit; ++i) {
        const long long tl0 = (long long)blockIdx.x + (long long)i * gridDim.x;
        const long long row0 = (p.reverse ? ntiles - 1 - tl0 : tl0) * kX5Rows;
        C v[16];
        if constexpr (!INV) {
            // ---------------------------------------------------------------- S1
            mbar_wait(&bar, parity);
            parity ^= 1;
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const C z = *reinterpret_cast<const C*>(rrow + 2 * (o + 16 * r));
                v[r] = h ? cmul(z, tin[r]) : z;                     // h = 1: z w512^n
            }
            dft16<false>(v);
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul(v[brev4(q)], t256[q]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * 256] = v[brev4(q)];
            if (tid < kX5Rows) bulk_wait_read();   // the previous tile's stores have left sbuf
            __syncthreads();
            issue(i + 1);                          // rbuf is in registers everywhere
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = xr[j * 16];
            dft16<false>(v);
            // Z[2 k' + h], k' = o + 16 k2, natural order into the staged row
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) srow[2 * (o + 16 * k2) + h] = v[brev4(k2)];
            __syncthreads();
            // split in place
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                C zk[5], zm[5];
#pragma unroll
                for (int mm = 0; mm < 5; ++mm) {
                    const int m = 4 * half + mm;
                    const int k = idx + 32 * m;
                    if (mm < 4 || (half == 1 && idx == 0)) { zk[mm] = srow[k]; zm[mm] = srow[(kX5N - k) & (kX5N - 1)]; }
                }
#pragma unroll
                for (int mm = 0; mm < 5; ++mm) {
                    const int m = 4 * half + mm;
                    const int k = idx + 32 * m;
                    if (mm < 4 || (half == 1 && idx == 0)) {
                        const C e = cadd(zk[mm], make_float2(zm[mm].x, -zm[mm].y));
                        const C d = csub(zk[mm], make_float2(zm[mm].x, -zm[mm].y));
                        const C wd = cmul(d, s_tsp[k]);   // w1024^k d
                        // X[k] = (e - i wd) / 2,  X[512 - k] = (conj e - i conj wd) / 2
                        srow[k] = cscale(cadd(e, make_float2(wd.y, -wd.x)), 0.5f);
                        srow[kX5N - k] = cscale(make_float2(e.x - wd.y, -e.y - wd.x), 0.5f);
                    }
                }
            }
            fence_async_smem();
            __syncthreads();
            if (tid < kX5Rows) {
                bulk_s2g(p.spec + (row0 + tid) * p.spec_pitch, sbuf + tid * kX5SpPitch, kX5SpPitch * (uint32_t)sizeof(C));
                bulk_commit();
            }
        } else {
            // ---------------------------------------------------------------- S5
            mbar_wait(&bar, parity);
            parity ^= 1;
            // merge in place: Z[k] = e + i conj(w1024^k) d, Z[512 - k] = conj e + i conj(conj(w1024^k) d)
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                C xk[5], xm[5];
#pragma unroll
                for (int mm = 0; mm < 5; ++mm) {
                    const int m = 4 * half + mm;
                    const int k = idx + 32 * m;
                    if (mm < 4 || (half == 1 && idx == 0)) { xk[mm] = srow[k]; xm[mm] = srow[kX5N - k]; }
                }
#pragma unroll
                for (int mm = 0; mm < 5; ++mm) {
                    const int m = 4 * half + mm;
                    const int k = idx + 32 * m;
                    if (mm < 4 || (half == 1 && idx == 0)) {
                        const C e = cadd(xk[mm], make_float2(xm[mm].x, -xm[mm].y));
                        const C d = csub(xk[mm], make_float2(xm[mm].x, -xm[mm].y));
                        const C wd = cmulc(d, s_tsp[k]);   // conj(w1024^k) d
                        srow[k] = cadd(e, make_float2(-wd.y, wd.x));
                        if (k > 0) srow[kX5N - k] = make_float2(e.x + wd.y, wd.x - e.y);
                    }
                }
            }
            __syncthreads();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = srow[2 * (o + 16 * j) + h];   // Z[2 k' + h], k' = o + 16 j
            dft16<true>(v);
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmulc(v[brev4(q)], t256[q]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * 256] = v[brev4(q)];
            if (tid < kX5Rows) bulk_wait_read();   // the previous tile's stores have left rbuf
            fence_async_smem();                    // the merged values in sbuf are overwritten by the next bulk load
            __syncthreads();
            issue(i + 1);                          // sbuf is in registers everywhere
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = xr[j * 16];
            dft16<true>(v);
            // z[n] = z0[n] + conj(w512^n) z1[n], n = o + 16 k2 < 256: h = 0 holds z0, h = 1 holds z1; the two lanes
            // swap half of their values: h = 0 finishes k2 < 8, h = 1 finishes k2 >= 8
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const C a = v[brev4(r)], b = v[brev4(r + 8)];
                const C tl = h ? cmulc(a, tin[r]) : a, th = h ? cmulc(b, tin[r + 8]) : b;
                const C send = h ? tl : th;
                const C keep = h ? th : tl;
                C recv;
                recv.x = __shfl_xor_sync(0xffffffffu, send.x, 1);
                recv.y = __shfl_xor_sync(0xffffffffu, send.y, 1);
                const C z = cadd(keep, recv);
                const int n = o + 16 * r + 128 * h;
                *reinterpret_cast<C*>(rrow + 2 * n) = z;   // (x[2n], x[2n+1])
            }
            fence_async_smem();
            __syncthreads();
            if (tid < kX5Rows) {
                bulk_s2g(p.real_out + (row0 + tid) * kX5N, rbuf + tid * kX5InPitch, kX5N * (uint32_t)sizeof(float));
                bulk_commit();
            }
        }
    }
    if (tid < kX5Rows) bulk_wait_read();
}

} // namespace sf2
