// sf_fast2p.cuh -- the fused pass S3 of sf_fast.cuh (Z forward x Green x Z backward for 256-long pencils padded to
// 512; PAPER.md:103-109 four-step solve, :181 / :213 padded and pruned transforms) with TWO neighbouring pencils
// per thread.
//
// fast_pad_kernel<FMODE_FUSED> is bound by instruction issue (profiles/r01_d.md: 1322 issue cycles per warp-tile,
// 370 of them not arithmetic: 8-byte shared-memory exchange accesses, 4-byte table loads, address arithmetic).
// Here a thread owns pencils 2 pp and 2 pp + 1 of the 16-pencil tile, so that every shared-memory exchange access,
// every read of the staged tile and every global store moves 16 bytes (both pencils), every Green's factor load 8,
// and one set of addresses and one twiddle operand serve two transforms: half the non-arithmetic instructions per
// pencil.  A CTA has 256 threads: half-warp = residue o of the 256-point transform (16 of them), its 16 lanes =
// 8 pencil pairs x 2 halves h of the padded problem; two CTAs per SM (<= 128 registers).  Everything else --
// radix 16 x 16 with one exchange per transform in alternating orientation, TMA-fed slot, dynamic tile queue,
// Nyquist-column tiles from the side array -- is as in sf_fast.cuh.
#pragma once
#include "sf_fast.cuh"

namespace sf2 {

constexpr int kT2 = 256;
constexpr int kXchg2Elems = 16 * 16 * 16;      // float4: both pencils of a thread
constexpr size_t kSmem2 = (size_t)kXchg2Elems * sizeof(float4) + (size_t)kL * kTile * sizeof(C);

// first half of a 256-point transform of both pencils: radix-16 over r, twiddle w256^(q o), write slots (q, o)
template <bool INV, bool ORIENT_B> __device__ __forceinline__ void fft256_a2(C (&va)[16], C (&vb)[16], const C* tw256, float4* x4, int ea, int eb)
{
    dft16<INV>(va);
    dft16<INV>(vb);
#pragma unroll
    for (int q = 1; q < 16; ++q) {
        const C w = tw256[q];
        va[brev4(q)] = cmul_sel<INV>(va[brev4(q)], w);
        vb[brev4(q)] = cmul_sel<INV>(vb[brev4(q)], w);
    }
    float4* w4 = x4 + (ORIENT_B ? eb : ea);
    constexpr int ws = (ORIENT_B ? 16 : 256);
#pragma unroll
    for (int q = 0; q < 16; ++q) w4[q * ws] = make_float4(va[brev4(q)].x, va[brev4(q)].y, vb[brev4(q)].x, vb[brev4(q)].y);
}
// second half (after a barrier): read slots (o, o'), radix-16 over o'.  X[o + 16 k2] at v[brev4(k2)] out.
template <bool INV, bool ORIENT_B> __device__ __forceinline__ void fft256_b2(C (&va)[16], C (&vb)[16], const float4* x4, int ea, int eb)
{
    const float4* r4 = x4 + (ORIENT_B ? ea : eb);
    constexpr int rs = (ORIENT_B ? 256 : 16);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const float4 t = r4[i * rs];
        va[i] = make_float2(t.x, t.y);
        vb[i] = make_float2(t.z, t.w);
    }
    dft16<INV>(va);
    dft16<INV>(vb);
}

// the same two halves with the exchange buffer as two planes of 8-byte slots (one per register set) instead of 16-byte
// slots: two 8-byte stores / loads per slot pair, but no moves that pack two register pairs into an aligned quad
constexpr int kPlane2 = 16 * 16 * 16;   // C elements per plane
template <bool INV, bool ORIENT_B> __device__ __forceinline__ void fft256_a2p(C (&va)[16], C (&vb)[16], const C* tw256, C* xp, int ea, int eb)
{
    dft16<INV>(va);
    dft16<INV>(vb);
#pragma unroll
    for (int q = 1; q < 16; ++q) {
        const C w = tw256[q];
        va[brev4(q)] = cmul_sel<INV>(va[brev4(q)], w);
        vb[brev4(q)] = cmul_sel<INV>(vb[brev4(q)], w);
    }
    C* w0 = xp + (ORIENT_B ? eb : ea);
    constexpr int ws = (ORIENT_B ? 16 : 256);
#pragma unroll
    for (int q = 0; q < 16; ++q) { w0[q * ws] = va[brev4(q)]; w0[kPlane2 + q * ws] = vb[brev4(q)]; }
}
template <bool INV, bool ORIENT_B> __device__ __forceinline__ void fft256_b2p(C (&va)[16], C (&vb)[16], const C* xp, int ea, int eb)
{
    const C* r0 = xp + (ORIENT_B ? ea : eb);
    constexpr int rs = (ORIENT_B ? 256 : 16);
#pragma unroll
    for (int i = 0; i < 16; ++i) { va[i] = r0[i * rs]; vb[i] = r0[kPlane2 + i * rs]; }
    dft16<INV>(va);
    dft16<INV>(vb);
}

__global__ void __launch_bounds__(kT2, 2) fast_fused2_kernel(const FastParams p, const __grid_constant__ CUtensorMap tm)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* x4 = reinterpret_cast<float4*>(smem_raw);
    C* slot = reinterpret_cast<C*>(smem_raw + (size_t)kXchg2Elems * sizeof(float4));
    __shared__ __align__(8) uint64_t bar;
    __shared__ __align__(16) C s_tab[768];   // [0, 256) tw256[o][q]; [256, 768) tw512[h][o][r] (g_tab_pad)
    __shared__ int s_tile[2];

    const int tid = threadIdx.x;
    const int l16 = tid & 15;
    const int pp = l16 & 7;          // pencils 2 pp, 2 pp + 1
    const int h = l16 >> 3;
    const int o = tid >> 4;
    const int ea = o * 16 + l16;
    const int eb = o * 256 + l16;
    const C* t256 = s_tab + o * 16;
    const C* t512 = s_tab + 256 + (h * 16 + o) * 16;

    const int ntiles = fast_ntiles(p.nb, p.nct, p.nyq_col);
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;
    uint32_t parity = 0;

    auto issue = [&](int t) {
        if (tid != 0 || t >= ntiles) return;
        const TileGeom g = tile_geom(p, t);
        if (!g.full) return;
        mbar_expect_tx(&bar, kL * kTile * (uint32_t)sizeof(C));
        tma_load_4d(slot, &tm, g.col, g.b, 0, 0, &bar);
    };
    auto advance = [&](int it) {
        if (tid != 0) return;
        issue(s_tile[(it + 1) & 1]);
        s_tile[it & 1] = atomicAdd(p.sched, 1) + 2 * (int)gridDim.x;
    };

    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s_tile[0] = (int)blockIdx.x;
        s_tile[1] = (int)(blockIdx.x + gridDim.x);
        issue(s_tile[0]);
    }
    for (int i = tid; i < 384; i += kT2) reinterpret_cast<float4*>(s_tab)[i] = reinterpret_cast<const float4*>(g_tab_pad)[i];
    __syncthreads();

    for (int it = 0;; ++it) {
        const int t = s_tile[it & 1];
        if (t >= ntiles) break;
        const TileGeom g = tile_geom(p, t);
        // a Nyquist-column tile is 16 batches of one column; in the side array [row][batch] they are neighbours too
        const bool side = !g.full && p.nyq_in != nullptr;
        const bool pvalid = g.full || (g.b + 2 * pp < p.nb);   // nb is even: both pencils of the pair or none
        C va[16], vb[16];
        if (g.full) {
            mbar_wait(&bar, parity);
            parity ^= 1;
            const float4* s4 = reinterpret_cast<const float4*>(slot) + (o * (kTile / 2) + pp);
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const float4 x = s4[r * 16 * (kTile / 2)];
                va[r] = make_float2(x.x, x.y);
                vb[r] = make_float2(x.z, x.w);
            }
        } else if (side) {
            const C* inp = p.nyq_in + ((size_t)o * p.nb + min(g.b + 2 * pp, p.nb - 2));
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const float4 x = __ldg(reinterpret_cast<const float4*>(inp + (size_t)r * 16 * p.nb));
                va[r] = make_float2(x.x, x.y);
                vb[r] = make_float2(x.z, x.w);
            }
        } else {
            const C* ia = p.in + (min(g.b + 2 * pp, p.nb - 1) * ibs + g.col + o * ips);
            const C* ib = p.in + (min(g.b + 2 * pp + 1, p.nb - 1) * ibs + g.col + o * ips);
#pragma unroll
            for (int r = 0; r < 16; ++r) { va[r] = __ldg(ia + r * 16 * ips); vb[r] = __ldg(ib + r * 16 * ips); }
        }
        // h = 0: x -> even outputs;  h = 1: x w512^n -> odd outputs (the table row of h = 0 is all ones)
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const C w = t512[r];
            va[r] = cmul(va[r], w);
            vb[r] = cmul(vb[r], w);
        }
        fft256_a2<false, false>(va, vb, t256, x4, ea, eb);
        __syncthreads();
        advance(it);
        // Green's factors of the spectral rows kp = 2 (o + 16 k2) + h, folded to min(kp, 512 - kp), both pencils
        float2 gm[16];
        {
            const float* gt = p.green_tiles + ((size_t)green_tile_index(p, g) * (kGreenRows * kTile) + 2 * pp);
            const float* glo = gt + (2 * o + h) * kTile;
            const float* ghi = gt + (2 * kL - 2 * o - h) * kTile;
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) gm[k2] = __ldg(reinterpret_cast<const float2*>(k2 < 8 ? glo + k2 * 32 * kTile : ghi - k2 * 32 * kTile));
        }
        fft256_b2<false, false>(va, vb, x4, ea, eb);
        {
            C ua[16], ub[16];
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) { ua[k2] = cscale(va[brev4(k2)], gm[k2].x); ub[k2] = cscale(vb[brev4(k2)], gm[k2].y); }
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) { va[k2] = ua[k2]; vb[k2] = ub[k2]; }
        }
        fft256_a2<true, true>(va, vb, t256, x4, ea, eb);
        __syncthreads();
        fft256_b2<true, true>(va, vb, x4, ea, eb);
        // x_j = e_j + conj(w512^j) o_j, j = o + 16 r: h = 0 holds e, h = 1 holds o; the two lanes swap half of
        // their values: h = 0 finishes r < 8, h = 1 finishes r >= 8
        C* outp;
        int ost;
        if (g.full) { outp = p.out + (g.b * obs + g.col + 2 * pp); ost = ops; }
        else if (side) { outp = p.nyq_out + (g.b + 2 * pp); ost = p.nb; }
        else { outp = p.out + ((g.b + 2 * pp) * obs + g.col); ost = ops; }
        outp += (size_t)(o + 128 * h) * ost;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const C wl = t512[r], wh = t512[r + 8];
            const C al = cmulc(va[brev4(r)], wl), ah = cmulc(va[brev4(r + 8)], wh);
            const C bl = cmulc(vb[brev4(r)], wl), bh = cmulc(vb[brev4(r + 8)], wh);
            const C sa = h ? al : ah, ka = h ? ah : al;
            const C sb = h ? bl : bh, kb = h ? bh : bl;
            C ra, rb;
            ra.x = __shfl_xor_sync(0xffffffffu, sa.x, 8);
            ra.y = __shfl_xor_sync(0xffffffffu, sa.y, 8);
            rb.x = __shfl_xor_sync(0xffffffffu, sb.x, 8);
            rb.y = __shfl_xor_sync(0xffffffffu, sb.y, 8);
            const C xa = cadd(ka, ra), xb = cadd(kb, rb);
            if (pvalid) {
                if (g.full || side) {
                    *reinterpret_cast<float4*>(outp + (size_t)r * 16 * ost) = make_float4(xa.x, xa.y, xb.x, xb.y);
                } else {
                    outp[(size_t)r * 16 * ost] = xa;
                    outp[(size_t)r * 16 * ost + obs] = xb;
                }
            }
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


// ------------------------------------------------------------------------------------ both halves per thread
// The same pass with the two register sets of a thread holding the EVEN and the ODD half of ONE pencil's padded
// transform instead of one half of two pencils: half-warp = residue o, its 16 lanes = the 16 pencils of the tile.
// The even half then needs no input factor and no output factor (in the kernel above every lane multiplies, the
// lanes of the even half by one), the combine x_j = e_j + conj(w512^j) o_j is local (no shuffles, no selects), and a
// tile needs no pairing of pencils (odd batch counts run here too).  Exchange, slot, tile queue as above.
__global__ void __launch_bounds__(kT2, 2) fast_fused2h_kernel(const FastParams p, const __grid_constant__ CUtensorMap tm)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* xp = reinterpret_cast<C*>(smem_raw);
    C* slot = reinterpret_cast<C*>(smem_raw + (size_t)kXchg2Elems * sizeof(float4));
    __shared__ __align__(8) uint64_t bar;
    __shared__ __align__(16) C s_tab[512];   // [0, 256) tw256[o][q]; [256, 512) tw512[o][r] = w512^(o + 16 r)
    __shared__ int s_tile[2];

    const int tid = threadIdx.x;
    const int pen = tid & 15;
    const int o = tid >> 4;
    const int ea = o * 16 + pen;
    const int eb = o * 256 + pen;
    const C* t256 = s_tab + o * 16;
    const C* t512 = s_tab + 256 + o * 16;

    const int ntiles = fast_ntiles(p.nb, p.nct, p.nyq_col);
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;
    uint32_t parity = 0;

    auto issue = [&](int t) {
        if (tid != 0 || t >= ntiles) return;
        const TileGeom g = tile_geom(p, t);
        if (!g.full) return;
        mbar_expect_tx(&bar, kL * kTile * (uint32_t)sizeof(C));
        tma_load_4d(slot, &tm, g.col, g.b, 0, 0, &bar);
    };
    auto advance = [&](int it) {
        if (tid != 0) return;
        issue(s_tile[(it + 1) & 1]);
        s_tile[it & 1] = atomicAdd(p.sched, 1) + 2 * (int)gridDim.x;
    };

    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s_tile[0] = (int)blockIdx.x;
        s_tile[1] = (int)(blockIdx.x + gridDim.x);
        issue(s_tile[0]);
    }
    // g_tab_pad: [0, 256) tw256, [256, 512) ones (row h = 0), [512, 768) tw512 (row h = 1)
    if (tid < 128) reinterpret_cast<float4*>(s_tab)[tid] = reinterpret_cast<const float4*>(g_tab_pad)[tid];
    else reinterpret_cast<float4*>(s_tab)[tid] = reinterpret_cast<const float4*>(g_tab_pad)[tid + 128];
    __syncthreads();

    for (int it = 0;; ++it) {
        const int t = s_tile[it & 1];
        if (t >= ntiles) break;
        const TileGeom g = tile_geom(p, t);
        // a Nyquist-column tile is 16 batches of one column; in the side array [row][batch] they are neighbours too
        const bool side = !g.full && p.nyq_in != nullptr;
        const bool pvalid = g.full || (g.b + pen < p.nb);
        C v0[16], v1[16];
        if (g.full) {
            mbar_wait(&bar, parity);
            parity ^= 1;
            const C* s = slot + (o * kTile + pen);
#pragma unroll
            for (int r = 0; r < 16; ++r) v0[r] = s[r * 16 * kTile];
        } else if (side) {
            const C* inp = p.nyq_in + ((size_t)o * p.nb + min(g.b + pen, p.nb - 1));
#pragma unroll
            for (int r = 0; r < 16; ++r) v0[r] = __ldg(inp + (size_t)r * 16 * p.nb);
        } else {
            const C* inp = p.in + (min(g.b + pen, p.nb - 1) * ibs + g.col + o * ips);
#pragma unroll
            for (int r = 0; r < 16; ++r) v0[r] = __ldg(inp + r * 16 * ips);
        }
        // even outputs: x;  odd outputs: x w512^n, n = o + 16 r
#pragma unroll
        for (int r = 0; r < 16; ++r) v1[r] = cmul(v0[r], t512[r]);
        fft256_a2p<false, false>(v0, v1, t256, xp, ea, eb);
        __syncthreads();
        advance(it);
        // Green's factors of the spectral rows kp = 2 (o + 16 k2) + h, folded to min(kp, 512 - kp)
        float g0[16], g1[16];
        {
            const float* gt = p.green_tiles + ((size_t)green_tile_index(p, g) * (kGreenRows * kTile) + pen);
            const float* glo = gt + (2 * o) * kTile;
            const float* ghi = gt + (2 * kL - 2 * o) * kTile;
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) {
                g0[k2] = __ldg(k2 < 8 ? glo + k2 * 32 * kTile : ghi - k2 * 32 * kTile);
                g1[k2] = __ldg(k2 < 8 ? glo + (k2 * 32 + 1) * kTile : ghi - (k2 * 32 + 1) * kTile);
            }
        }
        fft256_b2p<false, false>(v0, v1, xp, ea, eb);
        {
            C u0[16], u1[16];
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) { u0[k2] = cscale(v0[brev4(k2)], g0[k2]); u1[k2] = cscale(v1[brev4(k2)], g1[k2]); }
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) { v0[k2] = u0[k2]; v1[k2] = u1[k2]; }
        }
        fft256_a2p<true, true>(v0, v1, t256, xp, ea, eb);
        __syncthreads();
        fft256_b2p<true, true>(v0, v1, xp, ea, eb);
        // x_j = e_j + conj(w512^j) o_j, j = o + 16 r < 256
        C* outp;
        int ost;
        if (g.full) { outp = p.out + (g.b * obs + g.col + pen); ost = ops; }
        else if (side) { outp = p.nyq_out + (g.b + pen); ost = p.nb; }
        else { outp = p.out + ((g.b + pen) * obs + g.col); ost = ops; }
        outp += (size_t)o * ost;
        if (pvalid) {
#pragma unroll
            for (int r = 0; r < 16; ++r) outp[(size_t)r * 16 * ost] = cadd(v0[brev4(r)], cmulc(v1[brev4(r)], t512[r]));
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


// ------------------------------------------------------------------------------------ S4 with both halves per thread
// FMODE_INV of fast_pad_kernel (rows k < 512 -> rows j < 256) in the same mapping: a thread reads the even row 2 m
// and the odd row 2 m + 1, m = o + 16 k2, of its pencil (32 loads in flight), runs the two inverse 256-point
// transforms through one float4 exchange and combines them locally.  No slot (the rows go straight into registers);
// consecutive tiles alternate the orientation of the exchange buffer: one barrier per tile.
constexpr size_t kSmemInv2 = (size_t)kXchg2Elems * sizeof(float4);

__global__ void __launch_bounds__(kT2, 2) fast_inv2h_kernel(const FastParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* xbuf = reinterpret_cast<C*>(smem_raw);   // staging of a Nyquist tile image: 512 rows x 16 pencils = the same 64 KB
    __shared__ __align__(16) C s_tab[512];      // [0, 256) tw256[o][q]; [256, 512) tw512[o][r] = w512^(o + 16 r)
    __shared__ int s_tile[2];

    const int tid = threadIdx.x;
    const int pen = tid & 15;
    const int o = tid >> 4;
    const int ea = o * 16 + pen;
    const int eb = o * 256 + pen;
    const C* t256 = s_tab + o * 16;
    const C* t512 = s_tab + 256 + o * 16;

    const int ntiles = fast_ntiles(p.nb, p.nct, p.nyq_col);
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;
    auto stage = [&](int row, int pencil) -> C& { return xbuf[row * kTile + ((pencil + row) & 15)]; };

    if (tid == 0) {
        s_tile[0] = (int)blockIdx.x;
        s_tile[1] = (int)(blockIdx.x + gridDim.x);
    }
    if (tid < 128) reinterpret_cast<float4*>(s_tab)[tid] = reinterpret_cast<const float4*>(g_tab_pad)[tid];
    else reinterpret_cast<float4*>(s_tab)[tid] = reinterpret_cast<const float4*>(g_tab_pad)[tid + 128];
    __syncthreads();

    auto tile = [&](int t, int it, auto orient_tag) {
        constexpr bool OB = decltype(orient_tag)::value;
        const TileGeom g = tile_geom(p, t);
        const bool side = !g.full && p.nyq_in != nullptr;
        const bool pvalid = g.full || (g.b + pen < p.nb);
        C v0[16], v1[16];
        if (side) {
            // the producer (S3) left this column as [pencil of S4 = z][ky]: read 512 contiguous ky per z and transpose
            // through the exchange buffer (which the previous tile's second half may still be reading)
            if (it > 0) __syncthreads();
            for (int idx = tid; idx < 2 * kL * kTile; idx += kT2) {
                const int pp = idx >> 9, ky = idx & (2 * kL - 1);
                stage(ky, pp) = (g.b + pp < p.nb) ? __ldg(p.nyq_in + (g.b + pp) * (2 * kL) + ky) : make_float2(0.f, 0.f);
            }
            __syncthreads();
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) { v0[k2] = stage(2 * (o + 16 * k2), pen); v1[k2] = stage(2 * (o + 16 * k2) + 1, pen); }
            __syncthreads();   // before the exchange overwrites the staging
        } else {
            const C* inp = p.in + ((g.full ? (g.b * ibs + g.col + pen) : (min(g.b + pen, p.nb - 1) * ibs + g.col)) + 2 * o * ips);
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) { v0[k2] = __ldg(inp + k2 * 32 * ips); v1[k2] = __ldg(inp + ips + k2 * 32 * ips); }
        }
        fft256_a2p<true, OB>(v0, v1, t256, xbuf, ea, eb);
        __syncthreads();
        {
            // ask the next tile's 512 rows of 128 bytes into the L2 while this one is transformed
            const int tn = s_tile[(it + 1) & 1];
            if (tn < ntiles) {
                const TileGeom gn = tile_geom(p, tn);
                if (gn.full) {
                    const C* nx = p.in + (gn.b * ibs + gn.col);
                    prefetch_l2(nx + (size_t)tid * ips);
                    prefetch_l2(nx + (size_t)(tid + kT2) * ips);
                }
            }
        }
        if (tid == 0) s_tile[it & 1] = atomicAdd(p.sched, 1) + 2 * (int)gridDim.x;
        fft256_b2p<true, OB>(v0, v1, xbuf, ea, eb);
        // x_j = e_j + conj(w512^j) o_j, j = o + 16 r < 256
        C* outp;
        int ost;
        if (g.full) { outp = p.out + (g.b * obs + g.col + pen); ost = ops; }
        else if (side) { outp = p.nyq_out + (g.b + pen); ost = p.nb; }
        else { outp = p.out + ((g.b + pen) * obs + g.col); ost = ops; }
        outp += (size_t)o * ost;
        if (pvalid) {
#pragma unroll
            for (int r = 0; r < 16; ++r) outp[(size_t)r * 16 * ost] = cadd(v0[brev4(r)], cmulc(v1[brev4(r)], t512[r]));
        }
    };

    for (int it = 0;; it += 2) {
        int t = s_tile[0];
        if (t >= ntiles) break;
        tile(t, it, std::false_type());
        t = s_tile[1];
        if (t >= ntiles) break;
        tile(t, it + 1, std::true_type());
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


// ------------------------------------------------------------------------------------ S2 with both halves per thread
// FMODE_FWD of fast_pad_kernel (rows n < 256 -> rows k < 512) in the same mapping: the staged tile is read once per
// element (not once per half), the odd half's input factor is the only one applied, and a thread stores the even row
// 2 m and the odd row 2 m + 1, m = o + 16 k2, of its pencil.  TMA-fed slot and tile queue as in fast_fused2h_kernel;
// consecutive tiles alternate the orientation of the exchange buffer.  `tm`: dims (column, row, batch, 1).
__global__ void __launch_bounds__(kT2, 2) fast_fwd2h_kernel(const FastParams p, const __grid_constant__ CUtensorMap tm)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* xbuf = reinterpret_cast<C*>(smem_raw);   // staging of a Nyquist tile image (512 rows x 16 pencils)
    C* slot = reinterpret_cast<C*>(smem_raw + (size_t)kXchg2Elems * sizeof(float4));
    __shared__ __align__(8) uint64_t bar;
    __shared__ __align__(16) C s_tab[512];
    __shared__ int s_tile[2];

    const int tid = threadIdx.x;
    const int pen = tid & 15;
    const int o = tid >> 4;
    const int ea = o * 16 + pen;
    const int eb = o * 256 + pen;
    const C* t256 = s_tab + o * 16;
    const C* t512 = s_tab + 256 + o * 16;

    const int ntiles = fast_ntiles(p.nb, p.nct, p.nyq_col);
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;
    uint32_t parity = 0;
    auto stage = [&](int row, int pencil) -> C& { return xbuf[row * kTile + ((pencil + row) & 15)]; };
    auto issue = [&](int t) {
        if (tid != 0 || t >= ntiles) return;
        const TileGeom g = tile_geom(p, t);
        if (!g.full) return;
        mbar_expect_tx(&bar, kL * kTile * (uint32_t)sizeof(C));
        tma_load_4d(slot, &tm, g.col, 0, g.b, 0, &bar);
    };
    auto advance = [&](int it) {
        if (tid != 0) return;
        issue(s_tile[(it + 1) & 1]);
        s_tile[it & 1] = atomicAdd(p.sched, 1) + 2 * (int)gridDim.x;
    };

    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s_tile[0] = (int)blockIdx.x;
        s_tile[1] = (int)(blockIdx.x + gridDim.x);
        issue(s_tile[0]);
    }
    if (tid < 128) reinterpret_cast<float4*>(s_tab)[tid] = reinterpret_cast<const float4*>(g_tab_pad)[tid];
    else reinterpret_cast<float4*>(s_tab)[tid] = reinterpret_cast<const float4*>(g_tab_pad)[tid + 128];
    __syncthreads();

    auto tile = [&](int t, int it, auto orient_tag) {
        constexpr bool OB = decltype(orient_tag)::value;
        const TileGeom g = tile_geom(p, t);
        const bool side = !g.full && p.nyq_in != nullptr;
        const bool pvalid = g.full || (g.b + pen < p.nb);
        C v0[16], v1[16];
        if (g.full) {
            mbar_wait(&bar, parity);
            parity ^= 1;
            const C* s = slot + (o * kTile + pen);
#pragma unroll
            for (int r = 0; r < 16; ++r) v0[r] = s[r * 16 * kTile];
        } else if (side) {
            // Nyquist column from its side array [row][batch]: the 16 batches are contiguous
            const C* inp = p.nyq_in + ((size_t)o * p.nb + min(g.b + pen, p.nb - 1));
#pragma unroll
            for (int r = 0; r < 16; ++r) v0[r] = __ldg(inp + (size_t)r * 16 * p.nb);
        } else {
            const C* inp = p.in + (min(g.b + pen, p.nb - 1) * ibs + g.col + o * ips);
#pragma unroll
            for (int r = 0; r < 16; ++r) v0[r] = __ldg(inp + r * 16 * ips);
        }
        // even outputs: x;  odd outputs: x w512^n, n = o + 16 r
#pragma unroll
        for (int r = 0; r < 16; ++r) v1[r] = cmul(v0[r], t512[r]);
        fft256_a2p<false, OB>(v0, v1, t256, xbuf, ea, eb);
        __syncthreads();
        advance(it);
        fft256_b2p<false, OB>(v0, v1, xbuf, ea, eb);
        if (side) {
            // the consumer (S3) wants this column as [pencil of S2 = z][ky]: transpose through the exchange buffer and
            // write 512 contiguous ky per z
            __syncthreads();   // every thread is done reading the exchange buffer
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) {
                stage(2 * (o + 16 * k2), pen) = v0[brev4(k2)];
                stage(2 * (o + 16 * k2) + 1, pen) = v1[brev4(k2)];
            }
            __syncthreads();
            for (int idx = tid; idx < 2 * kL * kTile; idx += kT2) {
                const int pp = idx >> 9, ky = idx & (2 * kL - 1);
                if (g.b + pp < p.nb) p.nyq_out[(g.b + pp) * (2 * kL) + ky] = stage(ky, pp);
            }
            __syncthreads();   // before the next tile's exchange
        } else if (pvalid) {
            C* q = p.out + ((g.full ? (g.b * obs + g.col + pen) : ((g.b + pen) * obs + g.col)) + 2 * o * ops);   // row 2 (o + 16 k2) + h
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) {
                q[k2 * 32 * ops] = v0[brev4(k2)];
                q[k2 * 32 * ops + ops] = v1[brev4(k2)];
            }
        }
    };

    for (int it = 0;; it += 2) {
        int t = s_tile[0];
        if (t >= ntiles) break;
        tile(t, it, std::false_type());
        t = s_tile[1];
        if (t >= ntiles) break;
        tile(t, it + 1, std::true_type());
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

} // namespace sf2
