// sf_fastx5w.cuh -- S1 (X forward) and S5 (X backward) for rows of 512 reals zero-padded to 1024 (PAPER.md:87 real
// transform / half spectrum; PAPER.md:181 padding): fast_x5_kernel of sf_fast512.cuh with one pipeline PER WARP, the
// scheme of sf_fastxw.cuh one size up.  A warp owns ONE row per iteration:
//     lane = 2 o + h,   o = residue of the 256-point transform,  h = half of the padded problem.
// The padded real row is packed as z[n] = x[2n] + i x[2n+1], n < 512, non-zero for n < 256; Z = DFT512(z) is two
// 256-point transforms (radix 16 x 16, one exchange between the 16 lanes of a half), of z (even outputs, h = 0) and of
// z w512^n (odd outputs, h = 1).  Lane idx = 2 o + h then holds Z[idx + 32 j], j < 16; the partner 512 - k of
// k = idx + 32 m, m < 8, is j' = 15 - m of lane idx' = 32 - idx, so the real-transform split
//     X[k] = ((Z[k] + conj Z[512-k]) - i w1024^k (Z[k] - conj Z[512-k])) / 2,   k = 0..512
// (S1) and its mirror (S5) pair up through shuffles and the results leave by 8-byte stores, 256 consecutive bytes per
// warp.  Shared memory carries the bulk-copied input row and the exchange only; __syncwarp is the only barrier.
// Twiddles: the part of the odd half's factor that does not depend on the radix-16 index rides on the table
// (forward w512^((2 q + h) o), backward w512^(q (2 o + h))), the rest, w32^r, are immediates.
#pragma once
#include "sf_fast.cuh"
#include "sf_fast512.cuh"

namespace sf2 {

constexpr int kX5wWarps = 8;
constexpr int kX5wThreads = 32 * kX5wWarps;
constexpr int kX5wQP = 17;                                   // exchange: words per q (odd: conflict-free both ways)
constexpr int kX5wGP = 16 * kX5wQP + 8;                      // exchange: words per half, 8 (mod 16)
constexpr int kX5wTab = 1280;                                // forward tw[q][h][o] | backward tw[q][h][o] | twsp[m][idx]
constexpr int kX5wTabCta = 768;                              // what one kernel keeps in shared memory
constexpr size_t kX5wRealBytes = (size_t)kX5N * sizeof(float);          // 2 KB
constexpr size_t kX5wSpecBytes = (size_t)kX5SpPitch * sizeof(C);        // 4112 B
constexpr size_t kX5wXchBytes = 2 * (size_t)kX5wGP * sizeof(C);
// forward: two input rows (prefetch distance two) and the exchange;  backward: one input row and the exchange
constexpr size_t kX5wWarpBytesFwd = 2 * kX5wRealBytes + kX5wXchBytes;
constexpr size_t kX5wWarpBytesInv = kX5wSpecBytes + kX5wXchBytes;
constexpr size_t kX5wSmemFwd = kX5wWarps * kX5wWarpBytesFwd;
constexpr size_t kX5wSmemInv = kX5wWarps * kX5wWarpBytesInv;
static_assert(kX5wWarpBytesFwd % 16 == 0 && kX5wWarpBytesInv % 16 == 0, "bulk copies need 16-byte aligned rows");

__device__ float2 g_tab_x5w[kX5wTab];

template <bool INV, int R = 1> __device__ __forceinline__ void mul32_nat(C (&v)[16])
{
    if constexpr (R < 16) {
        v[R] = mul_w32<R, INV>(v[R]);
        mul32_nat<INV, R + 1>(v);
    }
}
template <bool INV, int R = 1> __device__ __forceinline__ void mul32_rev(C (&v)[16])
{
    if constexpr (R < 16) {
        v[brev4(R)] = mul_w32<R, INV>(v[brev4(R)]);
        mul32_rev<INV, R + 1>(v);
    }
}

template <bool INV> __global__ void __launch_bounds__(kX5wThreads, 2) fast_x5w_kernel(const FastXParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bars[kX5wWarps][2];
    __shared__ __align__(16) C s_tab[kX5wTabCta];

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int wid = tid >> 5;
    const int o = lane >> 1;
    const int h = lane & 1;
    const int idx = lane;                 // = 2 o + h: this lane ends up with Z[idx + 32 j]
    // the lane that holds the residue 32 - idx (mod 32): idx = 0 and idx = 16 are their own partners
    const int plane = (32 - idx) & 31;

    for (int i = tid; i < kX5wTabCta / 2; i += kX5wThreads)
        reinterpret_cast<float4*>(s_tab)[i] = reinterpret_cast<const float4*>(g_tab_x5w)[i + (i < 256 ? (INV ? 256 : 0) : 256)];
    if (lane == 0) {
        mbar_init(&bars[wid][0], 1);
        mbar_init(&bars[wid][1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const C* t256 = s_tab + h * 16 + o;   // [q * 32]
    __syncthreads();
    C tsp[8];                             // w1024^(idx + 32 m): the same in every iteration
#pragma unroll
    for (int m = 0; m < 8; ++m) tsp[m] = s_tab[512 + idx + 32 * m];

    unsigned char* wbase = smem_raw + (size_t)wid * (INV ? kX5wWarpBytesInv : kX5wWarpBytesFwd);
    float* rbuf = reinterpret_cast<float*>(wbase);
    const C* srow = reinterpret_cast<const C*>(wbase);
    C* xch = reinterpret_cast<C*>(wbase + (INV ? kX5wSpecBytes : 2 * kX5wRealBytes));
    C* xw = xch + h * kX5wGP + o;                 // slot (q, o) at q * kX5wQP
    const C* xr = xch + h * kX5wGP + o * kX5wQP;  // slots (o, o')

    const long long nrows = p.nrows;
    const long long gw = (long long)blockIdx.x * kX5wWarps + wid;
    const long long nw = (long long)gridDim.x * kX5wWarps;
    const int nit = gw < nrows ? (int)((nrows - gw + nw - 1) / nw) : 0;
    auto row_of = [&](int i) -> long long {
        const long long r = gw + (long long)i * nw;
        return p.reverse ? nrows - 1 - r : r;
    };
    // lane 0 starts the row copy of iteration i (forward: into input buffer i & 1)
    auto issue = [&](int i) {
        if (lane != 0 || i >= nit) return;
        const long long row = row_of(i);
        if (INV) {
            mbar_expect_tx(&bars[wid][0], (uint32_t)kX5wSpecBytes);
            bulk_g2s(wbase, p.spec + row * p.spec_pitch, (uint32_t)kX5wSpecBytes, &bars[wid][0]);
        } else {
            mbar_expect_tx(&bars[wid][i & 1], (uint32_t)kX5wRealBytes);
            bulk_g2s(wbase + (i & 1) * kX5wRealBytes, p.real_in + row * kX5N, (uint32_t)kX5wRealBytes, &bars[wid][i & 1]);
        }
    };

    issue(0);
    if (!INV) issue(1);
    for (int i = 0; i < nit; ++i) {
        const long long row = row_of(i);
        C v[16];
        if constexpr (!INV) {
            // ---------------------------------------------------------------- S1
            mbar_wait(&bars[wid][i & 1], (i >> 1) & 1);
            const C* zin = reinterpret_cast<const C*>(rbuf + (i & 1) * kX5N) + o;
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = zin[16 * r];
            if (h) mul32_nat<false>(v);   // h = 1: z w512^n, n = o + 16 r: w32^r here, w512^o with the twiddles
            dft16<false>(v);
#pragma unroll
            for (int q = 0; q < 16; ++q) v[brev4(q)] = cmul(v[brev4(q)], t256[q * 32]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * kX5wQP] = v[brev4(q)];
            __syncwarp();
            issue(i + 2);                 // this input buffer is in registers in every lane
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = xr[j];
            dft16<false>(v);
            // v[brev4(j)] = Z[idx + 32 j]
            C* orow = p.spec + row * p.spec_pitch;
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const C snd = v[brev4(15 - m)];
                C zm;
                zm.x = __shfl_sync(0xffffffffu, snd.x, plane);
                zm.y = __shfl_sync(0xffffffffu, snd.y, plane);
                if (idx == 0) zm = v[brev4((16 - m) & 15)];   // 512 - 32 m = 32 (16 - m) is its own
                const C zk = v[brev4(m)];
                const C e = cadd(zk, make_float2(zm.x, -zm.y));
                const C d = csub(zk, make_float2(zm.x, -zm.y));
                const C wd = cmul(d, tsp[m]);   // w1024^k d
                // X[k] = (e - i wd) / 2,  X[512 - k] = (conj e - i conj wd) / 2
                const int k = idx + 32 * m;
                orow[k] = cscale(cadd(e, make_float2(wd.y, -wd.x)), 0.5f);
                orow[kX5N - k] = cscale(make_float2(e.x - wd.y, -e.y - wd.x), 0.5f);
                if (m == 0 && idx == 0) orow[kX5N + 1] = make_float2(0.f, 0.f);   // pad column 513 leaves as zero
            }
            if (idx == 0) orow[kX5N / 2] = make_float2(v[brev4(8)].x, -v[brev4(8)].y);   // k = 256 pairs with itself
        } else {
            // ---------------------------------------------------------------- S5
            mbar_wait(&bars[wid][0], i & 1);
            // merge: Z[k] = e + i conj(w1024^k) d, Z[512 - k] = conj e + i conj(conj(w1024^k) d), k = idx + 32 m, m < 8.
            // Z[k] is this lane's v[m]; Z[512 - k] is v[15 - m] of the partner lane
            C zhi[8];
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int k = idx + 32 * m;
                const C xk = srow[k], xm = srow[kX5N - k];
                const C e = cadd(xk, make_float2(xm.x, -xm.y));
                const C d = csub(xk, make_float2(xm.x, -xm.y));
                const C wd = cmulc(d, tsp[m]);   // conj(w1024^k) d
                v[m] = cadd(e, make_float2(-wd.y, wd.x));
                zhi[m] = make_float2(e.x + wd.y, wd.x - e.y);
            }
            const C x256 = srow[kX5N / 2];
#pragma unroll
            for (int j = 8; j < 16; ++j) {
                C r;
                r.x = __shfl_sync(0xffffffffu, zhi[15 - j].x, plane);
                r.y = __shfl_sync(0xffffffffu, zhi[15 - j].y, plane);
                // idx = 0: 512 - 32 m = 32 (16 - m) is its own; Z[256] = 2 conj X[256]
                if (idx == 0) r = (j == 8) ? make_float2(2.f * x256.x, -2.f * x256.y) : zhi[(16 - j) & 7];
                v[j] = r;
            }
            dft16<true>(v);   // v[j] = Z[2 (o + 16 j) + h] in
#pragma unroll
            for (int q = 0; q < 16; ++q) v[brev4(q)] = cmulc(v[brev4(q)], t256[q * 32]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * kX5wQP] = v[brev4(q)];
            __syncwarp();
            issue(i + 1);                 // the staged row is in registers in every lane
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = xr[j];
            dft16<true>(v);
            // z[n] = z0[n] + conj(w512^n) z1[n], n = o + 16 k2 < 256: h = 0 holds z0, h = 1 holds z1 conj(w512^o) (the
            // factor came with the twiddles), conj(w32^k2) is applied here; the two lanes swap half of their values:
            // h = 0 finishes k2 < 8, h = 1 finishes k2 >= 8
            if (h) mul32_rev<true>(v);
            C* orow = reinterpret_cast<C*>(p.real_out + row * kX5N);
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const C a = v[brev4(r)], b = v[brev4(r + 8)];
                const C send = h ? a : b;
                const C keep = h ? b : a;
                C recv;
                recv.x = __shfl_xor_sync(0xffffffffu, send.x, 1);
                recv.y = __shfl_xor_sync(0xffffffffu, send.y, 1);
                orow[o + 16 * r + 128 * h] = cadd(keep, recv);   // (x[2n], x[2n+1])
            }
        }
    }
}

} // namespace sf2
