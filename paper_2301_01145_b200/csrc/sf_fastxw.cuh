// sf_fastxw.cuh -- S1 (X forward) and S5 (X backward) for rows of 256 reals zero-padded to 512 (PAPER.md:87 real
// transform / half spectrum; PAPER.md:181 padding, :268-272 Set_Input .. Get_Output) with one pipeline PER WARP.
//
// fast_x_kernel (sf_fast.cuh) maps a tile of 16 rows onto a 256-thread CTA with warp = residue of the 128-point
// transform, so every exchange crosses warps: three CTA barriers per tile, and a quarter of all warp time is spent
// in them (profiles/r02_a: barrier is the first stall reason of both X passes, 24 % warps active, DRAM 39 - 42 %).
// Rows are independent, so here the 16 threads that transform one row sit in ONE warp:
//     lane = w + 8 h + 16 rr,   w = residue 0..7,  h = half of the padded problem,  rr = row of the pair,
// a warp owns two neighbouring rows per iteration, has its own staging buffers, mbarriers and bulk copies, and the
// only synchronisation left is __syncwarp.  Sixteen such pipelines run per SM, each at its own phase.
//   forward: the padded real row is packed as z[n] = x[2n] + i x[2n+1], n < 256, non-zero for n < 128.
//   Z = DFT256(z) = two 128-point transforms, of z (even outputs, h = 0) and of z w256^n (odd outputs, h = 1);
//   then the real-transform split X[k] = ((Z[k] + conj Z[256-k]) - i w512^k (Z[k] - conj Z[256-k])) / 2.
//   backward: the mirror.
//   128-point transform: radix-16 over r (n = w + 8 r), twiddle w128^(q w), one exchange between the eight
//   threads of the group, two radix-8 over o' for q = w and q = w + 8.
// Both passes are bound by shared-memory bandwidth, not by HBM (ncu: l1tex 78 % with staged output rows), so the
// shared memory is used for the input rows and the one exchange only: the thread with lane index idx = 2 w + h ends
// up with Z[idx + 16 j], j < 16, the partner 256 - k of its k sits in the thread 16 - idx as j' = 15 - j, so the
// split (and the merge of S5) pair up through 16 shuffles, and the results leave by plain 8-byte stores: the 16
// lanes of a row write 128 consecutive bytes.
// Shared-memory words are 8 bytes (one complex); every access of a half-warp (one row, 8 residues x 2 halves) is
// either 16 consecutive words or 8 words with stride 9 plus the same 8 shifted by 8 (mod 16): no bank conflicts.
#pragma once
#include "sf_fast.cuh"
#include "sf_fast512.cuh"   // mul_w32

namespace sf2 {

constexpr int kXwWarps = 8;
constexpr int kXwThreads = 32 * kXwWarps;
constexpr int kXwInPitch = kXN + 16;          // floats per staged real row: 1088 B = 64 (mod 128)
constexpr int kXwQP = 9;                      // exchange: words per q
constexpr int kXwGP = 152;                    // exchange: words per (row, half) group, 8 (mod 16)
constexpr int kXwTab = 640;                   // forward tw[q][h][w] | backward tw[q][h][w] | twsp[m][2 w + h]
constexpr int kXwTabCta = 384;                // what one kernel keeps in shared memory: its tw and twsp
constexpr size_t kXwRealBytes = 2 * (size_t)kXwInPitch * sizeof(float);   // a pair of real rows
constexpr size_t kXwSpecBytes = 2 * (size_t)kXSpPitch * sizeof(C);        // a pair of spectrum rows
constexpr size_t kXwXchBytes = 4 * (size_t)kXwGP * sizeof(C);
// forward: two input pairs (prefetch distance two) and the exchange;  backward: one input pair and the exchange
constexpr size_t kXwWarpBytesFwd = 2 * kXwRealBytes + kXwXchBytes;
constexpr size_t kXwWarpBytesInv = kXwSpecBytes + kXwXchBytes;
// warps per CTA of the padded passes: the backward pass (90 registers under this bound) gains from twelve, the forward
// pass does not (measured: S5 40.8 -> 38.9 us, S1 41.8 -> 42.2 us)
__host__ __device__ constexpr int xw_warps(bool inv) { return inv ? 12 : 8; }
constexpr size_t kXwSmemFwd = xw_warps(false) * kXwWarpBytesFwd;
constexpr size_t kXwSmemInv = xw_warps(true) * kXwWarpBytesInv;

__device__ float2 g_tab_xw[kXwTab];

// v[r] = a[w + 8 r] in; writes the twiddled radix-16 outputs into the group's exchange slots (q, w).  The table row
// holds w128^(q w) times the factor of the odd half that does not depend on r (forward: w256^w of the input factor
// w256^(w + 8 r); backward: w256^q of the output factor w256^(q + 16 k2)); the rest of those factors are immediates
template <bool INV> __device__ __forceinline__ void fftw128_a(C (&v)[16], const C* t128, C* xw)
{
    dft16<INV>(v);
#pragma unroll
    for (int q = 0; q < 16; ++q) v[brev4(q)] = cmul_sel<INV>(v[brev4(q)], t128[q * 16]);
#pragma unroll
    for (int q = 0; q < 16; ++q) xw[q * kXwQP] = v[brev4(q)];
}
// after __syncwarp: A[w + 16 k2] at a[brev3(k2)], A[w + 8 + 16 k2] at b[brev3(k2)]
template <bool INV> __device__ __forceinline__ void fftw128_b(C (&a)[8], C (&b)[8], const C* xr)
{
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = xr[i]; b[i] = xr[8 * kXwQP + i]; }
    dft8<INV>(a);
    dft8<INV>(b);
}


template <bool INV> __global__ void __launch_bounds__(32 * xw_warps(INV), 2) fast_xw_kernel(const FastXParams p)
{
    constexpr int NW = xw_warps(INV), NT = 32 * NW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bars[NW][2];
    __shared__ __align__(16) C s_tab[kXwTabCta];

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int wid = tid >> 5;
    const int w = lane & 7;
    const int h = (lane >> 3) & 1;
    const int rr = lane >> 4;
    const int idx = 2 * w + h;
    // the thread that holds the residue 16 - idx (mod 16) of the same row: idx = 0 and idx = 8 are their own partners
    const int plane = ((8 - w - h) & 7) + 8 * h + 16 * rr;

    for (int i = tid; i < kXwTabCta / 2; i += NT)
        reinterpret_cast<float4*>(s_tab)[i] = reinterpret_cast<const float4*>(g_tab_xw)[i + (i < 128 ? (INV ? 128 : 0) : 128)];
    if (lane == 0) {
        mbar_init(&bars[wid][0], 1);
        mbar_init(&bars[wid][1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // [q * 16]: forward w256^((2 q + h) w), backward w256^(q (2 w + h))
    const C* t128 = s_tab + h * 8 + w;
    __syncthreads();
    C tsp[8];                                     // w512^(idx + 16 m): the same in every iteration
#pragma unroll
    for (int m = 0; m < 8; ++m) tsp[m] = s_tab[256 + idx + 16 * m];

    unsigned char* wbase = smem_raw + (size_t)wid * (INV ? kXwWarpBytesInv : kXwWarpBytesFwd);
    // forward: rin[2][2][kXwInPitch] | xch;   backward: sp[2][kXSpPitch] | xch
    float* rbuf = reinterpret_cast<float*>(wbase);
    C* sp = reinterpret_cast<C*>(wbase);
    C* xch = reinterpret_cast<C*>(wbase + (INV ? kXwSpecBytes : 2 * kXwRealBytes));
    C* xw = xch + (rr * 2 + h) * kXwGP + w;              // slot (q, w) at q * kXwQP
    const C* xr = xch + (rr * 2 + h) * kXwGP + w * kXwQP; // slots (w, o') and (w + 8, o')
    const C* srow = sp + rr * kXSpPitch;

    const long long npairs = p.nrows / 2;
    const long long gw = (long long)blockIdx.x * NW + wid;
    const long long nw = (long long)gridDim.x * NW;
    const int nit = gw < npairs ? (int)((npairs - gw + nw - 1) / nw) : 0;
    auto first_row = [&](int i) -> long long {
        const long long pr = gw + (long long)i * nw;
        return 2 * (p.reverse ? npairs - 1 - pr : pr);
    };
    // lane 0 starts the two row copies of iteration i (forward: into input buffer i & 1)
    auto issue = [&](int i) {
        if (lane != 0 || i >= nit) return;
        const long long row = first_row(i);
        if (INV) {
            mbar_expect_tx(&bars[wid][0], (uint32_t)kXwSpecBytes);
            bulk_g2s(sp, p.spec + row * p.spec_pitch, kXSpPitch * (uint32_t)sizeof(C), &bars[wid][0]);
            bulk_g2s(sp + kXSpPitch, p.spec + (row + 1) * p.spec_pitch, kXSpPitch * (uint32_t)sizeof(C), &bars[wid][0]);
        } else {
            float* dst = rbuf + (i & 1) * 2 * kXwInPitch;
            mbar_expect_tx(&bars[wid][i & 1], 2 * kXN * (uint32_t)sizeof(float));
            bulk_g2s(dst, p.real_in + row * kXN, kXN * (uint32_t)sizeof(float), &bars[wid][i & 1]);
            bulk_g2s(dst + kXwInPitch, p.real_in + (row + 1) * kXN, kXN * (uint32_t)sizeof(float), &bars[wid][i & 1]);
        }
    };
    // S5: X[256] of this thread's row of iteration i from the side array [y][z], for the owner of the pair (0, 256)
    auto load_nyq = [&](int i) -> C {
        if (!INV || !p.nyq || idx != 0 || i >= nit) return make_float2(0.f, 0.f);
        const int row = (int)first_row(i) + rr;
        return __ldg(p.nyq + (row % p.n1) * p.n2 + row / p.n1);
    };

    C xnyq_next = load_nyq(0);
    issue(0);
    if (!INV) issue(1);
    for (int i = 0; i < nit; ++i) {
        const long long row = first_row(i) + rr;
        C v[16];
        if constexpr (!INV) {
            // ---------------------------------------------------------------- S1
            mbar_wait(&bars[wid][i & 1], (i >> 1) & 1);
            const C* zin = reinterpret_cast<const C*>(rbuf + ((i & 1) * 2 + rr) * kXwInPitch) + w;
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = zin[8 * r];
            // h = 1: z w256^n, n = w + 8 r: the factor w32^r here, w256^w with the twiddles after the radix-16
            if (h) {
                v[1] = mul_w32<1, false>(v[1]);   v[2] = mul_w32<2, false>(v[2]);   v[3] = mul_w32<3, false>(v[3]);
                v[4] = mul_w32<4, false>(v[4]);   v[5] = mul_w32<5, false>(v[5]);   v[6] = mul_w32<6, false>(v[6]);
                v[7] = mul_w32<7, false>(v[7]);   v[8] = mul_w32<8, false>(v[8]);   v[9] = mul_w32<9, false>(v[9]);
                v[10] = mul_w32<10, false>(v[10]); v[11] = mul_w32<11, false>(v[11]); v[12] = mul_w32<12, false>(v[12]);
                v[13] = mul_w32<13, false>(v[13]); v[14] = mul_w32<14, false>(v[14]); v[15] = mul_w32<15, false>(v[15]);
            }
            fftw128_a<false>(v, t128, xw);
            __syncwarp();
            issue(i + 2);                         // this input buffer is in registers in every lane
            C a[8], b[8];
            fftw128_b<false>(a, b, xr);
            // this thread now holds Z[idx + 16 j]: j = 2 k2 in a[brev3(k2)], j = 2 k2 + 1 in b[brev3(k2)].
            // The real-transform split pairs k = idx + 16 m, m < 8, with 256 - k = (16 - idx) + 16 (15 - m): the
            // upper half j >= 8 of the partner thread, which arrives by shuffle (idx = 0: 256 - 16 m is its own)
            C* orow = p.spec + row * p.spec_pitch;
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int js = 15 - m, jo = (16 - m) & 15;
                const C snd = (js & 1) ? b[brev3(js >> 1)] : a[brev3(js >> 1)];
                const C own = (jo & 1) ? b[brev3(jo >> 1)] : a[brev3(jo >> 1)];
                C zm;
                zm.x = __shfl_sync(0xffffffffu, snd.x, plane);
                zm.y = __shfl_sync(0xffffffffu, snd.y, plane);
                if (idx == 0) zm = own;
                const C zk = (m & 1) ? b[brev3(m >> 1)] : a[brev3(m >> 1)];
                const C e = cadd(zk, make_float2(zm.x, -zm.y));
                const C d = csub(zk, make_float2(zm.x, -zm.y));
                const C wd = cmul(d, tsp[m]);   // w512^k d
                // X[k] = (e - i wd) / 2,  X[256 - k] = (conj e - i conj wd) / 2
                const int k = idx + 16 * m;
                const C xhi = cscale(make_float2(e.x - wd.y, -e.y - wd.x), 0.5f);
                orow[k] = cscale(cadd(e, make_float2(wd.y, -wd.x)), 0.5f);
                orow[kXN - k] = xhi;
                if (m == 0 && idx == 0) {
                    // the Nyquist coefficient X[256] of row (z, y) also goes to the side array [y][z] that the
                    // strided passes read it from in 128-byte runs; pad column 257 leaves as zero
                    orow[kXN + 1] = make_float2(0.f, 0.f);
                    if (p.nyq) p.nyq[((int)row % p.n1) * p.n2 + (int)row / p.n1] = xhi;
                }
            }
            if (idx == 0) orow[kXN / 2] = make_float2(a[brev3(4)].x, -a[brev3(4)].y);   // k = 128 pairs with itself: conj Z[128]
        } else {
            // ---------------------------------------------------------------- S5
            const C xnyq = xnyq_next;
            mbar_wait(&bars[wid][0], i & 1);
            // merge: Z[k] = e + i conj(w512^k) d, Z[256 - k] = conj e + i conj(conj(w512^k) d) for the pairs
            // k = idx + 16 m, m < 8.  Z[k] is this thread's v[m]; Z[256 - k] is v[15 - m] of the partner thread
            C zhi[8];
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int k = idx + 16 * m;
                const C xk = srow[k];
                C xm = srow[kXN - k];
                if (m == 0 && idx == 0 && p.nyq) xm = xnyq;
                const C e = cadd(xk, make_float2(xm.x, -xm.y));
                const C d = csub(xk, make_float2(xm.x, -xm.y));
                const C wd = cmulc(d, tsp[m]);   // conj(w512^k) d
                v[m] = cadd(e, make_float2(-wd.y, wd.x));
                zhi[m] = make_float2(e.x + wd.y, wd.x - e.y);
            }
            const C x128 = srow[kXN / 2];
#pragma unroll
            for (int j = 8; j < 16; ++j) {
                C r;
                r.x = __shfl_sync(0xffffffffu, zhi[15 - j].x, plane);
                r.y = __shfl_sync(0xffffffffu, zhi[15 - j].y, plane);
                // idx = 0: 256 - 16 m = 16 (16 - m) is its own; Z[128] = 2 conj X[128]
                if (idx == 0) r = (j == 8) ? make_float2(2.f * x128.x, -2.f * x128.y) : zhi[(16 - j) & 7];
                v[j] = r;
            }
            fftw128_a<true>(v, t128, xw);   // v[j] = Z[2 k' + h], k' = w + 8 j
            __syncwarp();
            issue(i + 1);                         // the staged rows are in registers in every lane
            xnyq_next = load_nyq(i + 1);
            C a[8], b[8];
            fftw128_b<true>(a, b, xr);
            // z[n] = z0[n] + conj(w256^n) z1[n], n = q + 16 k2, q = w (a) / w + 8 (b): h = 0 holds z0, h = 1 holds
            // z1 conj(w256^q) (the factor came with the twiddles), conj(w16^k2) is applied here; h = 0 finishes the
            // a set, h = 1 the b set
            if (h) {
                a[brev3(1)] = mul_w16<1, true>(a[brev3(1)]); b[brev3(1)] = mul_w16<1, true>(b[brev3(1)]);
                a[brev3(2)] = mul_w16<2, true>(a[brev3(2)]); b[brev3(2)] = mul_w16<2, true>(b[brev3(2)]);
                a[brev3(3)] = mul_w16<3, true>(a[brev3(3)]); b[brev3(3)] = mul_w16<3, true>(b[brev3(3)]);
                a[brev3(4)] = mul_w16<4, true>(a[brev3(4)]); b[brev3(4)] = mul_w16<4, true>(b[brev3(4)]);
                a[brev3(5)] = mul_w16<5, true>(a[brev3(5)]); b[brev3(5)] = mul_w16<5, true>(b[brev3(5)]);
                a[brev3(6)] = mul_w16<6, true>(a[brev3(6)]); b[brev3(6)] = mul_w16<6, true>(b[brev3(6)]);
                a[brev3(7)] = mul_w16<7, true>(a[brev3(7)]); b[brev3(7)] = mul_w16<7, true>(b[brev3(7)]);
            }
            C* orow = reinterpret_cast<C*>(p.real_out + row * kXN);
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                const C ta = a[brev3(k2)], tb = b[brev3(k2)];
                const C send = h ? ta : tb;
                const C keep = h ? tb : ta;
                C recv;
                recv.x = __shfl_xor_sync(0xffffffffu, send.x, 8);
                recv.y = __shfl_xor_sync(0xffffffffu, send.y, 8);
                orow[w + 8 * h + 16 * k2] = cadd(keep, recv);   // (x[2n], x[2n+1])
            }
        }
    }
}


// ==================================================================================== periodic rows of 256 reals
// S1 (real-to-complex) / S5 (complex-to-real) of periodic plans (PAPER.md:87 half spectrum), same scheme: the row is
// packed as z[n] = x[2n] + i x[2n+1], n < 128, Z = DFT128(z) by eight threads (lane = w + 8 rq, four rows per warp),
//     X[k] = ((Z[k] + conj Z[128-k]) - i w256^k (Z[k] - conj Z[128-k])) / 2,   k = 0..128.
// Thread w ends with Z[w + 8 j], j < 16; the partner 128 - k of k = w + 8 m, m < 8, is j' = 15 - m of thread 8 - w.
// X[0..127] go to the spectrum array, X[128] to the side array [row].
constexpr size_t kXpwRowBytes = (size_t)kXwInPitch * sizeof(float);   // 1088 B = 64 (mod 128): 256 reals or 128 complex
constexpr size_t kXpwWarpBytesFwd = 2 * 4 * kXpwRowBytes + kXwXchBytes;
constexpr size_t kXpwWarpBytesInv = 4 * kXpwRowBytes + kXwXchBytes;
constexpr size_t kXpwSmemFwd = kXwWarps * kXpwWarpBytesFwd;
constexpr size_t kXpwSmemInv = kXwWarps * kXpwWarpBytesInv;

template <bool INV> __device__ __forceinline__ void fftp128_a(C (&v)[16], const C* t128, C* xw)
{
    dft16<INV>(v);
#pragma unroll
    for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul_sel<INV>(v[brev4(q)], t128[q * 8]);   // w128^(q w)
#pragma unroll
    for (int q = 0; q < 16; ++q) xw[q * kXwQP] = v[brev4(q)];
}

template <bool INV> __global__ void __launch_bounds__(kXwThreads, 2) fast_xpw_kernel(const FastXPerParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bars[kXwWarps][2];
    __shared__ __align__(16) C s_t128[128];   // [q][w] = w128^(q w)

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int wid = tid >> 5;
    const int w = lane & 7;
    const int rq = lane >> 3;
    const int plane = ((8 - w) & 7) + 8 * rq;   // holds the residue 8 - w of the same row; 0 and 4 pair with themselves

    if (tid < 128) s_t128[tid] = c_tw1024[(8 * (tid >> 3) * (tid & 7)) & 1023];
    if (lane == 0) {
        mbar_init(&bars[wid][0], 1);
        mbar_init(&bars[wid][1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const C* t128 = s_t128 + w;   // [q * 8]
    C tsp[8];                     // w256^(w + 8 m): the same in every iteration
#pragma unroll
    for (int m = 0; m < 8; ++m) tsp[m] = c_tw1024[4 * (w + 8 * m)];
    __syncthreads();

    unsigned char* wbase = smem_raw + (size_t)wid * (INV ? kXpwWarpBytesInv : kXpwWarpBytesFwd);
    C* xch = reinterpret_cast<C*>(wbase + (INV ? 4 : 8) * kXpwRowBytes);
    C* xw = xch + rq * kXwGP + w;               // slot (q, w) at q * kXwQP
    const C* xr = xch + rq * kXwGP + w * kXwQP; // slots (w, o') and (w + 8, o')

    const long long nquads = p.nrows / 4;
    const long long gw = (long long)blockIdx.x * kXwWarps + wid;
    const long long nw = (long long)gridDim.x * kXwWarps;
    const int nit = gw < nquads ? (int)((nquads - gw + nw - 1) / nw) : 0;
    auto first_row = [&](int i) -> long long { return 4 * (gw + (long long)i * nw); };
    // lane 0 starts the four row copies of iteration i (forward: into input buffer i & 1)
    auto issue = [&](int i) {
        if (lane != 0 || i >= nit) return;
        const long long row = first_row(i);
        uint64_t* bar = &bars[wid][INV ? 0 : (i & 1)];
        unsigned char* dst = wbase + (INV ? 0 : (i & 1)) * 4 * kXpwRowBytes;
        mbar_expect_tx(bar, 4 * 1024u);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            if (INV) bulk_g2s(dst + r * kXpwRowBytes, p.spec + (row + r) * p.spec_pitch, 1024u, bar);
            else bulk_g2s(dst + r * kXpwRowBytes, p.real_in + (row + r) * kXN, 1024u, bar);
        }
    };
    // S5: X[128] of this thread's row of iteration i from the side array, for the owner of the pair (0, 128)
    auto load_nyq = [&](int i) -> C {
        if (!INV || w != 0 || i >= nit) return make_float2(0.f, 0.f);
        return __ldg(p.nyq + first_row(i) + rq);
    };

    C xnyq_next = load_nyq(0);
    issue(0);
    if (!INV) issue(1);
    for (int i = 0; i < nit; ++i) {
        const long long row = first_row(i) + rq;
        C v[16];
        if constexpr (!INV) {
            // ---------------------------------------------------------------- S1
            mbar_wait(&bars[wid][i & 1], (i >> 1) & 1);
            const C* zin = reinterpret_cast<const C*>(wbase + ((i & 1) * 4 + rq) * kXpwRowBytes) + w;
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = zin[8 * r];
            fftp128_a<false>(v, t128, xw);
            __syncwarp();
            issue(i + 2);                         // this input buffer is in registers in every lane
            C a[8], b[8];
            fftw128_b<false>(a, b, xr);
            // Z[w + 8 j]: j = 2 k2 in a[brev3(k2)], j = 2 k2 + 1 in b[brev3(k2)]
            C* orow = p.spec + row * p.spec_pitch;
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int js = 15 - m, jo = (16 - m) & 15;
                const C snd = (js & 1) ? b[brev3(js >> 1)] : a[brev3(js >> 1)];
                const C own = (jo & 1) ? b[brev3(jo >> 1)] : a[brev3(jo >> 1)];
                C zm;
                zm.x = __shfl_sync(0xffffffffu, snd.x, plane);
                zm.y = __shfl_sync(0xffffffffu, snd.y, plane);
                if (w == 0) zm = own;
                const C zk = (m & 1) ? b[brev3(m >> 1)] : a[brev3(m >> 1)];
                const C e = cadd(zk, make_float2(zm.x, -zm.y));
                const C d = csub(zk, make_float2(zm.x, -zm.y));
                const C wd = cmul(d, tsp[m]);   // w256^k d
                const int k = w + 8 * m;
                const C xhi = cscale(make_float2(e.x - wd.y, -e.y - wd.x), 0.5f);
                orow[k] = cscale(cadd(e, make_float2(wd.y, -wd.x)), 0.5f);
                if (m == 0) {
                    if (w == 0) p.nyq[row] = xhi;
                    else orow[128 - k] = xhi;
                } else {
                    orow[128 - k] = xhi;
                }
            }
            if (w == 0) orow[64] = make_float2(a[brev3(4)].x, -a[brev3(4)].y);   // k = 64 pairs with itself: conj Z[64]
        } else {
            // ---------------------------------------------------------------- S5
            const C xnyq = xnyq_next;
            mbar_wait(&bars[wid][0], i & 1);
            const C* srow = reinterpret_cast<const C*>(wbase + rq * kXpwRowBytes);
            C zhi[8];
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int k = w + 8 * m;
                const C xk = srow[k];
                C xm = srow[(128 - k) & 127];
                if (m == 0 && w == 0) xm = xnyq;
                const C e = cadd(xk, make_float2(xm.x, -xm.y));
                const C d = csub(xk, make_float2(xm.x, -xm.y));
                const C wd = cmulc(d, tsp[m]);   // conj(w256^k) d
                v[m] = cadd(e, make_float2(-wd.y, wd.x));
                zhi[m] = make_float2(e.x + wd.y, wd.x - e.y);
            }
            const C x64 = srow[64];
#pragma unroll
            for (int j = 8; j < 16; ++j) {
                C r;
                r.x = __shfl_sync(0xffffffffu, zhi[15 - j].x, plane);
                r.y = __shfl_sync(0xffffffffu, zhi[15 - j].y, plane);
                // w = 0: 128 - 8 m = 8 (16 - m) is its own; Z[64] = 2 conj X[64]
                if (w == 0) r = (j == 8) ? make_float2(2.f * x64.x, -2.f * x64.y) : zhi[(16 - j) & 7];
                v[j] = r;
            }
            fftp128_a<true>(v, t128, xw);   // v[j] = Z[w + 8 j]
            __syncwarp();
            issue(i + 1);                         // the staged rows are in registers in every lane
            xnyq_next = load_nyq(i + 1);
            C a[8], b[8];
            fftw128_b<true>(a, b, xr);
            C* orow = reinterpret_cast<C*>(p.real_out + row * kXN);
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                orow[w + 16 * k2] = a[brev3(k2)];        // (x[2n], x[2n+1]), n = w + 16 k2
                orow[w + 8 + 16 * k2] = b[brev3(k2)];
            }
        }
    }
}

} // namespace sf2
