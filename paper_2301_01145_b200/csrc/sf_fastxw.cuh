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
//   then the real-transform split X[k] = ((Z[k] + conj Z[256-k]) - i w512^k (Z[k] - conj Z[256-k])) / 2 in the
//   staged row, which leaves by one bulk store.  backward: the mirror.
//   128-point transform: radix-16 over r (n = w + 8 r), twiddle w128^(q w), one exchange between the eight
//   threads of the group, two radix-8 over o' for q = w and q = w + 8.
// Shared-memory words are 8 bytes (one complex); every access of a half-warp (one row, 8 residues x 2 halves) is
// either 16 consecutive words or 8 words with stride 9 plus the same 8 shifted by 8 (mod 16): no bank conflicts.
#pragma once
#include "sf_fast.cuh"

namespace sf2 {

constexpr int kXwWarps = 8;
constexpr int kXwThreads = 32 * kXwWarps;
constexpr int kXwInPitch = kXN + 16;          // floats per staged real row: 1088 B = 64 (mod 128)
constexpr int kXwQP = 9;                      // exchange: words per q
constexpr int kXwGP = 152;                    // exchange: words per (row, half) group, 8 (mod 16)
constexpr int kXwTab = 528;                   // tw128[q][w] | twin[j][h][w] | twsp[m][2 w + h]
constexpr size_t kXwRealBytes = 2 * (size_t)kXwInPitch * sizeof(float);   // a pair of real rows
constexpr size_t kXwSpecBytes = 2 * (size_t)kXSpPitch * sizeof(C);        // a pair of spectrum rows
constexpr size_t kXwXchBytes = 4 * (size_t)kXwGP * sizeof(C);
// forward: two input pairs (prefetch distance two), exchange, one output pair;  backward: one of each
constexpr size_t kXwWarpBytesFwd = 2 * kXwRealBytes + kXwXchBytes + kXwSpecBytes;
constexpr size_t kXwWarpBytesInv = kXwSpecBytes + kXwXchBytes + kXwRealBytes;
constexpr size_t kXwSmemFwd = kXwWarps * kXwWarpBytesFwd;
constexpr size_t kXwSmemInv = kXwWarps * kXwWarpBytesInv;

__device__ float2 g_tab_xw[kXwTab];

// v[r] = a[w + 8 r] in; writes the twiddled radix-16 outputs into the group's exchange slots (q, w)
template <bool INV> __device__ __forceinline__ void fftw128_a(C (&v)[16], const C* t128, C* xw)
{
    dft16<INV>(v);
#pragma unroll
    for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul_sel<INV>(v[brev4(q)], t128[q * 8]);   // w128^(q w)
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

template <bool INV> __global__ void __launch_bounds__(kXwThreads, 2) fast_xw_kernel(const FastXParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bars[kXwWarps][2];
    __shared__ __align__(16) C s_tab[kXwTab];

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int wid = tid >> 5;
    const int w = lane & 7;
    const int h = (lane >> 3) & 1;
    const int rr = lane >> 4;
    const int idx = 2 * w + h;

    for (int i = tid; i < kXwTab / 2; i += kXwThreads) reinterpret_cast<float4*>(s_tab)[i] = reinterpret_cast<const float4*>(g_tab_xw)[i];
    if (lane == 0) {
        mbar_init(&bars[wid][0], 1);
        mbar_init(&bars[wid][1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const C* t128 = s_tab + w;                    // [q * 8]
    const C* tin = s_tab + 128 + h * 8 + w;       // [j * 16]: w256^(w + 8 j) for h = 1, 1 for h = 0
    const C* tsp = s_tab + 384 + idx;             // [m * 16]: w512^(idx + 16 m)

    unsigned char* wbase = smem_raw + (size_t)wid * (INV ? kXwWarpBytesInv : kXwWarpBytesFwd);
    // forward: rin[2][2][kXwInPitch] | xch | sp[2][kXSpPitch];   backward: sp | xch | rout[2][kXwInPitch]
    float* rbuf = reinterpret_cast<float*>(INV ? wbase + kXwSpecBytes + kXwXchBytes : wbase);
    C* xch = reinterpret_cast<C*>(wbase + (INV ? kXwSpecBytes : 2 * kXwRealBytes));
    C* sp = reinterpret_cast<C*>(INV ? wbase : wbase + 2 * kXwRealBytes + kXwXchBytes);
    C* xw = xch + (rr * 2 + h) * kXwGP + w;              // slot (q, w) at q * kXwQP
    const C* xr = xch + (rr * 2 + h) * kXwGP + w * kXwQP; // slots (w, o') and (w + 8, o')
    C* srow = sp + rr * kXSpPitch;
    if (!INV && idx == 0) srow[kXN + 1] = make_float2(0.f, 0.f);   // pad column 257 leaves as zero
    __syncthreads();

    const long long npairs = p.nrows / 2;
    const long long gw = (long long)blockIdx.x * kXwWarps + wid;
    const long long nw = (long long)gridDim.x * kXwWarps;
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
        const long long row0 = first_row(i);
        C v[16];
        if constexpr (!INV) {
            // ---------------------------------------------------------------- S1
            mbar_wait(&bars[wid][i & 1], (i >> 1) & 1);
            const C* zin = reinterpret_cast<const C*>(rbuf + ((i & 1) * 2 + rr) * kXwInPitch) + w;
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = cmul(zin[8 * r], tin[16 * r]);   // h = 1: z w256^n
            fftw128_a<false>(v, t128, xw);
            __syncwarp();
            issue(i + 2);                         // this input buffer is in registers in every lane
            C a[8], b[8];
            fftw128_b<false>(a, b, xr);
            if (lane == 0) bulk_wait_read();      // the previous pair's stores have left the staged rows
            __syncwarp();
            // Z[2 k' + h], k' = w + 16 k2 (a) and w + 8 + 16 k2 (b), natural order into the staged row
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                srow[2 * (w + 16 * k2) + h] = a[brev3(k2)];
                srow[2 * (w + 8 + 16 * k2) + h] = b[brev3(k2)];
            }
            __syncwarp();
            // split in place: the 16 threads of a row own the pairs (k, 256 - k), k = idx + 16 m
            C xn = make_float2(0.f, 0.f);
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
                        const C wd = cmul(d, tsp[16 * m]);   // w512^k d
                        // X[k] = (e - i wd) / 2,  X[256 - k] = (conj e - i conj wd) / 2
                        const C xhi = cscale(make_float2(e.x - wd.y, -e.y - wd.x), 0.5f);
                        srow[k] = cscale(cadd(e, make_float2(wd.y, -wd.x)), 0.5f);
                        srow[kXN - k] = xhi;
                        if (m == 0) xn = xhi;
                    }
                }
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                bulk_s2g(p.spec + row0 * p.spec_pitch, sp, kXSpPitch * (uint32_t)sizeof(C));
                bulk_s2g(p.spec + (row0 + 1) * p.spec_pitch, sp + kXSpPitch, kXSpPitch * (uint32_t)sizeof(C));
                bulk_commit();
            }
            // the Nyquist coefficient X[256] of row (z, y) also goes to the side array [y][z] that the strided
            // passes read it from in 128-byte runs
            if (p.nyq && idx == 0) {
                const int row = (int)row0 + rr;
                p.nyq[(row % p.n1) * p.n2 + row / p.n1] = xn;
            }
        } else {
            // ---------------------------------------------------------------- S5
            const C xnyq = xnyq_next;
            mbar_wait(&bars[wid][0], i & 1);
            // merge in place: Z[k] = e + i conj(w512^k) d, Z[256 - k] = conj e + i conj(conj(w512^k) d)
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
                        const C wd = cmulc(d, tsp[16 * m]);   // conj(w512^k) d
                        srow[k] = cadd(e, make_float2(-wd.y, wd.x));
                        if (k > 0) srow[kXN - k] = make_float2(e.x + wd.y, wd.x - e.y);
                    }
                }
            }
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = srow[2 * (w + 8 * j) + h];   // Z[2 k' + h], k' = w + 8 j
            fftw128_a<true>(v, t128, xw);
            fence_async_smem();                   // the merged values in the staged rows are overwritten by the next bulk load
            __syncwarp();
            issue(i + 1);                         // the staged rows are in registers in every lane
            xnyq_next = load_nyq(i + 1);
            C a[8], b[8];
            fftw128_b<true>(a, b, xr);
            if (lane == 0) bulk_wait_read();      // the previous pair's stores have left the real rows
            __syncwarp();
            // z[n] = z0[n] + conj(w256^n) z1[n], n = w + 16 k2 (a) / w + 8 + 16 k2 (b): h = 0 holds z0, h = 1 holds
            // z1; h = 0 finishes the a set, h = 1 the b set
            float* rrow = rbuf + rr * kXwInPitch;
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                // (the table row of h = 0 is all ones)
                const C ta = cmulc(a[brev3(k2)], tin[32 * k2]), tb = cmulc(b[brev3(k2)], tin[32 * k2 + 16]);
                const C send = h ? ta : tb;
                const C keep = h ? tb : ta;
                C recv;
                recv.x = __shfl_xor_sync(0xffffffffu, send.x, 8);
                recv.y = __shfl_xor_sync(0xffffffffu, send.y, 8);
                const C z = cadd(keep, recv);
                const int n = w + 8 * h + 16 * k2;
                *reinterpret_cast<C*>(rrow + 2 * n) = z;   // (x[2n], x[2n+1])
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                bulk_s2g(p.real_out + row0 * kXN, rbuf, kXN * (uint32_t)sizeof(float));
                bulk_s2g(p.real_out + (row0 + 1) * kXN, rbuf + kXwInPitch, kXN * (uint32_t)sizeof(float));
                bulk_commit();
            }
        }
    }
    if (lane == 0) bulk_wait_read();
}

} // namespace sf2
