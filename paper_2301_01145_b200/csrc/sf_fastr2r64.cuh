// sf_fastr2r64.cuh -- kernel generation 2 for the strided passes S2 / S3 / S4 of Dirichlet and Neumann plans in double
// precision with 255- / 256-long y and z pencils (Table 1: DST-I on the cell-boundary grid, DCT-II
// forward / DCT-III backward on the cell-centre grid; BASELINE.json configs[2]).
//
// The work arrays of these plans are REAL.  Two neighbouring real columns are read as one complex column z = a + i b
// (the transforms are linear with real coefficients, so the real and imaginary parts stay the two columns), and the
// sine / cosine transform of a pencil is taken as the 512-point FFT F of its odd / even extension x~:
//     DST-I :  x~ = (0, z_0 .. z_254, 0, -z_254 .. -z_0),   Y_k = i F[k+1]               (= 2 sum_j z_j sin(pi (j+1)(k+1)/256))
//     DCT-II:  x~ = (z_0 .. z_255, z_255 .. z_0),           Y_k = e^{-i pi k / 512} F[k] (= 2 sum_j z_j cos(pi (j+1/2) k/256))
// F is computed as in sf_fast64.cuh: even outputs = FFT256(x~[n] + x~[n+256]), odd outputs = FFT256((x~[n] -
// x~[n+256]) w512^n), the two halves side by side in the two quarter-warps of a half-warp, a thread holding the 16
// elements n = o + 16 r.  With the extension written out, x~[n] +- x~[n+256] = z[n-1] -+ z[255-n] (DST-I) or
// z[n] +- z[255-n] (DCT-II): two reads of the staged tile per element instead of one, nothing else.
// The fused pass needs no sine / cosine bookkeeping at all: the backward transform is the inverse FFT of the same
// symmetric spectrum, so it is   extension -> FFT512 -> F[k] *= scale / (lambda_x + lambda_y + lambda_z[fold(k)])
// -> inverse FFT512 truncated to the stored rows   with fold(k) = min(k, 512 - k): the structure of the padded
// fused kernel with the multiplier computed on the fly (one reciprocal per real column and spectral row: fast_rcp of sf_fast64.cuh).  The two
// real columns have different multipliers and are separated in Y, not in F, so F is rotated to Y around the multiply
// (a swap of the two factors for DST-I, two complex multiplications by w1024^k for DCT).
// Tiles of 8 complex = 16 real columns (128-byte rows) arrive by TMA; 256 threads, two CTAs per SM.
#pragma once
#include "sf_fast64.cuh"

namespace sf2 {

enum { R2RK_DST1 = 0, R2RK_DCT = 1 };
enum { RMODE_FWD = 0, RMODE_INV = 1, RMODE_FUSED = 2 };   // FWD: x -> Y;  INV: Y -> x (DCT-III; DST-I uses FWD);  FUSED: S3

constexpr size_t kSmemR64 = ((size_t)kXchg64Elems + kSlot64Elems) * sizeof(D);

template <int KIND, int MODE>
__global__ void __launch_bounds__(kT64, 2) fast_r2r64_kernel(const FastR64Params p, const __grid_constant__ CUtensorMap tm)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    D* xbuf = reinterpret_cast<D*>(smem_raw);
    D* slot = xbuf + kXchg64Elems;                 // [row][8 complex columns]
    __shared__ __align__(8) uint64_t bar;
    __shared__ __align__(16) D s_t256[256];        // [o][q] = w256^(q o)
    __shared__ __align__(16) D s_t512[256];        // [o][r] = w512^(o + 16 r)
    __shared__ __align__(16) D s_t1024[(KIND == R2RK_DCT && MODE != RMODE_FUSED) ? 256 : 1];   // w1024^k, k < 256
    __shared__ double s_lamp[MODE == RMODE_FUSED ? 256 : 1];   // eigenvalue contribution of the pencil axis
    __shared__ int s_tile[2];

    const int tid = threadIdx.x;
    const int l16 = tid & 15;
    const int pen = l16 & 7;
    const int h = l16 >> 3;
    const int o = tid >> 4;
    const int ea = o * 16 + l16;
    const int eb = o * 256 + l16;
    const D* t256 = s_t256 + o * 16;
    const D* t512 = s_t512 + o * 16;
    const int n = p.n;                             // stored rows per pencil: 255 (DST-I) or 256 (DCT)
    const int ntiles = p.nb * p.nct;
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;
    uint32_t parity = 0;

    auto issue = [&](int t) {
        if (tid != 0 || t >= ntiles) return;
        const int b = t / p.nct, ct = t - b * p.nct;
        mbar_expect_tx(&bar, (uint32_t)n * kTile64 * (uint32_t)sizeof(D));
        if (p.batch_dim == 2) tma_load_4d(slot, &tm, 16 * ct, 0, b, 0, &bar);   // (column, row, batch)
        else tma_load_4d(slot, &tm, 16 * ct, b, 0, 0, &bar);                   // (column, batch, row)
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
    s_t256[tid] = c_tw1024d[(4 * (tid & 15) * (tid >> 4)) & 1023];
    s_t512[tid] = c_tw1024d[2 * ((tid >> 4) + 16 * (tid & 15))];
    if (KIND == R2RK_DCT && MODE != RMODE_FUSED) s_t1024[tid] = c_tw1024d[tid];
    if (MODE == RMODE_FUSED) s_lamp[tid] = (tid < n) ? __ldg(p.lam_p + tid) : 0.0;
    __syncthreads();

    // x~[nn] +- x~[nn + 256] of this thread's column from the staged tile, times w512^nn for the odd half
    auto load_sym = [&](D (&v)[16]) {
        mbar_wait(&bar, parity);
        parity ^= 1;
        // DST-I: h = 0 takes z[nn-1] - z[255-nn], h = 1 the sum;  DCT: h = 0 the sum z[nn] + z[255-nn], h = 1 the difference
        const double sg = ((KIND == R2RK_DST1) == (h == 1)) ? 1.0 : -1.0;
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int nn = o + 16 * r;
            D a, b;
            if (KIND == R2RK_DST1) {
                if (nn == 0) { a = make_double2(0.0, 0.0); b = a; }
                else { a = slot[(nn - 1) * kTile64 + pen]; b = slot[(255 - nn) * kTile64 + pen]; }
            } else {
                a = slot[nn * kTile64 + pen];
                b = slot[(255 - nn) * kTile64 + pen];
            }
            const D s = make_double2(fma(sg, b.x, a.x), fma(sg, b.y, a.y));
            v[r] = h ? cmul(s, t512[r]) : s;
        }
    };
    // truncated inverse of the 512-point spectrum held as two halves: x~[j] = e_j + conj(w512^j) o_j, j = o + 16 r;
    // h = 0 ends with j = o + 16 r, h = 1 with j = o + 128 + 16 r (r < 8); stored at row j - shift
    auto combine_store = [&](D (&v)[16], D* outp, bool valid) {
        constexpr int shift = (KIND == R2RK_DST1) ? 1 : 0;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const D a = v[brev4(r)], b = v[brev4(r + 8)];
            const D tl = h ? cmulc(a, t512[r]) : a, th = h ? cmulc(b, t512[r + 8]) : b;
            const D send = h ? tl : th;
            const D keep = h ? th : tl;
            D recv;
            recv.x = __shfl_xor_sync(0xffffffffu, send.x, 8);
            recv.y = __shfl_xor_sync(0xffffffffu, send.y, 8);
            const D x = cadd(keep, recv);
            const int j = o + 128 * h + 16 * r - shift;
            if (valid && j >= 0 && j < n) outp[(size_t)j * ops] = x;
        }
    };

    auto tile = [&](int t, int it, auto orient_tag) {
        constexpr bool OB = decltype(orient_tag)::value;
        const int b = t / p.nct, ct = t - b * p.nct;
        const int col = ct * kTile64;                       // first complex column
        D* outp = p.out + ((size_t)b * obs + col + pen);
        D v[16];
        if constexpr (MODE == RMODE_FWD) {
            load_sym(v);
            fft256d_a<false, OB>(v, t256, xbuf, ea, eb);
            __syncthreads();
            advance(it);
            fft256d_b<false, OB>(v, xbuf, ea, eb);
            // F[k], k = 2 (o + 16 k2) + h; the stored spectrum is k <= 255: k2 < 8
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                const int k = 2 * (o + 16 * k2) + h;
                const D f = v[brev4(k2)];
                if (KIND == R2RK_DST1) {
                    if (k >= 1) outp[(size_t)(k - 1) * ops] = cmuli(f);             // Y_{k-1} = i F[k]
                } else {
                    outp[(size_t)k * ops] = cmul(f, s_t1024[k]);                    // Y_k = e^{-i pi k / 512} F[k]
                }
            }
        } else if constexpr (MODE == RMODE_INV) {
            // DCT-III: F[k] = e^{+i pi k / 512} Y[k] (k < 256), 0 (k = 256), e^{-i pi (512-k) / 512} Y[512-k] (k > 256)
            mbar_wait(&bar, parity);
            parity ^= 1;
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) {
                const int k = 2 * (o + 16 * k2) + h;
                if (k < 256) v[k2] = cmulc(slot[k * kTile64 + pen], s_t1024[k]);
                else if (k == 256) v[k2] = make_double2(0.0, 0.0);
                else v[k2] = cmul(slot[(512 - k) * kTile64 + pen], s_t1024[512 - k]);
            }
            fft256d_a<true, OB>(v, t256, xbuf, ea, eb);
            __syncthreads();
            advance(it);
            fft256d_b<true, OB>(v, xbuf, ea, eb);
            combine_store(v, outp, true);
        } else {
            load_sym(v);
            fft256d_a<false, OB>(v, t256, xbuf, ea, eb);
            __syncthreads();
            advance(it);
            // multiplier of the two real columns of this complex column, per spectral row (requested before the second half)
            const int cx = 2 * (col + pen);
            const double lxa = __ldg(p.lam_x + min(cx, p.nx - 1)) + __ldg(p.lam_b + b);
            const double lxb = __ldg(p.lam_x + min(cx + 1, p.nx - 1)) + __ldg(p.lam_b + b);
            fft256d_b<false, OB>(v, xbuf, ea, eb);
            D u[16];
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) {
                const int k = 2 * (o + 16 * k2) + h;
                const int f = (k <= 256) ? k : 512 - k;                       // fold: the multiplier is even in k
                const int li = (KIND == R2RK_DST1) ? f - 1 : f;               // index of the stored spectral row
                double ma = 0.0, mb = 0.0;
                if (li >= 0 && li < n) {
                    const double lp = s_lamp[li];
                    ma = p.scale * fast_rcp(lxa + lp);
                    mb = p.scale * fast_rcp(lxb + lp);
                    if (p.zero_mode && li == 0 && b == 0) {                   // the all-zero index
                        if (cx == 0) ma = 0.0;
                        if (cx + 1 == 0) mb = 0.0;
                    }
                }
                // The two real columns are separated in Y = rot F, not in F itself: rot = i (DST-I: F = -i (Ya + i Yb))
                // or e^{-i pi k / 512} = w1024^k (DCT) for every k < 512.  Y' = (Ya ma, Yb mb), F' = conj(rot) Y'.
                const D f0 = v[brev4(k2)];
                if (KIND == R2RK_DST1) {
                    u[k2] = make_double2(f0.x * mb, f0.y * ma);       // i, then -i: the parts swap their multipliers
                } else {
                    D rot = t512[k2];                                 // w512^(o + 16 k2) = w1024^(k - h)
                    if (h) rot = cmul(rot, c_tw1024d[1]);
                    const D y = cmul(f0, rot);
                    u[k2] = cmulc(make_double2(y.x * ma, y.y * mb), rot);
                }
            }
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) v[k2] = u[k2];
            fft256d_a<true, !OB>(v, t256, xbuf, ea, eb);
            __syncthreads();
            fft256d_b<true, !OB>(v, xbuf, ea, eb);
            combine_store(v, outp, true);
        }
    };

    if constexpr (MODE == RMODE_FUSED) {
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

} // namespace sf2
