// sf_fastxw64.cuh -- the X passes S1 / S5 in double precision for rows whose extended real sequence has length 512
// (zero-padded rows of 256; DST-I rows of 255 and DCT-II / DCT-III rows of 256, Table 1 PAPER.md:160-167,
// boundary values folded into the source on load) with one pipeline PER WARP.
//
// fast_xg_kernel (sf_fastx64.cuh) stages rows, exchange and spectrum in the shared memory of a 128-thread CTA: seven
// CTA barriers per tile and every value crosses shared memory five times; ncu shows the shared-memory pipe as the limit
// (l1tex 64 - 72 %, DRAM 20 - 42 %).  Here, as in sf_fastxw.cuh, the 16 threads that transform a row sit in one warp
//     lane = o + 16 rr,   o = residue of the 256-point transform,  rr = row of the pair,
// a warp owns two rows per iteration with its own cp.async-fed input buffers and exchange buffer, and synchronises by
// __syncwarp only.  Shared memory carries the raw rows (extension rules are index arithmetic on them) and the one
// exchange of the 16 x 16 transform.  After the second radix-16 thread o holds Z[o + 16 j]; the partner 256 - k of its
// k sits in thread 16 - o as j' = 15 - j, so the real-transform split (S1) and merge (S5) pair up through shuffles
// and the results go straight to global memory: the 16 lanes of a row write consecutive elements.
#pragma once
#include "sf_fastx64.cuh"

namespace sf2 {

constexpr int kXw64Warps = 6;
constexpr int kXw64Threads = 32 * kXw64Warps;
constexpr int kXw64QP = 17;                                    // exchange: 16-byte words per q (odd: conflict-free reads)
constexpr int kXw64GP = 16 * kXw64QP;                          // exchange: words per row
constexpr size_t kXw64XchBytes = 2 * (size_t)kXw64GP * sizeof(D);
constexpr int kXw64RP = 258;   // doubles per staged real row
template <int MODE, bool INV> constexpr bool xw64_cplx_in() { return INV && MODE == sf::X_ZEROPAD; }
// raw rows: real rows are double-buffered (prefetch distance two), the 4 KB complex rows of the backward zero-padded
// pass single-buffered, so that twelve warps fit an SM in every mode
template <int MODE, bool INV> constexpr int xw64_nbuf() { return xw64_cplx_in<MODE, INV>() ? 1 : 2; }
template <int MODE, bool INV> constexpr size_t xw64_raw_bytes()
{
    return 2 * (xw64_cplx_in<MODE, INV>() ? (size_t)kXgSP * sizeof(D) : (size_t)kXw64RP * sizeof(double));
}
template <int MODE, bool INV> constexpr size_t xw64_warp_bytes() { return xw64_nbuf<MODE, INV>() * xw64_raw_bytes<MODE, INV>() + kXw64XchBytes; }
template <int MODE, bool INV> constexpr size_t xw64_smem() { return kXw64Warps * xw64_warp_bytes<MODE, INV>(); }

__device__ __forceinline__ void cp_async16(void* dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ D shfl_d(D v, int src)
{
    return make_double2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}

template <int MODE, bool INV> __global__ void __launch_bounds__(kXw64Threads, 2) fast_xgw_kernel(const sf::XParams<double> p)
{
    constexpr bool CIN = xw64_cplx_in<MODE, INV>();
    constexpr int NBUF = xw64_nbuf<MODE, INV>();
    constexpr size_t RAW = xw64_raw_bytes<MODE, INV>();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(16) D s_t256[256];   // [q][o] = w256^(q o)
    __shared__ __align__(16) D s_tsp[128];    // [m][o] = w512^(o + 16 m)
    __shared__ __align__(16) D s_ptw[MODE == sf::X_DCT2 ? 128 : 1];   // [m][o] = exp(-i pi (o + 16 m) / 512)

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int wid = tid >> 5;
    const int o = lane & 15;
    const int rr = lane >> 4;
    const int plane = ((16 - o) & 15) + 16 * rr;   // holds the residue 16 - o of the same row; 0 and 8 pair with themselves
    const int comp = blockIdx.y;
    const int n = p.n;
    for (int i = tid; i < 256; i += kXw64Threads) s_t256[i] = c_tw1024d[(4 * (i >> 4) * (i & 15)) & 1023];
    for (int i = tid; i < 128; i += kXw64Threads) s_tsp[i] = c_tw1024d[2 * i];
    if constexpr (MODE == sf::X_DCT2)
        for (int i = tid; i < 128; i += kXw64Threads) s_ptw[i] = ldg_d(reinterpret_cast<const D*>(p.ptw) + i);
    __syncthreads();
    const D* t256 = s_t256 + o;   // [q * 16]
    const D* tsp = s_tsp + o;     // [m * 16]
    const D* tpw = s_ptw + (MODE == sf::X_DCT2 ? o : 0);

    unsigned char* wbase = smem_raw + (size_t)wid * xw64_warp_bytes<MODE, INV>();
    D* xch = reinterpret_cast<D*>(wbase + NBUF * RAW);
    D* xw = xch + rr * kXw64GP + o;                    // slot (q, o) at q * kXw64QP
    const D* xr = xch + rr * kXw64GP + o * kXw64QP;    // slots (o, o')

    const long long nrows = (long long)p.ny * p.nz;
    const long long npairs = (nrows + 1) / 2;
    const long long gw = (long long)blockIdx.x * kXw64Warps + wid;
    const long long nw = (long long)gridDim.x * kXw64Warps;
    const int nit = gw < npairs ? (int)((npairs - gw + nw - 1) / nw) : 0;
    // the rows this pass reads: the source (S1), the real spectrum rows (S5, real-to-real) or the half spectra (S5, padded)
    const double* rsrc = INV ? reinterpret_cast<const double*>(p.spec_in) + comp * p.sp_pc : p.real_in + comp * p.rin_pc;

    // a lane's row of iteration i; past the end (odd row count) the last row is done twice, by both half-warps, with
    // identical stores: no validity tests anywhere
    struct Geom {
        int iy, iz;
    };
    const unsigned last_row = (unsigned)(nrows - 1);
    auto geometry = [&](int i) {
        const long long r = 2 * (gw + (long long)i * nw) + rr;
        const unsigned rc = r < (long long)last_row ? (unsigned)r : last_row;
        Geom g;
        g.iz = (int)(rc / (unsigned)p.ny);
        g.iy = (int)(rc - (unsigned)g.iz * (unsigned)p.ny);
        return g;
    };
    auto rin_of = [&](const Geom& g) { return g.iy * p.rin_py + g.iz * p.rin_pz; };
    auto sp_of = [&](const Geom& g) { return g.iy * p.sp_py + g.iz * p.sp_pz; };
    // the half-warp of a row copies it into buffer i % NBUF, lanes along the row
    auto prefetch = [&](int i, const Geom& g) {
        if (i < nit) {
            unsigned char* buf = wbase + (i % NBUF) * RAW;
            if constexpr (CIN) {
                D* dst = reinterpret_cast<D*>(buf) + rr * kXgSP;
                const D* src = reinterpret_cast<const D*>(p.spec_in) + comp * p.sp_pc + sp_of(g);
#pragma unroll
                for (int t = 0; t < 16; ++t) cp_async16(dst + o + 16 * t, src + o + 16 * t);
                if (o == 0) cp_async16(dst + 256, src + 256);
            } else {
                // 16-byte copies when both rows of the pair start at 0 (mod 16) bytes (the last chunk of an odd row
                // shrinks to the one element inside), 8-byte copies otherwise (dense rows of 255)
                double* dst = reinterpret_cast<double*>(buf) + rr * kXw64RP;
                const double* src = rsrc + (INV ? sp_of(g) : rin_of(g));
                if (__all_sync(0xffffffffu, (reinterpret_cast<unsigned long long>(src) & 15ull) == 0ull)) {
#pragma unroll
                    for (int t = 0; t < 8; ++t) {
                        const int j = 2 * (o + 16 * t);
                        if (t < 7 || j + 2 <= n) cp_async16(dst + j, src + j);
                        else if (j < n) cp_async8(dst + j, src + j);
                    }
                } else {
#pragma unroll
                    for (int t = 0; t < 16; ++t) {
                        const int j = o + 16 * t;
                        if (t < 15 || j < n) cp_async8(dst + j, src + j);
                    }
                }
            }
        }
        cp_async_commit();
    };

    // S1 with boundary values: a row off the y / z faces takes a term at its two ends only, which the lanes o < 2
    // fetch one iteration ahead (rows on a face are rare and fold the whole row when they come up)
    auto on_face = [&](const Geom& g) { return g.iy == 0 || g.iy == p.ny - 1 || g.iz == 0 || g.iz == p.nz - 1; };
    auto end_term = [&](const Geom& g) -> double {
        if (INV || !p.has_faces || o >= 2 || on_face(g)) return 0.0;
        return sf::x_face_term(p, o ? n - 1 : 0, g.iy, g.iz);
    };

    Geom g0 = geometry(0), g1 = geometry(1);
    prefetch(0, g0);
    if (NBUF == 2) prefetch(1, g1);
    double fterm_next = end_term(g0);
    for (int i = 0; i < nit; ++i) {
        const Geom g = g0;
        const Geom gpf = NBUF == 2 ? geometry(i + 2) : g1;   // the rows of the next prefetch
        g0 = g1;
        g1 = NBUF == 2 ? gpf : geometry(i + 2);
        const double fterm = fterm_next;
        fterm_next = end_term(g0);
        cp_async_wait<NBUF - 1>();
        __syncwarp();
        unsigned char* buf = wbase + (i % NBUF) * RAW;
        D v[16];
        if constexpr (!INV) {
            // ---------------------------------------------------------------- S1
            double* prow = reinterpret_cast<double*>(buf) + rr * kXw64RP;
            if (p.has_faces) {
                // boundary values folded into the staged row
                if (on_face(g)) {
                    for (int ix = o; ix < n; ix += 16) prow[ix] += sf::x_face_term(p, ix, g.iy, g.iz);
                } else if (o < 2) {
                    prow[o ? n - 1 : 0] += fterm;
                }
                __syncwarp();
            }
            // packed extended sequence z[nn] = x~[2 nn] + i x~[2 nn + 1], nn = o + 16 r (n = 255 or 256: for r < 8 both
            // positions lie in the stored half of the extension, for r >= 8 in the mirrored / padded half)
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const int nn = o + 16 * r;
                if (r < 8) {
                    if (MODE == sf::X_DST1) v[r] = make_double2(nn == 0 ? 0.0 : prow[max(2 * nn - 1, 0)], prow[2 * nn]);
                    else v[r] = *reinterpret_cast<const D*>(prow + 2 * nn);
                } else {
                    if (MODE == sf::X_ZEROPAD) {
                        v[r] = make_double2(0.0, 0.0);
                    } else {
                        const D t = *reinterpret_cast<const D*>(prow + 510 - 2 * nn);   // (row[510 - 2 nn], row[511 - 2 nn])
                        if (MODE == sf::X_DST1) v[r] = make_double2(nn == 128 ? 0.0 : -t.y, -t.x);
                        else v[r] = make_double2(t.y, t.x);
                    }
                }
            }
            __syncwarp();   // the raw rows are in registers: fetch the rows of two iterations ahead
            prefetch(i + NBUF, gpf);
            dft16<false>(v);
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul(v[brev4(q)], t256[q * 16]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * kXw64QP] = v[brev4(q)];
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = xr[j];
            dft16<false>(v);
            // Z[o + 16 k2] at v[brev4(k2)].  Split X[k] = ((Z[k] + conj Z[256-k]) - i w512^k (Z[k] - conj Z[256-k])) / 2
            // for the pairs k = o + 16 m, m < 8, and 256 - k = (16 - o) + 16 (15 - m) of the partner thread
            D* so = reinterpret_cast<D*>(p.spec_out) + comp * p.sp_pc + sp_of(g);
            double* ro = p.real_out + comp * p.sp_pc + sp_of(g);
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const D zk = v[brev4(m)];
                D zm = shfl_d(v[brev4(15 - m)], plane);
                if (o == 0) zm = v[brev4((16 - m) & 15)];
                const D e = make_double2(zk.x + zm.x, zk.y - zm.y);
                const D d = make_double2(zk.x - zm.x, zk.y + zm.y);
                const D wd = cmul(d, tsp[m * 16]);
                const int k = o + 16 * m;
                {
                    if constexpr (MODE == sf::X_ZEROPAD) {
                        so[k] = make_double2(0.5 * (e.x + wd.y), 0.5 * (e.y - wd.x));
                        so[256 - k] = make_double2(0.5 * (e.x - wd.y), 0.5 * (-e.y - wd.x));
                    } else if constexpr (MODE == sf::X_DST1) {
                        // DST-I: Y_k = -Im X~[k+1]
                        if (k >= 1) {
                            ro[k - 1] = -0.5 * (e.y - wd.x);
                            ro[255 - k] = 0.5 * (e.y + wd.x);
                        }
                    } else {
                        // DCT-II: Y_k = Re(e^{-i pi k / 512} X~[k]);  e^{-i pi (256 - k) / 512} = -i conj(e^{-i pi k / 512})
                        const D pw = tpw[m * 16];
                        ro[k] = 0.5 * (pw.x * (e.x + wd.y) - pw.y * (e.y - wd.x));
                        if (k >= 1) ro[256 - k] = 0.5 * (-pw.y * (e.x - wd.y) + pw.x * (-e.y - wd.x));
                    }
                }
            }
            if (o == 0) {
                // k = 128 pairs with itself: X~[128] = conj Z[128]
                const D z = v[brev4(8)];
                if constexpr (MODE == sf::X_ZEROPAD) so[128] = make_double2(z.x, -z.y);
                else if constexpr (MODE == sf::X_DST1) ro[127] = z.y;
                else ro[128] = 0.70710678118654752440 * (z.x - z.y);
            }
        } else {
            // ---------------------------------------------------------------- S5
            // half spectrum X~[k] of the extended sequence from the raw row, merged pairwise:
            // Z[k] = (X[k] + conj X[256-k]) + i conj(w512^k) (X[k] - conj X[256-k]); Z[k] is this thread's v[m],
            // Z[256 - k] the partner's v[15 - m]
            const D* sr = reinterpret_cast<const D*>(buf) + rr * kXgSP;
            const double* ri = reinterpret_cast<const double*>(buf) + rr * kXw64RP;
            D zhi[8];
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int k = o + 16 * m;
                D xk, xm;
                if constexpr (MODE == sf::X_ZEROPAD) {
                    xk = sr[k];
                    xm = sr[256 - k];
                } else if constexpr (MODE == sf::X_DST1) {
                    // X~[k] = -i Y[k-1], 1 <= k <= 255
                    xk = make_double2(0.0, k >= 1 ? -ri[max(k - 1, 0)] : 0.0);
                    xm = make_double2(0.0, k >= 1 ? -ri[255 - k] : 0.0);
                } else {
                    // X~[k] = e^{+i pi k / 512} Y[k], k <= 255
                    const D pw = tpw[m * 16];
                    const double y = ri[k], ym = k >= 1 ? ri[256 - k] : 0.0;
                    xk = make_double2(pw.x * y, -pw.y * y);
                    xm = make_double2(-pw.y * ym, pw.x * ym);
                }
                const D e = make_double2(xk.x + xm.x, xk.y - xm.y);
                const D d = make_double2(xk.x - xm.x, xk.y + xm.y);
                const D wd = cmulc(d, tsp[m * 16]);
                v[m] = make_double2(e.x - wd.y, e.y + wd.x);
                zhi[m] = make_double2(e.x + wd.y, wd.x - e.y);
            }
            D x128;
            if constexpr (MODE == sf::X_ZEROPAD) x128 = sr[128];
            else if constexpr (MODE == sf::X_DST1) x128 = make_double2(0.0, -ri[127]);
            else x128 = make_double2(0.70710678118654752440 * ri[128], 0.70710678118654752440 * ri[128]);
#pragma unroll
            for (int j = 8; j < 16; ++j) {
                D r = shfl_d(zhi[15 - j], plane);
                // o = 0: 256 - 16 m = 16 (16 - m) is its own; Z[128] = 2 conj X[128]
                if (o == 0) r = (j == 8) ? make_double2(2.0 * x128.x, -2.0 * x128.y) : zhi[(16 - j) & 7];
                v[j] = r;
            }
            __syncwarp();   // the raw rows have been consumed
            prefetch(i + NBUF, gpf);
            dft16<true>(v);   // v[j] = Z[o + 16 j]
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmulc(v[brev4(q)], t256[q * 16]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * kXw64QP] = v[brev4(q)];
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = xr[j];
            dft16<true>(v);
            // z[nn] = (x~[2 nn], x~[2 nn + 1]), nn = o + 16 k2; the stored unknowns lie in x~[0 .. 256): x_j = x~[j]
            // (zero-padded, DCT) or x~[j + 1] (DST-I)
            {
                double* dst = p.real_out + comp * p.rin_pc + rin_of(g);
                const bool al16 = ((reinterpret_cast<unsigned long long>(dst) & 15ull) == 0ull);
#pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) {
                    const int nn = o + 16 * k2;
                    const D z = v[brev4(k2)];
                    if constexpr (MODE == sf::X_DST1) {
                        if (nn > 0) dst[2 * nn - 1] = z.x;
                        dst[2 * nn] = z.y;
                    } else if (al16) {
                        *reinterpret_cast<D*>(dst + 2 * nn) = z;
                    } else {
                        dst[2 * nn] = z.x;
                        dst[2 * nn + 1] = z.y;
                    }
                }
            }
        }
    }
    cp_async_wait<0>();
}


// ==================================================================================== periodic rows of 256 reals, fp64
// S1 (real-to-complex) / S5 (complex-to-real) of periodic plans (PAPER.md:87 half spectrum), same scheme: the row is
// packed as z[n] = x[2n] + i x[2n+1], n < 128, Z = DFT128(z) by eight threads (lane = w + 8 rq, four rows per warp),
//     X[k] = ((Z[k] + conj Z[128-k]) - i w256^k (Z[k] - conj Z[128-k])) / 2,   k = 0..128.
// Thread w ends with Z[w + 8 j], j < 16; the partner 128 - k of k = w + 8 m, m < 8, is j' = 15 - m of thread 8 - w.
// X[128] goes to / comes from the side array of the strided passes when the plan has one.
constexpr int kXpw64QP = 9;                                          // exchange: 16-byte words per q
constexpr int kXpw64GP = 16 * kXpw64QP;                              // exchange: words per row
constexpr size_t kXpw64RawBytes = 4 * 256 * sizeof(double);          // four rows of 256 reals or 128 complex
constexpr size_t kXpw64WarpBytes = kXpw64RawBytes + 4 * (size_t)kXpw64GP * sizeof(D);
constexpr size_t kXpw64Smem = kXw64Warps * kXpw64WarpBytes;

template <bool INV> __global__ void __launch_bounds__(kXw64Threads, 2) fast_xpw64_kernel(const sf::XParams<double> p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(16) D s_t128[128];   // [q][w] = w128^(q w)
    __shared__ __align__(16) D s_tsp[64];     // [m][w] = w256^(w + 8 m)

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int wid = tid >> 5;
    const int w = lane & 7;
    const int rq = lane >> 3;
    const int plane = ((8 - w) & 7) + 8 * rq;   // holds the residue 8 - w of the same row; 0 and 4 pair with themselves
    const int comp = blockIdx.y;
    if (tid < 128) s_t128[tid] = c_tw1024d[(8 * (tid >> 3) * (tid & 7)) & 1023];
    if (tid < 64) s_tsp[tid] = c_tw1024d[4 * tid];
    __syncthreads();
    const D* t128 = s_t128 + w;   // [q * 8]
    const D* tsp = s_tsp + w;     // [m * 8]

    unsigned char* wbase = smem_raw + (size_t)wid * kXpw64WarpBytes;
    D* xch = reinterpret_cast<D*>(wbase + kXpw64RawBytes);
    D* xw = xch + rq * kXpw64GP + w;                     // slot (q, w) at q * kXpw64QP
    const D* xr = xch + rq * kXpw64GP + w * kXpw64QP;    // slots (w, o') and (w + 8, o')
    const D* srow = reinterpret_cast<const D*>(wbase) + rq * 128;

    const long long nrows = (long long)p.ny * p.nz;
    const long long nquads = (nrows + 3) / 4;
    const long long gw = (long long)blockIdx.x * kXw64Warps + wid;
    const long long nw = (long long)gridDim.x * kXw64Warps;
    const int nit = gw < nquads ? (int)((nquads - gw + nw - 1) / nw) : 0;
    D* nyq = reinterpret_cast<D*>(p.nyq_side);

    // a lane's row of iteration i; past the end the last row is done again, with identical stores
    struct Geom {
        int iy, iz;
        long long r;
    };
    const unsigned last_row = (unsigned)(nrows - 1);
    auto geometry = [&](int i) {
        const long long r = 4 * (gw + (long long)i * nw) + rq;
        const unsigned rc = r < (long long)last_row ? (unsigned)r : last_row;
        Geom g;
        g.r = rc;
        g.iz = (int)(rc / (unsigned)p.ny);
        g.iy = (int)(rc - (unsigned)g.iz * (unsigned)p.ny);
        return g;
    };
    auto rin_of = [&](const Geom& g) { return g.iy * p.rin_py + g.iz * p.rin_pz; };
    auto sp_of = [&](const Geom& g) { return g.iy * p.sp_py + g.iz * p.sp_pz; };
    // the eight lanes of a row copy it (256 reals or X[0..127]) into the staging buffer
    auto prefetch = [&](int i, const Geom& g) {
        if (i < nit) {
            double* dst = reinterpret_cast<double*>(wbase) + rq * 256;
            const double* src = INV ? reinterpret_cast<const double*>(reinterpret_cast<const D*>(p.spec_in) + comp * p.sp_pc + sp_of(g))
                                    : p.real_in + comp * p.rin_pc + rin_of(g);
            if (INV || __all_sync(0xffffffffu, (reinterpret_cast<unsigned long long>(src) & 15ull) == 0ull)) {
#pragma unroll
                for (int t = 0; t < 16; ++t) cp_async16(dst + 2 * (w + 8 * t), src + 2 * (w + 8 * t));
            } else {
#pragma unroll
                for (int t = 0; t < 32; ++t) cp_async8(dst + w + 8 * t, src + w + 8 * t);
            }
        }
        cp_async_commit();
    };
    // S5: X[128] of this thread's row, for the owner of the pair (0, 128)
    auto load_nyq = [&](int i, const Geom& g) -> D {
        if (!INV || w != 0 || i >= nit) return make_double2(0.0, 0.0);
        return nyq ? ldg_d(nyq + comp * nrows + g.r) : ldg_d(reinterpret_cast<const D*>(p.spec_in) + comp * p.sp_pc + sp_of(g) + 128);
    };

    Geom g0 = geometry(0);
    prefetch(0, g0);
    D xnyq_next = load_nyq(0, g0);
    for (int i = 0; i < nit; ++i) {
        const Geom g = g0;
        g0 = geometry(i + 1);
        cp_async_wait<0>();
        __syncwarp();
        D v[16], a[8], b[8];
        if constexpr (!INV) {
            // ---------------------------------------------------------------- S1
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = srow[w + 8 * r];
            __syncwarp();   // the raw rows are in registers: fetch the next ones
            prefetch(i + 1, g0);
            dft16<false>(v);
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul(v[brev4(q)], t128[q * 8]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * kXpw64QP] = v[brev4(q)];
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 8; ++j) { a[j] = xr[j]; b[j] = xr[8 * kXpw64QP + j]; }
            dft8<false>(a);
            dft8<false>(b);
            // Z[w + 8 j]: j = 2 k2 in a[brev3(k2)], j = 2 k2 + 1 in b[brev3(k2)]
            D* so = reinterpret_cast<D*>(p.spec_out) + comp * p.sp_pc + sp_of(g);
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int js = 15 - m, jo = (16 - m) & 15;
                D zm = shfl_d((js & 1) ? b[brev3(js >> 1)] : a[brev3(js >> 1)], plane);
                if (w == 0) zm = (jo & 1) ? b[brev3(jo >> 1)] : a[brev3(jo >> 1)];
                const D zk = (m & 1) ? b[brev3(m >> 1)] : a[brev3(m >> 1)];
                const D e = make_double2(zk.x + zm.x, zk.y - zm.y);
                const D d = make_double2(zk.x - zm.x, zk.y + zm.y);
                const D wd = cmul(d, tsp[m * 8]);
                const int k = w + 8 * m;
                const D xhi = make_double2(0.5 * (e.x - wd.y), 0.5 * (-e.y - wd.x));
                so[k] = make_double2(0.5 * (e.x + wd.y), 0.5 * (e.y - wd.x));
                if (m == 0 && w == 0) {
                    if (nyq) nyq[comp * nrows + g.r] = xhi;
                    else so[128] = xhi;
                } else {
                    so[128 - k] = xhi;
                }
            }
            if (w == 0) so[64] = make_double2(a[brev3(4)].x, -a[brev3(4)].y);   // k = 64 pairs with itself: conj Z[64]
        } else {
            // ---------------------------------------------------------------- S5
            const D xnyq = xnyq_next;
            D zhi[8];
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int k = w + 8 * m;
                const D xk = srow[k];
                D xm = srow[(128 - k) & 127];
                if (m == 0 && w == 0) xm = xnyq;
                const D e = make_double2(xk.x + xm.x, xk.y - xm.y);
                const D d = make_double2(xk.x - xm.x, xk.y + xm.y);
                const D wd = cmulc(d, tsp[m * 8]);
                v[m] = make_double2(e.x - wd.y, e.y + wd.x);
                zhi[m] = make_double2(e.x + wd.y, wd.x - e.y);
            }
            const D x64 = srow[64];
#pragma unroll
            for (int j = 8; j < 16; ++j) {
                D r = shfl_d(zhi[15 - j], plane);
                // w = 0: 128 - 8 m = 8 (16 - m) is its own; Z[64] = 2 conj X[64]
                if (w == 0) r = (j == 8) ? make_double2(2.0 * x64.x, -2.0 * x64.y) : zhi[(16 - j) & 7];
                v[j] = r;
            }
            __syncwarp();   // the raw rows have been consumed
            prefetch(i + 1, g0);
            xnyq_next = load_nyq(i + 1, g0);
            dft16<true>(v);   // v[j] = Z[w + 8 j]
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmulc(v[brev4(q)], t128[q * 8]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * kXpw64QP] = v[brev4(q)];
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 8; ++j) { a[j] = xr[j]; b[j] = xr[8 * kXpw64QP + j]; }
            dft8<true>(a);
            dft8<true>(b);
            double* dst = p.real_out + comp * p.rin_pc + rin_of(g);
            const bool al16 = ((reinterpret_cast<unsigned long long>(dst) & 15ull) == 0ull);
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                const int na = w + 16 * k2, nb = na + 8;   // (x[2n], x[2n+1])
                if (al16) {
                    *reinterpret_cast<D*>(dst + 2 * na) = a[brev3(k2)];
                    *reinterpret_cast<D*>(dst + 2 * nb) = b[brev3(k2)];
                } else {
                    dst[2 * na] = a[brev3(k2)].x; dst[2 * na + 1] = a[brev3(k2)].y;
                    dst[2 * nb] = b[brev3(k2)].x; dst[2 * nb + 1] = b[brev3(k2)].y;
                }
            }
        }
    }
    cp_async_wait<0>();
}

} // namespace sf2
