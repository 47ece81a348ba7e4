// sf_fastx64.cuh -- kernel generation 2 for the X passes S1 / S5 in double precision, rows whose extended real
// sequence has length 512 (complex transform length 256): zero-padded rows of 256 (unbounded plans),
// DST-I rows of 255 (Dirichlet, cell-boundary grid) and DCT-II / DCT-III rows of 256 (Neumann, cell-centre grid;
// Table 1, boundary values folded into the source on load).
//
// Same steps as sf_xpass.cuh (extension rule on load, packed real transform with split / merge, extraction rule on
// store; XParams and the folded source x_src are shared with it), with the register-resident 256-point transform
// of sf_fast.cuh in the middle: a CTA of 128 threads owns 8 contiguous rows; thread (o, row) holds the 16 packed
// elements n = o + 16 r of its row, radix-16 in registers, twiddle, one exchange through shared memory, radix-16
// in registers.  The rows are staged in shared memory both ways so that every global access is a coalesced run
// along a row (a warp per row), and the index rules of the boundary conditions touch shared memory only.  The
// exchange buffer and the staged spectrum rows and the staged real rows all share one 33 KB region (they are never live together): four CTAs per SM; persistent
// grid over the row tiles.
#pragma once
#include "sf_fast64.cuh"
#include "sf_fastper.cuh"
#include "sf_xpass.cuh"

namespace sf2 {

constexpr int kXgThreads = 128;
constexpr int kXgRows = 8;
constexpr int kXgRP = 258;     // doubles per staged real row: 2064 B = 16 (mod 128)
constexpr int kXgSP = 257;     // complex doubles per staged spectrum row: 4112 B = 16 (mod 128)
// the staged real rows, the exchange buffer and the staged spectrum rows are never live together: one region
constexpr size_t kXgSmem = (size_t)kXgRows * kXgSP * sizeof(D);
static_assert((size_t)kXgRows * kXgRP * sizeof(double) <= kXgSmem && (size_t)kXgRows * kXgSP >= 16 * 16 * 8, "staging layout");

// extended sequence x~[m], m < 512, from the staged row (the rules of sf_xpass.cuh: x_ext)
template <int MODE> __device__ __forceinline__ double xg_ext(const double* row, int m, int n)
{
    if constexpr (MODE == sf::X_ZEROPAD) {
        return m < n ? row[m] : 0.0;
    } else if constexpr (MODE == sf::X_DST1) {
        if (m == 0 || m == n + 1) return 0.0;
        return m <= n ? row[m - 1] : -row[511 - m];
    } else {   // X_DCT2
        return m < n ? row[m] : row[511 - m];
    }
}

// raw rows of the NEXT tile are fetched by asynchronous 8-byte copies (LDGSTS) into a buffer of their own while the
// current tile is transformed (all cases but the backward zero-padded pass, whose input rows are 4 KB each)
template <int MODE, bool INV> constexpr bool xg_prefetch() { return !(INV && MODE == sf::X_ZEROPAD); }
template <int MODE, bool INV> constexpr size_t xg_smem() { return kXgSmem + (xg_prefetch<MODE, INV>() ? (size_t)kXgRows * kXgRP * sizeof(double) : 0); }

template <int MODE, bool INV> __global__ void __launch_bounds__(kXgThreads, 4) fast_xg_kernel(const sf::XParams<double> p)
{
    constexpr bool PF = xg_prefetch<MODE, INV>();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* rbuf = reinterpret_cast<double*>(smem_raw);                                         // [8][kXgRP] reals
    D* sbuf = reinterpret_cast<D*>(smem_raw);                                                   // [8][kXgSP] complex, same storage
    D* xbuf = sbuf;                                                                             // exchange [16 q][16 o][8 rows]
    double* pbuf = reinterpret_cast<double*>(smem_raw + kXgSmem);                               // [8][kXgRP] raw rows of the next tile
    __shared__ __align__(16) D s_t256[256];   // [o][q] = w256^(q o)
    __shared__ __align__(16) D s_tsp[136];    // w512^k, k <= 128
    __shared__ int s_iy[2][kXgRows], s_iz[2][kXgRows];
    __shared__ long long s_rin[2][kXgRows], s_sp[2][kXgRows];

    const int tid = threadIdx.x;
    const int row = tid & 7;
    const int o = tid >> 3;
    const int warp = tid >> 5, lane = tid & 31;
    const int comp = blockIdx.y;
    const int n = p.n;
    for (int i = tid; i < 256; i += kXgThreads) s_t256[i] = c_tw1024d[(4 * (i & 15) * (i >> 4)) & 1023];
    for (int i = tid; i <= 128; i += kXgThreads) s_tsp[i] = c_tw1024d[2 * i];
    const D* t256 = s_t256 + o * 16;
    double* rrow = rbuf + row * kXgRP;
    const double* prow = pbuf + row * kXgRP;
    D* srow = sbuf + row * kXgSP;
    D* xw = xbuf + (o * 8 + row);            // slot (q, o) at stride 128
    const D* xr = xbuf + (o * 128 + row);    // slot (o, o') at stride 8

    const long long nrows = (long long)p.ny * p.nz;
    const long long ntiles = (nrows + kXgRows - 1) / kXgRows;
    // the rows this pass reads: the source (S1) or the real spectrum rows (S5, real-to-real modes)
    const double* rsrc = INV ? reinterpret_cast<const double*>(p.spec_in) + comp * p.sp_pc : p.real_in + comp * p.rin_pc;

    auto geometry = [&](long long tile, int g) {      // threads 0 .. 7
        const long long r = tile * kXgRows + tid;
        const int iy = (int)(r % p.ny), iz = (int)(r / p.ny);
        s_iy[g][tid] = (tile < ntiles && r < nrows) ? iy : -1;
        s_iz[g][tid] = iz;
        s_rin[g][tid] = iy * p.rin_py + iz * p.rin_pz;
        s_sp[g][tid] = iy * p.sp_py + iz * p.sp_pz;
    };
    auto prefetch = [&](int g) {                      // a warp per row, lanes along the row
        for (int r = warp; r < kXgRows; r += kXgThreads / 32) {
            double* dst = pbuf + r * kXgRP;
            if (s_iy[g][r] >= 0) {
                const double* src = rsrc + (INV ? s_sp[g][r] : s_rin[g][r]);
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (lane + 32 * j < n) cp_async8(dst + lane + 32 * j, src + lane + 32 * j);
            } else {
#pragma unroll
                for (int j = 0; j < 8; ++j) dst[lane + 32 * j] = 0.0;
            }
        }
        cp_async_commit();
    };

    int g = 0;
    if (tid < kXgRows) geometry(blockIdx.x, 0);
    __syncthreads();
    if (PF) prefetch(0);

    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, g ^= 1) {
        if (PF) cp_async_wait_all();
        __syncthreads();   // this tile's raw rows have landed; the previous tile's stores have read the staged rows
        D v[16];
        if constexpr (!INV) {
            // ---------------------------------------------------------------- S1
            if (p.has_faces) {
                // boundary values folded into the staged rows: a warp per row
                for (int r = warp; r < kXgRows; r += kXgThreads / 32) {
                    const int iy = s_iy[g][r];
                    if (iy < 0) continue;
                    const int iz = s_iz[g][r];
                    double* dst = pbuf + r * kXgRP;
                    if (iy == 0 || iy == p.ny - 1 || iz == 0 || iz == p.nz - 1) {
                        for (int ix = lane; ix < n; ix += 32) dst[ix] += sf::x_face_term(p, ix, iy, iz);
                    } else if (lane < 2) {
                        const int ix = lane ? n - 1 : 0;
                        dst[ix] += sf::x_face_term(p, ix, iy, iz);
                    }
                }
                __syncthreads();
            }
            // packed extended sequence z[nn] = x~[2 nn] + i x~[2 nn + 1], nn = o + 16 r
            // (n = 255 or 256: for r < 8 both positions 2 nn, 2 nn + 1 <= 255 lie in the stored half of the extension, for
            // r >= 8 in the mirrored / padded half -- the rules of xg_ext resolved at compile time)
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const int nn = o + 16 * r;
                if (r < 8) {
                    if (MODE == sf::X_DST1) v[r] = make_double2(nn == 0 ? 0.0 : prow[max(2 * nn - 1, 0)], prow[2 * nn]);
                    else v[r] = make_double2(prow[2 * nn], prow[2 * nn + 1]);
                } else {
                    if (MODE == sf::X_ZEROPAD) v[r] = make_double2(0.0, 0.0);
                    else if (MODE == sf::X_DST1) v[r] = make_double2(nn == 128 ? 0.0 : -prow[min(511 - 2 * nn, 254)], -prow[510 - 2 * nn]);
                    else v[r] = make_double2(prow[511 - 2 * nn], prow[510 - 2 * nn]);
                }
            }
            if (tid < kXgRows) geometry(tile + gridDim.x, g ^ 1);
            __syncthreads();   // the raw rows are in registers: fetch the next tile's while this one is transformed
            prefetch(g ^ 1);
            dft16<false>(v);
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul(v[brev4(q)], t256[q]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * 128] = v[brev4(q)];
            __syncthreads();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = xr[j * 8];
            dft16<false>(v);
            __syncthreads();   // everyone has read the exchange buffer: its storage becomes the spectrum rows
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) srow[o + 16 * k2] = v[brev4(k2)];   // Z[k], natural order
            __syncthreads();
            // split in place: X[k] = ((Z[k] + conj Z[256-k]) - i w512^k (Z[k] - conj Z[256-k])) / 2, pairs (k, 256 - k)
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                const int k = o + 16 * m;
                if (m < 8 || o == 0) {
                    const D zk = srow[k], zm = srow[(256 - k) & 255];
                    const D e = make_double2(zk.x + zm.x, zk.y - zm.y);
                    const D d = make_double2(zk.x - zm.x, zk.y + zm.y);
                    const D wd = cmul(d, s_tsp[k]);
                    srow[k] = make_double2(0.5 * (e.x + wd.y), 0.5 * (e.y - wd.x));
                    srow[256 - k] = make_double2(0.5 * (e.x - wd.y), 0.5 * (-e.y - wd.x));
                }
            }
            __syncthreads();
            // extraction rule and store, a warp per row
            for (int r = warp; r < kXgRows; r += kXgThreads / 32) {
                if (s_iy[g][r] < 0) continue;
                const D* sr = sbuf + r * kXgSP;
                if constexpr (MODE == sf::X_ZEROPAD) {
                    D* so = reinterpret_cast<D*>(p.spec_out) + comp * p.sp_pc + s_sp[g][r];
                    for (int k = lane; k <= 256; k += 32) so[k] = sr[k];
                } else {
                    double* ro = p.real_out + comp * p.sp_pc + s_sp[g][r];
                    for (int k = lane; k < n; k += 32) {
                        if constexpr (MODE == sf::X_DST1) {
                            ro[k] = -sr[k + 1].y;                        // DST-I: Y_k = -Im X~[k+1]
                        } else {
                            const D w = __ldg(p.ptw + k), x = sr[k];     // DCT-II: Y_k = Re(e^{-i pi k / 2n} X~[k])
                            ro[k] = w.x * x.x - w.y * x.y;
                        }
                    }
                }
            }
        } else {
            // ---------------------------------------------------------------- S5
            // half spectrum X~[0..256] of the extended sequence into the staged rows, a warp per row
            for (int r = warp; r < kXgRows; r += kXgThreads / 32) {
                D* sr = sbuf + r * kXgSP;
                const bool valid = s_iy[g][r] >= 0;
                if constexpr (MODE == sf::X_ZEROPAD) {
                    const D* si = reinterpret_cast<const D*>(p.spec_in) + comp * p.sp_pc + s_sp[g][r];
                    D t[9];
#pragma unroll
                    for (int j = 0; j < 9; ++j) t[j] = (valid && lane + 32 * j <= 256) ? ldg_d(si + lane + 32 * j) : make_double2(0.0, 0.0);
#pragma unroll
                    for (int j = 0; j < 9; ++j)
                        if (lane + 32 * j <= 256) sr[lane + 32 * j] = t[j];
                } else {
                    const double* ri = pbuf + r * kXgRP;     // the real spectrum row, prefetched
                    for (int k = lane; k <= 256; k += 32) {
                        D x = make_double2(0.0, 0.0);
                        if (valid) {
                            if constexpr (MODE == sf::X_DST1) {
                                if (k >= 1 && k <= n) x = make_double2(0.0, -ri[k - 1]);     // X~[k] = -i Y[k-1]
                            } else if (k < n) {
                                const D w = __ldg(p.ptw + k);                                // X~[k] = e^{+i pi k / 2n} Y[k]
                                const double y = ri[k];
                                x = make_double2(w.x * y, -w.y * y);
                            }
                        }
                        sr[k] = x;
                    }
                }
            }
            if (tid < kXgRows) geometry(tile + gridDim.x, g ^ 1);
            __syncthreads();
            if (PF) prefetch(g ^ 1);   // the raw rows have been consumed: fetch the next tile's
            // merge in place: Z[k] = (X[k] + conj X[256-k]) + i conj(w512^k) (X[k] - conj X[256-k]), pairs (k, 256 - k)
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                const int k = o + 16 * m;
                if (m < 8 || o == 0) {
                    const D xk = srow[k], xm = srow[256 - k];
                    const D e = make_double2(xk.x + xm.x, xk.y - xm.y);
                    const D d = make_double2(xk.x - xm.x, xk.y + xm.y);
                    const D wd = cmulc(d, s_tsp[k]);
                    srow[k] = make_double2(e.x - wd.y, e.y + wd.x);
                    if (k > 0) srow[256 - k] = make_double2(e.x + wd.y, wd.x - e.y);
                }
            }
            __syncthreads();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = srow[o + 16 * j];
            __syncthreads();   // the spectrum rows are in registers: their storage becomes the exchange buffer
            dft16<true>(v);
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmulc(v[brev4(q)], t256[q]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * 128] = v[brev4(q)];
            __syncthreads();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = xr[j * 8];
            __syncthreads();   // the exchange buffer has been read: its storage becomes the staged real rows
            dft16<true>(v);
            // unpack z[nn] = (x~[2 nn], x~[2 nn + 1]), nn = o + 16 k2; the stored unknowns lie in x~[0 .. 256)
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                const int nn = o + 16 * k2;
                rrow[2 * nn] = v[brev4(k2)].x;
                rrow[2 * nn + 1] = v[brev4(k2)].y;
            }
            __syncthreads();
            // extraction rule and store, a warp per row: x_j = x~[j] (zero-padded, DCT) or x~[j + 1] (DST-I)
            double* ro = p.real_out + comp * p.rin_pc;
            for (int r = warp; r < kXgRows; r += kXgThreads / 32) {
                if (s_iy[g][r] < 0) continue;
                const double* src = rbuf + r * kXgRP + (MODE == sf::X_DST1 ? 1 : 0);
                double* dst = ro + s_rin[g][r];
                for (int j = lane; j < n; j += 32) dst[j] = src[j];
            }
        }
    }
}

} // namespace sf2

namespace sf2 {

// ==================================================================================== periodic rows of 256 reals, fp64
// S1 (real-to-complex) / S5 (complex-to-real) of periodic plans (PAPER.md:87 half spectrum): the row is packed as
// z[n] = x[2n] + i x[2n+1], n < 128; Z = DFT128(z) = radix-16 over r (n = w + 8 r) in registers, twiddle w128^(q w), one
// exchange, two radix-8 (outputs k = w + 16 k2 and w + 8 + 16 k2); then the real-transform split to X[0..128].  A CTA of
// 128 threads owns 16 rows (thread = (w, row)); staged real rows, exchange buffer and staged spectrum rows share one
// 33 KB region.  X[128] goes to / comes from the side array of the strided passes when the plan has one.
constexpr int kXp64Threads = 128;
constexpr int kXp64Rows = 16;
constexpr int kXp64RP = 258;     // doubles per staged real row
constexpr int kXp64SP = 129;     // complex doubles per staged spectrum row (X[0..128])
constexpr size_t kXp64Smem = (size_t)kXp64Rows * kXp64RP * sizeof(double);
static_assert((size_t)kXp64Rows * kXp64SP * sizeof(D) <= kXp64Smem && (size_t)16 * 8 * 16 * sizeof(D) <= kXp64Smem, "one region");

template <bool INV> __global__ void __launch_bounds__(kXp64Threads, 4) fast_xp64_kernel(const sf::XParams<double> p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* rbuf = reinterpret_cast<double*>(smem_raw);
    D* sbuf = reinterpret_cast<D*>(smem_raw);
    D* xbuf = sbuf;
    __shared__ __align__(16) D s_t128[128];   // [w][q] = w128^(q w)
    __shared__ __align__(16) D s_tsp[72];     // w256^k, k <= 64
    __shared__ int s_ok[kXp64Rows];
    __shared__ long long s_rin[kXp64Rows], s_sp[kXp64Rows];

    const int tid = threadIdx.x;
    const int row = tid & 15;
    const int w = tid >> 4;
    const int warp = tid >> 5, lane = tid & 31;
    const int comp = blockIdx.y;
    s_t128[tid] = c_tw1024d[(8 * (tid & 15) * (tid >> 4)) & 1023];
    if (tid <= 64) s_tsp[tid] = c_tw1024d[4 * tid];
    const D* t128 = s_t128 + w * 16;
    double* rrow = rbuf + row * kXp64RP;
    D* srow = sbuf + row * kXp64SP;
    D* xw = xbuf + (w * 16 + row);                 // slot (q, w) at stride 128
    const D* xra = xbuf + (w * 128 + row);         // slot (w, o') at stride 16
    const D* xrb = xbuf + ((w + 8) * 128 + row);   // slot (w + 8, o')

    const long long nrows = (long long)p.ny * p.nz;
    const long long ntiles = (nrows + kXp64Rows - 1) / kXp64Rows;
    D* nyq = reinterpret_cast<D*>(p.nyq_side);

    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const long long row0 = tile * kXp64Rows;
        __syncthreads();
        if (tid < kXp64Rows) {
            const long long r = row0 + tid;
            const int iy = (int)(r % p.ny), iz = (int)(r / p.ny);
            s_ok[tid] = r < nrows;
            s_rin[tid] = iy * p.rin_py + iz * p.rin_pz;
            s_sp[tid] = iy * p.sp_py + iz * p.sp_pz;
        }
        __syncthreads();
        D v[16], a[8], b[8];
        if constexpr (!INV) {
            const double* rin = p.real_in + comp * p.rin_pc;
            for (int r = warp; r < kXp64Rows; r += kXp64Threads / 32) {
                double t[8];
                const double* rp = rin + s_rin[r];
#pragma unroll
                for (int j = 0; j < 8; ++j) t[j] = s_ok[r] ? __ldg(rp + lane + 32 * j) : 0.0;
#pragma unroll
                for (int j = 0; j < 8; ++j) rbuf[r * kXp64RP + lane + 32 * j] = t[j];
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = make_double2(rrow[2 * (w + 8 * r)], rrow[2 * (w + 8 * r) + 1]);
            __syncthreads();   // the staged rows are in registers: their storage becomes the exchange buffer
            dft16<false>(v);
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmul(v[brev4(q)], t128[q]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * 128] = v[brev4(q)];
            __syncthreads();
#pragma unroll
            for (int i = 0; i < 8; ++i) { a[i] = xra[i * 16]; b[i] = xrb[i * 16]; }
            dft8<false>(a);
            dft8<false>(b);
            __syncthreads();   // the exchange buffer has been read: its storage becomes the spectrum rows
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) { srow[w + 16 * k2] = a[brev3(k2)]; srow[w + 8 + 16 * k2] = b[brev3(k2)]; }
            __syncthreads();
            // split in place: pairs (k, 128 - k), k = w + 8 m
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                const int k = w + 8 * m;
                if (m < 8 || w == 0) {
                    const D zk = srow[k], zm = srow[(128 - k) & 127];
                    const D e = make_double2(zk.x + zm.x, zk.y - zm.y);
                    const D d = make_double2(zk.x - zm.x, zk.y + zm.y);
                    const D wd = cmul(d, s_tsp[k]);
                    srow[k] = make_double2(0.5 * (e.x + wd.y), 0.5 * (e.y - wd.x));
                    srow[128 - k] = make_double2(0.5 * (e.x - wd.y), 0.5 * (-e.y - wd.x));
                }
            }
            __syncthreads();
            D* so = reinterpret_cast<D*>(p.spec_out) + comp * p.sp_pc;
            for (int r = warp; r < kXp64Rows; r += kXp64Threads / 32) {
                if (!s_ok[r]) continue;
                const D* sr = sbuf + r * kXp64SP;
                D* dst = so + s_sp[r];
#pragma unroll
                for (int j = 0; j < 4; ++j) dst[lane + 32 * j] = sr[lane + 32 * j];
                if (lane == 0) {
                    if (nyq) nyq[comp * nrows + row0 + r] = sr[128];
                    else dst[128] = sr[128];
                }
            }
        } else {
            const D* si = reinterpret_cast<const D*>(p.spec_in) + comp * p.sp_pc;
            for (int r = warp; r < kXp64Rows; r += kXp64Threads / 32) {
                D* sr = sbuf + r * kXp64SP;
                const D* src = si + s_sp[r];
                D t[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) t[j] = s_ok[r] ? ldg_d(src + lane + 32 * j) : make_double2(0.0, 0.0);
#pragma unroll
                for (int j = 0; j < 4; ++j) sr[lane + 32 * j] = t[j];
                if (lane == 0) sr[128] = !s_ok[r] ? make_double2(0.0, 0.0) : (nyq ? nyq[comp * nrows + row0 + r] : src[128]);
            }
            __syncthreads();
            // merge in place: Z[k] = (X[k] + conj X[128-k]) + i conj(w256^k) (X[k] - conj X[128-k])
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                const int k = w + 8 * m;
                if (m < 8 || w == 0) {
                    const D xk = srow[k], xm = srow[128 - k];
                    const D e = make_double2(xk.x + xm.x, xk.y - xm.y);
                    const D d = make_double2(xk.x - xm.x, xk.y + xm.y);
                    const D wd = cmulc(d, s_tsp[k]);
                    srow[k] = make_double2(e.x - wd.y, e.y + wd.x);
                    if (k > 0) srow[128 - k] = make_double2(e.x + wd.y, wd.x - e.y);
                }
            }
            __syncthreads();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = srow[w + 8 * j];
            __syncthreads();
            dft16<true>(v);
#pragma unroll
            for (int q = 1; q < 16; ++q) v[brev4(q)] = cmulc(v[brev4(q)], t128[q]);
#pragma unroll
            for (int q = 0; q < 16; ++q) xw[q * 128] = v[brev4(q)];
            __syncthreads();
#pragma unroll
            for (int i = 0; i < 8; ++i) { a[i] = xra[i * 16]; b[i] = xrb[i * 16]; }
            __syncthreads();
            dft8<true>(a);
            dft8<true>(b);
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                const int na = w + 16 * k2, nb = w + 8 + 16 * k2;
                rrow[2 * na] = a[brev3(k2)].x; rrow[2 * na + 1] = a[brev3(k2)].y;
                rrow[2 * nb] = b[brev3(k2)].x; rrow[2 * nb + 1] = b[brev3(k2)].y;
            }
            __syncthreads();
            double* ro = p.real_out + comp * p.rin_pc;
            for (int r = warp; r < kXp64Rows; r += kXp64Threads / 32) {
                if (!s_ok[r]) continue;
                double* dst = ro + s_rin[r];
#pragma unroll
                for (int j = 0; j < 8; ++j) dst[lane + 32 * j] = rbuf[r * kXp64RP + lane + 32 * j];
            }
        }
    }
}

} // namespace sf2
