// sf_fastper.cuh -- kernel generation 2 for periodic fp32 plans whose y and z pencils are 256 long
// (BASELINE.json configs[1]): the strided passes S2 (Y forward), S3 (Z forward x 1 / eigenvalue x
// Z backward, fused) and S4 (Y backward) with the register-resident 256-point transform of
// sf_fast.cuh (PAPER.md:89-97 pencils, :103-109 four-step solve, Table 1 PAPER.md:160-167 periodic
// eigenvalues, zero mode PAPER.md:69).
//
// There is no padding here, so a thread has one transform to do instead of the two halves of the
// padded kernels: lane = pencil, and a CTA of 512 threads owns 32 neighbouring pencils -- every row
// of a tile is one 256-byte run, read straight into registers (the tile image is the 16 elements
// n = o + 16 r that thread (o, pencil) needs anyway) and written straight back.  Warp = o as in
// sf_fast.cuh; persistent CTAs, two per SM, tiles handed out by an atomic counter.
// The column count of a real-to-complex spectrum is n/2 + 1 = 4 * 32 + 1: the last (Nyquist)
// column is kept in a compact side array [z][y] that S1 writes and S5 reads instead of that column,
// and is handled 32 batches at a time (lane = batch), first in the queue.
#pragma once
#include "sf_fast.cuh"

namespace sf2 {

constexpr int kPerTile = 32;
constexpr size_t kPerSmem = (size_t)16 * 16 * 32 * sizeof(C);   // the exchange buffer

// tile t -> geometry
struct PerGeom {
    bool full;
    int b, col;   // full: batch, first column; else: first batch, the column
};
__device__ __forceinline__ PerGeom per_geom(const FastPerParams& p, int t)
{
    PerGeom g;
    const int nnyq = (p.nyq_col >= 0) ? (p.nb + kPerTile - 1) / kPerTile : 0;
    if (t < nnyq) {
        g.full = false;
        g.b = t * kPerTile;
        g.col = p.nyq_col;
    } else {
        const int tf = t - nnyq;
        g.full = true;
        g.b = tf / p.nct;
        g.col = (tf - g.b * p.nct) * kPerTile;
    }
    return g;
}

// backward transform of u (natural order in) and store of rows o + 16 j to q (row stride ors)
template <bool OB> __device__ __forceinline__ void per_inverse_store(C (&u)[16], const C* t256, int o, const Xchg& xc, C* q, int ors, bool valid)
{
    fft256_a<true, OB, true>(u, t256, o, xc);
    __syncthreads();
    fft256_b<true, OB>(u, xc);
    if (valid) {
#pragma unroll
        for (int j2 = 0; j2 < 16; ++j2) q[j2 * 16 * ors] = u[brev4(j2)];
    }
}

// 1 / d by the hardware approximation (one instruction, 1 ulp) for the spectral multiplier of fp32 plans; the correctly
// rounded __frcp_rn costs a fix-up sequence per element that the 2e-5 tolerance of these plans has no use for
__device__ __forceinline__ float rcp_approx(float d)
{
    float x;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(x) : "f"(d));
    return x;
}

// GRAD (fused mode only): besides psi, the three derivative spectra i kappa_a psi_hat (eq. (10))
// are transformed back from the same registers into fields 1..3 -- five transforms per tile, 32 more live
// registers, hence one CTA per SM
template <int MODE, bool GRAD = false>
__global__ void __launch_bounds__(kThreads, GRAD ? 1 : 2) fast_per_kernel(const FastPerParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* xbuf = reinterpret_cast<C*>(smem_raw);
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int o = (int)__reduce_max_sync(0xffffffffu, (unsigned)(tid >> 5));
    Xchg xc;
    xc.base = xbuf;
    xc.ea = o * 32 + lane;
    xc.eb = o * 512 + lane;

    __shared__ __align__(16) C s_t256[256];      // w256^(q o), row o
    __shared__ float s_lamp[256];                // fused: eigenvalue contribution of the pencil axis
    __shared__ float s_kapp[GRAD ? 256 : 1];     // gradient: wavenumber along the pencil axis
    __shared__ int s_tile[2];
    if (tid < 128) reinterpret_cast<float4*>(s_t256)[tid] = reinterpret_cast<const float4*>(g_tab_pad)[tid];
    if (MODE == FMODE_FUSED && tid < 256) s_lamp[tid] = __ldg(p.lam_p + tid);
    if (GRAD && tid < 256) s_kapp[tid] = __ldg(p.kap_p + tid);
    const C* t256 = s_t256 + o * 16;
    if (tid == 0) {   // the first two tiles are static, the rest come from the counter (+ 2 gridDim.x)
        s_tile[0] = (int)blockIdx.x;
        s_tile[1] = (int)(blockIdx.x + gridDim.x);
    }
    __syncthreads();

    const int ntiles = p.nb * p.nct + ((p.nyq_col >= 0) ? (p.nb + kPerTile - 1) / kPerTile : 0);
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;

    // one tile; OB = orientation of the exchange buffer its first transform starts with
    auto tile = [&](int t, int it, auto orient_tag) {
        constexpr bool OB = decltype(orient_tag)::value;
        const PerGeom g = per_geom(p, t);
        const bool valid = g.full ? (g.col + lane < p.nx) : (g.b + lane < p.nb);
        // Nyquist-column tiles live in a compact side array (element (row, batch) at row * nyq_ps +
        // batch * nyq_bs): column nyq_col of the work array itself would be gathered in 8-byte pieces a
        // whole plane apart, which costs more than all full tiles together (measured)
        const C* ibase = g.full ? p.in + (g.b * ibs + g.col + lane) : p.nyq + min(g.b + lane, p.nb - 1) * (int)p.nyq_bs;
        C* obase = g.full ? p.out + (g.b * obs + g.col + lane) : p.nyq + (g.b + lane) * (int)p.nyq_bs;
        const int irs = g.full ? ips : (int)p.nyq_ps, ors = g.full ? ops : (int)p.nyq_ps;
        // side-array tiles whose rows are contiguous in memory (the y passes: [z][y], lane = z) are moved as
        // 256-byte runs and transposed in the exchange buffer, idle at both ends of a tile: element
        // (row, pencil) at row * 32 + ((pencil + row) & 31), conflict-free along rows and along pencils
        const bool transposed = !g.full && p.nyq_ps == 1;
        auto stage = [&](int row, int pencil) -> C& { return xbuf[row * 32 + ((pencil + row) & 31)]; };
        C v[16];
        if (transposed) {
            if (it > 0) __syncthreads();   // the previous tile's second half may still be reading the exchange buffer
#pragma unroll 4
            for (int j = 0; j < 16; ++j) {
                const int idx = tid + kThreads * j, pl = idx >> 8, row = idx & 255;
                stage(row, pl) = (g.b + pl < p.nb) ? __ldg(p.nyq + (g.b + pl) * (int)p.nyq_bs + row) : make_float2(0.f, 0.f);
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = stage(o + 16 * r, lane);
            __syncthreads();
        } else {
            const C* ip = ibase + o * irs;
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = valid ? __ldg(ip + r * 16 * irs) : make_float2(0.f, 0.f);
        }
        // mirror of the transposing load for the results v[brev4(k)] = element o + 16 k
        auto store_transposed = [&](const C (&u)[16]) {
            __syncthreads();   // every thread is done reading the exchange buffer
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) stage(o + 16 * k2, lane) = u[brev4(k2)];
            __syncthreads();
#pragma unroll 4
            for (int j = 0; j < 16; ++j) {
                const int idx = tid + kThreads * j, pl = idx >> 8, row = idx & 255;
                if (g.b + pl < p.nb) p.nyq[(g.b + pl) * (int)p.nyq_bs + row] = stage(row, pl);
            }
            __syncthreads();   // before the next tile's exchange
        };
        // after the tile's first barrier every thread has read this tile's index: claim the tile after next
        // (the next tile's barrier publishes it)
        auto claim = [&]() { if (tid == 0) s_tile[it & 1] = atomicAdd(p.sched, 1) + 2 * (int)gridDim.x; };
        if constexpr (MODE == FMODE_FWD) {
            fft256_a<false, OB, false>(v, t256, o, xc);
            __syncthreads();
            claim();
            fft256_b<false, OB>(v, xc);
            if (transposed) {
                store_transposed(v);
            } else if (valid) {
                C* q = obase + o * ors;
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) q[k2 * 16 * ors] = v[brev4(k2)];
            }
        } else if constexpr (MODE == FMODE_INV) {
            fft256_a<true, OB, true>(v, t256, o, xc);
            __syncthreads();
            claim();
            fft256_b<true, OB>(v, xc);
            if (transposed) {
                store_transposed(v);
            } else if (valid) {
                C* q = obase + o * ors;
#pragma unroll
                for (int j2 = 0; j2 < 16; ++j2) q[j2 * 16 * ors] = v[brev4(j2)];
            }
        } else {
            fft256_a<false, OB, true>(v, t256, o, xc);
            __syncthreads();
            claim();
            fft256_b<false, OB>(v, xc);
            // X[k = o + 16 k2] at v[brev4(k2)]: multiply by scale / (lambda_x + lambda_b + lambda_p[k]), zero mode -> 0
            const int kx = g.full ? min(g.col + lane, p.nx - 1) : g.col;
            const int kb = g.full ? g.b : min(g.b + lane, p.nb - 1);
            const float lxb = __ldg(p.lam_x + kx) + __ldg(p.lam_b + kb);
            const bool zero0 = p.zero_mode && kx == 0 && kb == 0 && o == 0;
            C w[16];
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) {
                float m = p.scale * rcp_approx(lxb + s_lamp[o + 16 * k2]);
                if (k2 == 0 && zero0) m = 0.f;
                w[k2] = cscale(v[brev4(k2)], m);
            }
            if constexpr (GRAD) {
                const float qx = __ldg(p.kap_x + kx), qy = __ldg(p.kap_b + kb);
                const int ocs = g.full ? (int)p.out_cs : (int)p.nyq_cs;   // field stride
                C* q = obase + o * ors;
                C u[16];
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) u[k2] = cmuli(cscale(w[k2], s_kapp[o + 16 * k2]));
                per_inverse_store<!OB>(u, t256, o, xc, q + 3 * ocs, ors, valid);
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) u[k2] = cmuli(cscale(w[k2], qy));
                per_inverse_store<OB>(u, t256, o, xc, q + 2 * ocs, ors, valid);
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) u[k2] = cmuli(cscale(w[k2], qx));
                per_inverse_store<!OB>(u, t256, o, xc, q + ocs, ors, valid);
                per_inverse_store<OB>(w, t256, o, xc, q, ors, valid);
            } else {
                per_inverse_store<!OB>(w, t256, o, xc, obase + o * ors, ors, valid);
            }
        }
    };

    if constexpr (MODE == FMODE_FUSED && !GRAD) {
        // two transforms per tile: the orientation is back where it started
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

namespace sf2 {

// ==================================================================================== X passes, periodic
// S1 (real-to-complex) and S5 (complex-to-real) for rows of 256 reals (PAPER.md:87 half spectrum).
// A row is packed as z[n] = x[2n] + i x[2n+1], n < 128; Z = DFT128(z) by the 128-point transform of
// the padded X kernels (radix-16 over r, n = w + 8 r; twiddle; one exchange; two radix-8), then
//     X[k] = ( (Z[k] + conj Z[128-k]) - i w256^k (Z[k] - conj Z[128-k]) ) / 2,   k = 0..128.
// CTA of 256 threads = 8 warps (w) x 32 lanes, lane = row: a tile is 32 rows, staged in shared
// memory with odd 8-byte pitches (lanes on distinct banks) and moved to and from global memory as
// whole contiguous rows.  X[0..127] go to the spectrum array, X[128] to the side array [row].
constexpr int kXpThreads = 256;
constexpr int kXpRows = 32;
constexpr int kXpRealPitch = 258;   // floats: 1032 B = 8 (mod 128)
constexpr int kXpSpecPitch = 129;   // complex: 1032 B
constexpr size_t kXpSmem = (size_t)kXpRows * kXpRealPitch * sizeof(float) + (size_t)16 * 8 * 32 * sizeof(C) + (size_t)kXpRows * kXpSpecPitch * sizeof(C);

// 8-byte asynchronous copy global -> shared (LDGSTS), completion by cp.async groups
__device__ __forceinline__ void cp_async8(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <bool INV> __global__ void __launch_bounds__(kXpThreads, 2) fast_xper_kernel(const FastXPerParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* rbuf = reinterpret_cast<float*>(smem_raw);
    C* xbuf = reinterpret_cast<C*>(smem_raw + (size_t)kXpRows * kXpRealPitch * sizeof(float));
    C* sbuf = xbuf + 16 * 8 * 32;
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int w = (int)__reduce_max_sync(0xffffffffu, (unsigned)(tid >> 5));
    __shared__ __align__(16) C s_t128[128];     // w128^(q w), row w
    if (tid < 64) reinterpret_cast<float4*>(s_t128)[tid] = reinterpret_cast<const float4*>(g_tab_x)[tid];
    const C* t128 = s_t128 + w * 16;
    C* xw = xbuf + w * 32 + lane;
    const C* xr = xbuf + w * 8 * 32 + lane;
    C* srow = sbuf + lane * kXpSpecPitch;
    float* rrow = rbuf + lane * kXpRealPitch;
    __syncthreads();

    const int ntiles = p.nrows / kXpRows;
    // the rows of tile t arrive by asynchronous 8-byte copies (coalesced), issued one tile ahead as soon as
    // the staging buffer of the current tile has been read by every thread
    auto fetch = [&](int t) {
        if (t >= ntiles) return;
        const long long row0 = (long long)t * kXpRows;
        if constexpr (!INV) {
            const float2* gin = reinterpret_cast<const float2*>(p.real_in + row0 * 256);
#pragma unroll 4
            for (int j = 0; j < 16; ++j) {
                const int idx = tid + kXpThreads * j, r = idx >> 7, n = idx & 127;
                cp_async8(rbuf + r * kXpRealPitch + 2 * n, gin + idx);
            }
        } else {
#pragma unroll 4
            for (int j = 0; j < 16; ++j) {
                const int idx = tid + kXpThreads * j, r = idx >> 7, k = idx & 127;
                cp_async8(sbuf + r * kXpSpecPitch + k, p.spec + (row0 + r) * p.spec_pitch + k);
            }
            if (tid < kXpRows) cp_async8(sbuf + tid * kXpSpecPitch + 128, p.nyq + row0 + tid);
        }
        cp_async_commit();
    };
    fetch(blockIdx.x);
    for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const long long row0 = (long long)t * kXpRows;
        cp_async_wait_all();
        __syncthreads();
        if constexpr (!INV) {
            C v[16];
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = *reinterpret_cast<const C*>(rrow + 2 * (w + 8 * r));
            fft128_a<false>(v, t128, xw);
            __syncthreads();
            fetch(t + gridDim.x);   // rbuf is in registers everywhere
            C a[8], b[8];
            fft128_b<false>(a, b, xr);
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                srow[w + 16 * k2] = a[brev3(k2)];
                srow[w + 8 + 16 * k2] = b[brev3(k2)];
            }
            __syncthreads();
            // split in place: thread w owns the pairs (k, 128 - k), k = w + 8 m, m < 8 (and k = 64 for w = 0)
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                const int k = (m < 8) ? w + 8 * m : 64;
                if (m == 8 && w != 0) break;
                const C zk = srow[k], zm = srow[(128 - k) & 127];
                const C e = make_float2(zk.x + zm.x, zk.y - zm.y);
                const C d = make_float2(zk.x - zm.x, zk.y + zm.y);
                const C wd = cmul(d, c_tw1024[4 * k]);   // w256^k d
                srow[k] = make_float2(0.5f * (e.x + wd.y), 0.5f * (e.y - wd.x));
                if (k != 64) srow[128 - k] = make_float2(0.5f * (e.x - wd.y), 0.5f * (-e.y - wd.x));
            }
            __syncthreads();
#pragma unroll 4
            for (int j = 0; j < 16; ++j) {
                const int idx = tid + kXpThreads * j, r = idx >> 7, k = idx & 127;
                p.spec[(row0 + r) * p.spec_pitch + k] = sbuf[r * kXpSpecPitch + k];
            }
            if (tid < kXpRows) p.nyq[row0 + tid] = sbuf[tid * kXpSpecPitch + 128];
            // (sbuf is rewritten after the next tile's second barrier)
        } else {
            // merge in place: Z[k] = e + i conj(w256^k) d,  Z[128 - k] = conj e + i conj(conj(w256^k) d)
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                const int k = (m < 8) ? w + 8 * m : 64;
                if (m == 8 && w != 0) break;
                const C xk = srow[k], xm = srow[128 - k];
                const C e = make_float2(xk.x + xm.x, xk.y - xm.y);
                const C d = make_float2(xk.x - xm.x, xk.y + xm.y);
                const C wd = cmulc(d, c_tw1024[4 * k]);
                srow[k] = make_float2(e.x - wd.y, e.y + wd.x);
                if (k != 0 && k != 64) srow[128 - k] = make_float2(e.x + wd.y, -e.y + wd.x);
            }
            __syncthreads();
            C v[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = srow[w + 8 * j];
            fft128_a<true>(v, t128, xw);
            __syncthreads();
            fetch(t + gridDim.x);   // sbuf is in registers everywhere
            C a[8], b[8];
            fft128_b<true>(a, b, xr);
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                *reinterpret_cast<C*>(rrow + 2 * (w + 16 * k2)) = a[brev3(k2)];
                *reinterpret_cast<C*>(rrow + 2 * (w + 8 + 16 * k2)) = b[brev3(k2)];
            }
            __syncthreads();
            float2* gout = reinterpret_cast<float2*>(p.real_out + row0 * 256);
#pragma unroll 4
            for (int j = 0; j < 16; ++j) {
                const int idx = tid + kXpThreads * j, r = idx >> 7, n = idx & 127;
                gout[idx] = *reinterpret_cast<const float2*>(rbuf + r * kXpRealPitch + 2 * n);
            }
            // (rbuf is rewritten after the next tile's third barrier)
        }
    }
}

} // namespace sf2
