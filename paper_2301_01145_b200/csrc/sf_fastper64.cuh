// sf_fastper64.cuh -- kernel generation 2 in double precision for periodic plans whose y and z pencils are 256 long
// (BASELINE.json configs[1] in fp64): the strided passes S2 (Y forward), S3 (Z forward x 1 / eigenvalue x Z backward,
// fused; with sf_gradient also the three spectra i kappa_a psi_hat, eq. (10)) and S4 (Y backward);
// PAPER.md:89-97 pencils, :103-109 four-step solve, Table 1 PAPER.md:160-167 periodic eigenvalues, zero mode PAPER.md:69.
//
// sf_fastper.cuh with 16-byte elements: no padding, one 256-point transform per thread; a CTA of 256 threads owns 16
// neighbouring pencils (256-byte rows), half-warp = residue o, lane = pencil; rows are read straight into registers and
// written straight back; two CTAs per SM (<= 128 registers), dynamic tile queue.  The Nyquist column (129 = 8 x 16 + 1)
// lives in the compact side array that the X passes write and read, 16 batches per tile.
// The gradient needs psi_hat four times (psi and three derivatives), 64 registers that a 128-register thread does not
// have twice: psi_hat is parked in TENSOR MEMORY (tcgen05.st / ld 32x32b.x64: every thread parks and fetches its own
// 64 words; 128 columns per CTA) and fetched back for each of the four backward transforms.
#pragma once
#include "sf_fast64.cuh"
#include "sf_fast512.cuh"

namespace sf2 {

constexpr int kPer64Tile = 16;
constexpr size_t kPer64Smem = (size_t)kXchg64Elems * sizeof(D);   // the exchange buffer, 64 KB

// 16 doubles (32 words) of this thread to / from 32 consecutive columns of its tensor-memory lane
__device__ __forceinline__ void tmem_st16dbl(uint32_t addr, const double (&d)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(addr),
                 "r"(__double2loint(d[0])), "r"(__double2hiint(d[0])), "r"(__double2loint(d[1])), "r"(__double2hiint(d[1])), "r"(__double2loint(d[2])), "r"(__double2hiint(d[2])), "r"(__double2loint(d[3])), "r"(__double2hiint(d[3])), "r"(__double2loint(d[4])), "r"(__double2hiint(d[4])), "r"(__double2loint(d[5])), "r"(__double2hiint(d[5])), "r"(__double2loint(d[6])), "r"(__double2hiint(d[6])), "r"(__double2loint(d[7])), "r"(__double2hiint(d[7])), "r"(__double2loint(d[8])), "r"(__double2hiint(d[8])), "r"(__double2loint(d[9])), "r"(__double2hiint(d[9])), "r"(__double2loint(d[10])), "r"(__double2hiint(d[10])), "r"(__double2loint(d[11])), "r"(__double2hiint(d[11])), "r"(__double2loint(d[12])), "r"(__double2hiint(d[12])), "r"(__double2loint(d[13])), "r"(__double2hiint(d[13])), "r"(__double2loint(d[14])), "r"(__double2hiint(d[14])), "r"(__double2loint(d[15])), "r"(__double2hiint(d[15]))
                 : "memory");
}
__device__ __forceinline__ void tmem_ld16dbl(uint32_t addr, double (&d)[16])
{
    int w[32];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7]), "=r"(w[8]), "=r"(w[9]), "=r"(w[10]), "=r"(w[11]), "=r"(w[12]), "=r"(w[13]), "=r"(w[14]), "=r"(w[15]), "=r"(w[16]), "=r"(w[17]), "=r"(w[18]), "=r"(w[19]), "=r"(w[20]), "=r"(w[21]), "=r"(w[22]), "=r"(w[23]), "=r"(w[24]), "=r"(w[25]), "=r"(w[26]), "=r"(w[27]), "=r"(w[28]), "=r"(w[29]), "=r"(w[30]), "=r"(w[31])
                 : "r"(addr)
                 : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) d[i] = __hiloint2double(w[2 * i + 1], w[2 * i]);
}

struct Per64Geom { bool full; int b, col; };
__device__ __forceinline__ Per64Geom per64_geom(const FastPer64Params& p, int t)
{
    Per64Geom g;
    const int nnyq = (p.nyq_col >= 0) ? (p.nb + kPer64Tile - 1) / kPer64Tile : 0;
    if (t < nnyq) {
        g.full = false;
        g.b = t * kPer64Tile;
        g.col = p.nyq_col;
    } else {
        const int tf = t - nnyq;
        g.full = true;
        g.b = tf / p.nct;
        g.col = (tf - g.b * p.nct) * kPer64Tile;
    }
    return g;
}

template <int MODE, bool GRAD = false>
__global__ void __launch_bounds__(kT64, 2) fast_per64_kernel(const FastPer64Params p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    D* xbuf = reinterpret_cast<D*>(smem_raw);
    const int tid = threadIdx.x;
    const int pen = tid & 15;
    const int o = tid >> 4;
    const int ea = o * 16 + pen;
    const int eb = o * 256 + pen;
    __shared__ __align__(16) D s_t256[256];
    __shared__ double s_lamp[MODE == FMODE_FUSED ? 256 : 1];
    __shared__ double s_kapp[GRAD ? 256 : 1];
    __shared__ int s_tile[2];
    __shared__ uint32_t s_tmem;
    s_t256[tid] = c_tw1024d[(4 * (tid & 15) * (tid >> 4)) & 1023];
    if (MODE == FMODE_FUSED) s_lamp[tid] = __ldg(p.lam_p + tid);
    if (GRAD) s_kapp[tid] = __ldg(p.kap_p + tid);
    const D* t256 = s_t256 + o * 16;
    if (tid == 0) {
        s_tile[0] = (int)blockIdx.x;
        s_tile[1] = (int)(blockIdx.x + gridDim.x);
    }
    uint32_t tpark = 0;
    if (GRAD) {
        if (tid < 32) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(128u) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    __syncthreads();
    if (GRAD) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const int wq = tid >> 5;
        tpark = s_tmem + ((uint32_t)(wq & 3) << 21) + (uint32_t)(wq >> 2) * 64;   // lane quadrant of the warp, 64 columns
    }

    const int ntiles = p.nb * p.nct + ((p.nyq_col >= 0) ? (p.nb + kPer64Tile - 1) / kPer64Tile : 0);
    const int ips = (int)p.in_ps, ops = (int)p.out_ps, ibs = (int)p.in_bs, obs = (int)p.out_bs;

    auto tile = [&](int t, int it, auto orient_tag) {
        constexpr bool OB = decltype(orient_tag)::value;
        const Per64Geom g = per64_geom(p, t);
        const bool valid = g.full ? (g.col + pen < p.nx) : (g.b + pen < p.nb);
        // Nyquist-column tiles live in the compact side array: element (row, batch) at row * nyq_ps + batch * nyq_bs
        const D* ibase = g.full ? p.in + ((size_t)g.b * ibs + g.col + pen) : p.nyq + (size_t)min(g.b + pen, p.nb - 1) * (int)p.nyq_bs;
        D* obase = g.full ? p.out + ((size_t)g.b * obs + g.col + pen) : p.nyq + (size_t)(g.b + pen) * (int)p.nyq_bs;
        const int irs = g.full ? ips : (int)p.nyq_ps, ors = g.full ? ops : (int)p.nyq_ps;
        D v[16];
        {
            const D* ip = ibase + (size_t)o * irs;
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = valid ? ldg_d(ip + (size_t)r * 16 * irs) : make_double2(0.0, 0.0);
        }
        auto claim = [&]() { if (tid == 0) s_tile[it & 1] = atomicAdd(p.sched, 1) + 2 * (int)gridDim.x; };
        // backward transform of u (natural order) and store of rows o + 16 j
        auto inverse_store = [&](D (&u)[16], D* q, auto ob_tag) {
            constexpr bool OBI = decltype(ob_tag)::value;
            fft256d_a<true, OBI>(u, t256, xbuf, ea, eb);
            __syncthreads();
            fft256d_b<true, OBI>(u, xbuf, ea, eb);
            if (valid) {
#pragma unroll
                for (int j2 = 0; j2 < 16; ++j2) q[(size_t)j2 * 16 * ors] = u[brev4(j2)];
            }
        };
        if constexpr (MODE == FMODE_FWD || MODE == FMODE_INV) {
            fft256d_a<MODE == FMODE_INV, OB>(v, t256, xbuf, ea, eb);
            __syncthreads();
            claim();
            fft256d_b<MODE == FMODE_INV, OB>(v, xbuf, ea, eb);
            if (valid) {
                D* q = obase + (size_t)o * ors;
#pragma unroll
                for (int k2 = 0; k2 < 16; ++k2) q[(size_t)k2 * 16 * ors] = v[brev4(k2)];
            }
        } else {
            fft256d_a<false, OB>(v, t256, xbuf, ea, eb);
            __syncthreads();
            claim();
            fft256d_b<false, OB>(v, xbuf, ea, eb);
            // X[k = o + 16 k2] at v[brev4(k2)]: times scale / (lambda_x + lambda_b + lambda_p[k]), zero mode -> 0
            const int kx = g.full ? min(g.col + pen, p.nx - 1) : g.col;
            const int kb = g.full ? g.b : min(g.b + pen, p.nb - 1);
            const double lxb = __ldg(p.lam_x + kx) + __ldg(p.lam_b + kb);
            const bool zero0 = p.zero_mode && kx == 0 && kb == 0 && o == 0;
            D w[16];
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) {
                double m = p.scale * fast_rcp(lxb + s_lamp[o + 16 * k2]);
                if (k2 == 0 && zero0) m = 0.0;
                w[k2] = cscale(v[brev4(k2)], m);
            }
            D* q = obase + (size_t)o * ors;
            if constexpr (GRAD) {
                const double qx = __ldg(p.kap_x + kx), qy = __ldg(p.kap_b + kb);
                const size_t ocs = g.full ? (size_t)p.out_cs : (size_t)p.nyq_cs;   // field stride
                // park psi_hat in tensor memory: real parts in columns 0..31, imaginary parts in 32..63
                {
                    double re[16], im[16];
#pragma unroll
                    for (int k2 = 0; k2 < 16; ++k2) { re[k2] = w[k2].x; im[k2] = w[k2].y; }
                    tmem_st16dbl(tpark, re);
                    tmem_st16dbl(tpark + 32, im);
                    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                }
                // fields 3, 2, 1: i kappa psi_hat = (-kappa Im, kappa Re); then psi itself
#pragma unroll 1
                for (int fld = 3; fld >= 0; --fld) {
                    double re[16], im[16];
                    tmem_ld16dbl(tpark, re);
                    tmem_ld16dbl(tpark + 32, im);
                    D u[16];
#pragma unroll
                    for (int k2 = 0; k2 < 16; ++k2) {
                        if (fld == 0) {
                            u[k2] = make_double2(re[k2], im[k2]);
                        } else {
                            const double kk = (fld == 3) ? s_kapp[o + 16 * k2] : (fld == 2 ? qy : qx);
                            u[k2] = make_double2(-kk * im[k2], kk * re[k2]);
                        }
                    }
                    // four transforms follow the forward one: the orientation alternates !OB, OB, !OB, OB
                    if ((fld & 1) == 1) inverse_store(u, q + (size_t)fld * ocs, std::integral_constant<bool, !OB>());
                    else inverse_store(u, q + (size_t)fld * ocs, std::integral_constant<bool, OB>());
                }
            } else {
                inverse_store(w, q, std::integral_constant<bool, !OB>());
            }
        }
    };

    if constexpr (MODE == FMODE_FUSED && !GRAD) {
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
    if (GRAD) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem), "r"(128u) : "memory");
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
