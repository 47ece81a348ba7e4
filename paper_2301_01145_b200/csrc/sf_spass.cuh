// sf_spass.cuh -- steps S2 (Y forward), S3 (Z forward x multiplier x Z backward, fused) and
// S4 (Y backward) of the hot path: batched transforms along a strided axis
// (PAPER.md:89-97 pencils; PAPER.md:103-109 four-step solve; eq. (10) PAPER.md:141 spectral
// differentiation; Table 1 PAPER.md:160-167 eigenvalues; PAPER.md:181, :213 padded / pruned solve).
//
// One CTA owns a tile of TX neighbouring x-columns times the whole pencil: every global access is
// a run of TX consecutive elements (128 B for the headline configurations).  In shared memory the
// tile is s[position * TX + column]; butterflies run in place, decimation in frequency forward
// (natural order in, digit-reversed out) and its mirror backward (digit-reversed in, natural out),
// so the fused kernel multiplies in digit-reversed order and never reorders, and the unfused
// kernels fold the permutation into the global row address.
//   MODE 0: forward only   (S2; also plan-time transforms of the Green's function)
//   MODE 1: backward only  (S4)
//   MODE 2: forward, multiply, backward (S3) with 1 -> 1 (solve, Laplacian), 1 -> 1+d (gradient),
//           3 -> 3 (curl) or 3 -> 1 (divergence) fields
// Zero padding is fused into the load (rows >= n_in are zeros), truncation into the store (rows
// >= n_out are dropped).  Dirichlet / Neumann pencils are real: they are extended (odd / even) to
// length 2L on load, packed as L complex numbers, and the real-transform split / merge steps are
// done pairwise in place around the multiply.
#pragma once
#include "sf_common.cuh"

namespace sf {

enum { MUL_SYMBOL = 0, MUL_GREEN = 1 };
enum { OUT_SOLVE = 0, OUT_GRAD = 1, OUT_CURL = 2, OUT_DIV = 3, OUT_LAP = 4 };
enum { R2R_NONE = 0, R2R_DST1 = 1, R2R_DCT = 2, R2R_DST2 = 3, R2R_DCT1 = 4 };

template <typename T> struct SParams {
    typedef SF_CX C;
    const void* in;
    void* out;
    long long in_ps, in_bs, in_cs;    // pencil-axis / batch-axis / field strides, in elements
    long long out_ps, out_bs, out_cs;
    int nx;       // valid columns
    int n_in;     // complex: rows read (the rest are zero); real: stored unknowns n
    int n_out;    // rows written
    int r2r;      // R2R_*
    int LT;       // length of tw (a multiple of the transform length)
    const C* tw;  // exp(-2 pi i j / LT)
    const C* ptw; // R2R_DCT, R2R_DST2: exp(-i pi k / (2n)), k <= n
    // ---- fused multiply (MODE 2)
    int mul;          // MUL_*
    int outk;         // OUT_*
    int pencil_axis;  // 1: 2-D problem (pencil = y), 2: 3-D problem (pencil = z, batch = y)
    const T* lam_x; const T* lam_b; const T* lam_p;   // eigenvalue contribution per axis
    const T* kap_x; const T* kap_b; const T* kap_p;   // wavenumber per axis (0 at Nyquist)
    T scale;          // rhs_sign / (transform normalisation)
    int zero_mode;    // all-zero index -> 0
    const T* green;   // compact real table [fp][fb][kx], rhs_sign and normalisation folded in
    long long g_pb, g_pp;
    int Pb, Pp;       // transform lengths along batch / pencil axes (index folding k -> min(k, P-k))
    // ---- real pencils: spectral derivative along the pencil axis (sine <-> cosine series, eq. (10))
    int dfield1;      // MODE 1: 1 + index of the field (blockIdx.z) whose backward transform differentiates; 0: none
    const T* kap_ext; // wavenumber pi k / L_domain of slot k of the extended sequence, k <= L, zero at k = L
};

template <typename T, int L> __host__ __device__ constexpr int s_tx()
{
    constexpr int e = 2 * (int)sizeof(T);
    constexpr int t = 65536 / (L * e);
    return t >= 16 ? 16 : (t >= 8 ? 8 : 4);
}

template <typename T> __device__ __forceinline__ T s_multiplier(const SParams<T>& p, int kx, int kb, int kp)
{
    if (p.mul == MUL_SYMBOL) {
        if (p.zero_mode && kx == 0 && kb == 0 && kp == 0) return (T)0;
        const T lam = __ldg(p.lam_x + kx) + __ldg(p.lam_b + kb) + __ldg(p.lam_p + kp);
        return p.scale / lam;
    } else {
        const int fb = min(kb, p.Pb - kb), fp = min(kp, p.Pp - kp);
        return __ldg(p.green + kx + fb * p.g_pb + fp * p.g_pp);
    }
}

// real component m (0 .. 2L) of the packed tile
template <typename T, int TX> __device__ __forceinline__ T& s_real(SF_CX* s, int m, int tx)
{
    return reinterpret_cast<T*>(s + (m >> 1) * TX + tx)[m & 1];
}

template <typename T, int L, int TX, int NT, int MODE>
__global__ void __launch_bounds__(NT) spass_kernel(const SParams<T> p)
{
    typedef SF_CX C;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s0 = reinterpret_cast<C*>(smem_raw);
    constexpr int TILE = L * TX;

    const int x0 = blockIdx.x * TX;
    const int ib = blockIdx.y;
    const int tx_ = threadIdx.x % TX;
    const bool xok = (x0 + tx_) < p.nx;          // a thread keeps its column in every tx-fastest loop
    const bool div = (MODE == 2) && (p.outk == OUT_DIV);
    const bool curl = (MODE == 2) && (p.outk == OUT_CURL || div);   // all three spectra in one CTA
    const int nfield_in = curl ? 3 : 1;
    const long long fz = curl ? 0 : blockIdx.z;   // independent components ride on gridDim.z

    // ------------------------------------------------------------------ load
    if (p.r2r == R2R_NONE) {
        for (int c = 0; c < nfield_in; ++c) {
            const C* gin = reinterpret_cast<const C*>(p.in) + (fz + c) * p.in_cs + ib * p.in_bs + x0;
            C* s = s0 + c * TILE;
            for (int idx = threadIdx.x; idx < TILE; idx += NT) {
                const int tx = idx % TX, j = idx / TX;
                C v = mk<T>(0, 0);
                if (j < p.n_in && xok) v = gin[j * p.in_ps + tx];
                s[(MODE == 1 ? pos_of_k<L>(j) : j) * TX + tx] = v;
            }
        }
    } else if (MODE != 1) {
        // real pencils, extended to length 2L:  DST-I: 0, x, 0, -reverse(x);  DCT-II: x, reverse(x);
        // DST-II: x, -reverse(x);  DCT-I (n = L + 1): x_0 .. x_L, x_{L-1} .. x_1
        const T* gin = reinterpret_cast<const T*>(p.in) + fz * p.in_cs + ib * p.in_bs + x0;
        const int n = p.n_in;
        constexpr int M = 2 * L;
        if (p.r2r == R2R_DST1 && threadIdx.x < TX) {
            s_real<T, TX>(s0, 0, threadIdx.x) = (T)0;
            s_real<T, TX>(s0, L, threadIdx.x) = (T)0;
        }
        for (int idx = threadIdx.x; idx < n * TX; idx += NT) {
            const int tx = idx % TX, j = idx / TX;
            const T v = xok ? gin[j * p.in_ps + tx] : (T)0;
            if (p.r2r == R2R_DST1) {
                s_real<T, TX>(s0, j + 1, tx) = v;
                s_real<T, TX>(s0, M - 1 - j, tx) = -v;
            } else if (p.r2r == R2R_DCT1) {
                s_real<T, TX>(s0, j, tx) = v;
                if (j >= 1 && j < L) s_real<T, TX>(s0, M - j, tx) = v;
            } else {
                s_real<T, TX>(s0, j, tx) = v;
                s_real<T, TX>(s0, M - 1 - j, tx) = (p.r2r == R2R_DST2) ? -v : v;
            }
        }
    }
    if (!(p.r2r != R2R_NONE && MODE == 1)) __syncthreads();

    // ------------------------------------------------------------------ forward transform
    if constexpr (MODE != 1) {
        for (int c = 0; c < nfield_in; ++c) tile_fft_fwd<T, L, TX, NT>(s0 + c * TILE, p.tw, p.LT);
    }

    // ------------------------------------------------------------------ complex pencils
    if (p.r2r == R2R_NONE) {
        if constexpr (MODE == 0) {
            C* gout = reinterpret_cast<C*>(p.out) + fz * p.out_cs + ib * p.out_bs + x0;
            for (int idx = threadIdx.x; idx < TILE; idx += NT) {
                const int tx = idx % TX, pos = idx / TX;
                const int k = k_of_pos<L>(pos);
                if (k < p.n_out && xok) gout[k * p.out_ps + tx] = s0[idx];
            }
            return;
        }
        if constexpr (MODE == 2) {
            const int kx = min(x0 + tx_, p.nx - 1);
            if (!curl) {
                const bool lap = (p.outk == OUT_LAP);
                const T qx = __ldg(p.kap_x + kx), qy = __ldg(p.kap_b + ib);
                for (int idx = threadIdx.x; idx < TILE; idx += NT) {
                    const int kp = k_of_pos<L>(idx / TX);
                    T m = s_multiplier(p, kx, ib, kp);
                    if (lap) {
                        // NABLA = DIV of GRAD: (i kappa)^2 summed over the axes
                        const T qz = __ldg(p.kap_p + kp);
                        m *= -(qx * qx + qy * qy + qz * qz);
                    }
                    s0[idx] = cscale(s0[idx], m);
                }
            } else if (div) {
                const T qx = __ldg(p.kap_x + kx), qy = __ldg(p.kap_b + ib);
                for (int idx = threadIdx.x; idx < TILE; idx += NT) {
                    const int kp = k_of_pos<L>(idx / TX);
                    const T m = s_multiplier(p, kx, ib, kp);
                    const T qz = __ldg(p.kap_p + kp);
                    const C a = s0[idx], b = s0[TILE + idx], c = s0[2 * TILE + idx];
                    // div psi = i kappa . psi
                    s0[idx] = cmuli(mk<T>(m * (qx * a.x + qy * b.x + qz * c.x), m * (qx * a.y + qy * b.y + qz * c.y)));
                }
            } else {
                const T qx = __ldg(p.kap_x + kx), qy = __ldg(p.kap_b + ib);
                for (int idx = threadIdx.x; idx < TILE; idx += NT) {
                    const int kp = k_of_pos<L>(idx / TX);
                    const T m = s_multiplier(p, kx, ib, kp);
                    const T qz = __ldg(p.kap_p + kp);
                    const C a = cscale(s0[idx], m), b = cscale(s0[TILE + idx], m), c = cscale(s0[2 * TILE + idx], m);
                    // u = i kappa x psi
                    s0[idx] = cmuli(mk<T>(qy * c.x - qz * b.x, qy * c.y - qz * b.y));
                    s0[TILE + idx] = cmuli(mk<T>(qz * a.x - qx * c.x, qz * a.y - qx * c.y));
                    s0[2 * TILE + idx] = cmuli(mk<T>(qx * b.x - qy * a.x, qx * b.y - qy * a.y));
                }
            }
            __syncthreads();
        }
        if constexpr (MODE != 0) {
            const int nd = (MODE == 2 && p.outk == OUT_GRAD) ? p.pencil_axis + 1 : 0;
            const int nfield_out = div ? 1 : (curl ? 3 : 1 + nd);
            // gradient fields first (they are derived from buffer 0 into buffer 1), psi last
            for (int f = nfield_out - 1; f >= 0; --f) {
                C* s = s0;
                if (curl) s = s0 + f * TILE;
                if (MODE == 2 && !curl && f > 0) {
                    s = s0 + TILE;
                    const int a = f - 1;          // axis of the derivative
                    const int kx = min(x0 + tx_, p.nx - 1);
                    for (int idx = threadIdx.x; idx < TILE; idx += NT) {
                        T q;
                        if (a == 0) q = __ldg(p.kap_x + kx);
                        else if (a == p.pencil_axis) q = __ldg(p.kap_p + k_of_pos<L>(idx / TX));
                        else q = __ldg(p.kap_b + ib);
                        s[idx] = cmuli(cscale(s0[idx], q));
                    }
                    __syncthreads();
                }
                tile_fft_inv<T, L, TX, NT>(s, p.tw, p.LT);
                C* gout = reinterpret_cast<C*>(p.out) + (fz + f) * p.out_cs + ib * p.out_bs + x0;
                for (int idx = threadIdx.x; idx < p.n_out * TX; idx += NT) {
                    const int tx = idx % TX, j = idx / TX;
                    if (xok) gout[j * p.out_ps + tx] = s[idx];
                }
                if (f > 0 && !curl) __syncthreads(); // buffer 1 is reused by the next field
            }
        }
        return;
    }

    // ------------------------------------------------------------------ real pencils (DST / DCT)
    // Pair (k, L-k) of the packed transform Z is turned into the real-transform outputs, multiplied,
    // turned back and stored in the same two slots: no other thread touches them.  Slot k of the
    // half-spectrum X[0..L] of the extended sequence holds stored row k - sh:
    //   DST-I   Y[k-1] = -Im X[k],            1 <= k <= L-1        DST-II  Y[k-1] = -Im(ptw[k] X[k]),  1 <= k <= L
    //   DCT-II  Y[k]   = Re(ptw[k] X[k]),     0 <= k <= L-1        DCT-I   Y[k]   = Re X[k],           0 <= k <= L
    {
        constexpr int M = 2 * L;
        const int n = p.n_in;
        const int tws = p.LT / M;
        const T* yin = reinterpret_cast<const T*>(p.in) + fz * p.in_cs + ib * p.in_bs + x0;
        T* yout = reinterpret_cast<T*>(p.out) + fz * p.out_cs + ib * p.out_bs + x0;
        const int kx = min(x0 + tx_, p.nx - 1);
        const bool sine = (p.r2r == R2R_DST1 || p.r2r == R2R_DST2);
        const bool shifted = (p.r2r == R2R_DCT || p.r2r == R2R_DST2);     // outputs carry the half-sample phase ptw
        const int sh = sine ? 1 : 0;
        const bool has0 = !sine, hasL = (p.r2r == R2R_DST2 || p.r2r == R2R_DCT1);
        for (int idx = threadIdx.x; idx < (L / 2 + 1) * TX; idx += NT) {
            const int tx = idx % TX, k = idx / TX;
            const int km = L - k;
            const int ik = k - sh, im = km - sh;                          // stored row of slot k / slot L-k
            const bool vk = (k >= 1) || has0, vm = (k >= 1) || hasL;
            T yk = 0, ym = 0;
            C wk = mk<T>(1, 0), wm = mk<T>(1, 0);
            if (shifted) {
                wk = __ldg(p.ptw + k);
                wm = __ldg(p.ptw + km);
            }
            const C w = __ldg(p.tw + k * tws);
            if constexpr (MODE != 1) {
                C xk, xm;
                if (k == 0) {
                    const C z0 = s0[tx];
                    xk = mk<T>(z0.x + z0.y, 0);
                    xm = mk<T>(z0.x - z0.y, 0);
                } else {
                    const C zk = s0[pos_of_k<L>(k) * TX + tx], zm = s0[pos_of_k<L>(km) * TX + tx];
                    const C e = mk<T>(zk.x + zm.x, zk.y - zm.y);
                    const C d = mk<T>(zk.x - zm.x, zk.y + zm.y);
                    const C wd = cmul(w, d);
                    xk = mk<T>((T)0.5 * (e.x + wd.y), (T)0.5 * (e.y - wd.x));
                    xm = mk<T>((T)0.5 * (e.x - wd.y), (T)0.5 * (-e.y - wd.x));
                }
                if (sine) { yk = -(wk.x * xk.y + wk.y * xk.x); ym = -(wm.x * xm.y + wm.y * xm.x); }   // -Im(w X)
                else { yk = wk.x * xk.x - wk.y * xk.y; ym = wm.x * xm.x - wm.y * xm.y; }              //  Re(w X)
            } else {
                if (xok && vk) yk = yin[ik * p.in_ps + tx];
                if (xok && vm && km != k) ym = yin[im * p.in_ps + tx];
                if (km == k) ym = yk;
            }
            if constexpr (MODE == 0) {
                if (xok && vk) yout[ik * p.out_ps + tx] = yk;
                if (xok && vm && km != k) yout[im * p.out_ps + tx] = ym;
                continue;
            }
            if constexpr (MODE == 2) {
                if (vk) yk *= s_multiplier(p, kx, ib, ik);
                if (vm) ym *= s_multiplier(p, kx, ib, im);
            }
            // back to the packed spectrum: X'[k], X'[L-k] -> Z'[k], Z'[L-k]; slots that hold no row are zero
            if (!vk) yk = (T)0;
            if (!vm) ym = (T)0;
            C xk, xm;
            if (sine) { xk = mk<T>(-wk.y * yk, -wk.x * yk); xm = mk<T>(-wm.y * ym, -wm.x * ym); }     // -i conj(w) Y
            else { xk = mk<T>(wk.x * yk, -wk.y * yk); xm = mk<T>(wm.x * ym, -wm.y * ym); }            //    conj(w) Y
            // d/dx of the series: X'[k] -> i kappa_k X'[k] (a sine series becomes a cosine series and back)
            const bool dgrad = (MODE == 2 && p.outk == OUT_GRAD);
            const bool dthis = (MODE == 1 && p.dfield1 == (int)blockIdx.z + 1);
            if (dgrad || dthis) {
                const T qk = __ldg(p.kap_ext + k), qm = __ldg(p.kap_ext + km);
                const C dk = mk<T>(-qk * xk.y, qk * xk.x), dm = mk<T>(-qm * xm.y, qm * xm.x);
                if (dthis) { xk = dk; xm = dm; }
                else {
                    const C e = mk<T>(dk.x + dm.x, dk.y - dm.y);
                    const C d = mk<T>(dk.x - dm.x, dk.y + dm.y);
                    const C wd = cmulc(d, w);
                    s0[TILE + pos_of_k<L>(k) * TX + tx] = mk<T>(e.x - wd.y, e.y + wd.x);
                    if (k > 0) s0[TILE + pos_of_k<L>(km) * TX + tx] = mk<T>(e.x + wd.y, -e.y + wd.x);
                }
            }
            const C e = mk<T>(xk.x + xm.x, xk.y - xm.y);
            const C d = mk<T>(xk.x - xm.x, xk.y + xm.y);
            const C wd = cmulc(d, w);
            s0[pos_of_k<L>(k) * TX + tx] = mk<T>(e.x - wd.y, e.y + wd.x);
            if (k > 0) s0[pos_of_k<L>(km) * TX + tx] = mk<T>(e.x + wd.y, -e.y + wd.x);
        }
        if constexpr (MODE == 0) return;
        __syncthreads();
        tile_fft_inv<T, L, TX, NT>(s0, p.tw, p.LT);
        const bool grad = (MODE == 2 && p.outk == OUT_GRAD);
        if (grad) tile_fft_inv<T, L, TX, NT>(s0 + TILE, p.tw, p.LT);
        // extract the stored unknowns:  DST-I: x_j = x~[j+1];  the others: x_j = x~[j].  Gradient: the
        // field differentiated along this axis takes the second buffer, psi and the other derivative
        // fields (differentiated by the later passes) the first
        const int nfo = grad ? p.pencil_axis + 2 : 1;
        for (int f = 0; f < nfo; ++f) {
            const C* sb = (grad && f == p.pencil_axis + 1) ? s0 + TILE : s0;
            T* yo = yout + f * p.out_cs;
            for (int idx = threadIdx.x; idx < n * TX; idx += NT) {
                const int tx = idx % TX, j = idx / TX;
                if (xok) yo[j * p.out_ps + tx] = s_real<T, TX>(const_cast<C*>(sb), (p.r2r == R2R_DST1) ? j + 1 : j, tx);
            }
        }
    }
}

} // namespace sf
