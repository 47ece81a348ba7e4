// sf_xpass.cuh -- steps S1 (X forward) and S5 (X backward) of the hot path: the stride-1 real
// transforms along x (PAPER.md:87 R2C half-spectrum; PAPER.md:89-97 pencils; Table 1).
//
// One CTA owns ROWS contiguous-in-memory rows.  A real row of (extended) length M = 2L is packed
// as L complex numbers z[n] = x[2n] + i x[2n+1], transformed with a self-sorting (Stockham)
// mixed-radix FFT in shared memory, and split into the half-spectrum X[0..L]; the backward kernel
// is the exact mirror (merge, inverse FFT, unpack).  What differs between boundary conditions is
// only the rule that extends the stored row to length M on load and the rule that extracts the
// stored unknowns on store -- both are fused into the load / store loops (north_star items 4, 5):
//   X_PERIODIC  M = n            x~ = x
//   X_ZEROPAD   M = 2n           x~ = x, 0                      (Hockney-Eastwood)
//   X_DST1      M = 2(n+1)       x~ = 0, x, 0, -reverse(x)      DST-I:  Y_k = -Im X~[k+1]
//   X_DCT2      M = 2n           x~ = x, reverse(x)             DCT-II: Y_k = Re(e^{-i pi k/2n} X~[k])
//   X_DST2      M = 2n           x~ = x, -reverse(x)            DST-II: Y_k = -Im(e^{-i pi (k+1)/2n} X~[k+1])
//   X_DCT1      M = 2(n-1)       x~ = x_0..x_{n-1}, x_{n-2}..x_1  DCT-I:  Y_k = Re X~[k]
// and backward: DST-I again / DCT-III / DST-III / DCT-I again through the complex-to-real path.
// Inhomogeneous boundary values are folded into the source as it is loaded.
#pragma once
#include "sf_common.cuh"

namespace sf {

enum { X_PERIODIC = 0, X_ZEROPAD = 1, X_DST1 = 2, X_DCT2 = 3, X_DST2 = 4, X_DCT1 = 5 };

template <typename T> struct XParams {
    typedef SF_CX C;
    const T* real_in;   // forward: source rows (dense or pitched reals)
    T* real_out;        // backward: result rows; forward R2R: transformed rows
    const void* spec_in; // backward: half-spectrum rows (complex) or R2R rows (real)
    void* spec_out;      // forward: half-spectrum rows (complex)
    long long rin_py, rin_pz, rin_pc;   // real-side pitches in elements: row (y), plane (z), component
    long long sp_py, sp_pz, sp_pc;      // spectrum-side pitches in elements of its own type
    int n;              // stored reals per row
    int ny, nz;         // rows = ny * nz per component
    int mode;           // X_*
    int LT;             // length of tw
    const C* tw;        // exp(-2 pi i j / LT), LT = M
    const C* ptw;       // X_DCT2, X_DST2: exp(-i pi k / (2n)), k <= n
    // boundary-value folding (forward only): face[2*axis+side], weight w[2*axis+side]; NULL = none
    const T* face[6];
    T wface[6];
    int has_faces;
    // periodic / zero-padded: optional side array [field][row] that holds the last column (k = L, the Nyquist
    // coefficient) of every row instead of the spectrum array (sf_fastper.cuh)
    void* nyq_side;
    int nyq_side_yz;    // 0: [field][row = iz * ny + iy];  1: transposed, [iy][iz] (single field)
    // backward, real modes: spectral derivative along x of one field (sine <-> cosine series, eq. (10))
    int dfield1;        // 1 + index of the field (blockIdx.y) that is differentiated; 0: none
    const T* kap_ext;   // pi k / L_domain for slot k <= L of the extended sequence, zero at k = L
};

// rows per CTA: two Stockham buffers of ROWS x LP complex; prefer a footprint that lets several CTAs
// share an SM, never exceed the 227 KB a CTA may use
__host__ __device__ constexpr int x_bytes(int rows, int L, int csize) { return 2 * rows * (L + 16) * csize; }
template <typename T, int L> __host__ __device__ constexpr int x_rows()
{
    constexpr int cs = 2 * (int)sizeof(T);
    if (x_bytes(16, L, cs) <= 72 * 1024) return 16;
    if (x_bytes(8, L, cs) <= 72 * 1024) return 8;
    if (x_bytes(4, L, cs) <= 72 * 1024) return 4;
    if (x_bytes(2, L, cs) <= 136 * 1024) return 2;
    return 1;
}
// row pitch in complex elements: with P = 128 B / sizeof(complex) lanes served per shared-memory
// phase and lanes running over rows first, LP = P / ROWS (mod P) puts them on distinct banks
template <typename T, int L> __host__ __device__ constexpr int x_lp()
{
    constexpr int P = 128 / (2 * (int)sizeof(T));
    constexpr int R = x_rows<T, L>();
    return L + ((P / R) > 1 ? (P / R) : 1);
}

// value of the (folded) source at (ix, iy, iz)
// (only the two x faces depend on the position in the row; whether the row lies in a y / z boundary layer is the
// same for all its elements and is tested first)
template <typename T> __device__ __forceinline__ T x_face_term(const XParams<T>& p, int ix, int iy, int iz)
{
    T v = (T)0;
    if (ix == 0 && p.face[0]) v += p.wface[0] * p.face[0][iy + (long long)p.ny * iz];
    if (ix == p.n - 1 && p.face[1]) v += p.wface[1] * p.face[1][iy + (long long)p.ny * iz];
    if (iy == 0 || iy == p.ny - 1 || iz == 0 || iz == p.nz - 1) {
        if (iy == 0 && p.face[2]) v += p.wface[2] * p.face[2][ix + (long long)p.n * iz];
        if (iy == p.ny - 1 && p.face[3]) v += p.wface[3] * p.face[3][ix + (long long)p.n * iz];
        if (iz == 0 && p.face[4]) v += p.wface[4] * p.face[4][ix + (long long)p.n * iy];
        if (iz == p.nz - 1 && p.face[5]) v += p.wface[5] * p.face[5][ix + (long long)p.n * iy];
    }
    return v;
}
template <typename T> __device__ __forceinline__ T x_src(const XParams<T>& p, const T* row, int ix, int iy, int iz)
{
    T v = row[ix];
    if (p.has_faces) v += x_face_term(p, ix, iy, iz);
    return v;
}

// extended sequence x~[m], m < 2L
template <typename T> __device__ __forceinline__ T x_ext(const XParams<T>& p, const T* row, int m, int M, int iy, int iz)
{
    const int n = p.n;
    switch (p.mode) {
    case X_PERIODIC: return x_src(p, row, m, iy, iz);
    case X_ZEROPAD: return m < n ? x_src(p, row, m, iy, iz) : (T)0;
    case X_DST1:
        if (m == 0 || m == n + 1) return (T)0;
        return m <= n ? x_src(p, row, m - 1, iy, iz) : -x_src(p, row, M - m - 1, iy, iz);
    case X_DST2: return m < n ? x_src(p, row, m, iy, iz) : -x_src(p, row, M - 1 - m, iy, iz);
    case X_DCT1: return m < n ? x_src(p, row, m, iy, iz) : x_src(p, row, M - m, iy, iz);
    default: /* X_DCT2 */ return m < n ? x_src(p, row, m, iy, iz) : x_src(p, row, M - 1 - m, iy, iz);
    }
}

// ------------------------------------------------------------------------------------ S1
template <typename T, int L, int NT>
__global__ void __launch_bounds__(NT) xfwd_kernel(const XParams<T> p)
{
    typedef SF_CX C;
    constexpr int ROWS = x_rows<T, L>();
    constexpr int LP = x_lp<T, L>();
    constexpr int M = 2 * L;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* A = reinterpret_cast<C*>(smem_raw);
    C* B = A + ROWS * LP;

    const int comp = blockIdx.y;
    const long long row0 = (long long)blockIdx.x * ROWS;
    const long long nrows = (long long)p.ny * p.nz;
    const T* rin = p.real_in + comp * p.rin_pc;
    // row geometry once per row (the 64-bit divisions and pitch products do not belong in the element loops)
    __shared__ int s_iy[16], s_iz[16];
    __shared__ long long s_rin[16], s_sp[16];
    if (threadIdx.x < ROWS) {
        const long long row = row0 + threadIdx.x;
        const int iy = (int)(row % p.ny), iz = (int)(row / p.ny);
        s_iy[threadIdx.x] = (row < nrows) ? iy : -1;
        s_iz[threadIdx.x] = iz;
        s_rin[threadIdx.x] = iy * p.rin_py + iz * p.rin_pz;
        s_sp[threadIdx.x] = iy * p.sp_py + iz * p.sp_pz;
    }
    __syncthreads();

    // load + extend + fold (position index fastest: coalesced)
    const bool fast = (p.mode == X_PERIODIC || p.mode == X_ZEROPAD) && !p.has_faces;
    for (int idx = threadIdx.x; idx < ROWS * L; idx += NT) {
        const int r = idx / L, j = idx % L;
        C z = mk<T>(0, 0);
        const int iy = s_iy[r];
        if (iy >= 0) {
            const int iz = s_iz[r];
            const T* rp = rin + s_rin[r];
            if (fast) {
                if (2 * j < p.n) z = *reinterpret_cast<const C*>(rp + 2 * j);
            } else {
                z.x = x_ext(p, rp, 2 * j, M, iy, iz);
                z.y = x_ext(p, rp, 2 * j + 1, M, iy, iz);
            }
        }
        A[r * LP + j] = z;
    }
    __syncthreads();

    C* F = stockham_fft<T, L, ROWS, LP, NT, false>(A, B, p.tw, p.LT);
    C* G = (F == A) ? B : A;

    // split Z -> X (rows across lanes: conflict-free), out of place F -> G
    //   X[k] = ( (Z[k] + conj Z[L-k]) - i w_M^k (Z[k] - conj Z[L-k]) ) / 2,  Z[L] = Z[0]
    const int tws = p.LT / M;
    for (int idx = threadIdx.x; idx < ROWS * (L / 2 + 1); idx += NT) {
        const int r = idx % ROWS, k = idx / ROWS;
        const C* f = F + r * LP;
        C* g = G + r * LP;
        if (k == 0) {
            const C z0 = f[0];
            g[0] = mk<T>(z0.x + z0.y, 0);
            g[L] = mk<T>(z0.x - z0.y, 0);
        } else {
            const C zk = f[k], zm = f[L - k];
            const C w = __ldg(p.tw + k * tws);
            // k
            C e = mk<T>(zk.x + zm.x, zk.y - zm.y);          // Z[k] + conj Z[L-k]
            C d = mk<T>(zk.x - zm.x, zk.y + zm.y);          // Z[k] - conj Z[L-k]
            C wd = cmul(w, d);                               // w^k d
            g[k] = mk<T>((T)0.5 * (e.x + wd.y), (T)0.5 * (e.y - wd.x));   // e - i wd
            // L-k : w^(L-k) = -conj(w^k);  e' = conj(e), d' = -conj(d)  =>  w' d' = conj(w d)
            g[L - k] = mk<T>((T)0.5 * (e.x - wd.y), (T)0.5 * (-e.y - wd.x)); // conj(e) - i conj(wd)
        }
    }
    __syncthreads();

    // store
    if (p.mode == X_PERIODIC || p.mode == X_ZEROPAD) {
        constexpr int H = L + 1;
        C* so = reinterpret_cast<C*>(p.spec_out) + comp * p.sp_pc;
        for (int idx = threadIdx.x; idx < ROWS * H; idx += NT) {
            const int r = idx / H, k = idx % H;
            const int iy = s_iy[r];
            if (iy >= 0) {
                if (k == L && p.nyq_side) reinterpret_cast<C*>(p.nyq_side)[p.nyq_side_yz ? (long long)iy * p.nz + s_iz[r] : comp * nrows + row0 + r] = G[r * LP + k];
                else so[s_sp[r] + k] = G[r * LP + k];
            }
        }
    } else {
        T* ro = p.real_out + comp * p.sp_pc;
        const int n = p.n;
        // a warp per row, lanes along the row (n is a run-time number: no division per element)
        for (int r = threadIdx.x >> 5; r < ROWS; r += NT / 32)
        for (int k = threadIdx.x & 31; k < n; k += 32) {
            if (s_iy[r] >= 0) {
                T y;
                if (p.mode == X_DST1) {
                    y = -G[r * LP + k + 1].y;
                } else if (p.mode == X_DCT1) {
                    y = G[r * LP + k].x;
                } else if (p.mode == X_DST2) {
                    const C w = __ldg(p.ptw + k + 1);
                    const C x = G[r * LP + k + 1];
                    y = -(w.x * x.y + w.y * x.x);
                } else {
                    const C w = __ldg(p.ptw + k);
                    const C x = G[r * LP + k];
                    y = w.x * x.x - w.y * x.y;
                }
                ro[s_sp[r] + k] = y;
            }
        }
    }
}

// ------------------------------------------------------------------------------------ S5
template <typename T, int L, int NT>
__global__ void __launch_bounds__(NT) xinv_kernel(const XParams<T> p)
{
    typedef SF_CX C;
    constexpr int ROWS = x_rows<T, L>();
    constexpr int LP = x_lp<T, L>();
    constexpr int M = 2 * L;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* A = reinterpret_cast<C*>(smem_raw);
    C* B = A + ROWS * LP;

    const int comp = blockIdx.y;
    const long long row0 = (long long)blockIdx.x * ROWS;
    const long long nrows = (long long)p.ny * p.nz;

    // row geometry once per row
    __shared__ int s_iy[16], s_iz[16];
    __shared__ long long s_rin[16], s_sp[16];
    if (threadIdx.x < ROWS) {
        const long long row = row0 + threadIdx.x;
        const int iy = (int)(row % p.ny), iz = (int)(row / p.ny);
        s_iy[threadIdx.x] = (row < nrows) ? iy : -1;
        s_iz[threadIdx.x] = iz;
        s_rin[threadIdx.x] = iy * p.rin_py + iz * p.rin_pz;
        s_sp[threadIdx.x] = iy * p.sp_py + iz * p.sp_pz;
    }
    __syncthreads();
    // load the half-spectrum X[0..L] (natural order) into A
    if (p.mode == X_PERIODIC || p.mode == X_ZEROPAD) {
        constexpr int H = L + 1;
        const C* si = reinterpret_cast<const C*>(p.spec_in) + comp * p.sp_pc;
        for (int idx = threadIdx.x; idx < ROWS * H; idx += NT) {
            const int r = idx / H, k = idx % H;
            C x = mk<T>(0, 0);
            const int iy = s_iy[r];
            if (iy >= 0) {
                if (k == L && p.nyq_side) x = reinterpret_cast<const C*>(p.nyq_side)[p.nyq_side_yz ? (long long)iy * p.nz + s_iz[r] : comp * nrows + row0 + r];
                else x = si[s_sp[r] + k];
            }
            A[r * LP + k] = x;
        }
    } else {
        const T* ri = reinterpret_cast<const T*>(p.spec_in) + comp * p.sp_pc;
        const int n = p.n;
        for (int idx = threadIdx.x; idx < ROWS * (L + 1); idx += NT) {
            const int r = idx / (L + 1), k = idx % (L + 1);
            C x = mk<T>(0, 0);
            if (s_iy[r] >= 0) {
                const T* rp = ri + s_sp[r];
                if (p.mode == X_DST1) {
                    if (k >= 1 && k <= n) x = mk<T>(0, -rp[k - 1]);       // X~[k] = -i Y[k-1]
                } else if (p.mode == X_DCT1) {
                    if (k < n) x = mk<T>(rp[k], 0);                        // X~[k] = Y[k]
                } else if (p.mode == X_DST2) {
                    if (k >= 1 && k <= n) {                                // X~[k] = -i e^{+i pi k/2n} Y[k-1]
                        const C w = __ldg(p.ptw + k);
                        const T y = rp[k - 1];
                        x = mk<T>(-w.y * y, -w.x * y);
                    }
                } else {
                    if (k < n) {                                             // X~[k] = e^{+i pi k/2n} Y[k]
                        const C w = __ldg(p.ptw + k);
                        const T y = rp[k];
                        x = mk<T>(w.x * y, -w.y * y);
                    }
                }
                if (p.dfield1 == comp + 1) {                                // X~[k] -> i kappa_k X~[k]
                    const T q = __ldg(p.kap_ext + k);
                    x = mk<T>(-q * x.y, q * x.x);
                }
            }
            A[r * LP + k] = x;
        }
    }
    __syncthreads();

    // merge X -> Z (rows across lanes), out of place A -> B
    //   Z[k] = (X[k] + conj X[L-k]) + i conj(w_M^k) (X[k] - conj X[L-k]),  k < L
    const int tws = p.LT / M;
    for (int idx = threadIdx.x; idx < ROWS * (L / 2 + 1); idx += NT) {
        const int r = idx % ROWS, k = idx / ROWS;
        const C* a = A + r * LP;
        C* b = B + r * LP;
        const C xk = a[k], xm = a[L - k];
        const C w = __ldg(p.tw + k * tws);
        C e = mk<T>(xk.x + xm.x, xk.y - xm.y);          // X[k] + conj X[L-k]
        C d = mk<T>(xk.x - xm.x, xk.y + xm.y);          // X[k] - conj X[L-k]
        C wd = cmulc(d, w);                              // conj(w^k) d
        b[k] = mk<T>(e.x - wd.y, e.y + wd.x);            // e + i wd
        // L-k: e' = conj(e), d' = -conj(d), conj(w^(L-k)) = -w^k  =>  conj(w') d' = conj(conj(w) d)
        if (k > 0) b[L - k] = mk<T>(e.x + wd.y, -e.y + wd.x);   // conj(e) + i conj(wd)
    }
    __syncthreads();

    C* F = stockham_fft<T, L, ROWS, LP, NT, true>(B, A, p.tw, p.LT);

    // unpack + extract + store
    T* ro = p.real_out + comp * p.rin_pc;
    const int n = p.n;
    if (p.mode == X_PERIODIC || p.mode == X_ZEROPAD || p.mode == X_DCT2 || p.mode == X_DST2) {
        const int nc = n / 2; // stored reals are x~[0..n): the first n/2 packed complex values
        for (int r = threadIdx.x >> 5; r < ROWS; r += NT / 32)
        for (int j = threadIdx.x & 31; j < nc; j += 32) {
            if (s_iy[r] >= 0) *reinterpret_cast<C*>(ro + s_rin[r] + 2 * j) = F[r * LP + j];
        }
    } else { // X_DST1: x_j = x~[j+1];  X_DCT1 (n odd): x_j = x~[j]
        for (int r = threadIdx.x >> 5; r < ROWS; r += NT / 32)
        for (int j = threadIdx.x & 31; j < n; j += 32) {
            if (s_iy[r] >= 0) {
                const int m = (p.mode == X_DST1) ? j + 1 : j;
                const C z = F[r * LP + (m >> 1)];
                ro[s_rin[r] + j] = (m & 1) ? z.y : z.x;
            }
        }
    }
}

} // namespace sf
