// sf_api.cu -- the C ABI of include/sailffish.h: plan construction (tables, Green's spectrum,
// workspaces) and the five-launch solve sequence S1..S5.
// Host code plus the two small plan-time kernels (Green's function evaluation, compact-table
// extraction).  No CPU fallback exists anywhere: every step of the path is a CUDA kernel.
#include "../../include/sailffish.h"
#include "sf_fast_api.h"
#include "sf_launch.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <type_traits>
#include <utility>
#include <vector>

using namespace sf;

namespace {

thread_local std::string g_create_error = "";

constexpr int kMaxFields = 4;
constexpr long double PI_L = 3.14159265358979323846264338327950288L;

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
};

} // namespace

struct sf_plan_s {
    int ndim = 3;
    long long n[3] = { 1, 1, 1 };
    double h[3] = { 1, 1, 1 };
    sf_bc bc = SF_BC_PERIODIC;
    sf_grid grid = SF_GRID_CELL_CENTRE;
    sf_bc bca[3] = { SF_BC_PERIODIC, SF_BC_PERIODIC, SF_BC_PERIODIC };   // per axis (Dirichlet / Neumann may be mixed)
    bool mixed = false;
    int r2ra[3] = { 0, 0, 0 };   // R2R_* of the pass along each axis
    sf_operator op = SF_OP_PSEUDO_SPECTRAL;
    sf_precision prec = SF_F32;
    int ncomp = 1;
    cudaStream_t stream = nullptr;
    double rhs_sign = 1.0, eps_over_h = 2.0;
    size_t esize = 4;

    // transform geometry
    int xmode = X_PERIODIC, r2r = R2R_NONE;
    int Lx = 0;          // complex length of the packed x rows
    int Mx = 0;          // real transform length along x
    int La[3] = { 0, 0, 0 }; // complex FFT length of the strided passes along y, z (index 1, 2)
    int P[3] = { 1, 1, 1 };  // transform length per axis as seen by the multiplier (index folding)
    int nspec_x = 0;     // valid spectral columns (H = Lx + 1 complex, or n0 reals)
    long long pitch = 0; // padded column count of the work arrays
    int nfields = 1;     // fields the workspaces can hold
    long long w1_field = 0, w2_field = 0; // elements per field in W1 ([n2][n1][pitch]) / W2 ([n2][P1][pitch])
    bool padded = false; // unbounded: W2 differs from W1

    // device memory
    std::vector<void*> allocs;
    long long dev_bytes = 0;
    void* W1 = nullptr;
    void* W2 = nullptr;
    void* out = nullptr;       // nfields dense real fields
    // scalar unbounded plans: a second, four-field set of work / output arrays, allocated by the first
    // sf_gradient (the solve path keeps its single-field arrays and their tensor maps)
    void *gW1 = nullptr, *gW2 = nullptr, *gout = nullptr;
    void* out_last = nullptr;  // array the last compute call wrote its fields to
    void* tw[3] = { nullptr, nullptr, nullptr };
    void* ptw[3] = { nullptr, nullptr, nullptr };
    void* lam[3] = { nullptr, nullptr, nullptr };
    void* kap[3] = { nullptr, nullptr, nullptr };
    void* kap_ext[3] = { nullptr, nullptr, nullptr };   // Dirichlet / Neumann: pi k / L_domain per slot k <= L of the extended sequence
    void* zero1 = nullptr;
    int LT[3] = { 0, 0, 0 };
    void* green = nullptr;
    void* green_tiles = nullptr;   // fast path: the same table, tile-major (sf_fast_api.h)
    void* sched = nullptr;         // fast path: the dynamic tile counter of the strided kernels
    void *nyqA = nullptr, *nyqB = nullptr;   // fast path with fast X passes: the Nyquist column as [y][z] and [z][ky]
    double scale = 1.0;
    // kernel generation 2 (sf_fast.cuh): fp32 unbounded plans with 256-long y and z pencils
    bool fast = false;
    bool fast_x = false;   // S1 / S5 too (x extent 256)
    sf2::TileMap map_s2, map_s3, map_s4;
    // ... and with 512-long y and z pencils (sf_fast512.cuh), scalar or three components (sf_solve, sf_curl)
    bool fast5 = false;
    bool fast5_x = false;  // S1 / S5 too (x extent 512)
    // ... and in double precision with 256-long y and z pencils (sf_fast64.cuh), scalar
    bool fast64 = false;
    bool r2r64 = false;    // fp64 Dirichlet (DST-I, 255) / Neumann (DCT, 256) strided passes (sf_fastr2r64.cuh)
    bool xp64 = false;     // fp64 periodic X passes for rows of 256 reals (sf_fastx64.cuh)
    bool xg64 = false;     // fp64 X passes with complex length 256: zero-padded 256, DST-I 255, DCT-II / III 256 (sf_fastx64.cuh)

    // per-solve state
    const void* src = nullptr;
    void* src_own = nullptr;
    const void* face[6] = { nullptr, nullptr, nullptr, nullptr, nullptr, nullptr };
    void* face_own[6] = { nullptr, nullptr, nullptr, nullptr, nullptr, nullptr };
    int last_kind = -1; // OUT_* of the last compute call
    int launches = 0;
    int tslots = 0;               // step timing: compute calls remembered (0 = off)
    long long tcount = 0;         // compute calls recorded since timing was enabled
    int tstride = 1;              // record every tstride-th compute call
    bool fastper = false;         // periodic fp32 plans with 256-point y / z pencils: generation-2 strided passes
    bool fastper_x = false;       // ... and rows of 256 reals: generation-2 X passes
    bool fastper64 = false;       // the same strided passes in double precision (sf_fastper64.cuh)
    long long tcalls = 0;         // compute calls seen since timing was enabled
    std::vector<cudaEvent_t> ev;  // 6 events per slot
    // copy pipeline (sf_set_pipeline): host copies on streams of their own, two source and two result buffers
    int pipe = 1;
    int ss = 0, os = 0;           // slot of the last host source / of the last result
    bool src_piped = false;       // plan->src is psrc[ss], filled on st_h2d
    cudaStream_t st_h2d = nullptr, st_d2h = nullptr;
    void* psrc[2] = { nullptr, nullptr };
    void* pout[2] = { nullptr, nullptr };
    cudaEvent_t ev_src_ready[2] = { nullptr, nullptr }, ev_src_free[2] = { nullptr, nullptr };
    cudaEvent_t ev_done[2] = { nullptr, nullptr }, ev_out_free[2] = { nullptr, nullptr };
    bool src_free_set[2] = { false, false }, out_free_set[2] = { false, false }, done_set[2] = { false, false };
    std::string err = "";
};

namespace {

sf_status fail(sf_plan p, sf_status st, const std::string& msg)
{
    if (p) p->err = msg;
    else g_create_error = msg;
    return st;
}

sf_status dev_alloc(sf_plan p, void** out, size_t bytes)
{
    void* d = nullptr;
    cudaError_t e = cudaMalloc(&d, bytes ? bytes : 1);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(p, SF_ERR_ALLOC, std::string("cudaMalloc of ") + std::to_string(bytes) + " bytes failed: " + cudaGetErrorString(e));
    }
    p->allocs.push_back(d);
    p->dev_bytes += (long long)bytes;
    *out = d;
    return SF_OK;
}

void dev_free(sf_plan p, void* d)
{
    for (size_t i = 0; i < p->allocs.size(); ++i)
        if (p->allocs[i] == d) {
            cudaFree(d);
            p->allocs.erase(p->allocs.begin() + i);
            return;
        }
}

bool is_pow2(long long v) { return v >= 1 && (v & (v - 1)) == 0; }
long long round_up(long long v, long long m) { return (v + m - 1) / m * m; }

// exp(-2 pi i j / len), j < len, computed in extended precision and rounded once
template <typename T> sf_status upload_twiddles(sf_plan p, void** dst, int len)
{
    std::vector<T> h((size_t)2 * len);
    for (int j = 0; j < len; ++j) {
        long double a = 2.0L * PI_L * (long double)j / (long double)len;
        h[2 * j] = (T)cosl(a);
        h[2 * j + 1] = (T)(-sinl(a));
    }
    sf_status st = dev_alloc(p, dst, h.size() * sizeof(T));
    if (st != SF_OK) return st;
    if (cudaMemcpy(*dst, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess)
        return fail(p, SF_ERR_CUDA, "twiddle upload failed");
    return SF_OK;
}

// exp(-i pi k / (2 n)), k < n  (quarter-wave shift of the DCT-II / DCT-III)
template <typename T> sf_status upload_dct_shift(sf_plan p, void** dst, int n)
{
    std::vector<T> h((size_t)2 * (n + 1));   // k = 0 .. n (DST-II uses the entry k = n, -i)
    for (int k = 0; k <= n; ++k) {
        long double a = PI_L * (long double)k / (2.0L * (long double)n);
        h[2 * k] = (T)cosl(a);
        h[2 * k + 1] = (T)(-sinl(a));
    }
    sf_status st = dev_alloc(p, dst, h.size() * sizeof(T));
    if (st != SF_OK) return st;
    if (cudaMemcpy(*dst, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess)
        return fail(p, SF_ERR_CUDA, "table upload failed");
    return SF_OK;
}

template <typename T> sf_status upload_real(sf_plan p, void** dst, const std::vector<long double>& v)
{
    std::vector<T> h(v.size());
    for (size_t i = 0; i < v.size(); ++i) h[i] = (T)v[i];
    sf_status st = dev_alloc(p, dst, h.size() * sizeof(T));
    if (st != SF_OK) return st;
    if (cudaMemcpy(*dst, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess)
        return fail(p, SF_ERR_CUDA, "table upload failed");
    return SF_OK;
}

// Per-axis eigenvalue contribution and wavenumber (Table 1; readings A1, A4, A5,
// A20 of DESIGN.md).  count = number of spectral indices stored along the axis.
void axis_tables(const sf_plan_s& pl, int a, int count, std::vector<long double>& lam, std::vector<long double>& kap)
{
    lam.assign(count, 0.0L);
    kap.assign(count, 0.0L);
    const long long n = pl.n[a];
    const long double h = pl.h[a];
    for (int k = 0; k < count; ++k) {
        switch (pl.bca[a]) {
        case SF_BC_PERIODIC: {
            const long double Ld = (long double)n * h;
            const long long m = (2 * k < n) ? k : k - n;
            const long double kappa = 2.0L * PI_L * (long double)m / Ld;
            kap[k] = (2 * k == n) ? 0.0L : kappa;
            if (pl.op == SF_OP_PSEUDO_SPECTRAL) lam[k] = -kappa * kappa;
            else { long double s = sinl(PI_L * (long double)k / (long double)n); lam[k] = -(4.0L / (h * h)) * s * s; }
            break;
        }
        case SF_BC_DIRICHLET: {
            // cell-boundary: n interior nodes, L = (n+1) h (DST-I); cell-centre: n cells, L = n h (DST-II)
            const long double cells = (pl.grid == SF_GRID_CELL_BOUNDARY) ? (long double)(n + 1) : (long double)n;
            const long double Ld = cells * h;
            if (pl.op == SF_OP_PSEUDO_SPECTRAL) { long double kk = PI_L * (long double)(k + 1) / Ld; lam[k] = -kk * kk; }
            else { long double s = sinl(PI_L * (long double)(k + 1) / (2.0L * cells)); lam[k] = -(4.0L / (h * h)) * s * s; }
            break;
        }
        case SF_BC_NEUMANN: {
            // cell-centre: n cells, L = n h (DCT-II); cell-boundary: n nodes, L = (n-1) h (DCT-I)
            const long double cells = (pl.grid == SF_GRID_CELL_CENTRE) ? (long double)n : (long double)(n - 1);
            const long double Ld = cells * h;
            if (pl.op == SF_OP_PSEUDO_SPECTRAL) { long double kk = PI_L * (long double)k / Ld; lam[k] = -kk * kk; }
            else { long double s = sinl(PI_L * (long double)k / (2.0L * cells)); lam[k] = -(4.0L / (h * h)) * s * s; }
            break;
        }
        case SF_BC_UNBOUNDED: {
            const long long P = 2 * n;
            const long long m = (k < n) ? k : k - P;
            kap[k] = (k == n) ? 0.0L : 2.0L * PI_L * (long double)m / ((long double)P * h);
            break;
        }
        }
    }
}

// ---------------------------------------------------------------- plan-time kernels (fp64)
// G on the doubled grid at the mirrored distance min(i, P - i) h (reading A12), times
// the cell volume (reading A11).  Kernels (formulas: DESIGN.md readings A10, A25, A26, A28):
//   order 2      3-D  -erf(r / (sqrt 2 eps)) / (4 pi r)            2-D  (ln r + E_1(r^2 / 2 eps^2) / 2) / (2 pi)
//   order 4..10  G_P = G_2 - sum_{n=1}^{P/2-1} eps^2 / (2 n) L_{n-1}^(alpha)(x) g,  x = r^2 / (2 eps^2), g the unit
//                Gaussian of width eps, alpha = 1/2 in 3-D and 0 in 2-D
//   order 0      the spectrally compact kernel -Si(pi r / h) / (2 pi^2 r), h passed in `eps`
//
// The special functions are evaluated by routes of their own (no expansion shared with the checker):
//   Si(x), x < 50:   the Bessel-function series  Si(x) = x sum_{n>=0} j_n(x/2)^2  (Abramowitz & Stegun 5.2.15), the
//                    spherical Bessel functions by Miller's downward recurrence, normalised with sum (2n+1) j_n^2 = 1
//   Si(x), x >= 50:  Si = pi/2 - f cos x - g sin x with the asymptotic expansions of the auxiliary functions
//                    f ~ (1/x) sum (-1)^k (2k)! / x^2k,  g ~ (1/x^2) sum (-1)^k (2k+1)! / x^2k  (smallest term < 1e-19)
//   E_1(u), u < 50:  E_1 = -gamma - ln u + e^-u sum_{n>=1} H_n u^n / n!  (H_n harmonic numbers; all terms positive, so
//                    the ABSOLUTE error is a few ulp of ln u, which is what (ln r + E_1 / 2) needs)
//   E_1(u), u >= 50: e^-u / u (1 - 1/u + 2/u^2 - ...), below 1e-23
//   Laguerre polynomials by their three-term recurrence (k+1) L_{k+1} = (2k + 1 + alpha - x) L_k - (k + alpha) L_{k-1}
__device__ double sine_integral(double x)
{
    if (x >= 50.0) {
        const double x2 = 1.0 / (x * x);
        double tf = 1.0, tg = 1.0, f = 1.0, g = 1.0;
        for (int k = 1; k < 30; ++k) {
            const double nf = -tf * (2.0 * k) * (2.0 * k - 1.0) * x2, ng = -tg * (2.0 * k + 1.0) * (2.0 * k) * x2;
            if (fabs(nf) >= fabs(tf) || fabs(nf) < 1e-20) break;   // past the smallest term, or converged
            tf = nf; tg = ng;
            f += tf; g += tg;
        }
        double sn, cs;
        sincos(x, &sn, &cs);
        return 1.5707963267948966192 - (f / x) * cs - (g * x2) * sn;
    }
    const double z = 0.5 * x;
    // downward recurrence j_{n-1} = (2n + 1) / z j_n - j_{n+1} from far above the turning point n ~ z
    const int N = (int)z + 40;
    double jp = 0.0, jn = 1e-30, s1 = 0.0, s2 = 0.0;   // j_{n+1}, j_n (unnormalised); sum (2n+1) j_n^2, sum j_n^2
    for (int n = N; n >= 0; --n) {
        s1 += (2.0 * n + 1.0) * jn * jn;
        s2 += jn * jn;
        const double jm = (2.0 * n + 1.0) / z * jn - jp;
        jp = jn; jn = jm;
        if (fabs(jn) > 1e120) {   // rescale: only ratios matter
            jn *= 1e-120; jp *= 1e-120;
            s1 *= 1e-240; s2 *= 1e-240;
        }
    }
    return x * s2 / s1;
}
__device__ double exp_integral1(double u)
{
    if (u >= 50.0) {
        const double iu = 1.0 / u;
        return exp(-u) * iu * (1.0 - iu * (1.0 - 2.0 * iu * (1.0 - 3.0 * iu)));
    }
    double term = 1.0, hn = 0.0, sum = 0.0;
    for (int n = 1; n < 400; ++n) {
        term *= u / (double)n;     // u^n / n!
        hn += 1.0 / (double)n;     // H_n
        const double add = hn * term;
        sum += add;
        if ((double)n > u && add < 1e-17 * sum) break;
    }
    return (-0.57721566490153286061 - log(u)) + exp(-u) * sum;
}
// sum_{n=1}^{P/2-1} L_{n-1}^(alpha)(x) / (2 n)
__device__ double laguerre_tail(int order, double alpha, double x)
{
    double lm = 0.0, lk = 1.0, acc = 0.0;   // L_{k-1}, L_k
    for (int k = 0; k + 1 < order / 2; ++k) {
        acc += lk / (2.0 * (k + 1));
        const double ln = ((2.0 * k + 1.0 + alpha - x) * lk - (k + alpha) * lm) / (k + 1.0);
        lm = lk; lk = ln;
    }
    return acc;
}
// C(x) = int_0^x (1 - J0(t)) / t dt for the 2-D spectrally compact kernel, as a Neumann series: with 1 = J0 + 2 sum J_2k,
// J_2k / t = (J_{2k-1} + J_{2k+1}) / 4k and int_0^x J_m = 2 sum_{j>=0} J_{m+1+2j}(x) the integral collapses to
//     C(x) = sum_{i>=1} (2 H_i - 1/i) J_{2i}(x),   H_i the harmonic numbers,
// the Bessel functions by Miller's downward recurrence J_{n-1} = (2n / x) J_n - J_{n+1}, normalised with J0 + 2 sum J_2k = 1
__device__ double bessel_cin(double x)
{
    if (x < 1e-4) return 0.125 * x * x;                       // (x/2)^2 / 2, next term x^4 / 256
    // start at J_{2M} far above the turning point n ~ x: beyond it J_n(x) falls off like exp(-(2/3) sqrt(2/x) (n - x)^(3/2)),
    // so n - x ~ 14 x^(1/3) + 30 puts the start below 1e-20 of the values that matter
    const int M = ((int)(x + 30.0 + 14.0 * cbrt(x))) / 2 + 1;
    double hi = 0.0;
    for (int i = 1; i <= M; ++i) hi += 1.0 / (double)i;       // H_M
    double jp = 0.0, jn = 1e-30;                              // J_{n+1}, J_n (unnormalised), n = 2 M
    double norm = 0.0, acc = 0.0;
    const double ix = 1.0 / x;
    for (int i = M; i >= 1; --i) {
        // n = 2 i
        norm += 2.0 * jn;
        acc += (2.0 * hi - 1.0 / (double)i) * jn;
        hi -= 1.0 / (double)i;                                // H_{i-1}
        const double jo = (4.0 * i) * ix * jn - jp;           // J_{2i-1}
        const double je = (4.0 * i - 2.0) * ix * jo - jn;     // J_{2i-2}
        jp = jo; jn = je;
        if (fabs(jn) > 1e120 || fabs(jp) > 1e120) { jn *= 1e-120; jp *= 1e-120; norm *= 1e-120; acc *= 1e-120; }
    }
    norm += jn;                                               // J_0
    return acc / norm;
}
__device__ double green2d_value(double r, double eps, int order)
{
    if (order == 0) {
        // spectrally compact kernel (reading A30), the grid spacing passed in `eps`: k_c = pi / h
        const double kc = 3.14159265358979323846 / eps;
        const double c0 = log(0.5 * kc) + 0.57721566490153286061;
        return ((r == 0.0 ? 0.0 : bessel_cin(kc * r)) - c0) / 6.2831853071795864769;
    }
    const double x = r * r / (2.0 * eps * eps);
    double v = (r == 0.0) ? (log(2.0 * eps * eps) - 0.57721566490153286061) / 12.566370614359172954
                          : (log(r) + 0.5 * exp_integral1(x)) / 6.2831853071795864769;
    if (order >= 4) v -= laguerre_tail(order, 0.0, x) * exp(-x) / 6.2831853071795864769;   // eps^2 * g = e^-x / (2 pi)
    return v;
}
__global__ void green_eval_kernel(double* g, int Px, int Py, int Pz, double hx, double hy, double hz, double eps, double vol, int order,
                                  int dim2)
{
    const long long tot = (long long)Px * Py * Pz;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < tot; i += (long long)gridDim.x * blockDim.x) {
        const int ix = (int)(i % Px), iy = (int)((i / Px) % Py), iz = (int)(i / ((long long)Px * Py));
        const double dx = (double)min(ix, Px - ix) * hx, dy = (double)min(iy, Py - iy) * hy, dz = (double)min(iz, Pz - iz) * hz;
        const double r = sqrt(dx * dx + dy * dy + dz * dz);
        if (dim2) { g[i] = vol * green2d_value(sqrt(dx * dx + dy * dy), eps, order); continue; }
        double v;
        if (order == 0) v = (r == 0.0) ? -1.0 / (6.2831853071795864769 * eps) : -sine_integral(3.14159265358979323846 * r / eps) / (19.739208802178717238 * r);
        else if (r == 0.0) v = -1.0 / (15.749609945722419 * eps); // (2 pi)^(3/2)
        else v = -erf(r * 0.70710678118654752440 / eps) / (12.566370614359172954 * r);
        if (order >= 4) {
            const double x = r * r / (2.0 * eps * eps);
            v -= laguerre_tail(order, 0.5, x) * exp(-x) / (15.749609945722419 * eps);   // eps^2 * g = e^-x / ((2 pi)^(3/2) eps)
        }
        g[i] = vol * v;
    }
}

// real part of the spectrum on the non-negative wavenumbers -> compact table, scaled and rounded
template <typename T>
__global__ void green_compact_kernel(const double2* spec, long long s_py, long long s_pz, T* tab, long long t_py, long long t_pz,
                                     int gx, int gy, int gz, double factor)
{
    const long long tot = (long long)gx * gy * gz;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < tot; i += (long long)gridDim.x * blockDim.x) {
        const int kx = (int)(i % gx), ky = (int)((i / gx) % gy), kz = (int)(i / ((long long)gx * gy));
        tab[kx + ky * t_py + kz * t_pz] = (T)(spec[kx + ky * s_py + kz * s_pz].x * factor);
    }
}

#define SF_CUDA(p, call)                                                                                   \
    do {                                                                                                   \
        cudaError_t e__ = (call);                                                                          \
        if (e__ != cudaSuccess) {                                                                          \
            cudaGetLastError();                                                                            \
            return fail(p, SF_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__));             \
        }                                                                                                  \
    } while (0)

// Green's spectrum: evaluate on the doubled grid, transform with the library's own fp64 passes
// (periodic R2C along x, forward strided passes along y and z), keep Re on [0, n]^3.
template <typename T> sf_status build_green(sf_plan p)
{
    const bool two_d = (p->ndim == 2);
    const int Px = 2 * (int)p->n[0], Py = 2 * (int)p->n[1], Pz = two_d ? 1 : 2 * (int)p->n[2];
    const long long hp = p->pitch; // >= Px/2 + 1
    double* g = nullptr;
    double2* spec = nullptr;
    void *twx = nullptr, *twy = nullptr, *twz = nullptr;
    const size_t gbytes = (size_t)Px * Py * Pz * sizeof(double), sbytes = (size_t)hp * Py * Pz * sizeof(double2);
    sf_status st;
    if ((st = dev_alloc(p, (void**)&g, gbytes)) != SF_OK) return st;
    if ((st = dev_alloc(p, (void**)&spec, sbytes)) != SF_OK) return st;
    if ((st = upload_twiddles<double>(p, &twx, Px)) != SF_OK) return st;
    if ((st = upload_twiddles<double>(p, &twy, Py)) != SF_OK) return st;
    if (!two_d && (st = upload_twiddles<double>(p, &twz, Pz)) != SF_OK) return st;
    const double hmax = two_d ? fmax(p->h[0], p->h[1]) : fmax(p->h[0], fmax(p->h[1], p->h[2]));
    const double eps = (p->op == SF_OP_GREEN_SPECTRAL ? 1.0 : p->eps_over_h) * hmax;
    const double vol = two_d ? p->h[0] * p->h[1] : p->h[0] * p->h[1] * p->h[2];
    const int order = (p->op == SF_OP_GREEN_SPECTRAL) ? 0 : 2 * ((int)p->op - (int)SF_OP_GREEN_GAUSS2 + 1);
    // the table uploads above are synchronous copies from pageable memory on the legacy stream, which a
    // non-blocking plan stream does not wait for: drain the device once before the first kernel reads them
    SF_CUDA(p, cudaDeviceSynchronize());
    green_eval_kernel<<<148 * 8, 256, 0, p->stream>>>(g, Px, Py, Pz, p->h[0], p->h[1], p->h[2], eps, vol, order, two_d ? 1 : 0);
    SF_CUDA(p, cudaGetLastError());

    XParams<double> xp;
    memset(&xp, 0, sizeof(xp));
    xp.real_in = g; xp.spec_out = spec;
    xp.rin_py = Px; xp.rin_pz = (long long)Px * Py; xp.rin_pc = 0;
    xp.sp_py = hp; xp.sp_pz = hp * Py; xp.sp_pc = 0;
    xp.n = Px; xp.ny = Py; xp.nz = Pz; xp.mode = X_PERIODIC;
    xp.LT = Px; xp.tw = (const double2*)twx;
    SF_CUDA(p, launch_xfwd<double>(Px / 2, xp, 1, p->stream));

    SParams<double> sp;
    memset(&sp, 0, sizeof(sp));
    sp.in = spec; sp.out = spec;
    sp.nx = Px / 2 + 1; sp.r2r = R2R_NONE;
    // along y
    sp.in_ps = sp.out_ps = hp; sp.in_bs = sp.out_bs = hp * Py;
    sp.n_in = Py; sp.n_out = Py; sp.LT = Py; sp.tw = (const double2*)twy;
    SF_CUDA(p, launch_spass<double>(Py, 0, sp, Pz, 1, 1, p->stream));
    // along z
    if (!two_d) {
        sp.in_ps = sp.out_ps = hp * Py; sp.in_bs = sp.out_bs = hp;
        sp.n_in = Pz; sp.n_out = Pz; sp.LT = Pz; sp.tw = (const double2*)twz;
        SF_CUDA(p, launch_spass<double>(Pz, 0, sp, Py, 1, 1, p->stream));
    }

    const int gx = (int)p->n[0] + 1, gy = (int)p->n[1] + 1, gz = two_d ? 1 : (int)p->n[2] + 1;
    if ((st = dev_alloc(p, &p->green, (size_t)hp * gy * gz * sizeof(T))) != SF_OK) return st;
    SF_CUDA(p, cudaMemsetAsync(p->green, 0, (size_t)hp * gy * gz * sizeof(T), p->stream));
    const double factor = p->rhs_sign / ((double)Px * (double)Py * (double)Pz);
    green_compact_kernel<T><<<148 * 8, 256, 0, p->stream>>>(spec, hp, hp * Py, (T*)p->green, hp, hp * gy, gx, gy, gz, factor);
    SF_CUDA(p, cudaGetLastError());
    SF_CUDA(p, cudaStreamSynchronize(p->stream));
    dev_free(p, g); dev_free(p, spec); dev_free(p, twx); dev_free(p, twy);
    if (!two_d) dev_free(p, twz);
    p->dev_bytes -= (long long)(gbytes + sbytes + (size_t)(Px + Py + (two_d ? 0 : Pz)) * 16);
    return SF_OK;
}

template <typename T> sf_status build_tables(sf_plan p)
{
    sf_status st;
    // twiddles: x table has the real transform length; strided tables the complex length, or the
    // real-extension length 2L for DST / DCT pencils (their split / merge steps need w_2L)
    p->LT[0] = p->Mx;
    if ((st = upload_twiddles<T>(p, &p->tw[0], p->LT[0])) != SF_OK) return st;
    for (int a = 1; a < p->ndim; ++a) {
        p->LT[a] = (p->r2r == R2R_NONE) ? p->La[a] : 2 * p->La[a];
        if ((st = upload_twiddles<T>(p, &p->tw[a], p->LT[a])) != SF_OK) return st;
    }
    for (int a = 0; a < p->ndim; ++a)
        if (p->r2ra[a] == R2R_DCT || p->r2ra[a] == R2R_DST2)
            if ((st = upload_dct_shift<T>(p, &p->ptw[a], (int)p->n[a])) != SF_OK) return st;
    std::vector<long double> z1(1, 0.0L);
    if ((st = upload_real<T>(p, &p->zero1, z1)) != SF_OK) return st;
    for (int a = 0; a < p->ndim; ++a) {
        int count;
        if (p->bc == SF_BC_UNBOUNDED) count = (a == 0) ? (int)p->n[0] + 1 : 2 * (int)p->n[a];
        else if (p->bc == SF_BC_PERIODIC) count = (a == 0) ? (int)p->n[0] / 2 + 1 : (int)p->n[a];
        else count = (int)p->n[a];
        std::vector<long double> lam, kap;
        axis_tables(*p, a, count, lam, kap);
        if ((st = upload_real<T>(p, &p->lam[a], lam)) != SF_OK) return st;
        if ((st = upload_real<T>(p, &p->kap[a], kap)) != SF_OK) return st;
        if (p->r2r != R2R_NONE) {
            // the extended sequence of length 2L has period 2 L_domain: slot k carries pi k / L_domain;
            // the Nyquist slot k = L is taken as zero (reading A20)
            const int Lh = (a == 0) ? p->Lx : p->La[a];
            std::vector<long double> ke((size_t)Lh + 1, 0.0L);
            for (int k = 0; k < Lh; ++k) ke[k] = PI_L * (long double)k / ((long double)Lh * (long double)p->h[a]);
            if ((st = upload_real<T>(p, &p->kap_ext[a], ke)) != SF_OK) return st;
        }
    }
    if (p->bc == SF_BC_UNBOUNDED) return build_green<T>(p);
    return SF_OK;
}

// S1 / S5: kernel generation 2 where the plan has it, generation 1 otherwise
template <typename T> cudaError_t x_forward(sf_plan p, const XParams<T>& xp, int ncomp, cudaStream_t st)
{
    if constexpr (std::is_same<T, double>::value) {
        if (p->xg64 && !xp.nyq_side) return sf2::launch_fast_xg(false, xp, ncomp, st);
        if (p->xp64 && !xp.nyq_side_yz && !xp.has_faces) return sf2::launch_fast_xp64(false, xp, ncomp, st);
    }
    return launch_xfwd<T>(p->Lx, xp, ncomp, st);
}
template <typename T> cudaError_t x_backward(sf_plan p, const XParams<T>& xp, int nf, cudaStream_t st)
{
    if constexpr (std::is_same<T, double>::value) {
        if (p->xg64 && !xp.nyq_side && !xp.dfield1) return sf2::launch_fast_xg(true, xp, nf, st);
        if (p->xp64 && !xp.nyq_side_yz && !xp.dfield1) return sf2::launch_fast_xp64(true, xp, nf, st);
    }
    return launch_xinv<T>(p->Lx, xp, nf, st);
}

// ---------------------------------------------------------------- the solve sequence
template <typename T> sf_status run(sf_plan p, int outk)
{
    typedef SF_CX C;
    const int nd = p->ndim;
    const int n0 = (int)p->n[0], n1 = (int)p->n[1], n2 = (nd == 3) ? (int)p->n[2] : 1;
    const long long hp = p->pitch;
    const int ncomp = p->ncomp;
    const int nf_out = (outk == OUT_GRAD) ? 1 + nd : (outk == OUT_DIV ? 1 : ncomp);
    const int P1 = p->padded ? 2 * n1 : n1;
    cudaStream_t st = p->stream;
    p->launches = 0;
    const bool timed = p->tslots && (p->tcalls++ % p->tstride) == 0;
    const int slot = p->tslots ? (int)(p->tcount % p->tslots) : 0;
    auto mark = [&](int i) { if (timed) cudaEventRecord(p->ev[6 * slot + i], st); };

    // S1: X forward
    XParams<T> xp;
    memset(&xp, 0, sizeof(xp));
    xp.real_in = (const T*)p->src;
    xp.rin_py = n0; xp.rin_pz = (long long)n0 * n1; xp.rin_pc = (long long)n0 * n1 * n2;
    xp.spec_out = p->W1; xp.real_out = (T*)p->W1;
    xp.sp_py = hp; xp.sp_pz = hp * n1; xp.sp_pc = p->w1_field;
    xp.n = n0; xp.ny = n1; xp.nz = n2; xp.mode = p->xmode;
    xp.LT = p->LT[0]; xp.tw = (const C*)p->tw[0]; xp.ptw = (const C*)p->ptw[0];
    if (p->bc == SF_BC_DIRICHLET || p->bc == SF_BC_NEUMANN) {
        for (int a = 0; a < nd; ++a)
            for (int s = 0; s < 2; ++s) {
                xp.face[2 * a + s] = (const T*)p->face[2 * a + s];
                if (xp.face[2 * a + s]) xp.has_faces = 1;
                // reading A18: the face sits one spacing (cell-boundary Dirichlet, cell-centre Neumann: weight 1)
                // or half a spacing / a mirrored ghost node (the other two Table-1 rows: weight 2) from the layer
                const double wf = ((p->bca[a] == SF_BC_DIRICHLET) == (p->grid == SF_GRID_CELL_BOUNDARY)) ? 1.0 : 2.0;
                // the discrete equation is lap_h psi = rhs_sign f with the face value in the ghost layer (eq. (2)
                // PAPER.md:22, reading A8): interior stencil = rhs_sign f + w g.  The multiplier carries rhs_sign for
                // the whole folded source, so the fold adds (w / rhs_sign) g -- the face value keeps its sign.
                if (p->bca[a] == SF_BC_DIRICHLET) xp.wface[2 * a + s] = (T)(-wf / (p->h[a] * p->h[a]) / p->rhs_sign);
                else xp.wface[2 * a + s] = (T)((s ? -wf : wf) / p->h[a] / p->rhs_sign);
            }
    }
    mark(0);
    const bool fast_x = p->fast_x && outk == OUT_SOLVE && !xp.has_faces;
    sf2::FastXParams fx;
    memset(&fx, 0, sizeof(fx));
    const bool fast5_x = p->fast5 && p->fast5_x && (outk == OUT_SOLVE || (outk == OUT_CURL && ncomp == 3));
    if (fast_x) {
        fx.real_in = (const float*)p->src; fx.real_out = (float*)p->out;
        fx.spec = (sf2::C*)p->W1; fx.spec_pitch = hp; fx.nrows = n1 * n2;
        fx.nyq = (sf2::C*)p->nyqA; fx.n1 = n1; fx.n2 = n2;
        SF_CUDA(p, sf2::launch_fast_x(false, fx, st));
    } else if (fast5_x) {
        // the components are contiguous in the source, the work array and the output: more rows
        fx.real_in = (const float*)p->src; fx.real_out = (float*)p->out;
        fx.spec = (sf2::C*)p->W1; fx.spec_pitch = hp; fx.nrows = n1 * n2 * ncomp;
        SF_CUDA(p, sf2::launch_fast_x5(false, fx, st));
    } else if (p->fastper && p->fastper_x && (outk == OUT_SOLVE || outk == OUT_GRAD) && !xp.has_faces) {
        sf2::FastXPerParams px;
        memset(&px, 0, sizeof(px));
        px.real_in = (const float*)p->src; px.spec = (sf2::C*)p->W1; px.spec_pitch = hp; px.nrows = n1 * n2;
        px.nyq = (sf2::C*)p->nyqA;
        SF_CUDA(p, sf2::launch_fast_xper(false, px, st));
    } else {
        if ((p->fastper || p->fastper64) && (outk == OUT_SOLVE || outk == OUT_GRAD)) xp.nyq_side = p->nyqA;
        if (p->fast && outk == OUT_SOLVE && p->nyqA) { xp.nyq_side = p->nyqA; xp.nyq_side_yz = 1; }   // [y][z], as fast_x_kernel writes it
        SF_CUDA(p, x_forward<T>(p, xp, ncomp, st));
        xp.nyq_side = nullptr; xp.nyq_side_yz = 0;
    }
    p->launches++;
    mark(1);

    SParams<T> sp;
    memset(&sp, 0, sizeof(sp));
    sp.nx = p->nspec_x; sp.r2r = p->r2r;
    sp.mul = (p->bc == SF_BC_UNBOUNDED) ? MUL_GREEN : MUL_SYMBOL;
    sp.scale = (T)p->scale;
    {   // the all-zero index is singular only when no axis is Dirichlet
        bool all_neumann = (p->bc == SF_BC_NEUMANN);
        for (int a = 0; a < nd; ++a) all_neumann = all_neumann && p->bca[a] == SF_BC_NEUMANN;
        sp.zero_mode = (p->bc == SF_BC_PERIODIC || all_neumann) ? 1 : 0;
    }
    sp.green = (const T*)p->green;

    if (p->fast && outk == OUT_SOLVE) {
        // kernel generation 2: S2, S3, S4 as persistent TMA-fed register-FFT kernels
        sf2::FastParams fp;
        memset(&fp, 0, sizeof(fp));
        fp.sched = (int*)p->sched;
        fp.nct = p->nspec_x / sf2::kTile;
        for (fp.nct_shift = 0; (1 << fp.nct_shift) < fp.nct; ++fp.nct_shift) {}
        fp.nyq_col = (p->nspec_x % sf2::kTile) ? fp.nct * sf2::kTile : -1;
        // S2: W1 [z][y][hp] -> W2 [z][ky][hp]
        fp.in = (const sf2::C*)p->W1; fp.out = (sf2::C*)p->W2;
        fp.in_ps = hp; fp.in_bs = hp * n1; fp.out_ps = hp; fp.out_bs = hp * P1; fp.nb = n2;
        const bool side = p->nyqA != nullptr;   // Nyquist column in the side arrays (written by either X kernel)
        if (side) { fp.nyq_in = (const sf2::C*)p->nyqA; fp.nyq_out = (sf2::C*)p->nyqB; }
        fp.nyq_first = side ? 1 : 0;
        fp.reverse_batches = 1;   // S1 wrote plane z last: start there while it is in L2
        SF_CUDA(p, sf2::launch_fast_pad(sf2::FMODE_FWD, fp, p->map_s2, st));
        fp.reverse_batches = 0;
        p->launches++;
        mark(2);
        // S3: W2 in place along z
        fp.in = (const sf2::C*)p->W2; fp.out = (sf2::C*)p->W2;
        fp.in_ps = fp.out_ps = hp * P1; fp.in_bs = fp.out_bs = hp; fp.nb = P1;
        if (side) { fp.nyq_in = (const sf2::C*)p->nyqB; fp.nyq_out = (sf2::C*)p->nyqB; }
        fp.pair_batches = 1;
        fp.nyq_first = 1;
        fp.green_tiles = (const float*)p->green_tiles; fp.Pb = P1;
        SF_CUDA(p, sf2::launch_fast_pad(sf2::FMODE_FUSED, fp, p->map_s3, st));
        p->launches++;
        mark(3);
        // S4: W2 [z][ky][hp] -> W1 [z][y][hp]
        if (side) { fp.nyq_in = (const sf2::C*)p->nyqB; fp.nyq_out = (sf2::C*)p->nyqA; }
        fp.pair_batches = 0;
        fp.nyq_first = side ? 1 : 0;
        fp.in = (const sf2::C*)p->W2; fp.out = (sf2::C*)p->W1;
        fp.in_ps = hp; fp.in_bs = hp * P1; fp.out_ps = hp; fp.out_bs = hp * n1; fp.nb = n2;
        SF_CUDA(p, sf2::launch_fast_pad(sf2::FMODE_INV, fp, p->map_s4, st));
        p->launches++;
        mark(4);
        xp.spec_in = p->W1; xp.real_out = (T*)p->out;
        fx.reverse = 1;           // S4 wrote the last planes last
        if (fast_x) {
            SF_CUDA(p, sf2::launch_fast_x(true, fx, st));
        } else {
            if (side) { xp.nyq_side = p->nyqA; xp.nyq_side_yz = 1; }
            SF_CUDA(p, x_backward<T>(p, xp, nf_out, st));
            xp.nyq_side = nullptr; xp.nyq_side_yz = 0;
        }
        p->launches++;
        mark(5);
        if (timed) p->tcount++;
        p->last_kind = outk;
        p->out_last = p->out;
        return SF_OK;
    }

    if (p->r2r64 && outk == OUT_SOLVE) {
        // kernel generation 2 for the real-to-real strided passes, in place on W1 (pairs of real columns as complex columns)
        sf2::FastR64Params fp;
        memset(&fp, 0, sizeof(fp));
        const int kind = (p->r2r == R2R_DST1) ? 0 : 1;
        const long long hc = hp / 2;
        fp.sched = (int*)p->sched;
        fp.in = (const double2*)p->W1; fp.out = (double2*)p->W1;
        fp.n = n1; fp.nct = (int)(hp / 16); fp.nx = p->nspec_x;
        // S2 along y: batches = z planes
        fp.in_ps = fp.out_ps = hc; fp.in_bs = fp.out_bs = hc * n1; fp.nb = n2; fp.batch_dim = 2;
        SF_CUDA(p, sf2::launch_fast_r2r64(kind, 0, fp, p->map_s2, st));
        p->launches++;
        mark(2);
        // S3 along z: batches = ky
        fp.in_ps = fp.out_ps = hc * n1; fp.in_bs = fp.out_bs = hc; fp.nb = n1; fp.batch_dim = 1; fp.n = n2;
        fp.lam_x = (const double*)p->lam[0]; fp.lam_b = (const double*)p->lam[1]; fp.lam_p = (const double*)p->lam[2];
        fp.scale = p->scale; fp.zero_mode = sp.zero_mode;
        SF_CUDA(p, sf2::launch_fast_r2r64(kind, 2, fp, p->map_s3, st));
        p->launches++;
        mark(3);
        // S4 along y (DST-I: the same transform again; DCT: DCT-III)
        fp.in_ps = fp.out_ps = hc; fp.in_bs = fp.out_bs = hc * n1; fp.nb = n2; fp.batch_dim = 2; fp.n = n1;
        SF_CUDA(p, sf2::launch_fast_r2r64(kind, kind == 0 ? 0 : 1, fp, p->map_s2, st));
        p->launches++;
        mark(4);
        xp.spec_in = p->W1; xp.real_out = (T*)p->out;
        SF_CUDA(p, x_backward<T>(p, xp, nf_out, st));
        p->launches++;
        mark(5);
        if (timed) p->tcount++;
        p->last_kind = outk;
        p->out_last = p->out;
        return SF_OK;
    }

    if (p->fast64 && outk == OUT_SOLVE) {
        // kernel generation 2 in double precision: S2, S3, S4 as persistent TMA-fed register-FFT kernels (tiles of 8 columns)
        sf2::Fast64Params fp;
        memset(&fp, 0, sizeof(fp));
        fp.sched = (int*)p->sched;
        fp.nct = p->nspec_x / 8;
        for (fp.nct_shift = 0; (1 << fp.nct_shift) < fp.nct; ++fp.nct_shift) {}
        fp.nyq_col = (p->nspec_x % 8) ? fp.nct * 8 : -1;
        // S2: W1 [z][y][hp] -> W2 [z][ky][hp]
        fp.in = (const double2*)p->W1; fp.out = (double2*)p->W2;
        fp.in_ps = hp; fp.in_bs = hp * n1; fp.out_ps = hp; fp.out_bs = hp * P1; fp.nb = n2;
        fp.reverse_batches = 1;
        SF_CUDA(p, sf2::launch_fast64(sf2::FMODE_FWD, fp, p->map_s2, st));
        fp.reverse_batches = 0;
        p->launches++;
        mark(2);
        // S3: W2 in place along z
        fp.in = (const double2*)p->W2; fp.out = (double2*)p->W2;
        fp.in_ps = fp.out_ps = hp * P1; fp.in_bs = fp.out_bs = hp; fp.nb = P1;
        fp.pair_batches = 1;
        fp.green_tiles = (const double*)p->green_tiles; fp.Pb = P1;
        SF_CUDA(p, sf2::launch_fast64(sf2::FMODE_FUSED, fp, p->map_s3, st));
        fp.pair_batches = 0;
        p->launches++;
        mark(3);
        // S4: W2 [z][ky][hp] -> W1 [z][y][hp]
        fp.in = (const double2*)p->W2; fp.out = (double2*)p->W1;
        fp.in_ps = hp; fp.in_bs = hp * P1; fp.out_ps = hp; fp.out_bs = hp * n1; fp.nb = n2;
        SF_CUDA(p, sf2::launch_fast64(sf2::FMODE_INV, fp, p->map_s4, st));
        p->launches++;
        mark(4);
        xp.spec_in = p->W1; xp.real_out = (T*)p->out;
        SF_CUDA(p, x_backward<T>(p, xp, nf_out, st));
        p->launches++;
        mark(5);
        if (timed) p->tcount++;
        p->last_kind = outk;
        p->out_last = p->out;
        return SF_OK;
    }

    if (p->fast5 && (outk == OUT_SOLVE || (outk == OUT_CURL && ncomp == 3))) {
        // kernel generation 2 for 512-long pencils: S2, S3, S4 as persistent TMA-fed register-FFT kernels, one CTA per SM
        sf2::Fast5Params fp;
        memset(&fp, 0, sizeof(fp));
        fp.sched = (int*)p->sched;
        fp.nct = p->nspec_x / sf2::kTile;
        for (fp.nct_shift = 0; (1 << fp.nct_shift) < fp.nct; ++fp.nct_shift) {}
        fp.nyq_col = (p->nspec_x % sf2::kTile) ? fp.nct * sf2::kTile : -1;
        fp.ncomp = ncomp;
        // S2: W1 [c][z][y][hp] -> W2 [c][z][ky][hp]; the components are more batches
        fp.in = (const sf2::C*)p->W1; fp.out = (sf2::C*)p->W2;
        fp.in_ps = hp; fp.in_bs = hp * n1; fp.out_ps = hp; fp.out_bs = hp * P1; fp.nb = n2 * ncomp;
        fp.reverse_batches = 1;   // S1 wrote the last planes last: start there while they are in L2
        // (S2, S3 on tiles of 8 columns -- two CTAs per SM; S4 on tiles of 16)
        const int nct16 = fp.nct, shift16 = fp.nct_shift, nyq16 = fp.nyq_col;
        fp.nct = p->nspec_x / 8;
        for (fp.nct_shift = 0; (1 << fp.nct_shift) < fp.nct; ++fp.nct_shift) {}
        fp.nyq_col = (p->nspec_x % 8) ? fp.nct * 8 : -1;
        SF_CUDA(p, sf2::launch_fast5(sf2::F5_FWD, fp, p->map_s2, st));
        fp.reverse_batches = 0;
        p->launches++;
        mark(2);
        // S3: W2 in place along z, tiles of 8 columns
        fp.in = (const sf2::C*)p->W2; fp.out = (sf2::C*)p->W2;
        fp.in_ps = fp.out_ps = hp * P1; fp.in_bs = fp.out_bs = hp; fp.in_cs = fp.out_cs = p->w2_field; fp.nb = P1;
        fp.pair_batches = 1;
        fp.green_tiles = (const float*)p->green_tiles; fp.Pb = P1;
        fp.kap_x = (const float*)p->kap[0]; fp.kap_b = (const float*)p->kap[1]; fp.kap_p = (const float*)p->kap[2];
        SF_CUDA(p, sf2::launch_fast5(outk == OUT_CURL ? sf2::F5_CURL : sf2::F5_FUSED, fp, p->map_s3, st));
        fp.pair_batches = 0;
        fp.nct = nct16; fp.nct_shift = shift16; fp.nyq_col = nyq16;
        p->launches++;
        mark(3);
        // S4: W2 [c][z][ky][hp] -> W1 [c][z][y][hp]
        fp.in = (const sf2::C*)p->W2; fp.out = (sf2::C*)p->W1;
        fp.in_ps = hp; fp.in_bs = hp * P1; fp.out_ps = hp; fp.out_bs = hp * n1; fp.in_cs = fp.out_cs = 0; fp.nb = n2 * ncomp;
        SF_CUDA(p, sf2::launch_fast5(sf2::F5_INV, fp, p->map_s4, st));
        p->launches++;
        mark(4);
        xp.spec_in = p->W1; xp.real_out = (T*)p->out;
        if (fast5_x) {
            fx.reverse = 1;       // S4 wrote the last planes last
            SF_CUDA(p, sf2::launch_fast_x5(true, fx, st));
        } else {
            SF_CUDA(p, x_backward<T>(p, xp, nf_out, st));
        }
        p->launches++;
        mark(5);
        if (timed) p->tcount++;
        p->last_kind = outk;
        p->out_last = p->out;
        return SF_OK;
    }

    if (p->fastper64 && (outk == OUT_SOLVE || outk == OUT_GRAD)) {
        // kernel generation 2, periodic, double precision: S2, S3, S4 in place on W1 (tiles of 16 columns)
        sf2::FastPer64Params fp;
        memset(&fp, 0, sizeof(fp));
        fp.sched = (int*)p->sched;
        fp.in = (const double2*)p->W1; fp.out = (double2*)p->W1;
        fp.nx = p->nspec_x;
        fp.nct = p->nspec_x / 16;
        fp.nyq_col = (p->nspec_x % 16) ? fp.nct * 16 : -1;
        fp.nyq = (double2*)p->nyqA;
        fp.in_ps = fp.out_ps = hp; fp.in_bs = fp.out_bs = hp * n1; fp.nb = n2;
        fp.nyq_ps = 1; fp.nyq_bs = n1;
        SF_CUDA(p, sf2::launch_fast_per64(sf2::FMODE_FWD, fp, st));
        p->launches++;
        mark(2);
        fp.in_ps = fp.out_ps = hp * n1; fp.in_bs = fp.out_bs = hp; fp.nb = n1;
        fp.nyq_ps = n1; fp.nyq_bs = 1;
        fp.lam_x = (const double*)p->lam[0]; fp.lam_b = (const double*)p->lam[1]; fp.lam_p = (const double*)p->lam[2];
        fp.scale = p->scale; fp.zero_mode = 1;
        if (outk == OUT_GRAD) {
            fp.grad = 1;
            fp.kap_x = (const double*)p->kap[0]; fp.kap_b = (const double*)p->kap[1]; fp.kap_p = (const double*)p->kap[2];
            fp.out_cs = p->w1_field; fp.nyq_cs = (long long)n1 * n2;
        }
        SF_CUDA(p, sf2::launch_fast_per64(sf2::FMODE_FUSED, fp, st));
        fp.grad = 0;
        p->launches++;
        mark(3);
        fp.in_ps = fp.out_ps = hp; fp.in_bs = fp.out_bs = hp * n1; fp.nb = n2 * nf_out;
        fp.nyq_ps = 1; fp.nyq_bs = n1;
        SF_CUDA(p, sf2::launch_fast_per64(sf2::FMODE_INV, fp, st));
        p->launches++;
        mark(4);
        xp.spec_in = p->W1; xp.real_out = (T*)p->out;
        xp.nyq_side = p->nyqA;
        SF_CUDA(p, x_backward<T>(p, xp, nf_out, st));
        p->launches++;
        mark(5);
        if (timed) p->tcount++;
        p->last_kind = outk;
        p->out_last = p->out;
        return SF_OK;
    }

    if (p->fastper && (outk == OUT_SOLVE || outk == OUT_GRAD)) {
        // kernel generation 2, periodic: S2, S3, S4 in place on W1 as persistent register-FFT kernels
        sf2::FastPerParams fp;
        memset(&fp, 0, sizeof(fp));
        fp.sched = (int*)p->sched;
        fp.in = (const sf2::C*)p->W1; fp.out = (sf2::C*)p->W1;
        fp.nx = p->nspec_x;
        fp.nct = p->nspec_x / sf2::kPerTileCols;
        fp.nyq_col = (p->nspec_x % sf2::kPerTileCols) ? fp.nct * sf2::kPerTileCols : -1;
        fp.nyq = (sf2::C*)p->nyqA;
        // S2 along y: batches = z planes
        fp.in_ps = fp.out_ps = hp; fp.in_bs = fp.out_bs = hp * n1; fp.nb = n2;
        fp.nyq_ps = 1; fp.nyq_bs = n1;
        SF_CUDA(p, sf2::launch_fast_per(sf2::FMODE_FWD, fp, st));
        p->launches++;
        mark(2);
        // S3 along z: batches = ky
        fp.in_ps = fp.out_ps = hp * n1; fp.in_bs = fp.out_bs = hp; fp.nb = n1;
        fp.nyq_ps = n1; fp.nyq_bs = 1;
        fp.lam_x = (const float*)p->lam[0]; fp.lam_b = (const float*)p->lam[1]; fp.lam_p = (const float*)p->lam[2];
        fp.scale = (float)p->scale; fp.zero_mode = 1;
        if (outk == OUT_GRAD) {
            fp.grad = 1;
            fp.kap_x = (const float*)p->kap[0]; fp.kap_b = (const float*)p->kap[1]; fp.kap_p = (const float*)p->kap[2];
            fp.out_cs = p->w1_field; fp.nyq_cs = (long long)n1 * n2;
        }
        SF_CUDA(p, sf2::launch_fast_per(sf2::FMODE_FUSED, fp, st));
        fp.grad = 0;
        p->launches++;
        mark(3);
        // S4 along y; the fields are contiguous, so the output fields are just more batches
        fp.in_ps = fp.out_ps = hp; fp.in_bs = fp.out_bs = hp * n1; fp.nb = n2 * nf_out;
        fp.nyq_ps = 1; fp.nyq_bs = n1;
        SF_CUDA(p, sf2::launch_fast_per(sf2::FMODE_INV, fp, st));
        p->launches++;
        mark(4);
        xp.spec_in = p->W1; xp.real_out = (T*)p->out;
        xp.nyq_side = p->nyqA;
        if (p->fastper_x) {
            sf2::FastXPerParams px;
            memset(&px, 0, sizeof(px));
            px.real_out = (float*)p->out; px.spec = (sf2::C*)p->W1; px.spec_pitch = hp; px.nrows = n1 * n2 * nf_out;
            px.nyq = (sf2::C*)p->nyqA;
            SF_CUDA(p, sf2::launch_fast_xper(true, px, st));
        } else {
            SF_CUDA(p, x_backward<T>(p, xp, nf_out, st));
        }
        p->launches++;
        mark(5);
        if (timed) p->tcount++;
        p->last_kind = outk;
        p->out_last = p->out;
        return SF_OK;
    }

    if (nd == 3) {
        // S2: Y forward (W1 -> W2; in place when not padded)
        sp.in = p->W1; sp.out = p->W2;
        sp.in_ps = hp; sp.in_bs = hp * n1; sp.in_cs = p->w1_field;
        sp.out_ps = hp; sp.out_bs = hp * P1; sp.out_cs = p->w2_field;
        sp.n_in = n1; sp.n_out = (p->r2r == R2R_NONE) ? p->La[1] : n1;
        sp.LT = p->LT[1]; sp.tw = (const C*)p->tw[1]; sp.ptw = (const C*)p->ptw[1];
        sp.r2r = p->r2ra[1];
        SF_CUDA(p, launch_spass<T>(p->La[1], 0, sp, n2, ncomp, 1, st));
        p->launches++;
    }
    mark(2);
    {
        // S3: forward along the last axis, multiply, backward along the last axis
        const int ax = nd - 1;
        const int nlast = (int)p->n[ax];
        sp.outk = outk; sp.pencil_axis = ax;
        sp.in = p->W2; sp.out = p->W2;
        if (nd == 3) {
            sp.in_ps = sp.out_ps = hp * P1; sp.in_bs = sp.out_bs = hp;
            sp.lam_b = (const T*)p->lam[1]; sp.kap_b = (const T*)p->kap[1];
            sp.Pb = p->P[1];
            sp.g_pb = hp; sp.g_pp = hp * (n1 + 1);
        } else {
            // 2-D: the fused pass follows S1 directly, in place on W1 (rows >= n of a padded pencil exist only in shared memory)
            sp.in = p->W1; sp.out = p->W1;
            sp.in_ps = sp.out_ps = hp; sp.in_bs = sp.out_bs = 0;
            sp.lam_b = (const T*)p->zero1; sp.kap_b = (const T*)p->zero1;
            sp.Pb = 1;
            sp.g_pb = 0; sp.g_pp = hp;
        }
        sp.in_cs = sp.out_cs = (nd == 3) ? p->w2_field : p->w1_field;
        sp.lam_x = (const T*)p->lam[0]; sp.kap_x = (const T*)p->kap[0];
        sp.lam_p = (const T*)p->lam[ax]; sp.kap_p = (const T*)p->kap[ax];
        sp.Pp = p->P[ax];
        sp.n_in = nlast; sp.n_out = nlast;
        sp.LT = p->LT[ax]; sp.tw = (const C*)p->tw[ax]; sp.ptw = (const C*)p->ptw[ax];
        sp.kap_ext = (const T*)p->kap_ext[ax];
        const int nb = (nd == 3) ? P1 : 1;
        const int nbuf = (outk == OUT_CURL || outk == OUT_DIV) ? 3 : (outk == OUT_GRAD ? 2 : 1);
        const int gz = (outk == OUT_SOLVE || outk == OUT_LAP) ? ncomp : 1;
        sp.r2r = p->r2ra[ax];
        SF_CUDA(p, launch_spass<T>(p->La[ax], 2, sp, nb, gz, nbuf, st));
        p->launches++;
    }
    mark(3);
    if (nd == 3) {
        // S4: Y backward (W2 -> W1)
        sp.in = p->W2; sp.out = p->W1;
        sp.in_ps = hp; sp.in_bs = hp * P1; sp.in_cs = p->w2_field;
        sp.out_ps = hp; sp.out_bs = hp * n1; sp.out_cs = p->w1_field;
        sp.n_in = (p->r2r == R2R_NONE) ? p->La[1] : n1; sp.n_out = n1;
        sp.LT = p->LT[1]; sp.tw = (const C*)p->tw[1]; sp.ptw = (const C*)p->ptw[1];
        sp.kap_ext = (const T*)p->kap_ext[1];
        sp.dfield1 = (p->r2r != R2R_NONE && outk == OUT_GRAD) ? 3 : 0;   // field 2 = d psi / dy
        sp.r2r = p->r2ra[1];
        SF_CUDA(p, launch_spass<T>(p->La[1], 1, sp, n2, nf_out, 1, st));
        p->launches++;
    }
    mark(4);
    // S5: X backward
    xp.spec_in = p->W1; xp.real_out = (T*)p->out;
    xp.kap_ext = (const T*)p->kap_ext[0];
    xp.dfield1 = (p->r2r != R2R_NONE && outk == OUT_GRAD) ? 2 : 0;       // field 1 = d psi / dx
    SF_CUDA(p, x_backward<T>(p, xp, nf_out, st));
    p->launches++;
    mark(5);
    if (timed) p->tcount++;
    p->last_kind = outk;
    p->out_last = p->out;
    return SF_OK;
}

sf_status run_any(sf_plan p, int outk)
{
    if (!p) return SF_ERR_INVALID_ARG;
    if (!p->src) return fail(p, SF_ERR_STATE, "no source set: call sf_set_source first");
    if (p->pipe < 2) return p->prec == SF_F32 ? run<float>(p, outk) : run<double>(p, outk);
    // copy pipeline: this call reads the source slot filled last and writes the other result buffer than the
    // previous call, once the copy that still reads that buffer has finished
    p->os ^= 1;
    if (p->src_piped) SF_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_src_ready[p->ss], 0));
    const bool own_out = (p->out == p->pout[0] || p->out == p->pout[1]);
    if (own_out) {
        p->out = p->pout[p->os];
        if (p->out_free_set[p->os]) SF_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_out_free[p->os], 0));
    } else {
        // a work set of sf_gradient: one result buffer, every earlier copy out of it must have finished
        for (int i = 0; i < 2; ++i)
            if (p->out_free_set[i]) SF_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_out_free[i], 0));
    }
    const sf_status st = p->prec == SF_F32 ? run<float>(p, outk) : run<double>(p, outk);
    if (st != SF_OK) return st;
    SF_CUDA(p, cudaEventRecord(p->ev_done[p->os], p->stream));
    p->done_set[p->os] = true;
    if (p->src_piped) {
        SF_CUDA(p, cudaEventRecord(p->ev_src_free[p->ss], p->stream));
        p->src_free_set[p->ss] = true;
    }
    return SF_OK;
}

size_t field_elems(const sf_plan_s* p) { return (size_t)p->n[0] * (size_t)p->n[1] * (size_t)(p->ndim == 3 ? p->n[2] : 1); }

} // namespace

// ==================================================================================== C ABI
extern "C" {

const char* sf_version(void) { return "sailffish-b200 0.1 (sm_100a)"; }

const char* sf_last_error(sf_plan plan) { return plan ? plan->err.c_str() : g_create_error.c_str(); }

sf_status sf_plan_destroy(sf_plan plan)
{
    if (!plan) return SF_OK;
    for (void* d : plan->allocs) cudaFree(d);
    for (cudaEvent_t e : plan->ev) cudaEventDestroy(e);
    for (int i = 0; i < 2; ++i) {
        if (plan->ev_src_ready[i]) cudaEventDestroy(plan->ev_src_ready[i]);
        if (plan->ev_src_free[i]) cudaEventDestroy(plan->ev_src_free[i]);
        if (plan->ev_done[i]) cudaEventDestroy(plan->ev_done[i]);
        if (plan->ev_out_free[i]) cudaEventDestroy(plan->ev_out_free[i]);
    }
    if (plan->st_h2d) cudaStreamDestroy(plan->st_h2d);
    if (plan->st_d2h) cudaStreamDestroy(plan->st_d2h);
    delete plan;
    return SF_OK;
}

sf_status sf_plan_create(sf_plan* out, int ndim, const long long n[3], const double h[3], const sf_bc bc[3], sf_grid grid,
                         sf_operator op, sf_precision prec, const sf_options* opt)
{
    if (!out) return fail(nullptr, SF_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!n || !h || !bc) return fail(nullptr, SF_ERR_INVALID_ARG, "n, h and bc must not be NULL");
    if (ndim != 2 && ndim != 3) return fail(nullptr, ndim == 1 ? SF_ERR_UNSUPPORTED : SF_ERR_INVALID_ARG, "ndim must be 2 or 3");
    if (prec != SF_F32 && prec != SF_F64) return fail(nullptr, SF_ERR_INVALID_ARG, "unknown precision");
    if (grid != SF_GRID_CELL_BOUNDARY && grid != SF_GRID_CELL_CENTRE) return fail(nullptr, SF_ERR_INVALID_ARG, "unknown grid type");
    if (op < SF_OP_PSEUDO_SPECTRAL || op > SF_OP_GREEN_SPECTRAL) return fail(nullptr, SF_ERR_INVALID_ARG, "unknown operator");
    const bool green_op = (op >= SF_OP_GREEN_GAUSS2 && op <= SF_OP_GREEN_SPECTRAL);
    for (int a = 0; a < ndim; ++a) {
        if (bc[a] < SF_BC_PERIODIC || bc[a] > SF_BC_UNBOUNDED) return fail(nullptr, SF_ERR_INVALID_ARG, "unknown boundary condition");
        if (n[a] <= 0) return fail(nullptr, SF_ERR_INVALID_ARG, "sizes must be positive");
        if (!(h[a] > 0.0) || !std::isfinite(h[a])) return fail(nullptr, SF_ERR_INVALID_ARG, "spacings must be positive and finite");
        if (bc[a] != bc[0]) {
            // Dirichlet and Neumann may be mixed per axis (each axis takes its own row of Table 1); periodic and
            // unbounded axes cannot be combined with others (that is the paper's semi-unbounded future work)
            const bool dn = (bc[a] == SF_BC_DIRICHLET || bc[a] == SF_BC_NEUMANN) && (bc[0] == SF_BC_DIRICHLET || bc[0] == SF_BC_NEUMANN);
            if (!dn) return fail(nullptr, SF_ERR_UNSUPPORTED, "periodic / unbounded axes cannot be mixed with other boundary conditions (PAPER.md:126, :191-199)");
        }
    }
    int ncomp = (opt && opt->ncomp) ? opt->ncomp : 1;
    if (ncomp != 1 && ncomp != 3) return fail(nullptr, SF_ERR_UNSUPPORTED, "ncomp must be 1 or 3");
    if (ncomp == 3 && ndim != 3) return fail(nullptr, SF_ERR_UNSUPPORTED, "vector plans are 3-D");
    const sf_bc b = bc[0];
    if (b == SF_BC_UNBOUNDED) {
        if (!green_op) return fail(nullptr, SF_ERR_UNSUPPORTED, "unbounded plans use a Green's function operator");
    } else if (green_op) {
        return fail(nullptr, SF_ERR_UNSUPPORTED, "Green's function operators need unbounded boundary conditions");
    }

    sf_plan p = new (std::nothrow) sf_plan_s();
    if (!p) return fail(nullptr, SF_ERR_ALLOC, "host allocation failed");
    p->ndim = ndim;
    for (int a = 0; a < 3; ++a) { p->n[a] = (a < ndim) ? n[a] : 1; p->h[a] = (a < ndim) ? h[a] : 1.0; }
    p->bc = b; p->grid = grid; p->op = op; p->prec = prec; p->ncomp = ncomp;
    for (int a = 0; a < 3; ++a) {
        p->bca[a] = (a < ndim) ? bc[a] : b;
        if (p->bca[a] != b) p->mixed = true;
    }
    p->stream = opt ? (cudaStream_t)opt->stream : nullptr;
    p->rhs_sign = (opt && opt->rhs_sign != 0.0) ? opt->rhs_sign : 1.0;
    p->eps_over_h = (opt && opt->eps_over_h != 0.0) ? opt->eps_over_h : 2.0;
    p->esize = (prec == SF_F32) ? 4 : 8;

    auto bail = [&](sf_status st, const std::string& msg) {
        std::string m = msg.empty() ? p->err : msg;
        sf_plan_destroy(p);
        return fail(nullptr, st, m);
    };

    // transform lengths
    double norm = 1.0;
    for (int a = 0; a < ndim; ++a) {
        const long long na = p->n[a];
        long long len; // complex FFT length of the pass along this axis
        switch (p->bca[a]) {
        case SF_BC_PERIODIC:
            if (!is_pow2(na)) return bail(SF_ERR_UNSUPPORTED, "periodic sizes must be powers of two");
            len = (a == 0) ? na / 2 : na; p->P[a] = (int)na; norm *= (double)na; break;
        case SF_BC_UNBOUNDED:
            if (!is_pow2(na)) return bail(SF_ERR_UNSUPPORTED, "unbounded sizes must be powers of two");
            len = (a == 0) ? na : 2 * na; p->P[a] = (int)(2 * na); norm *= 2.0 * (double)na; break;
        case SF_BC_DIRICHLET:
            if (grid == SF_GRID_CELL_BOUNDARY) {
                if (!is_pow2(na + 1)) return bail(SF_ERR_UNSUPPORTED, "Dirichlet cell-boundary sizes must be 2^k - 1 interior nodes");
                len = na + 1;
            } else {
                if (!is_pow2(na)) return bail(SF_ERR_UNSUPPORTED, "Dirichlet cell-centre sizes must be powers of two");
                len = na;
            }
            p->P[a] = (int)na; norm *= 2.0 * (double)len; break;
        default:
            if (grid == SF_GRID_CELL_CENTRE) {
                if (!is_pow2(na)) return bail(SF_ERR_UNSUPPORTED, "Neumann cell-centre sizes must be powers of two");
                len = na;
            } else {
                if (na < 3 || !is_pow2(na - 1)) return bail(SF_ERR_UNSUPPORTED, "Neumann cell-boundary sizes must be 2^k + 1 nodes");
                len = na - 1;
            }
            p->P[a] = (int)na; norm *= 2.0 * (double)len; break;
        }
        if (!length_built((int)len) || len > 2048) return bail(SF_ERR_UNSUPPORTED, "transform length outside the built range (complex length 4..2048 per pass)");
        if (a == 0) p->Lx = (int)len; else p->La[a] = (int)len;
    }
    p->Mx = 2 * p->Lx;
    p->scale = p->rhs_sign / norm;
    p->padded = (b == SF_BC_UNBOUNDED);
    switch (b) {
    case SF_BC_PERIODIC: p->xmode = X_PERIODIC; p->r2r = R2R_NONE; break;
    case SF_BC_UNBOUNDED: p->xmode = X_ZEROPAD; p->r2r = R2R_NONE; break;
    case SF_BC_DIRICHLET:
        if (grid == SF_GRID_CELL_BOUNDARY) { p->xmode = X_DST1; p->r2r = R2R_DST1; }
        else { p->xmode = X_DST2; p->r2r = R2R_DST2; }
        break;
    default:
        if (grid == SF_GRID_CELL_CENTRE) { p->xmode = X_DCT2; p->r2r = R2R_DCT; }
        else { p->xmode = X_DCT1; p->r2r = R2R_DCT1; }
        break;
    }
    for (int a = 0; a < 3; ++a) {
        if (p->bca[a] == SF_BC_DIRICHLET) p->r2ra[a] = (grid == SF_GRID_CELL_BOUNDARY) ? R2R_DST1 : R2R_DST2;
        else if (p->bca[a] == SF_BC_NEUMANN) p->r2ra[a] = (grid == SF_GRID_CELL_CENTRE) ? R2R_DCT : R2R_DCT1;
        else p->r2ra[a] = R2R_NONE;
    }
    p->nspec_x = (p->r2r == R2R_NONE) ? p->Lx + 1 : (int)p->n[0];
    p->pitch = round_up(p->nspec_x, 16);
    p->nfields = (ncomp == 3) ? 3 : ((b == SF_BC_PERIODIC) ? 1 + ndim : 1);
    const long long n1 = p->n[1], n2 = (ndim == 3) ? p->n[2] : 1;
    const long long P1 = p->padded ? 2 * n1 : n1;
    p->w1_field = p->pitch * n1 * n2;
    p->w2_field = p->pitch * P1 * n2;
    const size_t welem = (p->r2r == R2R_NONE) ? 2 * p->esize : p->esize;

    // shared-memory feasibility of the fused kernel for this plan's worst case
    {
        const int ax = ndim - 1;
        const int nbuf = (ncomp == 3) ? 3 : 1;   // sf_gradient checks its own two tiles when it is called
        const size_t need = (prec == SF_F32) ? spass_smem_bytes<float>(p->La[ax], nbuf) : spass_smem_bytes<double>(p->La[ax], nbuf);
        if (need > 227 * 1024) return bail(SF_ERR_UNSUPPORTED, "fused pass does not fit in shared memory for this size / precision / field count");
    }

    sf_status st;
    if ((st = dev_alloc(p, &p->W1, (size_t)p->w1_field * p->nfields * welem)) != SF_OK) return bail(st, "");
    if (p->padded) {
        if ((st = dev_alloc(p, &p->W2, (size_t)p->w2_field * p->nfields * welem)) != SF_OK) return bail(st, "");
    } else {
        p->W2 = p->W1;
    }
    if ((st = dev_alloc(p, &p->out, field_elems(p) * p->nfields * p->esize)) != SF_OK) return bail(st, "");
    // pitch padding columns are read by the strided passes' neighbours only through masked loads,
    // but keep the workspaces defined
    if (cudaMemsetAsync(p->W1, 0, (size_t)p->w1_field * p->nfields * welem, p->stream) != cudaSuccess) return bail(SF_ERR_CUDA, "memset failed");
    if (p->padded && cudaMemsetAsync(p->W2, 0, (size_t)p->w2_field * p->nfields * welem, p->stream) != cudaSuccess) return bail(SF_ERR_CUDA, "memset failed");

    st = (prec == SF_F32) ? build_tables<float>(p) : build_tables<double>(p);
    if (st != SF_OK) return bail(st, "");

    // kernel generation 2 covers fp32 scalar unbounded plans whose y and z pencils are 256 long
    if (prec == SF_F32 && b == SF_BC_UNBOUNDED && ndim == 3 && ncomp == 1 && p->n[1] == 256 && p->n[2] == 256 &&
        (p->nspec_x % sf2::kTile) <= 1 && p->nspec_x >= sf2::kTile && is_pow2(p->nspec_x / sf2::kTile) && p->n[0] <= 2048 &&
        !getenv("SF_DISABLE_FAST")) {
        if (sf2::fast_init() != cudaSuccess) { cudaGetLastError(); return bail(SF_ERR_CUDA, "set-up of the fp32 fast path failed"); }
        const unsigned long long hpB = (unsigned long long)p->pitch * 8ull, N1 = 256, N2 = 256, PP = 512;
        const unsigned long long hpc = (unsigned long long)p->pitch;
        cudaError_t e1, e2, e3;
        {
            const unsigned long long d[4] = { hpc, N1, N2, 1 }, sb[3] = { hpB, hpB * N1, hpB * N1 * N2 };
            const unsigned bx[4] = { 16, 256, 1, 1 };
            e1 = sf2::fast_make_map(&p->map_s2, p->W1, d, sb, bx);
        }
        {
            const unsigned long long d[4] = { hpc, PP, N2, 1 }, sb[3] = { hpB, hpB * PP, hpB * PP * N2 };
            const unsigned bx[4] = { 16, 1, 256, 1 };
            e2 = sf2::fast_make_map(&p->map_s3, p->W2, d, sb, bx);
        }
        p->map_s4 = p->map_s3; e3 = cudaSuccess;   // S4 loads straight into registers: no map of its own
        if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess) return bail(SF_ERR_CUDA, "tensor map encoding failed");
        {
            const int nct = p->nspec_x / sf2::kTile, nyq = (p->nspec_x % sf2::kTile) ? nct * sf2::kTile : -1;
            const size_t ne = sf2::fast_green_tiles_elems(512, nct, nyq);
            if ((st = dev_alloc(p, &p->green_tiles, ne * sizeof(float))) != SF_OK) return bail(st, "");
            if (sf2::fast_green_tiles((float*)p->green_tiles, (const float*)p->green, p->pitch, p->pitch * (p->n[1] + 1), 512, nct, nyq,
                                      p->stream) != cudaSuccess)
                return bail(SF_ERR_CUDA, "building the tile-major Green's table failed");
        }
        if ((st = dev_alloc(p, &p->sched, 2 * sizeof(int))) != SF_OK) return bail(st, "");
        if (cudaMemsetAsync(p->sched, 0, 2 * sizeof(int), p->stream) != cudaSuccess) return bail(SF_ERR_CUDA, "memset failed");
        p->fast = true;
        p->fast_x = (p->n[0] == 256) && p->pitch >= 258 && !getenv("SF_DISABLE_FAST_X");
        if (p->nspec_x % sf2::kTile) {   // the Nyquist column lives in two side arrays ([y][z] and [z][ky])
            if ((st = dev_alloc(p, &p->nyqA, (size_t)256 * 256 * 8)) != SF_OK) return bail(st, "");
            if ((st = dev_alloc(p, &p->nyqB, (size_t)256 * 512 * 8)) != SF_OK) return bail(st, "");
        }
    }
    // ... fp64 scalar unbounded plans whose y and z pencils are 256 long (tiles of 8 columns)
    if (prec == SF_F64 && b == SF_BC_UNBOUNDED && ndim == 3 && ncomp == 1 && p->n[1] == 256 && p->n[2] == 256 && (p->nspec_x % 8) <= 1 &&
        p->nspec_x >= 8 && is_pow2(p->nspec_x / 8) && p->n[0] <= 1024 && !getenv("SF_DISABLE_FAST")) {
        if (sf2::fast_init() != cudaSuccess) { cudaGetLastError(); return bail(SF_ERR_CUDA, "set-up of the fast path failed"); }
        // the tensor maps address the complex doubles as pairs of 8-byte words
        const unsigned long long hpB = (unsigned long long)p->pitch * 16ull, N1 = 256, N2 = 256, PP = 512;
        const unsigned long long hpw = 2ull * (unsigned long long)p->pitch;
        cudaError_t e1, e2;
        {
            const unsigned long long d[4] = { hpw, N1, N2, 1 }, sb[3] = { hpB, hpB * N1, hpB * N1 * N2 };
            const unsigned bx[4] = { 16, 256, 1, 1 };
            e1 = sf2::fast_make_map(&p->map_s2, p->W1, d, sb, bx);
        }
        {
            const unsigned long long d[4] = { hpw, PP, N2, 1 }, sb[3] = { hpB, hpB * PP, hpB * PP * N2 };
            const unsigned bx[4] = { 16, 1, 256, 1 };
            e2 = sf2::fast_make_map(&p->map_s3, p->W2, d, sb, bx);
        }
        p->map_s4 = p->map_s3;
        if (e1 != cudaSuccess || e2 != cudaSuccess) return bail(SF_ERR_CUDA, "tensor map encoding failed");
        {
            const int nct = p->nspec_x / 8, nyq = (p->nspec_x % 8) ? nct * 8 : -1;
            const size_t ne = sf2::fast64_green_tiles_elems(512, nct, nyq);
            if ((st = dev_alloc(p, &p->green_tiles, ne * sizeof(double))) != SF_OK) return bail(st, "");
            if (sf2::fast64_green_tiles((double*)p->green_tiles, (const double*)p->green, p->pitch, p->pitch * (p->n[1] + 1), 512, nct, nyq,
                                        p->stream) != cudaSuccess)
                return bail(SF_ERR_CUDA, "building the tile-major Green's table failed");
        }
        if ((st = dev_alloc(p, &p->sched, 2 * sizeof(int))) != SF_OK) return bail(st, "");
        if (cudaMemsetAsync(p->sched, 0, 2 * sizeof(int), p->stream) != cudaSuccess) return bail(SF_ERR_CUDA, "memset failed");
        p->fast64 = true;
    }
    // ... fp32 unbounded plans whose y and z pencils are 512 long (BASELINE.json configs[4]: three components, curl)
    if (prec == SF_F32 && b == SF_BC_UNBOUNDED && ndim == 3 && p->n[1] == 512 && p->n[2] == 512 && (p->nspec_x % sf2::kTile) <= 1 &&
        p->nspec_x >= sf2::kTile && is_pow2(p->nspec_x / sf2::kTile) && p->n[0] <= 1024 && !getenv("SF_DISABLE_FAST")) {
        if (sf2::fast_init() != cudaSuccess) { cudaGetLastError(); return bail(SF_ERR_CUDA, "set-up of the fp32 fast path failed"); }
        const unsigned long long hpB = (unsigned long long)p->pitch * 8ull, N1 = 512, N2 = 512, PP = 1024;
        const unsigned long long hpc = (unsigned long long)p->pitch;
        cudaError_t e1, e2;
        {
            // S2: W1 as (column, y, batch = component * n2 + z)
            const unsigned long long d[4] = { hpc, N1, N2 * (unsigned long long)ncomp, 1 }, sb[3] = { hpB, hpB * N1, hpB * N1 * N2 * ncomp };
            const unsigned bx[4] = { 8, 256, 1, 1 };
            e1 = sf2::fast_make_map(&p->map_s2, p->W1, d, sb, bx);
        }
        {
            // S3: W2 as (column, ky, z, component); the multiplying passes work on tiles of 8 columns
            const unsigned long long d[4] = { hpc, PP, N2, (unsigned long long)ncomp }, sb[3] = { hpB, hpB * PP, hpB * PP * N2 };
            const unsigned bx[4] = { 8, 1, 256, 1 };
            e2 = sf2::fast_make_map(&p->map_s3, p->W2, d, sb, bx);
        }
        p->map_s4 = p->map_s3;   // S4 loads straight into registers: no map of its own
        if (e1 != cudaSuccess || e2 != cudaSuccess) return bail(SF_ERR_CUDA, "tensor map encoding failed");
        {
            const int nct = p->nspec_x / 8, nyq = (p->nspec_x % 8) ? nct * 8 : -1;
            const size_t ne = sf2::fast_green_tiles_elems_rows_w(1024, nct, nyq, sf2::kGreenRows5, 8);
            if ((st = dev_alloc(p, &p->green_tiles, ne * sizeof(float))) != SF_OK) return bail(st, "");
            if (sf2::fast_green_tiles_rows_w((float*)p->green_tiles, (const float*)p->green, p->pitch, p->pitch * (p->n[1] + 1), 1024, nct, nyq,
                                             sf2::kGreenRows5, 8, p->stream) != cudaSuccess)
                return bail(SF_ERR_CUDA, "building the tile-major Green's table failed");
        }
        if ((st = dev_alloc(p, &p->sched, 2 * sizeof(int))) != SF_OK) return bail(st, "");
        if (cudaMemsetAsync(p->sched, 0, 2 * sizeof(int), p->stream) != cudaSuccess) return bail(SF_ERR_CUDA, "memset failed");
        p->fast5 = true;
        p->fast5_x = (p->n[0] == 512) && p->pitch >= 514 && !getenv("SF_DISABLE_FAST_X");
    }
    // ... and periodic fp32 scalar plans with 256-point y and z pencils (strided passes only)
    if (prec == SF_F32 && b == SF_BC_PERIODIC && ndim == 3 && ncomp == 1 && p->n[1] == 256 && p->n[2] == 256 &&
        p->nspec_x >= sf2::kPerTileCols && (p->nspec_x % sf2::kPerTileCols) <= 1 && p->n[0] <= 4096 && !getenv("SF_DISABLE_FAST")) {
        if (sf2::fast_init() != cudaSuccess) { cudaGetLastError(); return bail(SF_ERR_CUDA, "set-up of the fp32 fast path failed"); }
        if ((st = dev_alloc(p, &p->sched, 2 * sizeof(int))) != SF_OK) return bail(st, "");
        if (cudaMemsetAsync(p->sched, 0, 2 * sizeof(int), p->stream) != cudaSuccess) return bail(SF_ERR_CUDA, "memset failed");
        if ((st = dev_alloc(p, &p->nyqA, (size_t)p->nfields * p->n[1] * p->n[2] * 8)) != SF_OK) return bail(st, "");   // Nyquist column [field][z][y]
        p->fastper = true;
        p->fastper_x = (p->n[0] == 256) && !getenv("SF_DISABLE_FAST_X");
    }
    // ... and the same in double precision
    if (prec == SF_F64 && b == SF_BC_PERIODIC && ndim == 3 && ncomp == 1 && p->n[1] == 256 && p->n[2] == 256 && p->nspec_x >= 16 &&
        (p->nspec_x % 16) <= 1 && p->n[0] <= 4096 && !getenv("SF_DISABLE_FAST")) {
        if (sf2::fast_init() != cudaSuccess) { cudaGetLastError(); return bail(SF_ERR_CUDA, "set-up of the fast path failed"); }
        if ((st = dev_alloc(p, &p->sched, 2 * sizeof(int))) != SF_OK) return bail(st, "");
        if (cudaMemsetAsync(p->sched, 0, 2 * sizeof(int), p->stream) != cudaSuccess) return bail(SF_ERR_CUDA, "memset failed");
        if ((st = dev_alloc(p, &p->nyqA, (size_t)p->nfields * p->n[1] * p->n[2] * 16)) != SF_OK) return bail(st, "");   // Nyquist column [field][z][y]
        p->fastper64 = true;
    }
    // fp64 Dirichlet / Neumann plans with 255- / 256-long y and z pencils: generation-2 strided passes
    if (prec == SF_F64 && ndim == 3 && ncomp == 1 && !p->mixed && !getenv("SF_DISABLE_FAST") &&
        ((p->r2r == R2R_DST1 && p->n[1] == 255 && p->n[2] == 255) || (p->r2r == R2R_DCT && p->n[1] == 256 && p->n[2] == 256))) {
        if (sf2::fast_init() != cudaSuccess) { cudaGetLastError(); return bail(SF_ERR_CUDA, "set-up of the fast path failed"); }
        // the real work array as 8-byte words: (column, y, z); a tile is 16 words x all rows of a pencil
        const unsigned long long hpw = (unsigned long long)p->pitch, hpB = hpw * 8ull, N1 = (unsigned long long)p->n[1], N2 = (unsigned long long)p->n[2];
        const unsigned long long d[4] = { hpw, N1, N2, 1 }, sb[3] = { hpB, hpB * N1, hpB * N1 * N2 };
        const unsigned bx2[4] = { 16, (unsigned)N1, 1, 1 }, bx3[4] = { 16, 1, (unsigned)N2, 1 };
        if (sf2::fast_make_map(&p->map_s2, p->W1, d, sb, bx2) != cudaSuccess || sf2::fast_make_map(&p->map_s3, p->W1, d, sb, bx3) != cudaSuccess)
            return bail(SF_ERR_CUDA, "tensor map encoding failed");
        if (!p->sched) {
            if ((st = dev_alloc(p, &p->sched, 2 * sizeof(int))) != SF_OK) return bail(st, "");
            if (cudaMemsetAsync(p->sched, 0, 2 * sizeof(int), p->stream) != cudaSuccess) return bail(SF_ERR_CUDA, "memset failed");
        }
        p->r2r64 = true;
    }
    // fp64 X passes of generation 2: rows whose extended sequence is 512 long
    if (prec == SF_F64 && p->Lx == 256 && (p->xmode == X_ZEROPAD || p->xmode == X_DST1 || p->xmode == X_DCT2) && !getenv("SF_DISABLE_FAST") &&
        !getenv("SF_DISABLE_FAST_X")) {
        if (sf2::fast_init() != cudaSuccess) { cudaGetLastError(); return bail(SF_ERR_CUDA, "set-up of the fast path failed"); }
        p->xg64 = true;
    }
    if (prec == SF_F64 && p->xmode == X_PERIODIC && p->n[0] == 256 && !getenv("SF_DISABLE_FAST") && !getenv("SF_DISABLE_FAST_X")) {
        if (sf2::fast_init() != cudaSuccess) { cudaGetLastError(); return bail(SF_ERR_CUDA, "set-up of the fast path failed"); }
        p->xp64 = true;
    }
    // everything the plan built (uploads on the legacy stream, kernels and memsets on the plan's stream) is complete
    // before the first compute call can be enqueued
    if (cudaDeviceSynchronize() != cudaSuccess) return bail(SF_ERR_CUDA, "plan construction failed on the device");
    *out = p;
    return SF_OK;
}

sf_status sf_set_source(sf_plan plan, const void* src, sf_mem where)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (!src) return fail(plan, SF_ERR_INVALID_ARG, "src is NULL");
    if (where == SF_MEM_DEVICE) {
        if (((uintptr_t)src & 15) != 0) return fail(plan, SF_ERR_INVALID_ARG, "device source must be 16-byte aligned");
        plan->src = src;
        plan->src_piped = false;
        return SF_OK;
    }
    if (where != SF_MEM_HOST) return fail(plan, SF_ERR_INVALID_ARG, "unknown memory space");
    const size_t bytes = field_elems(plan) * plan->ncomp * plan->esize;
    if (plan->pipe >= 2) {
        // the copy runs on its own stream into the slot the compute call before last read
        plan->ss ^= 1;
        const int s = plan->ss;
        if (plan->src_free_set[s]) SF_CUDA(plan, cudaStreamWaitEvent(plan->st_h2d, plan->ev_src_free[s], 0));
        SF_CUDA(plan, cudaMemcpyAsync(plan->psrc[s], src, bytes, cudaMemcpyHostToDevice, plan->st_h2d));
        SF_CUDA(plan, cudaEventRecord(plan->ev_src_ready[s], plan->st_h2d));
        plan->src = plan->psrc[s];
        plan->src_piped = true;
        return SF_OK;
    }
    if (!plan->src_own) {
        sf_status st = dev_alloc(plan, &plan->src_own, bytes);
        if (st != SF_OK) return st;
    }
    SF_CUDA(plan, cudaMemcpyAsync(plan->src_own, src, bytes, cudaMemcpyHostToDevice, plan->stream));
    plan->src = plan->src_own;
    return SF_OK;
}

sf_status sf_set_bc_values(sf_plan plan, int axis, int side, const void* face, sf_mem where)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (axis < 0 || axis >= plan->ndim || side < 0 || side > 1) return fail(plan, SF_ERR_INVALID_ARG, "axis / side out of range");
    if (plan->bca[axis] != SF_BC_DIRICHLET && plan->bca[axis] != SF_BC_NEUMANN)
        return fail(plan, SF_ERR_UNSUPPORTED, "boundary values apply to Dirichlet / Neumann plans only (PAPER.md:302)");
    if (plan->op != SF_OP_FD2) return fail(plan, SF_ERR_UNSUPPORTED, "boundary values need the FD2 operator (PAPER.md:173)");
    const int i = 2 * axis + side;
    if (!face) { plan->face[i] = nullptr; return SF_OK; }
    if (where == SF_MEM_DEVICE) { plan->face[i] = face; return SF_OK; }
    if (where != SF_MEM_HOST) return fail(plan, SF_ERR_INVALID_ARG, "unknown memory space");
    size_t cnt = 1;
    for (int a = 0; a < plan->ndim; ++a) if (a != axis) cnt *= (size_t)plan->n[a];
    if (!plan->face_own[i]) {
        sf_status st = dev_alloc(plan, &plan->face_own[i], cnt * plan->esize);
        if (st != SF_OK) return st;
    }
    SF_CUDA(plan, cudaMemcpyAsync(plan->face_own[i], face, cnt * plan->esize, cudaMemcpyHostToDevice, plan->stream));
    plan->face[i] = plan->face_own[i];
    return SF_OK;
}

sf_status sf_solve(sf_plan plan) { return run_any(plan, OUT_SOLVE); }

sf_status sf_gradient(sf_plan plan)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (plan->ncomp != 1) return fail(plan, SF_ERR_UNSUPPORTED, "sf_gradient is built for scalar plans");
    if (plan->mixed) return fail(plan, SF_ERR_UNSUPPORTED, "sf_gradient is not built for plans with mixed boundary conditions");
    {
        // the fused pass holds two tiles (psi and one derivative)
        const int ax = plan->ndim - 1;
        const size_t need = (plan->prec == SF_F32) ? spass_smem_bytes<float>(plan->La[ax], 2) : spass_smem_bytes<double>(plan->La[ax], 2);
        if (need > 227 * 1024 && !plan->fastper && !plan->fastper64)
            return fail(plan, SF_ERR_UNSUPPORTED, "gradient: the fused pass does not fit in shared memory for this size / precision");
    }
    if (plan->bc == SF_BC_PERIODIC) return run_any(plan, OUT_GRAD);
    if (plan->ndim != 3 && plan->bc != SF_BC_UNBOUNDED)
        return fail(plan, SF_ERR_UNSUPPORTED, "sf_gradient on Dirichlet / Neumann plans is built for 3-D");
    // unbounded, Dirichlet, Neumann: psi and its derivatives need 1 + ndim fields of work space
    const int nf = 1 + plan->ndim;
    const size_t welem = (plan->r2r == R2R_NONE) ? 2 * plan->esize : plan->esize;
    if (!plan->gout) {
        // all three arrays or none: a half-made set must never be swapped in (the next call would launch on NULL)
        sf_status st;
        const size_t b1 = (size_t)plan->w1_field * nf * welem, b2 = (size_t)plan->w2_field * nf * welem;
        void *w1 = nullptr, *w2 = nullptr, *go = nullptr;
        st = dev_alloc(plan, &w1, b1);
        if (st == SF_OK && plan->padded) st = dev_alloc(plan, &w2, b2);
        if (st == SF_OK) st = dev_alloc(plan, &go, field_elems(plan) * nf * plan->esize);
        if (st != SF_OK) {
            const std::string msg = plan->err;
            if (w1) { dev_free(plan, w1); plan->dev_bytes -= (long long)b1; }
            if (w2) { dev_free(plan, w2); plan->dev_bytes -= (long long)b2; }
            plan->err = msg;
            return st;
        }
        SF_CUDA(plan, cudaMemsetAsync(w1, 0, b1, plan->stream));
        if (w2) SF_CUDA(plan, cudaMemsetAsync(w2, 0, b2, plan->stream));
        plan->gW1 = w1;
        plan->gW2 = plan->padded ? w2 : w1;
        plan->gout = go;
    }
    std::swap(plan->W1, plan->gW1);
    std::swap(plan->W2, plan->gW2);
    std::swap(plan->out, plan->gout);
    const sf_status st = run_any(plan, OUT_GRAD);
    std::swap(plan->W1, plan->gW1);
    std::swap(plan->W2, plan->gW2);
    std::swap(plan->out, plan->gout);
    return st;
}

sf_status sf_curl(sf_plan plan)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (plan->ncomp != 3) return fail(plan, SF_ERR_UNSUPPORTED, "sf_curl needs an ncomp == 3 plan");
    if (plan->bc != SF_BC_PERIODIC && plan->bc != SF_BC_UNBOUNDED)
        return fail(plan, SF_ERR_UNSUPPORTED, "sf_curl is built for periodic and unbounded plans");
    return run_any(plan, OUT_CURL);
}

sf_status sf_divergence(sf_plan plan)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (plan->ncomp != 3) return fail(plan, SF_ERR_UNSUPPORTED, "sf_divergence needs an ncomp == 3 plan");
    if (plan->bc != SF_BC_PERIODIC && plan->bc != SF_BC_UNBOUNDED)
        return fail(plan, SF_ERR_UNSUPPORTED, "sf_divergence is built for periodic and unbounded plans");
    return run_any(plan, OUT_DIV);
}

sf_status sf_laplacian(sf_plan plan)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (plan->bc != SF_BC_PERIODIC && plan->bc != SF_BC_UNBOUNDED)
        return fail(plan, SF_ERR_UNSUPPORTED, "sf_laplacian is built for periodic and unbounded plans");
    if (plan->bc == SF_BC_UNBOUNDED && plan->ndim != 3) return fail(plan, SF_ERR_UNSUPPORTED, "sf_laplacian on unbounded plans is built for 3-D");
    return run_any(plan, OUT_LAP);
}

sf_status sf_output_device_ptr(sf_plan plan, int field, int comp, void** ptr)
{
    if (!plan || !ptr) return SF_ERR_INVALID_ARG;
    int idx = -1;
    if (plan->last_kind < 0) return fail(plan, SF_ERR_STATE, "no result yet: call sf_solve / sf_gradient / sf_curl first");
    if (field == SF_OUT_PSI) {
        if (plan->last_kind != OUT_SOLVE && plan->last_kind != OUT_GRAD)
            return fail(plan, SF_ERR_STATE, "psi was not produced by the last call (sf_curl, sf_divergence and sf_laplacian return only their own field)");
        if (comp < 0 || comp >= plan->ncomp) return fail(plan, SF_ERR_INVALID_ARG, "component out of range");
        idx = comp;
    } else if (field == SF_OUT_GRAD) {
        if (plan->last_kind != OUT_GRAD) return fail(plan, SF_ERR_STATE, "gradient was not produced by the last call");
        if (comp < 0 || comp >= plan->ndim) return fail(plan, SF_ERR_INVALID_ARG, "axis out of range");
        idx = 1 + comp;
    } else if (field == SF_OUT_CURL) {
        if (plan->last_kind != OUT_CURL) return fail(plan, SF_ERR_STATE, "curl was not produced by the last call");
        if (comp < 0 || comp >= 3) return fail(plan, SF_ERR_INVALID_ARG, "component out of range");
        idx = comp;
    } else if (field == SF_OUT_DIV) {
        if (plan->last_kind != OUT_DIV) return fail(plan, SF_ERR_STATE, "divergence was not produced by the last call");
        if (comp != 0) return fail(plan, SF_ERR_INVALID_ARG, "the divergence is one field: comp must be 0");
        idx = 0;
    } else if (field == SF_OUT_LAP) {
        if (plan->last_kind != OUT_LAP) return fail(plan, SF_ERR_STATE, "Laplacian was not produced by the last call");
        if (comp < 0 || comp >= plan->ncomp) return fail(plan, SF_ERR_INVALID_ARG, "component out of range");
        idx = comp;
    } else {
        return fail(plan, SF_ERR_INVALID_ARG, "unknown field");
    }
    *ptr = (char*)plan->out_last + (size_t)idx * field_elems(plan) * plan->esize;
    return SF_OK;
}

sf_status sf_get_output(sf_plan plan, int field, int comp, void* dst, sf_mem where)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (!dst) return fail(plan, SF_ERR_INVALID_ARG, "dst is NULL");
    void* src = nullptr;
    sf_status st = sf_output_device_ptr(plan, field, comp, &src);
    if (st != SF_OK) return st;
    const size_t bytes = field_elems(plan) * plan->esize;
    if (where == SF_MEM_DEVICE) {
        SF_CUDA(plan, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, plan->stream));
    } else if (where == SF_MEM_HOST) {
        SF_CUDA(plan, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, plan->stream));
        SF_CUDA(plan, cudaStreamSynchronize(plan->stream));
    } else {
        return fail(plan, SF_ERR_INVALID_ARG, "unknown memory space");
    }
    return SF_OK;
}

sf_status sf_synchronize(sf_plan plan)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    SF_CUDA(plan, cudaStreamSynchronize(plan->stream));
    if (plan->st_h2d) SF_CUDA(plan, cudaStreamSynchronize(plan->st_h2d));
    if (plan->st_d2h) SF_CUDA(plan, cudaStreamSynchronize(plan->st_d2h));
    return SF_OK;
}

sf_status sf_set_pipeline(sf_plan plan, int depth)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (depth != 1 && depth != 2) return fail(plan, SF_ERR_INVALID_ARG, "pipeline depth must be 1 or 2");
    sf_status st = sf_synchronize(plan);
    if (st != SF_OK) return st;
    if (depth == 2 && !plan->st_h2d) {
        // second source and result buffers, two copy streams, the events that order them against the plan's stream
        const size_t sbytes = field_elems(plan) * plan->ncomp * plan->esize, obytes = field_elems(plan) * plan->nfields * plan->esize;
        if (!plan->src_own && (st = dev_alloc(plan, &plan->src_own, sbytes)) != SF_OK) return st;
        void *s1 = nullptr, *o1 = nullptr;
        if ((st = dev_alloc(plan, &s1, sbytes)) != SF_OK) return st;
        if ((st = dev_alloc(plan, &o1, obytes)) != SF_OK) { dev_free(plan, s1); plan->dev_bytes -= (long long)sbytes; return st; }
        plan->psrc[0] = plan->src_own; plan->psrc[1] = s1;
        plan->pout[0] = plan->out; plan->pout[1] = o1;
        SF_CUDA(plan, cudaStreamCreateWithFlags(&plan->st_h2d, cudaStreamNonBlocking));
        SF_CUDA(plan, cudaStreamCreateWithFlags(&plan->st_d2h, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            SF_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_src_ready[i], cudaEventDisableTiming));
            SF_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_src_free[i], cudaEventDisableTiming));
            SF_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_done[i], cudaEventDisableTiming));
            SF_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_out_free[i], cudaEventDisableTiming));
        }
    }
    if (depth == 1 && plan->pipe == 2) {
        // back to one stream: results land in the first buffer again; a piped source stays where it is (the device is idle)
        if (plan->out == plan->pout[1]) plan->out = plan->pout[0];
        plan->src_piped = false;
        for (int i = 0; i < 2; ++i) plan->src_free_set[i] = plan->out_free_set[i] = plan->done_set[i] = false;
    }
    plan->pipe = depth;
    return SF_OK;
}

sf_status sf_get_output_async(sf_plan plan, int field, int comp, void* dst_host)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (!dst_host) return fail(plan, SF_ERR_INVALID_ARG, "dst is NULL");
    void* src = nullptr;
    sf_status st = sf_output_device_ptr(plan, field, comp, &src);
    if (st != SF_OK) return st;
    const size_t bytes = field_elems(plan) * plan->esize;
    if (plan->pipe < 2) {
        SF_CUDA(plan, cudaMemcpyAsync(dst_host, src, bytes, cudaMemcpyDeviceToHost, plan->stream));
        return SF_OK;
    }
    const int o = plan->os;
    if (plan->done_set[o]) SF_CUDA(plan, cudaStreamWaitEvent(plan->st_d2h, plan->ev_done[o], 0));
    SF_CUDA(plan, cudaMemcpyAsync(dst_host, src, bytes, cudaMemcpyDeviceToHost, plan->st_d2h));
    SF_CUDA(plan, cudaEventRecord(plan->ev_out_free[o], plan->st_d2h));
    plan->out_free_set[o] = true;
    return SF_OK;
}

sf_status sf_pipeline_join(sf_plan plan)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (plan->pipe < 2) return SF_OK;
    for (int i = 0; i < 2; ++i) {
        if (plan->out_free_set[i]) SF_CUDA(plan, cudaStreamWaitEvent(plan->stream, plan->ev_out_free[i], 0));
    }
    if (plan->src_piped) SF_CUDA(plan, cudaStreamWaitEvent(plan->stream, plan->ev_src_ready[plan->ss], 0));
    return SF_OK;
}

sf_status sf_probe_dft16_stage(int variant, int reps, int ntiles, const void* in_dev, void* out_dev, float* ms)
{
    if (sf2::fast_init() != cudaSuccess) { cudaGetLastError(); return fail(nullptr, SF_ERR_CUDA, "set-up of the fast path failed"); }
    const cudaError_t e = sf2::probe_dft16_stage(variant, reps, ntiles, in_dev, out_dev, ms, nullptr);
    if (e == cudaErrorInvalidValue) { cudaGetLastError(); return fail(nullptr, SF_ERR_INVALID_ARG, "probe: bad argument"); }
    if (e != cudaSuccess) { cudaGetLastError(); return fail(nullptr, SF_ERR_CUDA, std::string("probe: ") + cudaGetErrorString(e)); }
    return SF_OK;
}

int sf_last_launch_count(sf_plan plan) { return plan ? plan->launches : 0; }
long long sf_device_bytes(sf_plan plan) { return plan ? plan->dev_bytes : 0; }

sf_status sf_enable_step_timing(sf_plan plan, int slots)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (slots < 0 || slots > 4096) return fail(plan, SF_ERR_INVALID_ARG, "slots must be in [0, 4096]");
    while ((int)plan->ev.size() < 6 * slots) {
        cudaEvent_t e = nullptr;
        SF_CUDA(plan, cudaEventCreate(&e));
        plan->ev.push_back(e);
    }
    plan->tslots = slots;
    plan->tcount = 0;
    plan->tcalls = 0;
    return SF_OK;
}

sf_status sf_set_step_timing_stride(sf_plan plan, int stride)
{
    if (!plan) return SF_ERR_INVALID_ARG;
    if (stride < 1) return fail(plan, SF_ERR_INVALID_ARG, "stride must be >= 1");
    plan->tstride = stride;
    return SF_OK;
}

sf_status sf_step_times_ms(sf_plan plan, float ms[5])
{
    if (!plan || !ms) return SF_ERR_INVALID_ARG;
    if (!plan->tslots || plan->tcount == 0) return fail(plan, SF_ERR_STATE, "no timed compute call: enable step timing, then solve");
    const int nrec = (int)(plan->tcount < plan->tslots ? plan->tcount : plan->tslots);
    double acc[5] = { 0, 0, 0, 0, 0 };
    for (int s = 0; s < nrec; ++s) {
        SF_CUDA(plan, cudaEventSynchronize(plan->ev[6 * s + 5]));
        for (int i = 0; i < 5; ++i) {
            float t = 0.f;
            SF_CUDA(plan, cudaEventElapsedTime(&t, plan->ev[6 * s + i], plan->ev[6 * s + i + 1]));
            acc[i] += t;
        }
    }
    for (int i = 0; i < 5; ++i) ms[i] = (float)(acc[i] / nrec);
    return SF_OK;
}

} // extern "C"
