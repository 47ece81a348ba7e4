/*
 * sf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision CPU restatement of the spectral Poisson solve of
 * SailFFish (arxiv 2301.01145), written from the paper only.  It shares no code with the
 * CUDA path under paper_2301_01145_b200/ and must never be imported, linked or executed by
 * it.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md):
 *   - the four-step solve: forward DFT, multiply by the spectral multiplier, optional
 *     spectral operations, backward DFT                         (sec 2.2)
 *   - DFT definitions, unnormalised forward, 1/N on the inverse  (eq. 8)
 *   - N-D transforms as successive 1-D pencils, inverse in reverse order
 *   - Table 1: transform type and eigenvalues per BC / grid type
 *   - k = 0 mode set to zero
 *   - spectral differentiation by multiplying with ik            (eq. 10)
 *   - inhomogeneous BC values folded into boundary-adjacent source cells, FD2 only
 *
 *   - Hockney-Eastwood: doubled domain, mirrored Green's function, zero-padded source,
 *     periodic solve, extraction                                 (sec 2.5)
 *   - Green's function evaluated in real space and forward transformed once
 *   - 3-D vector solver = component-wise scalar solves
 * Readings of silent / garbled passages are those of SURVEY.md sec 8(c) (A1-A24), restated in
 * DESIGN.md.
 *
 * Structure: transforms are a recursive radix-2 FFT (power-of-two lengths) and direct O(N^2)
 * sine / cosine sums (DST-I, DCT-II, DCT-III); every trigonometric argument is reduced in
 * integer arithmetic before sin/cos is called.  N-D transforms copy one pencil at a time to a
 * contiguous buffer, transform it and copy it back; OpenMP runs independent pencils in
 * parallel and nothing else.  The unbounded solver treats the WHOLE doubled domain, as the
 * paper does: no pruning.
 *
 * Array layout everywhere: x fastest, index = ix + nx*(iy + ny*iz); vector fields are
 * component-major.
 *
 * Pins (tests/test_oracle_*.py): P1-P12 of SURVEY.md sec 8(c).  No function here is
 * "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;
typedef long long i64;

#define ORC_OK 0
#define ORC_ERR_ARG (-1)
#define ORC_ERR_ALLOC (-3)

static const double PI = 3.14159265358979323846264338327950288;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------------------------------
 * sin(2 pi p/q), cos(2 pi p/q) with the argument reduced exactly: p mod q in integers, then
 * reflections down to the first octant so that libm only ever sees an angle in [0, pi/4].
 * ---------------------------------------------------------------------------------------- */
static void sincos2pi(i64 p, i64 q, double *s, double *c)
{
    int neg_s = 0, neg_c = 0, swap = 0;
    p %= q;
    if (p < 0) p += q;
    if (2 * p > q) { p = q - p; neg_s = 1; }               /* a -> 2pi - a                 */
    if (4 * p > q) { p = q - 2 * p; q = 2 * q; neg_c = 1; } /* a -> pi - a   (p/q in [0,1/4]) */
    if (8 * p > q) { p = q - 4 * p; q = 4 * q; swap = 1; }  /* a -> pi/2 - a (p/q in [0,1/8]) */
    double a = 2.0 * PI * ((double)p / (double)q);
    double sv = sin(a), cv = cos(a);
    if (swap) { double t = sv; sv = cv; cv = t; }
    *s = neg_s ? -sv : sv;
    *c = neg_c ? -cv : cv;
}

/* ------------------------------------------------------------------------------------------
 * 1-D transforms
 * ---------------------------------------------------------------------------------------- */

/* Brute-force DFT straight from eq. (8), unnormalised in both directions:
 * out[k] = sum_n in[n] exp(sign * 2 pi i n k / N), sign = -1 forward, +1 backward. */
void orc_dft_direct(int n, int sign, const cplx *in, cplx *out)
{
    for (int k = 0; k < n; ++k) {
        long double sr = 0.0L, si = 0.0L;
        for (int j = 0; j < n; ++j) {
            double s, c;
            sincos2pi((i64)j * k, n, &s, &c);
            if (sign < 0) s = -s;
            double xr = creal(in[j]), xi = cimag(in[j]);
            sr += (long double)xr * c - (long double)xi * s;
            si += (long double)xr * s + (long double)xi * c;
        }
        out[k] = (double)sr + I * (double)si;
    }
}

/* twiddle table for a power-of-two length: tw[j] = exp(-2 pi i j / n), j < n */
static cplx *make_twiddles(int n)
{
    cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)(n > 0 ? n : 1));
    if (!tw) return NULL;
    for (int j = 0; j < n; ++j) {
        double s, c;
        sincos2pi(j, n, &s, &c);
        tw[j] = c - I * s;
    }
    return tw;
}

/* Recursive decimation-in-time radix-2 FFT (Cooley-Tukey, PAPER.md ref. [16]):
 *   X[k]       = E[k] + w^k O[k]
 *   X[k + n/2] = E[k] - w^k O[k],  w = exp(sign 2 pi i / n)
 * with E, O the transforms of the even / odd samples.  tw holds exp(-2 pi i j / ntop) and is
 * read with stride ntop/n; the backward transform conjugates it.  scratch has n entries. */
static void fft_rec(int n, int sign, const cplx *in, int istride, cplx *out, cplx *scratch,
                    const cplx *tw, int twstride)
{
    if (n == 1) { out[0] = in[0]; return; }
    int h = n / 2;
    fft_rec(h, sign, in, 2 * istride, scratch, out, tw, 2 * twstride);
    fft_rec(h, sign, in + istride, 2 * istride, scratch + h, out + h, tw, 2 * twstride);
    for (int k = 0; k < h; ++k) {
        cplx w = tw[(size_t)k * twstride];
        if (sign > 0) w = conj(w);
        cplx e = scratch[k], o = w * scratch[k + h];
        out[k] = e + o;
        out[k + h] = e - o;
    }
}

static int is_pow2(i64 n) { return n >= 1 && (n & (n - 1)) == 0; }

/* power-of-two FFT, unnormalised, sign = -1 forward / +1 backward. */
int orc_fft_pow2(int n, int sign, const cplx *in, cplx *out)
{
    if (!is_pow2(n)) return ORC_ERR_ARG;
    cplx *tw = make_twiddles(n);
    cplx *scratch = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    cplx *tmp = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!tw || !scratch || !tmp) { free(tw); free(scratch); free(tmp); return ORC_ERR_ALLOC; }
    memcpy(tmp, in, sizeof(cplx) * (size_t)n);
    fft_rec(n, sign, tmp, 1, out, scratch, tw, 1);
    free(tw); free(scratch); free(tmp);
    return ORC_OK;
}

/* DST-I:  Y_k = 2 sum_{j=0}^{N-1} X_j sin(pi (j+1)(k+1)/(N+1))   (Table 1 row 1; odd extension) */
void orc_dst1_direct(int n, const double *in, double *out)
{
    i64 q = 2 * ((i64)n + 1);
    for (int k = 0; k < n; ++k) {
        long double acc = 0.0L;
        for (int j = 0; j < n; ++j) {
            double s, c;
            sincos2pi((i64)(j + 1) * (k + 1), q, &s, &c);
            acc += (long double)in[j] * s;
        }
        out[k] = (double)(2.0L * acc);
    }
}

/* DCT-II: Y_k = 2 sum_{j=0}^{N-1} X_j cos(pi (j+1/2) k / N)      (Table 1 row 4; even extension) */
void orc_dct2_direct(int n, const double *in, double *out)
{
    i64 q = 4 * (i64)n;
    for (int k = 0; k < n; ++k) {
        long double acc = 0.0L;
        for (int j = 0; j < n; ++j) {
            double s, c;
            sincos2pi((i64)(2 * j + 1) * k, q, &s, &c);
            acc += (long double)in[j] * c;
        }
        out[k] = (double)(2.0L * acc);
    }
}

/* DCT-III: Y_j = X_0 + 2 sum_{k=1}^{N-1} X_k cos(pi k (j+1/2) / N)   (inverse of DCT-II up to 2N) */
void orc_dct3_direct(int n, const double *in, double *out)
{
    i64 q = 4 * (i64)n;
    for (int j = 0; j < n; ++j) {
        long double acc = 0.0L;
        for (int k = 1; k < n; ++k) {
            double s, c;
            sincos2pi((i64)(2 * j + 1) * k, q, &s, &c);
            acc += (long double)in[k] * c;
        }
        out[j] = (double)((long double)in[0] + 2.0L * acc);
    }
}

/* DST-II: Y_k = 2 sum_{j=0}^{N-1} X_j sin(pi (j+1/2) (k+1) / N)   (Table 1 row 2; odd extension about the
 * faces of a cell-centre grid) */
void orc_dst2_direct(int n, const double *in, double *out)
{
    i64 q = 4 * (i64)n;
    for (int k = 0; k < n; ++k) {
        long double acc = 0.0L;
        for (int j = 0; j < n; ++j) {
            double s, c;
            sincos2pi((i64)(2 * j + 1) * (k + 1), q, &s, &c);
            acc += (long double)in[j] * s;
        }
        out[k] = (double)(2.0L * acc);
    }
}

/* DST-III: Y_j = (-1)^j X_{N-1} + 2 sum_{k=0}^{N-2} X_k sin(pi (k+1) (j+1/2) / N)   (inverse of DST-II up to 2N) */
void orc_dst3_direct(int n, const double *in, double *out)
{
    i64 q = 4 * (i64)n;
    for (int j = 0; j < n; ++j) {
        long double acc = 0.0L;
        for (int k = 0; k + 1 < n; ++k) {
            double s, c;
            sincos2pi((i64)(2 * j + 1) * (k + 1), q, &s, &c);
            acc += (long double)in[k] * s;
        }
        out[j] = (double)(((j & 1) ? -1.0L : 1.0L) * (long double)in[n - 1] + 2.0L * acc);
    }
}

/* DCT-I: Y_k = X_0 + (-1)^k X_{N-1} + 2 sum_{j=1}^{N-2} X_j cos(pi j k / (N-1))   (Table 1 row 3; even extension
 * about the end nodes of a cell-boundary grid; its own inverse up to 2 (N-1)) */
void orc_dct1_direct(int n, const double *in, double *out)
{
    i64 q = 2 * (i64)(n - 1);
    for (int k = 0; k < n; ++k) {
        long double acc = 0.0L;
        for (int j = 1; j + 1 < n; ++j) {
            double s, c;
            sincos2pi((i64)j * k, q, &s, &c);
            acc += (long double)in[j] * c;
        }
        out[k] = (double)((long double)in[0] + ((k & 1) ? -1.0L : 1.0L) * (long double)in[n - 1] + 2.0L * acc);
    }
}

/* ------------------------------------------------------------------------------------------
 * Table-driven versions of the same sums for the N-D solvers (the table is the list of all
 * sin / cos values of the reduced integer argument; the sum is unchanged).
 * ---------------------------------------------------------------------------------------- */
typedef struct { int n; i64 q; double *sn; double *cs; } trig_table;

static int trig_table_init(trig_table *t, int n, i64 q)
{
    t->n = n; t->q = q;
    t->sn = (double *)malloc(sizeof(double) * (size_t)q);
    t->cs = (double *)malloc(sizeof(double) * (size_t)q);
    if (!t->sn || !t->cs) return ORC_ERR_ALLOC;
    for (i64 m = 0; m < q; ++m) sincos2pi(m, q, &t->sn[m], &t->cs[m]);
    return ORC_OK;
}
static void trig_table_free(trig_table *t) { free(t->sn); free(t->cs); t->sn = t->cs = NULL; }

static void dst1_tab(const trig_table *t, const double *in, double *out)
{
    int n = t->n;
    for (int k = 0; k < n; ++k) {
        long double acc = 0.0L;
        for (int j = 0; j < n; ++j)
            acc += (long double)in[j] * t->sn[((i64)(j + 1) * (k + 1)) % t->q];
        out[k] = (double)(2.0L * acc);
    }
}
static void dct2_tab(const trig_table *t, const double *in, double *out)
{
    int n = t->n;
    for (int k = 0; k < n; ++k) {
        long double acc = 0.0L;
        for (int j = 0; j < n; ++j)
            acc += (long double)in[j] * t->cs[((i64)(2 * j + 1) * k) % t->q];
        out[k] = (double)(2.0L * acc);
    }
}
static void dct3_tab(const trig_table *t, const double *in, double *out)
{
    int n = t->n;
    for (int j = 0; j < n; ++j) {
        long double acc = 0.0L;
        for (int k = 1; k < n; ++k)
            acc += (long double)in[k] * t->cs[((i64)(2 * j + 1) * k) % t->q];
        out[j] = (double)((long double)in[0] + 2.0L * acc);
    }
}

static void dst2_tab(const trig_table *t, const double *in, double *out)
{
    int n = t->n;
    for (int k = 0; k < n; ++k) {
        long double acc = 0.0L;
        for (int j = 0; j < n; ++j)
            acc += (long double)in[j] * t->sn[((i64)(2 * j + 1) * (k + 1)) % t->q];
        out[k] = (double)(2.0L * acc);
    }
}
static void dst3_tab(const trig_table *t, const double *in, double *out)
{
    int n = t->n;
    for (int j = 0; j < n; ++j) {
        long double acc = 0.0L;
        for (int k = 0; k + 1 < n; ++k)
            acc += (long double)in[k] * t->sn[((i64)(2 * j + 1) * (k + 1)) % t->q];
        out[j] = (double)(((j & 1) ? -1.0L : 1.0L) * (long double)in[n - 1] + 2.0L * acc);
    }
}
static void dct1_tab(const trig_table *t, const double *in, double *out)
{
    int n = t->n;
    for (int k = 0; k < n; ++k) {
        long double acc = 0.0L;
        for (int j = 1; j + 1 < n; ++j)
            acc += (long double)in[j] * t->cs[((i64)j * k) % t->q];
        out[k] = (double)((long double)in[0] + ((k & 1) ? -1.0L : 1.0L) * (long double)in[n - 1] + 2.0L * acc);
    }
}

/* ------------------------------------------------------------------------------------------
 * N-D helpers: apply a 1-D transform to every pencil along one axis of a dense array
 * (PAPER.md:89-97).  One pencil is copied to a contiguous buffer, transformed, copied back.
 * ---------------------------------------------------------------------------------------- */
static void axis_geometry(const i64 dims[3], int axis, i64 *len, i64 *stride, i64 *na, i64 *sa,
                          i64 *nb, i64 *sb)
{
    i64 st[3] = { 1, dims[0], dims[0] * dims[1] };
    int a = (axis + 1) % 3, b = (axis + 2) % 3;
    *len = dims[axis]; *stride = st[axis];
    *na = dims[a]; *sa = st[a];
    *nb = dims[b]; *sb = st[b];
}

/* complex FFT (power of two) along one axis, in place, unnormalised */
static int fft_axis(cplx *a, const i64 dims[3], int axis, int sign)
{
    i64 len, stride, na, sa, nb, sb;
    axis_geometry(dims, axis, &len, &stride, &na, &sa, &nb, &sb);
    if (!is_pow2(len)) return ORC_ERR_ARG;
    if (len == 1) return ORC_OK;
    cplx *tw = make_twiddles((int)len);
    if (!tw) return ORC_ERR_ALLOC;
    int err = ORC_OK;
#pragma omp parallel
    {
        cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)len * 3);
        if (!buf) {
#pragma omp critical
            err = ORC_ERR_ALLOC;
        }
#pragma omp for collapse(2) schedule(static)
        for (i64 ib = 0; ib < nb; ++ib)
            for (i64 ia = 0; ia < na; ++ia) {
                if (!buf) continue;
                cplx *p = a + ia * sa + ib * sb;
                cplx *in = buf, *out = buf + len, *scr = buf + 2 * len;
                for (i64 j = 0; j < len; ++j) in[j] = p[j * stride];
                fft_rec((int)len, sign, in, 1, out, scr, tw, 1);
                for (i64 j = 0; j < len; ++j) p[j * stride] = out[j];
            }
        free(buf);
    }
    free(tw);
    return err;
}

typedef void (*real_xform)(const trig_table *, const double *, double *);

/* real-to-real transform along one axis of a dense real array, in place */
static int r2r_axis(double *a, const i64 dims[3], int axis, real_xform fn, const trig_table *t)
{
    i64 len, stride, na, sa, nb, sb;
    axis_geometry(dims, axis, &len, &stride, &na, &sa, &nb, &sb);
    int err = ORC_OK;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * (size_t)len * 2);
        if (!buf) {
#pragma omp critical
            err = ORC_ERR_ALLOC;
        }
#pragma omp for collapse(2) schedule(static)
        for (i64 ib = 0; ib < nb; ++ib)
            for (i64 ia = 0; ia < na; ++ia) {
                if (!buf) continue;
                double *p = a + ia * sa + ib * sb;
                double *in = buf, *out = buf + len;
                for (i64 j = 0; j < len; ++j) in[j] = p[j * stride];
                fn(t, in, out);
                for (i64 j = 0; j < len; ++j) p[j * stride] = out[j];
            }
        free(buf);
    }
    return err;
}

/* ------------------------------------------------------------------------------------------
 * O-PER: periodic solver (configs 1, 2).
 *
 * nd = 2 or 3 (unused axes have n = 1).  Real data are stored as complex with zero imaginary
 * part and transformed with the plain C2C DFT, as the paper does.
 *   op = 0: pseudo-spectral  Lambda = - sum_a kappa_a^2, kappa_a = 2 pi m_a / L_a,
 *           m_a = k_a (k_a < N_a/2) else k_a - N_a             (Table 1)
 *   op = 1: FD2              Lambda = - sum_a (4/h_a^2) sin^2(pi k_a / N_a)
 * psi_hat = rhs_sign * F / Lambda, zero at the all-zero index; the 1/N of eq. (8)
 * is applied on the inverse.  Gradient: g_a = IDFT(i kappa_a psi_hat) (eq. 10) with
 * kappa_a := 0 at the Nyquist index (reading A20).
 * f, psi: n0*n1*n2 reals; grad (may be NULL): nd fields of that size, component-major.
 * ---------------------------------------------------------------------------------------- */
int orc_periodic(int nd, const i64 n[3], const double L[3], int op, double rhs_sign,
                 const double *f, double *psi, double *grad)
{
    if (nd < 1 || nd > 3) return ORC_ERR_ARG;
    i64 dims[3] = { n[0], nd > 1 ? n[1] : 1, nd > 2 ? n[2] : 1 };
    i64 tot = dims[0] * dims[1] * dims[2];
    for (int a = 0; a < 3; ++a) if (!is_pow2(dims[a])) return ORC_ERR_ARG;

    cplx *F = (cplx *)malloc(sizeof(cplx) * (size_t)tot);
    cplx *W = grad ? (cplx *)malloc(sizeof(cplx) * (size_t)tot) : NULL;
    double *kap[3] = { 0, 0, 0 }, *lam[3] = { 0, 0, 0 };
    int err = ORC_OK;
    if (!F || (grad && !W)) { err = ORC_ERR_ALLOC; goto done; }

    /* per-axis wavenumbers and eigenvalue contributions */
    for (int a = 0; a < 3; ++a) {
        i64 N = dims[a];
        kap[a] = (double *)calloc((size_t)N, sizeof(double));
        lam[a] = (double *)calloc((size_t)N, sizeof(double));
        if (!kap[a] || !lam[a]) { err = ORC_ERR_ALLOC; goto done; }
        if (a >= nd) continue; /* unused axis: single zero mode */
        double h = L[a] / (double)N;
        for (i64 k = 0; k < N; ++k) {
            i64 m = (2 * k < N) ? k : k - N;
            double kappa = 2.0 * PI * (double)m / L[a];
            kap[a][k] = (2 * k == N) ? 0.0 : kappa; /* used for ik only */
            if (op == 0) {
                lam[a][k] = -kappa * kappa;
            } else {
                double s, c;
                sincos2pi(k, 2 * N, &s, &c); /* sin(pi k / N) */
                lam[a][k] = -(4.0 / (h * h)) * s * s;
            }
        }
    }

    /* 1. forward transform (x, then y, then z) */
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < tot; ++i) F[i] = f[i];
    for (int a = 0; a < nd; ++a)
        if ((err = fft_axis(F, dims, a, -1)) != ORC_OK) goto done;

    /* 2. convolution: divide by the eigenvalue, zero mode -> 0 */
#pragma omp parallel for collapse(2) schedule(static)
    for (i64 kz = 0; kz < dims[2]; ++kz)
        for (i64 ky = 0; ky < dims[1]; ++ky)
            for (i64 kx = 0; kx < dims[0]; ++kx) {
                i64 i = kx + dims[0] * (ky + dims[1] * kz);
                if (kx == 0 && ky == 0 && kz == 0) { F[i] = 0.0; continue; }
                double Lam = lam[0][kx] + lam[1][ky] + lam[2][kz];
                F[i] = rhs_sign * F[i] / Lam;
            }

    /* 3. spectral operations + 4. backward transform (z, y, x), 1/N on the inverse */
    double inv_n = 1.0 / (double)tot;
    if (grad) {
        for (int g = 0; g < nd; ++g) {
#pragma omp parallel for collapse(2) schedule(static)
            for (i64 kz = 0; kz < dims[2]; ++kz)
                for (i64 ky = 0; ky < dims[1]; ++ky)
                    for (i64 kx = 0; kx < dims[0]; ++kx) {
                        i64 i = kx + dims[0] * (ky + dims[1] * kz);
                        i64 kk[3] = { kx, ky, kz };
                        W[i] = I * kap[g][kk[g]] * F[i];
                    }
            for (int a = nd - 1; a >= 0; --a)
                if ((err = fft_axis(W, dims, a, +1)) != ORC_OK) goto done;
            double *out = grad + (size_t)g * (size_t)tot;
#pragma omp parallel for schedule(static)
            for (i64 i = 0; i < tot; ++i) out[i] = creal(W[i]) * inv_n;
        }
    }
    for (int a = nd - 1; a >= 0; --a)
        if ((err = fft_axis(F, dims, a, +1)) != ORC_OK) goto done;
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < tot; ++i) psi[i] = creal(F[i]) * inv_n;

done:
    for (int a = 0; a < 3; ++a) { free(kap[a]); free(lam[a]); }
    free(F); free(W);
    return err;
}

/* ------------------------------------------------------------------------------------------
 * Boundary-value folding (weights: reading A18).
 * The discrete equation is lap_h psi = rhs_sign f with the face values in the ghost layer (eq. (2)
 * and reading A8), i.e. interior stencil = rhs_sign f + w g; the solvers below multiply the folded source by
 * rhs_sign, so the fold adds (w / rhs_sign) g to f: the face value itself never changes sign.
 * faces[2*axis + side] (side 0 = lower, 1 = upper) holds the values on that face over the two
 * remaining axes, lower axis fastest; NULL = homogeneous.
 * ---------------------------------------------------------------------------------------- */
static void fold_faces(double *fp, const i64 n[3], const double h[3], const double *const faces[6],
                       int neumann, double rhs_sign)
{
    for (int axis = 0; axis < 3; ++axis) {
        int a = (axis == 0) ? 1 : 0;           /* lower remaining axis (fastest in the face) */
        int b = (axis == 2) ? 1 : 2;           /* upper remaining axis */
        i64 st[3] = { 1, n[0], n[0] * n[1] };
        for (int side = 0; side < 2; ++side) {
            const double *g = faces ? faces[2 * axis + side] : NULL;
            if (!g) continue;
            i64 ic = side ? n[axis] - 1 : 0;   /* boundary-adjacent layer */
            double w;
            if (!neumann) w = -1.0 / (h[axis] * h[axis]);          /* Dirichlet, cell-boundary */
            else w = side ? -1.0 / h[axis] : +1.0 / h[axis];       /* Neumann, cell-centre     */
            w /= rhs_sign;                                         /* the equation is lap_h psi = rhs_sign f (A8) */
            for (i64 jb = 0; jb < n[b]; ++jb)
                for (i64 ja = 0; ja < n[a]; ++ja)
                    fp[ic * st[axis] + ja * st[a] + jb * st[b]] += w * g[ja + n[a] * jb];
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * O-DIR: Dirichlet, cell-boundary (REGULAR) grid, DST-I forward and backward (Table 1 row 1).
 * n = interior nodes per axis; node j sits at (j+1) h; L = (n+1) h.
 *   op = 1 (FD2): Lambda = -sum_a (4/h_a^2) sin^2(pi (k_a+1) / (2 (N_a+1)))
 *   op = 0 (PS):  Lambda = -sum_a (pi (k_a+1) / L_a)^2       (homogeneous faces only)
 * psi = DST-I_3(rhs_sign * DST-I_3(f') / Lambda) / prod_a (2 (N_a+1)).
 * ---------------------------------------------------------------------------------------- */
int orc_dirichlet_regular(const i64 n[3], const double h[3], int op, double rhs_sign, const double *f,
                          const double *const faces[6], double *psi)
{
    i64 tot = n[0] * n[1] * n[2];
    trig_table tab[3];
    double *lam[3] = { 0, 0, 0 };
    int err = ORC_OK, ntab = 0;
    memcpy(psi, f, sizeof(double) * (size_t)tot);
    if (op == 1) fold_faces(psi, n, h, faces, 0, rhs_sign);
    for (int a = 0; a < 3; ++a) {
        if ((err = trig_table_init(&tab[a], (int)n[a], 2 * (n[a] + 1))) != ORC_OK) { ntab = a + 1; goto done; }
        ntab = a + 1;
        lam[a] = (double *)malloc(sizeof(double) * (size_t)n[a]);
        if (!lam[a]) { err = ORC_ERR_ALLOC; goto done; }
        double Ldom = (double)(n[a] + 1) * h[a];
        for (i64 k = 0; k < n[a]; ++k) {
            if (op == 0) {
                double kk = PI * (double)(k + 1) / Ldom;
                lam[a][k] = -kk * kk;
            } else {
                double s, c;
                sincos2pi(k + 1, 4 * (n[a] + 1), &s, &c); /* sin(pi (k+1) / (2(N+1))) */
                lam[a][k] = -(4.0 / (h[a] * h[a])) * s * s;
            }
        }
    }
    for (int a = 0; a < 3; ++a)
        if ((err = r2r_axis(psi, n, a, dst1_tab, &tab[a])) != ORC_OK) goto done;
    double norm = 1.0;
    for (int a = 0; a < 3; ++a) norm *= 2.0 * (double)(n[a] + 1);
#pragma omp parallel for collapse(2) schedule(static)
    for (i64 kz = 0; kz < n[2]; ++kz)
        for (i64 ky = 0; ky < n[1]; ++ky)
            for (i64 kx = 0; kx < n[0]; ++kx) {
                i64 i = kx + n[0] * (ky + n[1] * kz);
                psi[i] = rhs_sign * psi[i] / (lam[0][kx] + lam[1][ky] + lam[2][kz]);
            }
    for (int a = 2; a >= 0; --a)
        if ((err = r2r_axis(psi, n, a, dst1_tab, &tab[a])) != ORC_OK) goto done;
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < tot; ++i) psi[i] /= norm;
done:
    for (int a = 0; a < ntab; ++a) trig_table_free(&tab[a]);
    for (int a = 0; a < 3; ++a) free(lam[a]);
    return err;
}

/* ------------------------------------------------------------------------------------------
 * O-NEU: Neumann, cell-centre (STAGGERED) grid, DCT-II forward, DCT-III backward (Table 1 row 4;
 * the printed "DST-III" is read as DCT-III, reading A2).  n = cells per axis, x_j = (j+1/2) h.
 *   op = 1 (FD2): Lambda = -sum_a (4/h_a^2) sin^2(pi k_a / (2 N_a))
 *   op = 0 (PS):  Lambda = -sum_a (pi k_a / L_a)^2, L_a = N_a h_a   (reading A1)
 * Zero mode -> 0.  psi = DCT-III_3(rhs_sign * DCT-II_3(f') / Lambda) / prod_a (2 N_a).
 * ---------------------------------------------------------------------------------------- */
int orc_neumann_staggered(const i64 n[3], const double h[3], int op, double rhs_sign, const double *f,
                          const double *const faces[6], double *psi)
{
    i64 tot = n[0] * n[1] * n[2];
    trig_table tab[3];
    double *lam[3] = { 0, 0, 0 };
    int err = ORC_OK, ntab = 0;
    memcpy(psi, f, sizeof(double) * (size_t)tot);
    if (op == 1) fold_faces(psi, n, h, faces, 1, rhs_sign);
    for (int a = 0; a < 3; ++a) {
        if ((err = trig_table_init(&tab[a], (int)n[a], 4 * n[a])) != ORC_OK) { ntab = a + 1; goto done; }
        ntab = a + 1;
        lam[a] = (double *)malloc(sizeof(double) * (size_t)n[a]);
        if (!lam[a]) { err = ORC_ERR_ALLOC; goto done; }
        double Ldom = (double)n[a] * h[a];
        for (i64 k = 0; k < n[a]; ++k) {
            if (op == 0) {
                double kk = PI * (double)k / Ldom;
                lam[a][k] = -kk * kk;
            } else {
                double s, c;
                sincos2pi(k, 4 * n[a], &s, &c); /* sin(pi k / (2N)) */
                lam[a][k] = -(4.0 / (h[a] * h[a])) * s * s;
            }
        }
    }
    for (int a = 0; a < 3; ++a)
        if ((err = r2r_axis(psi, n, a, dct2_tab, &tab[a])) != ORC_OK) goto done;
    double norm = 1.0;
    for (int a = 0; a < 3; ++a) norm *= 2.0 * (double)n[a];
#pragma omp parallel for collapse(2) schedule(static)
    for (i64 kz = 0; kz < n[2]; ++kz)
        for (i64 ky = 0; ky < n[1]; ++ky)
            for (i64 kx = 0; kx < n[0]; ++kx) {
                i64 i = kx + n[0] * (ky + n[1] * kz);
                if (kx == 0 && ky == 0 && kz == 0) { psi[i] = 0.0; continue; }
                psi[i] = rhs_sign * psi[i] / (lam[0][kx] + lam[1][ky] + lam[2][kz]);
            }
    for (int a = 2; a >= 0; --a)
        if ((err = r2r_axis(psi, n, a, dct3_tab, &tab[a])) != ORC_OK) goto done;
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < tot; ++i) psi[i] /= norm;
done:
    for (int a = 0; a < ntab; ++a) trig_table_free(&tab[a]);
    for (int a = 0; a < 3; ++a) free(lam[a]);
    return err;
}

/* ------------------------------------------------------------------------------------------
 * The other two rows of Table 1.
 *
 * O-DIRS: Dirichlet, cell-centre (STAGGERED) grid, DST-II forward, DST-III backward.  n = cells per axis,
 * x_j = (j+1/2) h, faces at 0 and L = n h.  The ghost cell psi_ghost = 2 g - psi_first puts the face value g
 * between the two cell centres, so the folded source is f' = f - 2 g / h^2 in the boundary-adjacent layer
 * (reading A18).
 *   op = 1 (FD2): Lambda = -sum_a (4/h_a^2) sin^2(pi (k_a+1) / (2 N_a))
 *   op = 0 (PS):  Lambda = -sum_a (pi (k_a+1) / L_a)^2                     (homogeneous faces only)
 * psi = DST-III_3(rhs_sign * DST-II_3(f') / Lambda) / prod_a (2 N_a).
 *
 * O-NEUR: Neumann, cell-boundary (REGULAR) grid, DCT-I forward and backward.  n = nodes per axis including the
 * two boundary nodes, x_j = j h, L = (n-1) h.  The ghost node psi_ghost = psi_second -/+ 2 h g mirrors about
 * the boundary node, so f' = f + 2 g_lo / h on the first layer and f - 2 g_hi / h on the last (reading A18).
 *   op = 1 (FD2): Lambda = -sum_a (4/h_a^2) sin^2(pi k_a / (2 (N_a-1)))
 *   op = 0 (PS):  Lambda = -sum_a (pi k_a / L_a)^2
 * Zero mode -> 0.  psi = DCT-I_3(rhs_sign * DCT-I_3(f') / Lambda) / prod_a (2 (N_a-1)).
 * ---------------------------------------------------------------------------------------- */
static void fold_faces_f3(double *fp, const i64 n[3], const double h[3], const double *const faces[6], int neumann,
                          double rhs_sign)
{
    for (int axis = 0; axis < 3; ++axis) {
        int a = (axis == 0) ? 1 : 0;
        int b = (axis == 2) ? 1 : 2;
        i64 st[3] = { 1, n[0], n[0] * n[1] };
        for (int side = 0; side < 2; ++side) {
            const double *g = faces ? faces[2 * axis + side] : NULL;
            if (!g) continue;
            i64 ic = side ? n[axis] - 1 : 0;
            double w;
            if (!neumann) w = -2.0 / (h[axis] * h[axis]);          /* Dirichlet, cell-centre   */
            else w = side ? -2.0 / h[axis] : +2.0 / h[axis];       /* Neumann, cell-boundary   */
            w /= rhs_sign;
            for (i64 jb = 0; jb < n[b]; ++jb)
                for (i64 ja = 0; ja < n[a]; ++ja)
                    fp[ic * st[axis] + ja * st[a] + jb * st[b]] += w * g[ja + n[a] * jb];
        }
    }
}

int orc_dirichlet_staggered(const i64 n[3], const double h[3], int op, double rhs_sign, const double *f,
                            const double *const faces[6], double *psi)
{
    i64 tot = n[0] * n[1] * n[2];
    trig_table tab[3];
    double *lam[3] = { 0, 0, 0 };
    int err = ORC_OK, ntab = 0;
    memcpy(psi, f, sizeof(double) * (size_t)tot);
    if (op == 1) fold_faces_f3(psi, n, h, faces, 0, rhs_sign);
    for (int a = 0; a < 3; ++a) {
        if ((err = trig_table_init(&tab[a], (int)n[a], 4 * n[a])) != ORC_OK) { ntab = a + 1; goto done; }
        ntab = a + 1;
        lam[a] = (double *)malloc(sizeof(double) * (size_t)n[a]);
        if (!lam[a]) { err = ORC_ERR_ALLOC; goto done; }
        double Ldom = (double)n[a] * h[a];
        for (i64 k = 0; k < n[a]; ++k) {
            if (op == 0) {
                double kk = PI * (double)(k + 1) / Ldom;
                lam[a][k] = -kk * kk;
            } else {
                double s, c;
                sincos2pi(k + 1, 4 * n[a], &s, &c); /* sin(pi (k+1) / (2N)) */
                lam[a][k] = -(4.0 / (h[a] * h[a])) * s * s;
            }
        }
    }
    for (int a = 0; a < 3; ++a)
        if ((err = r2r_axis(psi, n, a, dst2_tab, &tab[a])) != ORC_OK) goto done;
    double norm = 1.0;
    for (int a = 0; a < 3; ++a) norm *= 2.0 * (double)n[a];
#pragma omp parallel for collapse(2) schedule(static)
    for (i64 kz = 0; kz < n[2]; ++kz)
        for (i64 ky = 0; ky < n[1]; ++ky)
            for (i64 kx = 0; kx < n[0]; ++kx) {
                i64 i = kx + n[0] * (ky + n[1] * kz);
                psi[i] = rhs_sign * psi[i] / (lam[0][kx] + lam[1][ky] + lam[2][kz]);
            }
    for (int a = 2; a >= 0; --a)
        if ((err = r2r_axis(psi, n, a, dst3_tab, &tab[a])) != ORC_OK) goto done;
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < tot; ++i) psi[i] /= norm;
done:
    for (int a = 0; a < ntab; ++a) trig_table_free(&tab[a]);
    for (int a = 0; a < 3; ++a) free(lam[a]);
    return err;
}

int orc_neumann_regular(const i64 n[3], const double h[3], int op, double rhs_sign, const double *f,
                        const double *const faces[6], double *psi)
{
    i64 tot = n[0] * n[1] * n[2];
    trig_table tab[3];
    double *lam[3] = { 0, 0, 0 };
    int err = ORC_OK, ntab = 0;
    for (int a = 0; a < 3; ++a) if (n[a] < 2) return ORC_ERR_ARG;
    memcpy(psi, f, sizeof(double) * (size_t)tot);
    if (op == 1) fold_faces_f3(psi, n, h, faces, 1, rhs_sign);
    for (int a = 0; a < 3; ++a) {
        if ((err = trig_table_init(&tab[a], (int)n[a], 2 * (n[a] - 1))) != ORC_OK) { ntab = a + 1; goto done; }
        ntab = a + 1;
        lam[a] = (double *)malloc(sizeof(double) * (size_t)n[a]);
        if (!lam[a]) { err = ORC_ERR_ALLOC; goto done; }
        double Ldom = (double)(n[a] - 1) * h[a];
        for (i64 k = 0; k < n[a]; ++k) {
            if (op == 0) {
                double kk = PI * (double)k / Ldom;
                lam[a][k] = -kk * kk;
            } else {
                double s, c;
                sincos2pi(k, 4 * (n[a] - 1), &s, &c); /* sin(pi k / (2 (N-1))) */
                lam[a][k] = -(4.0 / (h[a] * h[a])) * s * s;
            }
        }
    }
    for (int a = 0; a < 3; ++a)
        if ((err = r2r_axis(psi, n, a, dct1_tab, &tab[a])) != ORC_OK) goto done;
    double norm = 1.0;
    for (int a = 0; a < 3; ++a) norm *= 2.0 * (double)(n[a] - 1);
#pragma omp parallel for collapse(2) schedule(static)
    for (i64 kz = 0; kz < n[2]; ++kz)
        for (i64 ky = 0; ky < n[1]; ++ky)
            for (i64 kx = 0; kx < n[0]; ++kx) {
                i64 i = kx + n[0] * (ky + n[1] * kz);
                if (kx == 0 && ky == 0 && kz == 0) { psi[i] = 0.0; continue; }
                psi[i] = rhs_sign * psi[i] / (lam[0][kx] + lam[1][ky] + lam[2][kz]);
            }
    for (int a = 2; a >= 0; --a)
        if ((err = r2r_axis(psi, n, a, dct1_tab, &tab[a])) != ORC_OK) goto done;
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < tot; ++i) psi[i] /= norm;
done:
    for (int a = 0; a < ntab; ++a) trig_table_free(&tab[a]);
    for (int a = 0; a < 3; ++a) free(lam[a]);
    return err;
}

/* ------------------------------------------------------------------------------------------
 * O-MIX: Dirichlet and Neumann conditions mixed per axis (PAPER.md:191-199 describes the approach --
 * 1-D transforms chosen per direction -- and leaves it as future work).  Nothing new is computed:
 * axis a uses the row of Table 1 that its own condition selects on the plan's grid type,
 *   kind 0: Dirichlet, cell-boundary   DST-I  / DST-I    n interior nodes, L = (n+1) h, index k+1, norm 2 (n+1)
 *   kind 1: Neumann,   cell-centre     DCT-II / DCT-III  n cells,          L = n h,     index k,   norm 2 n
 *   kind 2: Dirichlet, cell-centre     DST-II / DST-III  n cells,          L = n h,     index k+1, norm 2 n
 *   kind 3: Neumann,   cell-boundary   DCT-I  / DCT-I    n nodes,          L = (n-1) h, index k,   norm 2 (n-1)
 * (kinds 0 and 3 share the cell-boundary grid, kinds 1 and 2 the cell-centre grid), its eigenvalue column and its
 * fold weight (reading A18).  The zero mode exists only when every axis is Neumann.
 * psi = B_z B_y B_x ( rhs_sign * F_x F_y F_z f' / (lam_x + lam_y + lam_z) ) / prod_a norm_a.
 * ---------------------------------------------------------------------------------------- */
int orc_bounded_mixed(const int kind[3], const i64 n[3], const double h[3], int op, double rhs_sign, const double *f,
                      const double *const faces[6], double *psi)
{
    i64 tot = n[0] * n[1] * n[2];
    trig_table tab[3];
    double *lam[3] = { 0, 0, 0 };
    real_xform fwd[3], bwd[3];
    int err = ORC_OK, ntab = 0, all_neumann = 1;
    double norm = 1.0;
    for (int a = 0; a < 3; ++a)
        if (kind[a] < 0 || kind[a] > 3) return ORC_ERR_ARG;
    memcpy(psi, f, sizeof(double) * (size_t)tot);
    /* fold the face values of every axis with the weight of that axis' own condition */
    if (op == 1 && faces) {
        i64 st[3] = { 1, n[0], n[0] * n[1] };
        for (int axis = 0; axis < 3; ++axis) {
            int a = (axis == 0) ? 1 : 0, b = (axis == 2) ? 1 : 2;
            for (int side = 0; side < 2; ++side) {
                const double *g = faces[2 * axis + side];
                if (!g) continue;
                i64 ic = side ? n[axis] - 1 : 0;
                double w;
                switch (kind[axis]) {
                case 0: w = -1.0 / (h[axis] * h[axis]); break;
                case 1: w = side ? -1.0 / h[axis] : +1.0 / h[axis]; break;
                case 2: w = -2.0 / (h[axis] * h[axis]); break;
                default: w = side ? -2.0 / h[axis] : +2.0 / h[axis]; break;
                }
                w /= rhs_sign;
                for (i64 jb = 0; jb < n[b]; ++jb)
                    for (i64 ja = 0; ja < n[a]; ++ja)
                        psi[ic * st[axis] + ja * st[a] + jb * st[b]] += w * g[ja + n[a] * jb];
            }
        }
    }
    for (int a = 0; a < 3; ++a) {
        i64 period, cells, shift;
        switch (kind[a]) {
        case 0: period = 2 * (n[a] + 1); cells = n[a] + 1; shift = 1; fwd[a] = dst1_tab; bwd[a] = dst1_tab; break;
        case 1: period = 4 * n[a];       cells = n[a];     shift = 0; fwd[a] = dct2_tab; bwd[a] = dct3_tab; break;
        case 2: period = 4 * n[a];       cells = n[a];     shift = 1; fwd[a] = dst2_tab; bwd[a] = dst3_tab; break;
        default: period = 2 * (n[a] - 1); cells = n[a] - 1; shift = 0; fwd[a] = dct1_tab; bwd[a] = dct1_tab; break;
        }
        if (cells < 1) { err = ORC_ERR_ARG; goto done; }
        if (kind[a] == 0 || kind[a] == 2) all_neumann = 0;
        norm *= 2.0 * (double)cells;
        if ((err = trig_table_init(&tab[a], (int)n[a], period)) != ORC_OK) { ntab = a + 1; goto done; }
        ntab = a + 1;
        lam[a] = (double *)malloc(sizeof(double) * (size_t)n[a]);
        if (!lam[a]) { err = ORC_ERR_ALLOC; goto done; }
        double Ldom = (double)cells * h[a];
        for (i64 k = 0; k < n[a]; ++k) {
            if (op == 0) {
                double kk = PI * (double)(k + shift) / Ldom;
                lam[a][k] = -kk * kk;
            } else {
                double sn, cs;
                sincos2pi(k + shift, 4 * cells, &sn, &cs);   /* sin(pi (k + shift) / (2 cells)) */
                lam[a][k] = -(4.0 / (h[a] * h[a])) * sn * sn;
            }
        }
    }
    for (int a = 0; a < 3; ++a)
        if ((err = r2r_axis(psi, n, a, fwd[a], &tab[a])) != ORC_OK) goto done;
#pragma omp parallel for collapse(2) schedule(static)
    for (i64 kz = 0; kz < n[2]; ++kz)
        for (i64 ky = 0; ky < n[1]; ++ky)
            for (i64 kx = 0; kx < n[0]; ++kx) {
                i64 i = kx + n[0] * (ky + n[1] * kz);
                if (all_neumann && kx == 0 && ky == 0 && kz == 0) { psi[i] = 0.0; continue; }
                psi[i] = rhs_sign * psi[i] / (lam[0][kx] + lam[1][ky] + lam[2][kz]);
            }
    for (int a = 2; a >= 0; --a)
        if ((err = r2r_axis(psi, n, a, bwd[a], &tab[a])) != ORC_OK) goto done;
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < tot; ++i) psi[i] /= norm;
done:
    for (int a = 0; a < ntab; ++a) trig_table_free(&tab[a]);
    for (int a = 0; a < 3; ++a) free(lam[a]);
    return err;
}

/* ------------------------------------------------------------------------------------------
 * Spectral gradient on Dirichlet / Neumann plans (eq. (10), applied to the sine / cosine
 * series of Table 1; SURVEY f3 "sine <-> cosine on the inverse").  The solve gives the coefficients
 * c_k = rhs_sign * T_3(f') / Lambda of the series psi = (1/norm) S_3(c), S the synthesis (backward) sum of
 * the row.  d psi / d x_a differentiates the basis functions of axis a analytically and evaluates them at
 * the same grid points; the other axes keep their synthesis sums.  With kappa_k the wavenumber of term k:
 *   kind 0  Dirichlet cell-boundary  psi_j = 2 sum_k c_k sin(kappa_k x_j),  x_j = (j+1) h,   kappa_k = pi (k+1) / ((n+1) h)
 *   kind 1  Neumann   cell-centre    psi_j = c_0 + 2 sum_{k>=1} c_k cos(kappa_k x_j),  x_j = (j+1/2) h,  kappa_k = pi k / (n h)
 *   kind 2  Dirichlet cell-centre    psi_j = (-1)^j c_{n-1} + 2 sum_{k<n-1} c_k sin(kappa_k x_j),  x_j = (j+1/2) h,  kappa_k = pi (k+1) / (n h)
 *   kind 3  Neumann   cell-boundary  psi_j = c_0 + (-1)^j c_{n-1} + 2 sum_{1<=k<=n-2} c_k cos(kappa_k x_j),  x_j = j h,  kappa_k = pi k / ((n-1) h)
 * The alternating terms of kinds 2 and 3 are the Nyquist terms sin / cos(pi x / h): their derivatives vanish at
 * every grid point of their grids (consistent with reading A20).
 *   sin -> kappa cos,  cos -> -kappa sin.
 * psi, grad[3] (d/dx, d/dy, d/dz).
 * ---------------------------------------------------------------------------------------- */
typedef struct { int kind; int n; double h; } dsyn_par;

/* derivative synthesis along one pencil: out_j = d/dx [ S(c) ](x_j) */
static void dsyn_pencil(const dsyn_par *q, const double *c, double *out)
{
    int n = q->n;
    for (int j = 0; j < n; ++j) {
        long double acc = 0.0L;
        for (int k = 0; k < n; ++k) {
            long double kappa, x;
            switch (q->kind) {
            case 0: kappa = (long double)PI * (k + 1) / ((long double)(n + 1) * q->h); x = (long double)(j + 1) * q->h;
                    acc += 2.0L * c[k] * kappa * cosl(kappa * x); break;
            case 1: if (k == 0) break;
                    kappa = (long double)PI * k / ((long double)n * q->h); x = ((long double)j + 0.5L) * q->h;
                    acc -= 2.0L * c[k] * kappa * sinl(kappa * x); break;
            case 2: if (k == n - 1) break;
                    kappa = (long double)PI * (k + 1) / ((long double)n * q->h); x = ((long double)j + 0.5L) * q->h;
                    acc += 2.0L * c[k] * kappa * cosl(kappa * x); break;
            default: if (k == 0 || k == n - 1) break;
                    kappa = (long double)PI * k / ((long double)(n - 1) * q->h); x = (long double)j * q->h;
                    acc -= 2.0L * c[k] * kappa * sinl(kappa * x); break;
            }
        }
        out[j] = (double)acc;
    }
}

static int dsyn_axis(double *a, const i64 dims[3], int axis, const dsyn_par *q)
{
    i64 len, stride, na, sa, nb, sb;
    axis_geometry(dims, axis, &len, &stride, &na, &sa, &nb, &sb);
    int err = ORC_OK;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * (size_t)len * 2);
        if (!buf) {
#pragma omp critical
            err = ORC_ERR_ALLOC;
        }
#pragma omp for collapse(2) schedule(static)
        for (i64 ib = 0; ib < nb; ++ib)
            for (i64 ia = 0; ia < na; ++ia) {
                if (!buf) continue;
                double *p = a + ia * sa + ib * sb;
                double *in = buf, *out = buf + len;
                for (i64 j = 0; j < len; ++j) in[j] = p[j * stride];
                dsyn_pencil(q, in, out);
                for (i64 j = 0; j < len; ++j) p[j * stride] = out[j];
            }
        free(buf);
    }
    return err;
}

int orc_bounded_gradient(int kind, const i64 n[3], const double h[3], int op, double rhs_sign, const double *f,
                         const double *const faces[6], double *psi, double *grad)
{
    if (kind < 0 || kind > 3) return ORC_ERR_ARG;
    i64 tot = n[0] * n[1] * n[2];
    trig_table tab[3];
    double *lam[3] = { 0, 0, 0 };
    double *coef = (double *)malloc(sizeof(double) * (size_t)tot);
    int err = ORC_OK, ntab = 0;
    real_xform fwd = (kind == 0) ? dst1_tab : (kind == 1) ? dct2_tab : (kind == 2) ? dst2_tab : dct1_tab;
    real_xform bwd = (kind == 0) ? dst1_tab : (kind == 1) ? dct3_tab : (kind == 2) ? dst3_tab : dct1_tab;
    int neumann = (kind == 1 || kind == 3);
    if (!coef) return ORC_ERR_ALLOC;
    memcpy(coef, f, sizeof(double) * (size_t)tot);
    if (op == 1) { if (kind < 2) fold_faces(coef, n, h, faces, neumann, rhs_sign); else fold_faces_f3(coef, n, h, faces, neumann, rhs_sign); }
    double norm = 1.0;
    for (int a = 0; a < 3; ++a) {
        i64 N = n[a];
        i64 q = (kind == 0) ? 2 * (N + 1) : (kind == 3) ? 2 * (N - 1) : 4 * N;
        double cells = (kind == 0) ? (double)(N + 1) : (kind == 3) ? (double)(N - 1) : (double)N;
        if ((err = trig_table_init(&tab[a], (int)N, q)) != ORC_OK) { ntab = a + 1; goto done; }
        ntab = a + 1;
        lam[a] = (double *)malloc(sizeof(double) * (size_t)N);
        if (!lam[a]) { err = ORC_ERR_ALLOC; goto done; }
        norm *= 2.0 * cells;
        for (i64 k = 0; k < N; ++k) {
            double idx = neumann ? (double)k : (double)(k + 1);
            if (op == 0) {
                double kk = PI * idx / (cells * h[a]);
                lam[a][k] = -kk * kk;
            } else {
                double sn, cs;
                sincos2pi((i64)idx, 4 * (i64)cells, &sn, &cs);   /* sin(pi idx / (2 cells)), integer-reduced like every other eigenvalue */
                lam[a][k] = -(4.0 / (h[a] * h[a])) * sn * sn;
            }
        }
    }
    for (int a = 0; a < 3; ++a)
        if ((err = r2r_axis(coef, n, a, fwd, &tab[a])) != ORC_OK) goto done;
#pragma omp parallel for collapse(2) schedule(static)
    for (i64 kz = 0; kz < n[2]; ++kz)
        for (i64 ky = 0; ky < n[1]; ++ky)
            for (i64 kx = 0; kx < n[0]; ++kx) {
                i64 i = kx + n[0] * (ky + n[1] * kz);
                if (neumann && kx == 0 && ky == 0 && kz == 0) { coef[i] = 0.0; continue; }
                coef[i] = rhs_sign * coef[i] / (lam[0][kx] + lam[1][ky] + lam[2][kz]) / norm;
            }
    for (int g = 0; g < 3; ++g) {
        double *out = grad + (size_t)g * (size_t)tot;
        memcpy(out, coef, sizeof(double) * (size_t)tot);
        for (int a = 2; a >= 0; --a) {
            if (a == g) {
                dsyn_par q = { kind, (int)n[a], h[a] };
                if ((err = dsyn_axis(out, n, a, &q)) != ORC_OK) goto done;
            } else if ((err = r2r_axis(out, n, a, bwd, &tab[a])) != ORC_OK) goto done;
        }
    }
    memcpy(psi, coef, sizeof(double) * (size_t)tot);
    for (int a = 2; a >= 0; --a)
        if ((err = r2r_axis(psi, n, a, bwd, &tab[a])) != ORC_OK) goto done;
done:
    for (int a = 0; a < ntab; ++a) trig_table_free(&tab[a]);
    for (int a = 0; a < 3; ++a) free(lam[a]);
    free(coef);
    return err;
}

/* ------------------------------------------------------------------------------------------
 * O-UNB / O-VEC: unbounded solver, Hockney-Eastwood on the whole doubled domain.
 *
 * Real-space kernel: 2nd-order Gaussian-regularised Green's function of Hejlesen (
 * formula not printed in the paper -- reading A10):
 *     G(r) = -erf(r / (sqrt(2) eps)) / (4 pi r),   G(0) = -1 / ((2 pi)^(3/2) eps),
 * so that lap G -> delta (sign of PAPER.md:38).
 * Definition being computed (discretised eq. (3); weight hx hy hz: reading A11):
 *     psi_i = rhs_sign * hx hy hz * sum_j G(|x_i - x_j|) f_j .
 * ---------------------------------------------------------------------------------------- */
double orc_green_gauss2(double r, double eps)
{
    if (r == 0.0) return -1.0 / (pow(2.0 * PI, 1.5) * eps);
    return -erf(r / (sqrt(2.0) * eps)) / (4.0 * PI * r);
}

/* Hejlesen's Gaussian kernels of order P = 2, 4, ... 10 ("Gaussian approximations of
 * order P = 2, 4, ... 10"; formulas not printed -- reading A25 of DESIGN.md).  In spectral space the
 * order-P kernel is  G^_P(k) = -zeta^_P(eps k) / k^2  with
 *     zeta^_P(s) = exp(-s^2/2) * sum_{n < P/2} (s^2/2)^n / n! ,
 * i.e. the Gaussian times the Taylor polynomial that cancels its deviation from 1 up to s^(P-2).
 * Term n >= 1 is  -(eps^2/2)^n / n! * k^(2n-2) exp(-eps^2 k^2 / 2)  <->  -(eps^2/2)^n / n! (-lap)^(n-1) g,
 * g(r) = (2 pi eps^2)^(-3/2) exp(-r^2 / (2 eps^2)) the unit Gaussian of width eps, and in 3-D
 *     lap^m g = (-1)^m 2^m m! / eps^(2m) * L_m^(1/2)(r^2 / (2 eps^2)) * g      (generalised Laguerre)
 * so term n = -(eps^2 / (2 n)) L_(n-1)^(1/2)(x) g,  x = r^2 / (2 eps^2):
 *     G_4 = G_2 - (eps^2/2) g,   G_6 = G_4 - (eps^2/4) L_1 g,   G_8 = G_6 - (eps^2/6) L_2 g,   G_10 = G_8 - (eps^2/8) L_3 g
 *     L_1 = 3/2 - x,  L_2 = x^2/2 - 5x/2 + 15/8,  L_3 = -x^3/6 + 7x^2/4 - 35x/8 + 35/16 . */
double orc_green_gauss(int order, double r, double eps)
{
    double G = orc_green_gauss2(r, eps);
    double x = r * r / (2.0 * eps * eps);
    double g = pow(2.0 * PI * eps * eps, -1.5) * exp(-x);
    double L[4] = { 1.0, 1.5 - x, x * x / 2.0 - 2.5 * x + 15.0 / 8.0, -x * x * x / 6.0 + 7.0 * x * x / 4.0 - 35.0 * x / 8.0 + 35.0 / 16.0 };
    for (int n = 1; n < order / 2 && n <= 4; ++n) G -= eps * eps / (2.0 * n) * L[n - 1] * g;
    return G;
}

/* Sine integral Si(x) = int_0^x sin(t)/t dt, x >= 0: Maclaurin series sum (-1)^n x^(2n+1)/((2n+1)(2n+1)!)
 * for x < 3, else from the exponential integral, E1(i x) = -Ci(x) + i (Si(x) - pi/2), with E1 by its
 * continued fraction e^(-z) / (z + 1 - 1^2/(z + 3 - 2^2/(z + 5 - ...))) (modified Lentz). */
double orc_sine_integral(double x)
{
    if (x < 3.0) {
        double term = x, sum = x, x2 = x * x;
        for (int n = 1; n < 40; ++n) {
            term *= -x2 / ((2.0 * n) * (2.0 * n + 1.0));
            double add = term / (2.0 * n + 1.0);
            sum += add;
            if (fabs(add) < 1e-18 * fabs(sum)) break;
        }
        return sum;
    }
    double complex z = I * x;
    double complex b = z + 1.0, c = 1e300, d = 1.0 / b, hh = d;
    for (int i = 1; i < 500; ++i) {
        double a = -(double)i * (double)i;
        b += 2.0;
        d = 1.0 / (a * d + b);
        c = b + a / c;
        double complex del = c * d;
        hh *= del;
        if (cabs(del - 1.0) < 1e-16) break;
    }
    double complex e1 = hh * cexp(-z);
    return PI / 2.0 + cimag(e1);   /* E1(ix) = -Ci(x) + i (Si(x) - pi/2)  =>  Si = pi/2 + Im E1(ix) */
}

/* Hejlesen's spectrally compact kernel, 3-D ("spectrally compact kernel which achieves
 * spectral accuracy"; formula not printed -- reading A26): the singular spectrum -1/k^2 kept inside the
 * ball |k| <= pi/h that the grid resolves and dropped outside; its radial inverse transform is
 *     G(r) = -1/(2 pi^2 r) int_0^(pi/h) sin(k r)/k dk = -Si(pi r / h) / (2 pi^2 r),   G(0) = -1/(2 pi h). */
double orc_green_spectral(double r, double h)
{
    if (r == 0.0) return -1.0 / (2.0 * PI * h);
    return -orc_sine_integral(PI * r / h) / (2.0 * PI * PI * r);
}

/* half-spectrum geometry on the doubled grid: [P2][P1][N0+1] complex, x fastest */
static i64 unb_spec_size(const i64 n[3]) { return (n[0] + 1) * (2 * n[1]) * (2 * n[2]); }
i64 orc_unbounded_spec_size(const i64 n[3]) { return unb_spec_size(n); }

/* forward transform of a real field given on the doubled grid by a callback-free rule:
 * src is either the n-sized source (zero-padded, pad = 1) or a full doubled real array (pad = 0).
 * x: full complex DFT of length P0 of each (padded) row, outputs k = 0..N0 kept (the rest follow
 * from Hermitian symmetry); then y; then z. */
static int unb_forward(const i64 n[3], const double *src, int pad, cplx *spec)
{
    i64 P0 = 2 * n[0], P1 = 2 * n[1], P2 = 2 * n[2], H0 = n[0] + 1;
    cplx *tw = make_twiddles((int)P0);
    if (!tw) return ORC_ERR_ALLOC;
    int err = ORC_OK;
#pragma omp parallel
    {
        cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)P0 * 3);
        if (!buf) {
#pragma omp critical
            err = ORC_ERR_ALLOC;
        }
#pragma omp for collapse(2) schedule(static)
        for (i64 iz = 0; iz < P2; ++iz)
            for (i64 iy = 0; iy < P1; ++iy) {
                if (!buf) continue;
                cplx *in = buf, *out = buf + P0, *scr = buf + 2 * P0;
                for (i64 ix = 0; ix < P0; ++ix) {
                    double v;
                    if (pad) v = (ix < n[0] && iy < n[1] && iz < n[2]) ? src[ix + n[0] * (iy + n[1] * iz)] : 0.0;
                    else v = src[ix + P0 * (iy + P1 * iz)];
                    in[ix] = v;
                }
                fft_rec((int)P0, -1, in, 1, out, scr, tw, 1);
                cplx *row = spec + H0 * (iy + P1 * iz);
                for (i64 k = 0; k < H0; ++k) row[k] = out[k];
            }
        free(buf);
    }
    free(tw);
    if (err != ORC_OK) return err;
    i64 sdims[3] = { H0, P1, P2 };
    if ((err = fft_axis(spec, sdims, 1, -1)) != ORC_OK) return err;
    return fft_axis(spec, sdims, 2, -1);
}

/* backward transform of a half-spectrum (z, then y, then x), 1/(P0 P1 P2) applied, first octant
 * extracted.  spec is destroyed. */
static int unb_backward_extract(const i64 n[3], cplx *spec, double *out)
{
    i64 P0 = 2 * n[0], P1 = 2 * n[1], P2 = 2 * n[2], H0 = n[0] + 1;
    i64 sdims[3] = { H0, P1, P2 };
    int err;
    if ((err = fft_axis(spec, sdims, 2, +1)) != ORC_OK) return err;
    if ((err = fft_axis(spec, sdims, 1, +1)) != ORC_OK) return err;
    cplx *tw = make_twiddles((int)P0);
    if (!tw) return ORC_ERR_ALLOC;
    double inv = 1.0 / ((double)P0 * (double)P1 * (double)P2);
#pragma omp parallel
    {
        cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)P0 * 3);
        if (!buf) {
#pragma omp critical
            err = ORC_ERR_ALLOC;
        }
#pragma omp for collapse(2) schedule(static)
        for (i64 iz = 0; iz < n[2]; ++iz)
            for (i64 iy = 0; iy < n[1]; ++iy) {
                if (!buf) continue;
                cplx *in = buf, *o = buf + P0, *scr = buf + 2 * P0;
                const cplx *row = spec + H0 * (iy + P1 * iz);
                for (i64 k = 0; k < H0; ++k) in[k] = row[k];
                for (i64 k = 1; k < n[0]; ++k) in[P0 - k] = conj(row[k]); /* Hermitian half */
                fft_rec((int)P0, +1, in, 1, o, scr, tw, 1);
                for (i64 ix = 0; ix < n[0]; ++ix) out[ix + n[0] * (iy + n[1] * iz)] = creal(o[ix]) * inv;
            }
        free(buf);
    }
    free(tw);
    return err;
}

/* Green's spectrum: G on the doubled grid at mirrored distance d_a = min(i_a, P_a - i_a) h_a
 * (reading A12), times the cell volume, forward transformed once.
 * ghat: (n0+1) * 2 n1 * 2 n2 complex. */
int orc_unbounded_green_order(const i64 n[3], const double h[3], double eps, int order, cplx *ghat);
int orc_unbounded_green(const i64 n[3], const double h[3], double eps, cplx *ghat)
{
    return orc_unbounded_green_order(n, h, eps, 2, ghat);
}
/* the same with the kernel of order 2, 4, 6, 8 or 10 */
int orc_unbounded_green_order(const i64 n[3], const double h[3], double eps, int order, cplx *ghat)
{
    if (order != 0 && (order < 2 || order > 10 || (order & 1))) return ORC_ERR_ARG;   /* 0: spectrally compact kernel, eps = h */
    for (int a = 0; a < 3; ++a) if (!is_pow2(n[a])) return ORC_ERR_ARG;
    i64 P0 = 2 * n[0], P1 = 2 * n[1], P2 = 2 * n[2];
    double *g = (double *)malloc(sizeof(double) * (size_t)(P0 * P1 * P2));
    if (!g) return ORC_ERR_ALLOC;
    double vol = h[0] * h[1] * h[2];
#pragma omp parallel for collapse(2) schedule(static)
    for (i64 iz = 0; iz < P2; ++iz)
        for (i64 iy = 0; iy < P1; ++iy)
            for (i64 ix = 0; ix < P0; ++ix) {
                double dx = (double)(ix < P0 - ix ? ix : P0 - ix) * h[0];
                double dy = (double)(iy < P1 - iy ? iy : P1 - iy) * h[1];
                double dz = (double)(iz < P2 - iz ? iz : P2 - iz) * h[2];
                double rr = sqrt(dx * dx + dy * dy + dz * dz);
                g[ix + P0 * (iy + P1 * iz)] = vol * (order ? orc_green_gauss(order, rr, eps) : orc_green_spectral(rr, eps));
            }
    int err = unb_forward(n, g, 0, ghat);
    free(g);
    return err;
}

/* Solve with a stored Green's spectrum.
 * f: ncomp fields of n0*n1*n2 (component-major).  out: ncomp fields; if want_curl (ncomp == 3)
 * out = u = curl psi computed in the same spectral pass: u_hat = i kappa x psi_hat, with
 * kappa_a = 2 pi m_a / (P_a h_a), m_a in [-N_a, N_a) on the DOUBLED grid, Nyquist -> 0
 * (reading A20).  Otherwise out = psi. */
int orc_unbounded_solve(const i64 n[3], const double h[3], const cplx *ghat, int ncomp, double rhs_sign,
                        const double *f, int want_curl, double *out)
{
    if (want_curl && ncomp != 3) return ORC_ERR_ARG;
    for (int a = 0; a < 3; ++a) if (!is_pow2(n[a])) return ORC_ERR_ARG;
    i64 tot = n[0] * n[1] * n[2], ns = unb_spec_size(n);
    i64 P[3] = { 2 * n[0], 2 * n[1], 2 * n[2] }, H0 = n[0] + 1;
    cplx *spec[3] = { 0, 0, 0 };
    cplx *work = NULL;
    double *kap[3] = { 0, 0, 0 };
    int err = ORC_OK;

    for (int c = 0; c < ncomp; ++c) {
        spec[c] = (cplx *)malloc(sizeof(cplx) * (size_t)ns);
        if (!spec[c]) { err = ORC_ERR_ALLOC; goto done; }
        if ((err = unb_forward(n, f + (size_t)c * (size_t)tot, 1, spec[c])) != ORC_OK) goto done;
#pragma omp parallel for schedule(static)
        for (i64 i = 0; i < ns; ++i) spec[c][i] = rhs_sign * ghat[i] * spec[c][i];
        if (!want_curl) {
            if ((err = unb_backward_extract(n, spec[c], out + (size_t)c * (size_t)tot)) != ORC_OK) goto done;
            free(spec[c]); spec[c] = NULL;
        }
    }
    if (want_curl) {
        for (int a = 0; a < 3; ++a) {
            kap[a] = (double *)malloc(sizeof(double) * (size_t)P[a]);
            if (!kap[a]) { err = ORC_ERR_ALLOC; goto done; }
            for (i64 k = 0; k < P[a]; ++k) {
                i64 m = (k < n[a]) ? k : k - P[a];
                kap[a][k] = (k == n[a]) ? 0.0 : 2.0 * PI * (double)m / ((double)P[a] * h[a]);
            }
        }
        work = (cplx *)malloc(sizeof(cplx) * (size_t)ns);
        if (!work) { err = ORC_ERR_ALLOC; goto done; }
        for (int a = 0; a < 3; ++a) {
            int b = (a + 1) % 3, c = (a + 2) % 3; /* u_a = d_b psi_c - d_c psi_b */
#pragma omp parallel for collapse(2) schedule(static)
            for (i64 kz = 0; kz < P[2]; ++kz)
                for (i64 ky = 0; ky < P[1]; ++ky)
                    for (i64 kx = 0; kx < H0; ++kx) {
                        i64 i = kx + H0 * (ky + P[1] * kz);
                        i64 kk[3] = { kx, ky, kz };
                        work[i] = I * (kap[b][kk[b]] * spec[c][i] - kap[c][kk[c]] * spec[b][i]);
                    }
            if ((err = unb_backward_extract(n, work, out + (size_t)a * (size_t)tot)) != ORC_OK) goto done;
        }
    }
done:
    for (int c = 0; c < 3; ++c) { free(spec[c]); free(kap[c]); }
    free(work);
    return err;
}

/* Scalar solve with spectral gradient (eq. (10)): psi as above and
 * g_a = IDFT(i kappa_a psi_hat) extracted on the first octant, kappa on the DOUBLED grid as for the
 * curl (kappa_a = 2 pi m_a / (P_a h_a), Nyquist -> 0; reading A20).  grad: 3 fields (d/dx, d/dy, d/dz). */
int orc_unbounded_gradient(const i64 n[3], const double h[3], const cplx *ghat, double rhs_sign, const double *f,
                           double *psi, double *grad)
{
    for (int a = 0; a < 3; ++a) if (!is_pow2(n[a])) return ORC_ERR_ARG;
    i64 tot = n[0] * n[1] * n[2], ns = unb_spec_size(n);
    i64 P[3] = { 2 * n[0], 2 * n[1], 2 * n[2] }, H0 = n[0] + 1;
    int err = ORC_OK;
    cplx *spec = (cplx *)malloc(sizeof(cplx) * (size_t)ns), *work = (cplx *)malloc(sizeof(cplx) * (size_t)ns);
    double *kap = (double *)malloc(sizeof(double) * (size_t)(P[0] > P[1] ? (P[0] > P[2] ? P[0] : P[2]) : (P[1] > P[2] ? P[1] : P[2])));
    if (!spec || !work || !kap) { err = ORC_ERR_ALLOC; goto done; }
    if ((err = unb_forward(n, f, 1, spec)) != ORC_OK) goto done;
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < ns; ++i) spec[i] = rhs_sign * ghat[i] * spec[i];
    for (int a = 0; a < 3; ++a) {
        for (i64 k = 0; k < P[a]; ++k) {
            i64 m = (k < n[a]) ? k : k - P[a];
            kap[k] = (k == n[a]) ? 0.0 : 2.0 * PI * (double)m / ((double)P[a] * h[a]);
        }
#pragma omp parallel for collapse(2) schedule(static)
        for (i64 kz = 0; kz < P[2]; ++kz)
            for (i64 ky = 0; ky < P[1]; ++ky)
                for (i64 kx = 0; kx < H0; ++kx) {
                    i64 i = kx + H0 * (ky + P[1] * kz);
                    i64 kk[3] = { kx, ky, kz };
                    work[i] = I * kap[kk[a]] * spec[i];
                }
        if ((err = unb_backward_extract(n, work, grad + (size_t)a * (size_t)tot)) != ORC_OK) goto done;
    }
    err = unb_backward_extract(n, spec, psi);   /* last: the backward transform works in place */
done:
    free(spec); free(work); free(kap);
    return err;
}

/* DIV and NABLA on an unbounded plan ("DIV: resolves the divergence ... NABLA: resolves
 * the Laplacian of the input field", applied with the convolution kernel as eq. (10) is, PAPER.md:141-143;
 * reading A27): psi_c = rhs_sign G * f_c per component, then in the same spectral pass
 *   kind 0 (DIV,   ncomp == 3): out = sum_a IDFT(i kappa_a psi_hat_a)                 one field
 *   kind 1 (NABLA, any ncomp):  out_c = IDFT(sum_a (i kappa_a)^2 psi_hat_c)           ncomp fields
 * with the kappa_a of the gradient and the curl (doubled grid, Nyquist -> 0, reading A20): NABLA is DIV of
 * GRAD, two successive multiplications by i kappa. */
int orc_unbounded_divlap(const i64 n[3], const double h[3], const cplx *ghat, int ncomp, double rhs_sign,
                         const double *f, int kind, double *out)
{
    if (kind != 0 && kind != 1) return ORC_ERR_ARG;
    if (kind == 0 && ncomp != 3) return ORC_ERR_ARG;
    for (int a = 0; a < 3; ++a) if (!is_pow2(n[a])) return ORC_ERR_ARG;
    i64 tot = n[0] * n[1] * n[2], ns = unb_spec_size(n);
    i64 P[3] = { 2 * n[0], 2 * n[1], 2 * n[2] }, H0 = n[0] + 1;
    int err = ORC_OK;
    cplx *spec = (cplx *)malloc(sizeof(cplx) * (size_t)ns), *acc = NULL;
    double *kap[3] = { 0, 0, 0 };
    if (!spec) { err = ORC_ERR_ALLOC; goto done; }
    for (int a = 0; a < 3; ++a) {
        kap[a] = (double *)malloc(sizeof(double) * (size_t)P[a]);
        if (!kap[a]) { err = ORC_ERR_ALLOC; goto done; }
        for (i64 k = 0; k < P[a]; ++k) {
            i64 m = (k < n[a]) ? k : k - P[a];
            kap[a][k] = (k == n[a]) ? 0.0 : 2.0 * PI * (double)m / ((double)P[a] * h[a]);
        }
    }
    if (kind == 0) {
        acc = (cplx *)calloc((size_t)ns, sizeof(cplx));
        if (!acc) { err = ORC_ERR_ALLOC; goto done; }
    }
    for (int c = 0; c < ncomp; ++c) {
        if ((err = unb_forward(n, f + (size_t)c * (size_t)tot, 1, spec)) != ORC_OK) goto done;
#pragma omp parallel for collapse(2) schedule(static)
        for (i64 kz = 0; kz < P[2]; ++kz)
            for (i64 ky = 0; ky < P[1]; ++ky)
                for (i64 kx = 0; kx < H0; ++kx) {
                    i64 i = kx + H0 * (ky + P[1] * kz);
                    i64 kk[3] = { kx, ky, kz };
                    cplx psi = rhs_sign * ghat[i] * spec[i];
                    if (kind == 0) {
                        acc[i] += I * kap[c][kk[c]] * psi;
                    } else {
                        cplx s = 0.0;
                        for (int a = 0; a < 3; ++a) s += (I * kap[a][kk[a]]) * (I * kap[a][kk[a]]) * psi;
                        spec[i] = s;
                    }
                }
        if (kind == 1 && (err = unb_backward_extract(n, spec, out + (size_t)c * (size_t)tot)) != ORC_OK) goto done;
    }
    if (kind == 0) err = unb_backward_extract(n, acc, out);
done:
    for (int a = 0; a < 3; ++a) free(kap[a]);
    free(spec); free(acc);
    return err;
}

/* DIV and NABLA on a periodic plan (same passage; reading A27): psi_hat_c = rhs_sign F_c / Lambda as in
 * orc_periodic (zero mode -> 0), then
 *   kind 0 (DIV,   ncomp == nd): out = sum_a IDFT(i kappa_a psi_hat_a)
 *   kind 1 (NABLA):              out_c = IDFT(sum_a (i kappa_a)^2 psi_hat_c)
 * kappa_a = 2 pi m_a / L_a, zero at the Nyquist index (reading A20).  With op = 0 NABLA returns the source
 * less its mean and its Nyquist planes; with op = 1 it returns the source filtered by kappa^2 / |Lambda_FD|. */
int orc_periodic_divlap(int nd, const i64 n[3], const double L[3], int op, double rhs_sign, int ncomp,
                        const double *f, int kind, double *out)
{
    if (nd < 1 || nd > 3 || (kind != 0 && kind != 1)) return ORC_ERR_ARG;
    if (kind == 0 && ncomp != nd) return ORC_ERR_ARG;
    i64 dims[3] = { n[0], nd > 1 ? n[1] : 1, nd > 2 ? n[2] : 1 };
    i64 tot = dims[0] * dims[1] * dims[2];
    for (int a = 0; a < 3; ++a) if (!is_pow2(dims[a])) return ORC_ERR_ARG;
    cplx *F = (cplx *)malloc(sizeof(cplx) * (size_t)tot);
    cplx *A = (kind == 0) ? (cplx *)calloc((size_t)tot, sizeof(cplx)) : NULL;
    double *kap[3] = { 0, 0, 0 }, *lam[3] = { 0, 0, 0 };
    int err = ORC_OK;
    if (!F || (kind == 0 && !A)) { err = ORC_ERR_ALLOC; goto done; }
    for (int a = 0; a < 3; ++a) {
        i64 N = dims[a];
        kap[a] = (double *)calloc((size_t)N, sizeof(double));
        lam[a] = (double *)calloc((size_t)N, sizeof(double));
        if (!kap[a] || !lam[a]) { err = ORC_ERR_ALLOC; goto done; }
        if (a >= nd) continue;
        double hh = L[a] / (double)N;
        for (i64 k = 0; k < N; ++k) {
            i64 m = (2 * k < N) ? k : k - N;
            double kappa = 2.0 * PI * (double)m / L[a];
            kap[a][k] = (2 * k == N) ? 0.0 : kappa;
            if (op == 0) lam[a][k] = -kappa * kappa;
            else {
                double sn, cs;
                sincos2pi(k, 2 * N, &sn, &cs);
                lam[a][k] = -(4.0 / (hh * hh)) * sn * sn;
            }
        }
    }
    double inv_n = 1.0 / (double)tot;
    for (int c = 0; c < ncomp; ++c) {
        const double *fc = f + (size_t)c * (size_t)tot;
#pragma omp parallel for schedule(static)
        for (i64 i = 0; i < tot; ++i) F[i] = fc[i];
        for (int a = 0; a < nd; ++a)
            if ((err = fft_axis(F, dims, a, -1)) != ORC_OK) goto done;
#pragma omp parallel for collapse(2) schedule(static)
        for (i64 kz = 0; kz < dims[2]; ++kz)
            for (i64 ky = 0; ky < dims[1]; ++ky)
                for (i64 kx = 0; kx < dims[0]; ++kx) {
                    i64 i = kx + dims[0] * (ky + dims[1] * kz);
                    i64 kk[3] = { kx, ky, kz };
                    cplx psi = 0.0;
                    if (kx || ky || kz) psi = rhs_sign * F[i] / (lam[0][kx] + lam[1][ky] + lam[2][kz]);
                    if (kind == 0) {
                        A[i] += I * kap[c][kk[c]] * psi;
                    } else {
                        cplx s = 0.0;
                        for (int a = 0; a < 3; ++a) s += (I * kap[a][kk[a]]) * (I * kap[a][kk[a]]) * psi;
                        F[i] = s;
                    }
                }
        if (kind == 1) {
            for (int a = nd - 1; a >= 0; --a)
                if ((err = fft_axis(F, dims, a, +1)) != ORC_OK) goto done;
            double *oc = out + (size_t)c * (size_t)tot;
#pragma omp parallel for schedule(static)
            for (i64 i = 0; i < tot; ++i) oc[i] = creal(F[i]) * inv_n;
        }
    }
    if (kind == 0) {
        for (int a = nd - 1; a >= 0; --a)
            if ((err = fft_axis(A, dims, a, +1)) != ORC_OK) goto done;
#pragma omp parallel for schedule(static)
        for (i64 i = 0; i < tot; ++i) out[i] = creal(A[i]) * inv_n;
    }
done:
    for (int a = 0; a < 3; ++a) { free(kap[a]); free(lam[a]); }
    free(F); free(A);
    return err;
}

/* CURL on a periodic 3-D vector plan (eq. (10); component-wise vector solve PAPER.md:119):
 * psi_hat_c = rhs_sign F_c / Lambda for each component as in orc_periodic (zero mode -> 0), then
 *   u_hat = i kappa x psi_hat,  u_a = IDFT(i (kappa_b psi_hat_c - kappa_c psi_hat_b)),  (a, b, c) cyclic,
 * kappa_a = 2 pi m_a / L_a, zero at the Nyquist index (reading A20).  f, out: three fields, component-major. */
int orc_periodic_curl(const i64 n[3], const double L[3], int op, double rhs_sign, const double *f, double *out)
{
    i64 tot = n[0] * n[1] * n[2];
    for (int a = 0; a < 3; ++a) if (!is_pow2(n[a])) return ORC_ERR_ARG;
    cplx *P[3] = { 0, 0, 0 }, *W = NULL;
    double *kap[3] = { 0, 0, 0 }, *lam[3] = { 0, 0, 0 };
    int err = ORC_OK;
    for (int a = 0; a < 3; ++a) {
        i64 N = n[a];
        kap[a] = (double *)calloc((size_t)N, sizeof(double));
        lam[a] = (double *)calloc((size_t)N, sizeof(double));
        P[a] = (cplx *)malloc(sizeof(cplx) * (size_t)tot);
        if (!kap[a] || !lam[a] || !P[a]) { err = ORC_ERR_ALLOC; goto done; }
        double hh = L[a] / (double)N;
        for (i64 k = 0; k < N; ++k) {
            i64 m = (2 * k < N) ? k : k - N;
            double kappa = 2.0 * PI * (double)m / L[a];
            kap[a][k] = (2 * k == N) ? 0.0 : kappa;
            if (op == 0) lam[a][k] = -kappa * kappa;
            else {
                double sn, cs;
                sincos2pi(k, 2 * N, &sn, &cs);
                lam[a][k] = -(4.0 / (hh * hh)) * sn * sn;
            }
        }
    }
    W = (cplx *)malloc(sizeof(cplx) * (size_t)tot);
    if (!W) { err = ORC_ERR_ALLOC; goto done; }
    for (int c = 0; c < 3; ++c) {
        const double *fc = f + (size_t)c * (size_t)tot;
#pragma omp parallel for schedule(static)
        for (i64 i = 0; i < tot; ++i) P[c][i] = fc[i];
        for (int a = 0; a < 3; ++a)
            if ((err = fft_axis(P[c], n, a, -1)) != ORC_OK) goto done;
#pragma omp parallel for collapse(2) schedule(static)
        for (i64 kz = 0; kz < n[2]; ++kz)
            for (i64 ky = 0; ky < n[1]; ++ky)
                for (i64 kx = 0; kx < n[0]; ++kx) {
                    i64 i = kx + n[0] * (ky + n[1] * kz);
                    if (kx || ky || kz) P[c][i] = rhs_sign * P[c][i] / (lam[0][kx] + lam[1][ky] + lam[2][kz]);
                    else P[c][i] = 0.0;
                }
    }
    double inv_n = 1.0 / (double)tot;
    for (int a = 0; a < 3; ++a) {
        int b = (a + 1) % 3, c = (a + 2) % 3;   /* u_a = d_b psi_c - d_c psi_b */
#pragma omp parallel for collapse(2) schedule(static)
        for (i64 kz = 0; kz < n[2]; ++kz)
            for (i64 ky = 0; ky < n[1]; ++ky)
                for (i64 kx = 0; kx < n[0]; ++kx) {
                    i64 i = kx + n[0] * (ky + n[1] * kz);
                    i64 kk[3] = { kx, ky, kz };
                    W[i] = I * (kap[b][kk[b]] * P[c][i] - kap[c][kk[c]] * P[b][i]);
                }
        for (int ax = 2; ax >= 0; --ax)
            if ((err = fft_axis(W, n, ax, +1)) != ORC_OK) goto done;
        double *oa = out + (size_t)a * (size_t)tot;
#pragma omp parallel for schedule(static)
        for (i64 i = 0; i < tot; ++i) oa[i] = creal(W[i]) * inv_n;
    }
done:
    for (int a = 0; a < 3; ++a) { free(kap[a]); free(lam[a]); free(P[a]); }
    free(W);
    return err;
}

/* ------------------------------------------------------------------------------------------
 * O-UNB2: 2-D unbounded solver (PAPER.md:189 lists the regularised kernels for 1-D, 2-D and 3-D,
 * formulas not printed -- reading A28).  Free-space kernel of the 2-D Laplacian: G_0 = ln(r) / (2 pi)
 * (lap G_0 = delta, sign of PAPER.md:38).  Regularised with the unit Gaussian of width eps,
 * G_2 = G_0 * zeta_eps: the radial field is G_2'(r) = (1 - exp(-r^2 / (2 eps^2))) / (2 pi r), hence
 *     G_2(r) = ( ln r + E_1(r^2 / (2 eps^2)) / 2 ) / (2 pi),    G_2(0) = ( ln(2 eps^2) - gamma ) / (4 pi),
 * E_1 the exponential integral, gamma Euler's constant.  Higher orders as in 3-D (reading A25): term n >= 1 of
 * zeta^_P is -(eps^2/2)^n / n! (-lap)^(n-1) g with g the 2-D unit Gaussian and, in 2-D,
 * lap^m g = (-1)^m 2^m m! / eps^(2m) L_m(x) g, x = r^2 / (2 eps^2), L_m the ordinary Laguerre polynomial:
 *     G_P = G_2 - sum_{n=1}^{P/2-1} eps^2 / (2 n) L_{n-1}(x) g .
 * Definition computed: psi_i = rhs_sign hx hy sum_j G(|x_i - x_j|) f_j, by Hockney-Eastwood doubling.
 * ---------------------------------------------------------------------------------------- */
#define EULER_GAMMA 0.57721566490153286060651209008240243
/* E_1(u), u > 0: series -gamma - ln u - sum_{k>=1} (-u)^k / (k k!) for u <= 1, else the continued fraction
 * e^-u / (u + 1 - 1/(u + 3 - 4/(u + 5 - ...))) by the modified Lentz method */
double orc_exp1(double u)
{
    if (u <= 1.0) {
        double sum = 0.0, term = 1.0;
        for (int k = 1; k < 60; ++k) {
            term *= -u / (double)k;
            double add = term / (double)k;
            sum += add;
            if (fabs(add) < 1e-18 * fabs(sum)) break;
        }
        return -EULER_GAMMA - log(u) - sum;
    }
    double b = u + 1.0, c = 1e300, d = 1.0 / b, hh = d;
    for (int i = 1; i < 500; ++i) {
        double a = -(double)i * (double)i;
        b += 2.0;
        d = 1.0 / (a * d + b);
        c = b + a / c;
        double del = c * d;
        hh *= del;
        if (fabs(del - 1.0) < 1e-16) break;
    }
    return hh * exp(-u);
}

double orc_green2d_gauss(int order, double r, double eps)
{
    double x = r * r / (2.0 * eps * eps);
    double G = (r == 0.0) ? (log(2.0 * eps * eps) - EULER_GAMMA) / (4.0 * PI) : (log(r) + 0.5 * orc_exp1(x)) / (2.0 * PI);
    double g = exp(-x) / (2.0 * PI * eps * eps);
    double L[4] = { 1.0, 1.0 - x, 1.0 - 2.0 * x + x * x / 2.0, 1.0 - 3.0 * x + 1.5 * x * x - x * x * x / 6.0 };
    for (int n = 1; n < order / 2 && n <= 4; ++n) G -= eps * eps / (2.0 * n) * L[n - 1] * g;
    return G;
}

/* forward transform on the doubled 2-D grid, half spectrum [P1][N0+1] (x first, then y) */
static int unb2_forward(const i64 n[2], const double *src, int pad, cplx *spec)
{
    i64 P0 = 2 * n[0], P1 = 2 * n[1], H0 = n[0] + 1;
    cplx *tw = make_twiddles((int)P0);
    cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)P0 * 3);
    if (!tw || !buf) { free(tw); free(buf); return ORC_ERR_ALLOC; }
    for (i64 iy = 0; iy < P1; ++iy) {
        cplx *in = buf, *out = buf + P0, *scr = buf + 2 * P0;
        for (i64 ix = 0; ix < P0; ++ix) {
            double v;
            if (pad) v = (ix < n[0] && iy < n[1]) ? src[ix + n[0] * iy] : 0.0;
            else v = src[ix + P0 * iy];
            in[ix] = v;
        }
        fft_rec((int)P0, -1, in, 1, out, scr, tw, 1);
        for (i64 k = 0; k < H0; ++k) spec[k + H0 * iy] = out[k];
    }
    free(tw); free(buf);
    i64 sdims[3] = { H0, P1, 1 };
    return fft_axis(spec, sdims, 1, -1);
}

/* backward (y, then x), 1/(P0 P1), first quadrant extracted; spec is destroyed */
static int unb2_backward_extract(const i64 n[2], cplx *spec, double *out)
{
    i64 P0 = 2 * n[0], P1 = 2 * n[1], H0 = n[0] + 1;
    i64 sdims[3] = { H0, P1, 1 };
    int err = fft_axis(spec, sdims, 1, +1);
    if (err != ORC_OK) return err;
    cplx *tw = make_twiddles((int)P0);
    cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)P0 * 3);
    if (!tw || !buf) { free(tw); free(buf); return ORC_ERR_ALLOC; }
    double inv = 1.0 / ((double)P0 * (double)P1);
    for (i64 iy = 0; iy < n[1]; ++iy) {
        cplx *in = buf, *o = buf + P0, *scr = buf + 2 * P0;
        const cplx *row = spec + H0 * iy;
        for (i64 k = 0; k < H0; ++k) in[k] = row[k];
        for (i64 k = 1; k < n[0]; ++k) in[P0 - k] = conj(row[k]);
        fft_rec((int)P0, +1, in, 1, o, scr, tw, 1);
        for (i64 ix = 0; ix < n[0]; ++ix) out[ix + n[0] * iy] = creal(o[ix]) * inv;
    }
    free(tw); free(buf);
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------
 * The spectrally compact kernel in 2-D ("1D, 2D and 3D"; reading A30 = A26 in the plane): the singular
 * spectrum -1/k^2 kept inside the disc |k| <= k_c = pi/h and dropped outside.  Its radial inverse transform diverges
 * logarithmically at k -> 0 (a 2-D potential is defined up to a constant); with the constant fixed so that
 * G -> ln(r) / (2 pi) far away, as for the Gaussian kernels of reading A28,
 *     G(r) = ( C(k_c r) - ln(k_c / 2) - gamma ) / (2 pi),   C(x) = int_0^x (1 - J0(t)) / t dt,
 *     G(0) = -( ln(k_c / 2) + gamma ) / (2 pi).
 * C(x) is computed from its definition: the power series sum_{m>=1} (-1)^(m+1) (x/2)^(2m) / (2m (m!)^2) in extended
 * precision up to x = 12, beyond that C(12) + ln(x / 12) - int_12^x J0(t) / t dt with composite 16-point Gauss-Legendre
 * panels of length <= 2 on the library's j0().
 * ---------------------------------------------------------------------------------------- */
extern double j0(double);   /* POSIX Bessel function of the C library (not declared under strict ISO C) */
static double cin_series(double x)
{
    long double q = 0.25L * (long double)x * (long double)x, term = 1.0L, sum = 0.0L;
    for (int m = 1; m < 200; ++m) {
        term *= -q / ((long double)m * (long double)m);          /* (-1)^m (x/2)^(2m) / (m!)^2 */
        long double add = -term / (2.0L * (long double)m);
        sum += add;
        if (fabsl(add) < 1e-22L * fabsl(sum) && m > (int)x) break;
    }
    return (double)sum;
}
double orc_bessel_cin(double x)
{
    static const double gx[8] = { 0.0950125098376374401853193, 0.2816035507792589132304605, 0.4580167776572273863424194,
                                  0.6178762444026437484466718, 0.7554044083550030338951012, 0.8656312023878317438804679,
                                  0.9445750230732325760779884, 0.9894009349916499325961542 };
    static const double gw[8] = { 0.1894506104550684962853967, 0.1826034150449235888667637, 0.1691565193950025381893121,
                                  0.1495959888165767320815017, 0.1246289712555338720524763, 0.0951585116824927848099251,
                                  0.0622535239386478928628438, 0.0271524594117540948517806 };
    if (x < 0.0) x = -x;
    if (x <= 12.0) return cin_series(x);
    double acc = 0.0;
    int panels = (int)ceil((x - 12.0) / 2.0);
    double len = (x - 12.0) / (double)panels;
    for (int p = 0; p < panels; ++p) {
        double a = 12.0 + len * (double)p, mid = a + 0.5 * len, half = 0.5 * len, s = 0.0;
        for (int i = 0; i < 8; ++i) {
            double t1 = mid + half * gx[i], t2 = mid - half * gx[i];
            s += gw[i] * (j0(t1) / t1 + j0(t2) / t2);
        }
        acc += s * half;
    }
    return cin_series(12.0) + log(x / 12.0) - acc;
}
double orc_green2d_spectral(double r, double h)
{
    const double kc = PI / h, euler = 0.57721566490153286061;
    if (r == 0.0) return -(log(0.5 * kc) + euler) / (2.0 * PI);
    return (orc_bessel_cin(kc * r) - log(0.5 * kc) - euler) / (2.0 * PI);
}

/* order 2 .. 10: Gaussian-regularised kernels (reading A28); order 0: the spectrally compact kernel above with
 * h = max spacing (eps ignored, as for the 3-D kernel) */
int orc_unbounded2d_green(const i64 n[2], const double h[2], double eps, int order, cplx *ghat)
{
    if (order != 0 && (order < 2 || order > 10 || (order & 1))) return ORC_ERR_ARG;
    for (int a = 0; a < 2; ++a) if (!is_pow2(n[a])) return ORC_ERR_ARG;
    i64 P0 = 2 * n[0], P1 = 2 * n[1];
    double *g = (double *)malloc(sizeof(double) * (size_t)(P0 * P1));
    if (!g) return ORC_ERR_ALLOC;
    double area = h[0] * h[1];
    double hmax = h[0] > h[1] ? h[0] : h[1];
#pragma omp parallel for schedule(dynamic, 1)
    for (i64 iy = 0; iy < P1; ++iy)
        for (i64 ix = 0; ix < P0; ++ix) {
            double dx = (double)(ix < P0 - ix ? ix : P0 - ix) * h[0];
            double dy = (double)(iy < P1 - iy ? iy : P1 - iy) * h[1];
            double r = sqrt(dx * dx + dy * dy);
            g[ix + P0 * iy] = area * (order == 0 ? orc_green2d_spectral(r, hmax) : orc_green2d_gauss(order, r, eps));
        }
    int err = unb2_forward(n, g, 0, ghat);
    free(g);
    return err;
}

int orc_unbounded2d_solve(const i64 n[2], const double h[2], const cplx *ghat, double rhs_sign, const double *f,
                          double *psi, double *grad)
{
    for (int a = 0; a < 2; ++a) if (!is_pow2(n[a])) return ORC_ERR_ARG;
    i64 P[2] = { 2 * n[0], 2 * n[1] }, H0 = n[0] + 1, ns = H0 * P[1], tot = n[0] * n[1];
    cplx *spec = (cplx *)malloc(sizeof(cplx) * (size_t)ns), *work = (cplx *)malloc(sizeof(cplx) * (size_t)ns);
    int err = ORC_OK;
    if (!spec || !work) { err = ORC_ERR_ALLOC; goto done; }
    if ((err = unb2_forward(n, f, 1, spec)) != ORC_OK) goto done;
    for (i64 i = 0; i < ns; ++i) spec[i] = rhs_sign * ghat[i] * spec[i];
    if (grad) {
        for (int a = 0; a < 2; ++a) {
            for (i64 ky = 0; ky < P[1]; ++ky)
                for (i64 kx = 0; kx < H0; ++kx) {
                    i64 kk = a ? ky : kx;
                    i64 m = (kk < n[a]) ? kk : kk - P[a];
                    double kap = (kk == n[a]) ? 0.0 : 2.0 * PI * (double)m / ((double)P[a] * h[a]);
                    work[kx + H0 * ky] = I * kap * spec[kx + H0 * ky];
                }
            if ((err = unb2_backward_extract(n, work, grad + (size_t)a * (size_t)tot)) != ORC_OK) goto done;
        }
    }
    err = unb2_backward_extract(n, spec, psi);
done:
    free(spec); free(work);
    return err;
}

/* the definition by direct O(N^4) summation, tiny grids only */
void orc_unbounded2d_direct(const i64 n[2], const double h[2], double eps, int order, double rhs_sign, const double *f,
                            double *psi)
{
    double area = h[0] * h[1];
    for (i64 iy = 0; iy < n[1]; ++iy)
        for (i64 ix = 0; ix < n[0]; ++ix) {
            long double acc = 0.0L;
            for (i64 jy = 0; jy < n[1]; ++jy)
                for (i64 jx = 0; jx < n[0]; ++jx) {
                    double dx = (double)(ix - jx) * h[0], dy = (double)(iy - jy) * h[1];
                    acc += (long double)orc_green2d_gauss(order, sqrt(dx * dx + dy * dy), eps) * f[jx + n[0] * jy];
                }
            psi[ix + n[0] * iy] = (double)(rhs_sign * area * acc);
        }
}

/* Direct O(N^6) evaluation of the definition above (scalar), for tiny grids only (pin P6). */
void orc_unbounded_direct(const i64 n[3], const double h[3], double eps, double rhs_sign, const double *f,
                          double *psi)
{
    double vol = h[0] * h[1] * h[2];
#pragma omp parallel for collapse(2) schedule(static)
    for (i64 iz = 0; iz < n[2]; ++iz)
        for (i64 iy = 0; iy < n[1]; ++iy)
            for (i64 ix = 0; ix < n[0]; ++ix) {
                long double acc = 0.0L;
                for (i64 jz = 0; jz < n[2]; ++jz)
                    for (i64 jy = 0; jy < n[1]; ++jy)
                        for (i64 jx = 0; jx < n[0]; ++jx) {
                            double dx = (double)(ix - jx) * h[0], dy = (double)(iy - jy) * h[1],
                                   dz = (double)(iz - jz) * h[2];
                            acc += (long double)orc_green_gauss2(sqrt(dx * dx + dy * dy + dz * dz), eps) *
                                   f[jx + n[0] * (jy + n[1] * jz)];
                        }
                psi[ix + n[0] * (iy + n[1] * iz)] = (double)(rhs_sign * vol * acc);
            }
}

/* Direct evaluation of the definition at a list of output points (full-size sampled parity):
 * psi(idx[s]) for s < ns, idx = linear grid indices. */
void orc_unbounded_direct_samples(const i64 n[3], const double h[3], double eps, double rhs_sign,
                                  const double *f, i64 ns, const i64 *idx, double *psi)
{
    double vol = h[0] * h[1] * h[2];
    for (i64 s = 0; s < ns; ++s) {
        i64 ix = idx[s] % n[0], iy = (idx[s] / n[0]) % n[1], iz = idx[s] / (n[0] * n[1]);
        double acc = 0.0;
#pragma omp parallel for reduction(+ : acc) schedule(static)
        for (i64 jz = 0; jz < n[2]; ++jz) {
            long double a = 0.0L;
            for (i64 jy = 0; jy < n[1]; ++jy)
                for (i64 jx = 0; jx < n[0]; ++jx) {
                    double fv = f[jx + n[0] * (jy + n[1] * jz)];
                    if (fv == 0.0) continue;
                    double dx = (double)(ix - jx) * h[0], dy = (double)(iy - jy) * h[1],
                           dz = (double)(iz - jz) * h[2];
                    a += (long double)orc_green_gauss2(sqrt(dx * dx + dy * dy + dz * dz), eps) * fv;
                }
            acc += (double)a;
        }
        psi[s] = rhs_sign * vol * acc;
    }
}
