// sf_common.cuh -- shared device building blocks of the sm_100a spectral Poisson kernels.
//
//   * complex arithmetic on float2 / double2
//   * register-resident radix-2/4/8/16 DFTs (decimation in frequency, compile-time constants)
//   * the per-length stage plan (mixed radix 16/8/4/2) and the digit-reversal maps that go with an
//     in-place decimation-in-frequency transform
//   * one in-place butterfly stage on a shared-memory tile laid out [position][pencil]
//   * one Stockham (self-sorting) stage on a shared-memory tile laid out [row][position]
//
// The transforms are those of PAPER.md eq. (8): forward exp(-2 pi i nk/N),
// backward exp(+2 pi i nk/N), both unnormalised here; the 1/N is folded into the spectral
// multiplier by the host.
#pragma once
#include "sf_trig.cuh"
#include <cuda_runtime.h>
#include <stdint.h>

namespace sf {

// ------------------------------------------------------------------------------------ complex
template <typename T> struct cx_of;
template <> struct cx_of<float> { typedef float2 type; };
template <> struct cx_of<double> { typedef double2 type; };

template <typename T> __host__ __device__ __forceinline__ typename cx_of<T>::type mk(T a, T b)
{
    typename cx_of<T>::type r;
    r.x = a;
    r.y = b;
    return r;
}
#define SF_CX typename cx_of<T>::type

template <typename C> __device__ __forceinline__ C cadd(C a, C b) { a.x += b.x; a.y += b.y; return a; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename C> __device__ __forceinline__ C cconj(C a) { a.y = -a.y; return a; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b)
{
    C r;
    r.x = a.x * b.x - a.y * b.y;
    r.y = a.x * b.y + a.y * b.x;
    return r;
}
// a * conj(b)
template <typename C> __device__ __forceinline__ C cmulc(C a, C b)
{
    C r;
    r.x = a.x * b.x + a.y * b.y;
    r.y = a.y * b.x - a.x * b.y;
    return r;
}
template <typename C, typename T> __device__ __forceinline__ C cscale(C a, T s) { a.x *= s; a.y *= s; return a; }
// multiply by +i / -i
template <typename C> __device__ __forceinline__ C cmuli(C a) { C r; r.x = -a.y; r.y = a.x; return r; }
template <typename C> __device__ __forceinline__ C cmulmi(C a) { C r; r.x = a.y; r.y = -a.x; return r; }

// ------------------------------------------------------------------------------------ radix DFTs
using sftrig::cos16;   // cos / sin of 2 pi i / 16 (sf_trig.cuh)
using sftrig::sin16;

// multiply d by exp(-/+ 2 pi i * I16 / 16) (forward: minus) with the trivial cases special-cased
template <int I16, bool INV, typename C> __device__ __forceinline__ C mul_w16(C d)
{
    typedef decltype(d.x) T;
    if constexpr (I16 == 0) {
        return d;
    } else if constexpr (I16 == 4) {
        return INV ? cmuli(d) : cmulmi(d);
    } else if constexpr (I16 == 2) {
        constexpr T h = (T)0.70710678118654752440;
        C r; // (1 -/+ i)/sqrt2 * d
        if (INV) { r.x = (d.x - d.y) * h; r.y = (d.x + d.y) * h; }
        else     { r.x = (d.x + d.y) * h; r.y = (d.y - d.x) * h; }
        return r;
    } else if constexpr (I16 == 6) {
        constexpr T h = (T)0.70710678118654752440;
        C r; // (-1 -/+ i)/sqrt2 * d
        if (INV) { r.x = (-d.x - d.y) * h; r.y = (d.x - d.y) * h; }
        else     { r.x = (d.y - d.x) * h; r.y = (-d.x - d.y) * h; }
        return r;
    } else {
        constexpr T c = (T)cos16(I16);
        constexpr T s = (T)(INV ? sin16(I16) : -sin16(I16));
        C r;
        r.x = d.x * c - d.y * s;
        r.y = d.x * s + d.y * c;
        return r;
    }
}

// In-place radix-2 decimation-in-frequency recursion on v[0], v[S], ..., v[(R-1)S]: result q of the
// length-R DFT ends at v[brev_R(q) * S].
template <int R, int S, bool INV, typename C> struct dft_rec {
    template <int I> static __device__ __forceinline__ void level(C* v)
    {
        if constexpr (I < R / 2) {
            C a = v[I * S], b = v[(I + R / 2) * S];
            v[I * S] = cadd(a, b);
            v[(I + R / 2) * S] = mul_w16<I * (16 / R), INV>(csub(a, b));
            level<I + 1>(v);
        }
    }
    static __device__ __forceinline__ void run(C* v)
    {
        level<0>(v);
        dft_rec<R / 2, S, INV, C>::run(v);
        dft_rec<R / 2, S, INV, C>::run(v + (R / 2) * S);
    }
};
template <int S, bool INV, typename C> struct dft_rec<1, S, INV, C> {
    static __device__ __forceinline__ void run(C*) {}
};

__host__ __device__ constexpr int brev(int q, int R)
{
    int r = 0;
    for (int b = 1; b < R; b <<= 1) { r = (r << 1) | (q & 1); q >>= 1; }
    return r;
}

// v[0..R): natural order in, result q at v[brev(q, R)]
template <int R, bool INV, typename C> __device__ __forceinline__ void dft_reg(C (&v)[R])
{
    dft_rec<R, 1, INV, C>::run(v);
}

// ------------------------------------------------------------------------------------ stage plan
struct StagePlan { int ns; int r[4]; };
__host__ __device__ constexpr StagePlan make_plan(int L)
{
    switch (L) {
    case 1: return { 0, { 1, 1, 1, 1 } };
    case 2: return { 1, { 2, 1, 1, 1 } };
    case 4: return { 1, { 4, 1, 1, 1 } };
    case 8: return { 1, { 8, 1, 1, 1 } };
    case 16: return { 1, { 16, 1, 1, 1 } };
    case 32: return { 2, { 8, 4, 1, 1 } };
    case 64: return { 2, { 8, 8, 1, 1 } };
    case 128: return { 2, { 16, 8, 1, 1 } };
    case 256: return { 2, { 16, 16, 1, 1 } };
    case 512: return { 3, { 8, 8, 8, 1 } };
    case 1024: return { 3, { 16, 8, 8, 1 } };
    case 2048: return { 3, { 16, 16, 8, 1 } };
    case 4096: return { 3, { 16, 16, 16, 1 } };
    default: return { 0, { 1, 1, 1, 1 } };
    }
}
// block length at the start of stage s (product of the radices from s on)
__host__ __device__ constexpr int stage_len(int L, int s)
{
    StagePlan p = make_plan(L);
    int m = L;
    for (int i = 0; i < s; ++i) m /= p.r[i];
    return m;
}

// After the in-place DIF transform, output k = k1 + R1 k2 + R1 R2 k3 sits at position
// p = k1 (L/R1) + k2 (L/(R1 R2)) + k3 (L/(R1 R2 R3)).
template <int L> __host__ __device__ __forceinline__ int pos_of_k(int k)
{
    constexpr StagePlan pl = make_plan(L);
    int p = 0, m = L;
#pragma unroll
    for (int s = 0; s < pl.ns; ++s) {
        m /= pl.r[s];
        p += (k % pl.r[s]) * m;
        k /= pl.r[s];
    }
    return p;
}
template <int L> __host__ __device__ __forceinline__ int k_of_pos(int p)
{
    constexpr StagePlan pl = make_plan(L);
    int k = 0, m = L, mult = 1;
#pragma unroll
    for (int s = 0; s < pl.ns; ++s) {
        m /= pl.r[s];
        k += ((p / m) % pl.r[s]) * mult;
        mult *= pl.r[s];
    }
    return k;
}

// ------------------------------------------------------------------------------------ tile stages
// One butterfly stage, in place, on a tile s[position * TX + pencil] (pencil index fastest: every
// access of a warp is to consecutive addresses whatever the position permutation, so no stage has
// shared-memory bank conflicts).
//   forward (INV = false): Gentleman-Sande: v = DFT_R(s[base + r Q]);  v[q] *= w_M^(q o)
//   backward (INV = true): the exact mirror: v[q] = s[base + q Q] * conj(w_M^(q o));  v = IDFT_R(v)
// M = block length of this stage, Q = M / R, base = block * M + o.
// tw: table of exp(-2 pi i j / LT), j < LT; w_M^(q o) = tw[q * o * (LT / M)].
template <typename T, int L, int M, int R, int TX, int NT, bool INV>
__device__ __forceinline__ void tile_stage(SF_CX* __restrict__ s, const SF_CX* __restrict__ tw, int LT)
{
    typedef SF_CX C;
    constexpr int Q = M / R;
    constexpr int NB = L / R;
    const int tstep = LT / M;
    for (int item = threadIdx.x; item < NB * TX; item += NT) {
        const int tx = item % TX;
        const int b = item / TX;
        const int o = b % Q;
        const int base = (b / Q) * M + o;
        C* p = s + base * TX + tx;
        C v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = p[r * Q * TX];
        if constexpr (INV) {
            if constexpr (Q > 1) {
#pragma unroll
                for (int q = 1; q < R; ++q) v[q] = cmulc(v[q], __ldg(tw + q * o * tstep));
            }
            dft_reg<R, true>(v);
#pragma unroll
            for (int r = 0; r < R; ++r) p[r * Q * TX] = v[brev(r, R)];
        } else {
            dft_reg<R, false>(v);
            if constexpr (Q > 1) {
#pragma unroll
                for (int q = 1; q < R; ++q) v[brev(q, R)] = cmul(v[brev(q, R)], __ldg(tw + q * o * tstep));
            }
#pragma unroll
            for (int q = 0; q < R; ++q) p[q * Q * TX] = v[brev(q, R)];
        }
    }
}

// all stages, forward: natural order in, X[k] at pos_of_k<L>(k) out.  Ends with a barrier.
template <typename T, int L, int TX, int NT, int S = 0>
__device__ __forceinline__ void tile_fft_fwd(SF_CX* s, const SF_CX* tw, int LT)
{
    constexpr StagePlan pl = make_plan(L);
    if constexpr (S < pl.ns) {
        tile_stage<T, L, stage_len(L, S), pl.r[S], TX, NT, false>(s, tw, LT);
        __syncthreads();
        tile_fft_fwd<T, L, TX, NT, S + 1>(s, tw, LT);
    }
}
// all stages, backward: X[k] at pos_of_k<L>(k) in, natural order out (unnormalised).  Ends with a barrier.
template <typename T, int L, int TX, int NT, int S = -1>
__device__ __forceinline__ void tile_fft_inv(SF_CX* s, const SF_CX* tw, int LT)
{
    constexpr StagePlan pl = make_plan(L);
    constexpr int SS = (S < 0) ? pl.ns - 1 : S;
    if constexpr (pl.ns > 0) {
        tile_stage<T, L, stage_len(L, SS), pl.r[SS], TX, NT, true>(s, tw, LT);
        __syncthreads();
        if constexpr (SS > 0) tile_fft_inv<T, L, TX, NT, SS - 1>(s, tw, LT);
    }
}

// One Stockham stage a -> b on tiles laid out [row * LP + position] (LP odd multiple keeps the
// row-strided accesses of a warp on distinct banks).  NS = product of the radices already done.
template <typename T, int L, int NS, int R, int ROWS, int LP, int NT, bool INV>
__device__ __forceinline__ void stockham_stage(const SF_CX* __restrict__ a, SF_CX* __restrict__ b,
                                               const SF_CX* __restrict__ tw, int LT)
{
    typedef SF_CX C;
    constexpr int NB = L / R;
    const int tstep = LT / (NS * R);
    for (int item = threadIdx.x; item < NB * ROWS; item += NT) {
        const int row = item % ROWS;
        const int j = item / ROWS;
        const int k = j % NS;
        const C* pa = a + row * LP + j;
        C v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = pa[r * NB];
        if constexpr (NS > 1) {
#pragma unroll
            for (int r = 1; r < R; ++r) {
                C w = __ldg(tw + r * k * tstep);
                v[r] = INV ? cmulc(v[r], w) : cmul(v[r], w);
            }
        }
        dft_reg<R, INV>(v);
        C* pb = b + row * LP + (j / NS) * NS * R + k;
#pragma unroll
        for (int q = 0; q < R; ++q) pb[q * NS] = v[brev(q, R)];
    }
}

// all Stockham stages; returns the buffer that holds the result (natural order).  Ends with a barrier.
template <typename T, int L, int ROWS, int LP, int NT, bool INV, int S = 0, int NS = 1>
__device__ __forceinline__ SF_CX* stockham_fft(SF_CX* a, SF_CX* b, const SF_CX* tw, int LT)
{
    constexpr StagePlan pl = make_plan(L);
    if constexpr (S < pl.ns) {
        stockham_stage<T, L, NS, pl.r[S], ROWS, LP, NT, INV>(a, b, tw, LT);
        __syncthreads();
        return stockham_fft<T, L, ROWS, LP, NT, INV, S + 1, NS * pl.r[S]>(b, a, tw, LT);
    } else {
        return a;
    }
}

} // namespace sf
