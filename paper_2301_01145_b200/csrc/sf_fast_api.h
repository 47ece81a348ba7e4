// sf_fast_api.h -- host-visible interface of kernel generation 2 (sf_fast.cuh / sf_fast.cu):
// parameter block and launchers of the fp32 256 -> 512 padded strided passes.
#pragma once
#include <cuda_runtime.h>

namespace sf {
template <typename T> struct XParams;   // sf_xpass.cuh
}

namespace sf2 {

typedef float2 C;

constexpr int kTile = 16;            // pencils per tile
constexpr int kGreenRows = 257;      // folded spectral indices along the pencil axis (0 .. 256)

enum { FMODE_FWD = 0, FMODE_INV = 1, FMODE_FUSED = 2 };

// opaque storage of a CUtensorMap (TMA descriptor): 128 bytes, 64-byte aligned
struct alignas(64) TileMap { unsigned char bytes[128]; };

struct FastParams {
    const C* in;
    C* out;
    long long in_ps, in_bs;     // row (pencil-axis) and batch strides of the input, complex elements
    long long out_ps, out_bs;
    int nb;                     // batches
    int nct;                    // full 16-column tiles per batch: a power of two
    int nct_shift;              // log2(nct)
    int nyq_col;                // column handled 16 batches at a time (the Nyquist column), -1: none
    // Optional side arrays that hold the Nyquist column instead of column nyq_col of in / out, laid out
    // so that its tiles move in 128-byte runs too (NULL: gather / scatter column nyq_col):
    //   FWD   nyq_in [row y][batch z]   -> nyq_out [batch z][row ky] (512 per z)
    //   FUSED nyq_in = nyq_out [row z][batch ky]
    //   INV   nyq_in [batch z][row ky]  -> nyq_out [row y][batch z]
    const C* nyq_in;
    C* nyq_out;
    int reverse_batches;        // visit batches last to first (the producer kernel wrote them first to last)
    int* sched;                 // device: { next unclaimed tile, CTAs finished }, zero between launches
    int nyq_first;              // Nyquist-column tiles at the head of the tile queue instead of its tail
    int pair_batches;           // fused: visit batches as 0, P/2, 1, P-1, 2, P-2, ... (mirror pairs share table rows)
    // fused multiply: real Green's table (rhs sign and normalisation folded in), tile-major:
    // chunk [kGreenRows fp][16 pencils] per tile, see green_tile_index / fast_green_tiles
    const float* green_tiles;
    int Pb;                     // transform length along the batch axis (index folding k -> min(k, P-k))
};


__host__ __device__ inline int fast_ntiles(int nb, int nct, int nyq_col) { return nb * nct + (nyq_col >= 0 ? (nb + kTile - 1) / kTile : 0); }

// S1 / S5 for rows of 256 reals padded to 512 (fast_x_kernel)
struct FastXParams {
    const float* real_in;   // S1: [rows][256]
    float* real_out;        // S5: [rows][256]
    C* spec;                // half spectra, row pitch spec_pitch complex (>= 258, rows 16-byte aligned)
    long long spec_pitch;
    int nrows;              // multiple of 16
    int reverse;            // visit row tiles last to first
    C* nyq;                 // optional side array [y][z] (n1 x n2) of the Nyquist coefficient X[256] of row z * n1 + y:
    int n1, n2;             // S1 writes it (besides column 256 of spec), S5 reads it (instead); NULL: column 256 only
};

constexpr int kPerTileCols = 32;
// strided passes of periodic plans with 256-point pencils (fast_per_kernel): tiles of 32 columns
struct FastPerParams {
    const C* in;
    C* out;
    long long in_ps, in_bs, out_ps, out_bs;   // row and batch strides, complex elements
    int nb;          // batches
    int nx;          // valid columns
    int nct;         // full 32-column tiles per batch
    int nyq_col;     // column handled 32 batches at a time, -1: none
    int* sched;      // device: { next unclaimed tile, CTAs finished }, zero between launches
    C* nyq;          // side array that holds column nyq_col: element (row, batch) at row * nyq_ps + batch * nyq_bs
    long long nyq_ps, nyq_bs;
    // fused multiply: scale / (lam_x[column] + lam_b[batch] + lam_p[row]), zero mode -> 0
    const float* lam_x; const float* lam_b; const float* lam_p;
    float scale;
    int zero_mode;
    // gradient (fused mode): fields 1 .. 3 = d/dx, d/dy (batch axis), d/dz (pencil axis) of the result
    int grad;
    const float* kap_x; const float* kap_b; const float* kap_p;   // wavenumbers, zero at the Nyquist index
    long long out_cs, nyq_cs;                                     // field strides of out and of the side array
};

// S1 / S5 of periodic plans for rows of 256 reals (fast_xper_kernel)
struct FastXPerParams {
    const float* real_in;   // S1: [rows][256]
    float* real_out;        // S5: [rows][256]
    C* spec;                // half spectra X[0..127], row pitch spec_pitch complex
    long long spec_pitch;
    int nrows;              // multiple of 32
    C* nyq;                 // side array [row] of X[128]
};

// strided passes of fp32 unbounded plans with 512-point y / z pencils padded to 1024 (fast5_kernel, sf_fast512.cuh)
constexpr int kGreenRows5 = 513;     // folded spectral indices along the pencil axis (0 .. 512)
enum { F5_FWD = 0, F5_INV = 1, F5_FUSED = 2, F5_CURL = 3 };
struct Fast5Params {
    const C* in;
    C* out;
    long long in_ps, in_bs, in_cs;     // row (pencil-axis), batch and component strides, complex elements
    long long out_ps, out_bs, out_cs;
    int nb;                     // batches (FWD / INV: components are more batches)
    int nct, nct_shift;         // full 16-column tiles per batch: a power of two
    int nyq_col;                // column handled 16 batches at a time (the Nyquist column), -1: none
    int ncomp;                  // FUSED: independent components (more tiles); CURL: 3
    int reverse_batches;        // visit batches last to first
    int pair_batches;           // visit batches as 0, P/2, 1, P-1, 2, P-2, ... (mirror pairs share the Green's chunk)
    int* sched;                 // device: { next unclaimed tile, CTAs finished }, zero between launches
    const float* green_tiles;   // tile-major real Green's table: chunk [kGreenRows5 fp][16 pencils] per tile
    int Pb;                     // transform length along the batch axis (index folding k -> min(k, P - k))
    // CURL: wavenumbers of the doubled grid (zero at the Nyquist index): per column, per batch, per pencil row (1024)
    const float* kap_x; const float* kap_b; const float* kap_p;
};
// strided passes of fp64 unbounded plans with 256-point y / z pencils padded to 512 (fast64_kernel, sf_fast64.cuh):
// tiles of 8 pencils
struct Fast64Params {
    const double2* in;
    double2* out;
    long long in_ps, in_bs;     // row (pencil-axis) and batch strides, complex elements
    long long out_ps, out_bs;
    int nb;                     // batches
    int nct, nct_shift;         // full 8-column tiles per batch: a power of two
    int nyq_col;                // column handled 8 batches at a time (the Nyquist column), -1: none
    int reverse_batches, pair_batches;
    int* sched;                 // device: { next unclaimed tile, CTAs finished }, zero between launches
    const double* green_tiles;  // tile-major real Green's table: chunk [kGreenRows fp][8 pencils] per tile
    int Pb;
};
inline size_t fast64_green_tiles_elems(int Pb, int nct, int nyq_col)
{
    return ((size_t)(Pb / 2 + 1) * nct + (nyq_col >= 0 ? (size_t)(Pb + 7) / 8 : 0)) * kGreenRows * 8;
}
cudaError_t fast64_green_tiles(double* tiles, const double* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                               cudaStream_t st);
// launch one fp64 padded pass (mode = FMODE_*) as a persistent grid of two 256-thread CTAs per SM; `in_map` describes
// p.in in 8-byte words as documented at fast64_kernel
cudaError_t launch_fast64(int mode, const Fast64Params& p, const TileMap& in_map, cudaStream_t st);

// number of floats of the tile-major Green's table with `rows` folded pencil indices per chunk
inline size_t fast_green_tiles_elems_rows(int Pb, int nct, int nyq_col, int rows)
{
    return ((size_t)(Pb / 2 + 1) * nct + (nyq_col >= 0 ? (size_t)(Pb + kTile - 1) / kTile : 0)) * rows * kTile;
}
cudaError_t fast_green_tiles_rows(float* tiles, const float* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                                  int rows, cudaStream_t st);
// the same for tiles of `width` pencils (nct = tiles of that width per batch; Nyquist tiles of `width` batches)
inline size_t fast_green_tiles_elems_rows_w(int Pb, int nct, int nyq_col, int rows, int width)
{
    return ((size_t)(Pb / 2 + 1) * nct + (nyq_col >= 0 ? (size_t)(Pb + width - 1) / width : 0)) * rows * width;
}
cudaError_t fast_green_tiles_rows_w(float* tiles, const float* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                                    int rows, int width, cudaStream_t st);
// launch one 512 -> 1024 padded pass (mode = F5_*) as a persistent grid of one 1024-thread CTA per SM; `in_map`
// describes p.in as documented at fast5_kernel
cudaError_t launch_fast5(int mode, const Fast5Params& p, const TileMap& in_map, cudaStream_t st);


// one-time per-process set-up: twiddle constants, shared-memory opt-in, SM count, driver entry point
cudaError_t fast_init();
// rank-4 tensor map over 8-byte elements: dims[0] fastest; strides_bytes[i] = stride of dims[i+1]
// (multiples of 16); box = tile image moved by one TMA instruction (dense, no swizzle)
cudaError_t fast_make_map(TileMap* out, const void* base, const unsigned long long dims[4],
                          const unsigned long long strides_bytes[3], const unsigned box[4]);
// number of floats of the tile-major Green's table for nb = P batches, nct column tiles (+ Nyquist column)
inline size_t fast_green_tiles_elems(int Pb, int nct, int nyq_col)
{
    return ((size_t)(Pb / 2 + 1) * nct + (nyq_col >= 0 ? (size_t)(Pb + kTile - 1) / kTile : 0)) * kGreenRows * kTile;
}
// re-lay the compact table green[fp][fb][kx] (pitches g_pp, g_pb) tile-major into `tiles`
cudaError_t fast_green_tiles(float* tiles, const float* green, long long g_pb, long long g_pp, int Pb, int nct, int nyq_col,
                             cudaStream_t st);
// launch one padded pass (mode = FMODE_*) as a persistent grid of two CTAs per SM; `in_map`
// describes p.in as documented at fast_pad_kernel
cudaError_t launch_fast_pad(int mode, const FastParams& p, const TileMap& in_map, cudaStream_t st);

// launch S1 (inv = false) or S5 (inv = true) as a persistent grid of two CTAs per SM
cudaError_t launch_fast_x(bool inv, const FastXParams& p, cudaStream_t st);
// the same for rows of 512 reals padded to 1024 (fast_x5_kernel; spec_pitch >= 514, no side array: p.nyq must be NULL;
// nrows a multiple of 8)
cudaError_t launch_fast_x5(bool inv, const FastXParams& p, cudaStream_t st);
// launch one periodic strided pass (mode = FMODE_*) as a persistent grid of two CTAs per SM
cudaError_t launch_fast_per(int mode, const FastPerParams& p, cudaStream_t st);
cudaError_t launch_fast_xper(bool inv, const FastXPerParams& p, cudaStream_t st);

// strided passes of fp64 periodic plans with 256-point pencils (fast_per64_kernel, sf_fastper64.cuh): tiles of 16 columns
struct FastPer64Params {
    const double2* in;
    double2* out;
    long long in_ps, in_bs, out_ps, out_bs;   // row and batch strides, complex elements
    int nb, nx, nct;            // batches, valid columns, full 16-column tiles per batch
    int nyq_col;                // column handled 16 batches at a time, -1: none
    int* sched;
    double2* nyq;               // side array that holds column nyq_col: element (row, batch) at row * nyq_ps + batch * nyq_bs
    long long nyq_ps, nyq_bs;
    const double* lam_x; const double* lam_b; const double* lam_p;
    double scale;
    int zero_mode;
    int grad;                   // fused mode: fields 1 .. 3 = d/dx, d/dy (batch axis), d/dz (pencil axis)
    const double* kap_x; const double* kap_b; const double* kap_p;
    long long out_cs, nyq_cs;   // field strides of out and of the side array
};
cudaError_t launch_fast_per64(int mode, const FastPer64Params& p, cudaStream_t st);

// strided passes of fp64 Dirichlet (DST-I, 255 rows) / Neumann (DCT-II / III, 256 rows) plans (fast_r2r64_kernel,
// sf_fastr2r64.cuh): the real work array is addressed as complex columns (pairs of real columns), tiles of 8
struct FastR64Params {
    const double2* in;
    double2* out;
    long long in_ps, in_bs, out_ps, out_bs;   // row and batch strides in complex columns (= real strides / 2)
    int n;                      // stored rows per pencil: 255 (DST-I) or 256 (DCT)
    int nb;                     // batches
    int nct;                    // 8-column tiles per batch (pitch / 16)
    int batch_dim;              // 2: the tensor map is (column, row, batch); 1: (column, batch, row)
    int* sched;
    // fused: scale / (lam_x[real column] + lam_b[batch] + lam_p[row]); zero mode -> 0
    const double* lam_x; const double* lam_b; const double* lam_p;
    int nx;                     // valid real columns
    double scale;
    int zero_mode;
};
// kind 0: DST-I, 1: DCT;  mode 0: forward (x -> Y), 1: backward (DCT-III; DST-I uses forward), 2: fused S3
cudaError_t launch_fast_r2r64(int kind, int mode, const FastR64Params& p, const TileMap& in_map, cudaStream_t st);

// S1 (inv = false) / S5 (inv = true) in double precision for rows whose extended sequence is 512 long (fast_xg_kernel,
// sf_fastx64.cuh): p.mode X_ZEROPAD (n = 256), X_DST1 (n = 255) or X_DCT2 (n = 256); no side array, no differentiated field
cudaError_t launch_fast_xg(bool inv, const sf::XParams<double>& p, int ncomp, cudaStream_t st);

// the same for periodic fp64 rows of 256 reals (fast_xp64_kernel): p.mode X_PERIODIC, n = 256; the side array [field][row] of
// the Nyquist coefficient is honoured when p.nyq_side is set
cudaError_t launch_fast_xp64(bool inv, const sf::XParams<double>& p, int ncomp, cudaStream_t st);

// tensor-core probe (sf_tcprobe.cuh): `reps` applications of one radix-16 exchange + DFT stage on `ntiles` tiles
cudaError_t probe_dft16_stage(int variant, int reps, int ntiles, const void* in, void* out, float* ms, cudaStream_t st);

} // namespace sf2
