// sf_static.cu -- sf_periodic2d_solve_static of include/sailffish.h: the periodic 2-D solve (PAPER.md:103-109 four-step
// solve, eq. (8) :79-81, Table 1 periodic row :166-167, zero mode :69) for callers that may not allocate: one kernel
// launch, no plan, no cudaMalloc / cudaFree, no allocating library call.
//
// The plan path runs this solve as X forward -> work array -> fused Y pass -> X backward with a cudaMalloc'ed work
// array between the launches.  Here the three steps are the phases of ONE kernel (one CTA: its barrier separates the
// phases) and the work array -- the half spectra [n1][n0/2 + 1] between the phases -- is the file-scope array
// g_static_scratch below: kStaticScratchBytes = 528 384 bytes that every device which loads this library holds until
// the process exits.  Every call on a device shares that array: calls that overlap on the GPU (two streams, two host
// threads) race on it; calls on one stream are ordered and safe.  Nothing in it has to start at zero and nothing is
// carried from call to call: phase 1 writes every word that phases 2 and 3 read.
#include "../../include/sailffish.h"

#include <cuda_runtime.h>

#include <mutex>
#include <string>

namespace {

constexpr int kStaticMaxN = SF_STATIC_MAX_N;                          // grid points per axis
constexpr int kStaticHalf = kStaticMaxN / 2 + 1;
constexpr size_t kStaticScratchBytes = (size_t)kStaticMaxN * kStaticHalf * sizeof(double2);
constexpr int kStaticThreads = 1024;
constexpr int kStaticWarps = kStaticThreads / 32;
// dynamic shared memory: twiddles [N/2], eigenvalues of both axes, one pencil buffer per warp
constexpr size_t kStaticSmem = (size_t)(kStaticMaxN / 2) * sizeof(double2) + (size_t)(kStaticHalf + 1 + kStaticMaxN) * sizeof(double) +
                               (size_t)kStaticWarps * kStaticMaxN * sizeof(double2);

// In host code this name is a host-side stand-in, not a device address: the launch below passes the pointer that
// cudaGetSymbolAddress returned for the current device (static_setup).
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

struct StaticParams {
    const double* src;   // [n1][n0]
    double* psi;         // [n1][n0]
    double2* spec;       // scratch [n1][n0 / 2 + 1]
    int n0, n1, l0, l1;  // sizes and their base-2 logarithms
    double h0, h1;
    int op;              // SF_OP_PSEUDO_SPECTRAL or SF_OP_FD2
};

__device__ __forceinline__ double2 zmul(double2 a, double2 w) { return make_double2(fma(a.x, w.x, -a.y * w.y), fma(a.x, w.y, a.y * w.x)); }
__device__ __forceinline__ double2 zmulc(double2 a, double2 w) { return make_double2(fma(a.x, w.x, a.y * w.y), fma(a.y, w.x, -a.x * w.y)); }

// radix-2 decimation in frequency by one warp, forward sign: natural order in, X[k] at position bitrev(k) out.
// tw[j] = exp(-2 pi i j / N), j < N / 2, N a multiple of n.
__device__ void warp_dif_forward(double2* x, int n, const double2* tw, int N, int lane)
{
    for (int m = n >> 1; m >= 1; m >>= 1) {
        const int ts = N / (2 * m);
        for (int j = lane; j < (n >> 1); j += 32) {
            const int pos = j & (m - 1), i0 = ((j - pos) << 1) + pos, i1 = i0 + m;
            const double2 a = x[i0], b = x[i1];
            x[i0] = make_double2(a.x + b.x, a.y + b.y);
            x[i1] = zmul(make_double2(a.x - b.x, a.y - b.y), tw[pos * ts]);
        }
        __syncwarp();
    }
}
// radix-2 decimation in time by one warp, backward sign, unnormalised: X[k] at position bitrev(k) in, natural order out
__device__ void warp_dit_backward(double2* x, int n, const double2* tw, int N, int lane)
{
    for (int m = 1; m < n; m <<= 1) {
        const int ts = N / (2 * m);
        for (int j = lane; j < (n >> 1); j += 32) {
            const int pos = j & (m - 1), i0 = ((j - pos) << 1) + pos, i1 = i0 + m;
            const double2 a = x[i0], t = zmulc(x[i1], tw[pos * ts]);
            x[i0] = make_double2(a.x + t.x, a.y + t.y);
            x[i1] = make_double2(a.x - t.x, a.y - t.y);
        }
        __syncwarp();
    }
}
__device__ __forceinline__ int bitrev(int i, int bits) { return (int)(__brev((unsigned)i) >> (32 - bits)); }

// Table 1, periodic row: PS  -kappa^2, kappa = 2 pi m / L, m = k (k < n/2) or k - n;  FD2  -(4 / h^2) sin^2(pi k / n)
__device__ double static_eigenvalue(int k, int n, double h, int op)
{
    if (op == SF_OP_FD2) {
        const double s = sinpi((double)k / (double)n);
        return -4.0 * s * s / (h * h);
    }
    const int m = (k < n / 2) ? k : k - n;
    const double kap = 2.0 * 3.14159265358979323846 * (double)m / ((double)n * h);
    return -kap * kap;
}

__global__ void __launch_bounds__(kStaticThreads, 1) periodic2d_static_kernel(const StaticParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* tw = reinterpret_cast<double2*>(smem_raw);
    double* ev0 = reinterpret_cast<double*>(tw + kStaticMaxN / 2);   // k <= n0 / 2
    double* ev1 = ev0 + kStaticHalf + 1;                               // k < n1
    double2* bufs = reinterpret_cast<double2*>(ev1 + kStaticMaxN);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n0 = p.n0, n1 = p.n1, hp = n0 / 2 + 1;
    const int N = n0 > n1 ? n0 : n1;
    for (int j = tid; j < N / 2; j += kStaticThreads) {
        double s, c;
        sincospi(-2.0 * (double)j / (double)N, &s, &c);
        tw[j] = make_double2(c, s);
    }
    for (int k = tid; k < hp; k += kStaticThreads) ev0[k] = static_eigenvalue(k, n0, p.h0, p.op);
    for (int k = tid; k < n1; k += kStaticThreads) ev1[k] = static_eigenvalue(k, n1, p.h1, p.op);
    __syncthreads();
    double2* buf = bufs + (size_t)warp * N;

    // phase 1: rows forward along x, half spectrum k <= n0 / 2 into the scratch
    for (int y = warp; y < n1; y += kStaticWarps) {
        for (int i = lane; i < n0; i += 32) buf[i] = make_double2(p.src[(size_t)y * n0 + i], 0.0);
        __syncwarp();
        warp_dif_forward(buf, n0, tw, N, lane);
        for (int i = lane; i < n0; i += 32) {
            const int k = bitrev(i, p.l0);
            if (k < hp) p.spec[(size_t)y * hp + k] = buf[i];
        }
        __syncwarp();
    }
    __syncthreads();   // the CTA's writes to the scratch are visible to all of its threads
    // phase 2: columns forward along y, times 1 / Lambda (zero mode -> 0) and 1 / (n0 n1), backward
    const double scale = 1.0 / ((double)n0 * (double)n1);
    for (int k = warp; k < hp; k += kStaticWarps) {
        for (int i = lane; i < n1; i += 32) buf[i] = p.spec[(size_t)i * hp + k];
        __syncwarp();
        warp_dif_forward(buf, n1, tw, N, lane);
        for (int i = lane; i < n1; i += 32) {
            const int ky = bitrev(i, p.l1);
            const double m = (k == 0 && ky == 0) ? 0.0 : scale / (ev0[k] + ev1[ky]);
            buf[i] = make_double2(buf[i].x * m, buf[i].y * m);
        }
        __syncwarp();
        warp_dit_backward(buf, n1, tw, N, lane);
        for (int i = lane; i < n1; i += 32) p.spec[(size_t)i * hp + k] = buf[i];
        __syncwarp();
    }
    __syncthreads();
    // phase 3: rows backward along x from the half spectrum (X[n0 - k] = conj X[k]: the row is real)
    for (int y = warp; y < n1; y += kStaticWarps) {
        for (int i = lane; i < n0; i += 32) {
            const int k = bitrev(i, p.l0);
            const double2 v = p.spec[(size_t)y * hp + (k < hp ? k : n0 - k)];
            buf[i] = make_double2(v.x, k < hp ? v.y : -v.y);
        }
        __syncwarp();
        warp_dit_backward(buf, n0, tw, N, lane);
        for (int i = lane; i < n0; i += 32) p.psi[(size_t)y * n0 + i] = buf[i].x;
        __syncwarp();
    }
}

thread_local std::string g_static_error = "";
sf_status static_fail(sf_status st, const std::string& msg)
{
    g_static_error = msg;
    return st;
}

// once per device, with that device current: the device address of the scratch array and the kernel's shared-memory limit
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_ptr[kMaxDevices] = { nullptr };

sf_status static_setup(int dev, void** ptr)
{
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* d = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&d, g_static_scratch);
        if (e != cudaSuccess || !d) {
            cudaGetLastError();
            return static_fail(SF_ERR_CUDA, std::string("cudaGetSymbolAddress of the static scratch failed: ") + cudaGetErrorString(e));
        }
        e = cudaFuncSetAttribute(periodic2d_static_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kStaticSmem);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return static_fail(SF_ERR_CUDA, std::string("shared-memory set-up of the static kernel failed: ") + cudaGetErrorString(e));
        }
        g_static_ptr[dev] = d;
    }
    *ptr = g_static_ptr[dev];
    return SF_OK;
}

int log2_exact(long long n)
{
    int l = 0;
    while ((1ll << l) < n) ++l;
    return ((1ll << l) == n) ? l : -1;
}

} // namespace

extern "C" {

const char* sf_static_last_error(void) { return g_static_error.c_str(); }

sf_status sf_periodic2d_solve_static(const long long n[2], const double h[2], sf_operator op, const void* src_dev, void* psi_dev, void* stream)
{
    if (!n || !h || !src_dev || !psi_dev) return static_fail(SF_ERR_INVALID_ARG, "null argument");
    if (op != SF_OP_PSEUDO_SPECTRAL && op != SF_OP_FD2) return static_fail(SF_ERR_UNSUPPORTED, "periodic solves take SF_OP_PSEUDO_SPECTRAL or SF_OP_FD2");
    const int l0 = log2_exact(n[0]), l1 = log2_exact(n[1]);
    if (n[0] < 4 || n[1] < 4 || l0 < 0 || l1 < 0) return static_fail(SF_ERR_INVALID_ARG, "n[0], n[1] must be powers of two >= 4");
    if (n[0] > kStaticMaxN || n[1] > kStaticMaxN)
        return static_fail(SF_ERR_INVALID_ARG, "grid " + std::to_string(n[0]) + " x " + std::to_string(n[1]) + " exceeds the static scratch: at most " +
                                                   std::to_string(kStaticMaxN) + " points per axis (SF_STATIC_MAX_N); use a plan for larger grids");
    if (!(h[0] > 0.0) || !(h[1] > 0.0)) return static_fail(SF_ERR_INVALID_ARG, "h must be positive");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) return static_fail(SF_ERR_CUDA, "no usable current device");
    void* scratch = nullptr;
    sf_status st = static_setup(dev, &scratch);
    if (st != SF_OK) return st;
    StaticParams p;
    p.src = static_cast<const double*>(src_dev);
    p.psi = static_cast<double*>(psi_dev);
    p.spec = static_cast<double2*>(scratch);
    p.n0 = (int)n[0]; p.n1 = (int)n[1]; p.l0 = l0; p.l1 = l1;
    p.h0 = h[0]; p.h1 = h[1];
    p.op = (int)op;
    periodic2d_static_kernel<<<1, kStaticThreads, kStaticSmem, static_cast<cudaStream_t>(stream)>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(SF_ERR_CUDA, std::string("launch failed: ") + cudaGetErrorString(e));
    return SF_OK;
}

} // extern "C"
