// edge.cu — edge correction of the raw multiplets:
//
//   f_Lam'(B) = R^B_Lam' / R^B_0,   M_{Lam Lam''}(B) = sum_Lam' f_Lam'(B) E(Lam'') G^{Lam Lam' Lam''}        eq. 41
//   sum_Lam zeta^B_Lam M_{Lam Lam''}(B) = N^B_Lam'' / R^B_0   ->   zeta^B = M(B)^{-T} N^B / R^B_0              eq. 42
//
// The paper does this in Python with sympy tables and one matrix inversion per bin tuple.  Here the
// tensor T = E G (host tables from App. A's closed forms) sits in HBM; one CTA per bin tuple assembles A = M^T and solves
// A zeta = rhs by LU with partial pivoting (fixed order of operations: deterministic).  Tiny next to the pair stage:
// 120 systems of 69 unknowns at c3/c4.
#include "../../include/encore.h"
#include "device.cuh"

#include <mutex>

namespace {

constexpr int kEdgeThreads = 256;

// A[b][k][i] = sum_j f_j(b) T[i][j][k]  (row k = Lam'', column i = Lam),  rhs[b][k] = N[k][b] / R[0][b]
__global__ void __launch_bounds__(kEdgeThreads) k_edge_assemble(const double *__restrict__ T, const double *__restrict__ Nraw,
                                                                const double *__restrict__ Rraw, int n, int nB, double *__restrict__ A,
                                                                double *__restrict__ rhs)
{
    extern __shared__ double f[]; // n
    const int b = blockIdx.x;
    const double r0 = Rraw[b];
    for (int j = threadIdx.x; j < n; j += blockDim.x) f[j] = Rraw[(size_t)j * nB + b] / r0;
    __syncthreads();
    double *Ab = A + (size_t)b * n * n;
    for (int e = threadIdx.x; e < n * n; e += blockDim.x) {
        const int i = e / n, k = e - i * n;         // consecutive threads: consecutive k (contiguous in T)
        const double *t = T + (size_t)i * n * n + k;
        double s = 0.0;
        for (int j = 0; j < n; ++j) s = fma(f[j], t[(size_t)j * n], s);
        Ab[(size_t)k * n + i] = s;
    }
    for (int k = threadIdx.x; k < n; k += blockDim.x) rhs[(size_t)b * n + k] = Nraw[(size_t)k * nB + b] / r0;
}

// one CTA per bin tuple: in-place LU with partial pivoting on A[b] (n x n, row-major, global memory: L2-resident),
// then forward / back substitution; zeta[i][b] = x[i]
__global__ void __launch_bounds__(kEdgeThreads) k_edge_solve(double *__restrict__ A, double *__restrict__ rhs, int n, int nB,
                                                             double *__restrict__ zeta)
{
    __shared__ double red_v[kEdgeThreads];
    __shared__ int red_i[kEdgeThreads];
    __shared__ int piv;
    const int b = blockIdx.x, tid = threadIdx.x;
    double *M = A + (size_t)b * n * n;
    double *y = rhs + (size_t)b * n;
    for (int c = 0; c < n; ++c) {
        // pivot: largest |M[r][c]|, r >= c (ties: smallest r)
        double best = -1.0;
        int bi = c;
        for (int r = c + tid; r < n; r += kEdgeThreads) {
            const double v = fabs(M[(size_t)r * n + c]);
            if (v > best) { best = v; bi = r; }
        }
        red_v[tid] = best; red_i[tid] = bi;
        __syncthreads();
        for (int st = kEdgeThreads / 2; st > 0; st >>= 1) {
            if (tid < st) {
                const double v = red_v[tid + st];
                const int i2 = red_i[tid + st];
                if (v > red_v[tid] || (v == red_v[tid] && i2 < red_i[tid])) { red_v[tid] = v; red_i[tid] = i2; }
            }
            __syncthreads();
        }
        if (tid == 0) piv = red_i[0];
        __syncthreads();
        const int p = piv;
        if (p != c) {
            for (int j = tid; j < n; j += kEdgeThreads) {
                const double t = M[(size_t)c * n + j];
                M[(size_t)c * n + j] = M[(size_t)p * n + j];
                M[(size_t)p * n + j] = t;
            }
            if (tid == 0) { const double t = y[c]; y[c] = y[p]; y[p] = t; }
        }
        __syncthreads();
        const double inv = 1.0 / M[(size_t)c * n + c];
        // multipliers, then the rank-1 update of the trailing block and of the right-hand side
        for (int r = c + 1 + tid; r < n; r += kEdgeThreads) M[(size_t)r * n + c] *= inv;
        __syncthreads();
        const int m = n - c - 1;
        for (int e = tid; e < m * m; e += kEdgeThreads) {
            const int r = c + 1 + e / m, j = c + 1 + e % m;
            M[(size_t)r * n + j] = fma(-M[(size_t)r * n + c], M[(size_t)c * n + j], M[(size_t)r * n + j]);
        }
        for (int r = c + 1 + tid; r < n; r += kEdgeThreads) y[r] = fma(-M[(size_t)r * n + c], y[c], y[r]);
        __syncthreads();
    }
    // back substitution (U x = y), one unknown at a time, the dot product over the threads in a fixed tree
    for (int c = n - 1; c >= 0; --c) {
        double s = 0.0;
        for (int j = c + 1 + tid; j < n; j += kEdgeThreads) s = fma(M[(size_t)c * n + j], y[j], s);
        red_v[tid] = s;
        __syncthreads();
        for (int st = kEdgeThreads / 2; st > 0; st >>= 1) {
            if (tid < st) red_v[tid] += red_v[tid + st];
            __syncthreads();
        }
        if (tid == 0) y[c] = (y[c] - red_v[0]) / M[(size_t)c * n + c];
        __syncthreads();
    }
    for (int i = tid; i < n; i += kEdgeThreads) zeta[(size_t)i * nB + b] = y[i];
}

} // namespace

cudaError_t launch_edge_correct(const double *T, const double *Nraw, const double *Rraw, int n, int nB, double *A, double *rhs,
                                double *zeta, cudaStream_t s)
{
    k_edge_assemble<<<nB, kEdgeThreads, sizeof(double) * n, s>>>(T, Nraw, Rraw, n, nB, A, rhs);
    k_edge_solve<<<nB, kEdgeThreads, 0, s>>>(A, rhs, n, nB, zeta);
    return cudaGetLastError();
}

// ---- edge correction without allocating (encore_edge_correct_noalloc, include/encore.h) ---------------------------------
// For callers that may not cudaMalloc (all of HBM handed to a pool allocator, a fixed memory quota, a loop that cannot
// afford the device-wide stalls of cudaMalloc / cudaFree).  The A and rhs scratch of the two kernels above sits in one
// file-scope device array of fixed size; every GPU that loads this library holds its 8 MiB until the process exits.
// NOTE for host code in this file: `g_edge_scratch` below is the HOST-side handle of the symbol, not a device address.
// Only cudaGetSymbolAddress turns it into a pointer a kernel may be given; that pointer differs from device to device.
namespace {

static __device__ __align__(256) double g_edge_scratch[ENCORE_EDGE_NOALLOC_MAX_DOUBLES];

constexpr int kCachedDevices = 64;
std::mutex g_edge_scratch_mu;
double *g_edge_scratch_addr[kCachedDevices]; // device address of g_edge_scratch on device d; nullptr: not looked up yet

// address of the scratch array on the CURRENT device; looked up once per device (devices >= 64: every call)
cudaError_t edge_scratch_address(double **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cache = dev >= 0 && dev < kCachedDevices;
    std::lock_guard<std::mutex> lock(g_edge_scratch_mu);
    if (cache && g_edge_scratch_addr[dev]) {
        *out = g_edge_scratch_addr[dev];
        return cudaSuccess;
    }
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_edge_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (cache) g_edge_scratch_addr[dev] = static_cast<double *>(p);
    *out = static_cast<double *>(p);
    return cudaSuccess;
}

} // namespace

// The caller (api.cu) has checked nB * n * (n + 1) <= ENCORE_EDGE_NOALLOC_MAX_DOUBLES.  No allocation on any path.
// A[b] and rhs[b] are written in full by k_edge_assemble before k_edge_solve reads them: stale contents of the shared
// array never matter, and nothing has to be cleared.  Calls that overlap on the GPU would race on the array.
cudaError_t launch_edge_correct_noalloc(const double *T, const double *Nraw, const double *Rraw, int n, int nB, double *zeta,
                                        cudaStream_t s)
{
    double *scratch = nullptr;
    const cudaError_t e = edge_scratch_address(&scratch);
    if (e != cudaSuccess) return e;
    double *A = scratch, *rhs = scratch + (size_t)nB * n * n;
    k_edge_assemble<<<nB, kEdgeThreads, sizeof(double) * n, s>>>(T, Nraw, Rraw, n, nB, A, rhs);
    k_edge_solve<<<nB, kEdgeThreads, 0, s>>>(A, rhs, n, nB, zeta);
    return cudaGetLastError();
}
