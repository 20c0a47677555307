// grid.cu — steps a1 (cell assignment) and a2 (sort by cell) of the ENCORE hot path.
// The paper only says particles are placed "onto a Cartesian grid" for neighbour look-ups;
// the geometry is this build's (R11).  The sort is a single-digit radix (counting) sort on the cell
// id: histogram -> exclusive scan -> scatter -> rank-by-original-index inside each cell, which makes the
// result the stable sort (within a cell, input order) without depending on atomic arrival order.
// All HBM-bound, a few tens of bytes per particle.
#include "device.cuh"

#include <algorithm>

namespace {

constexpr int kThreads = 256;
constexpr int kScanThreads = 512;
constexpr int kScanItems = 4;                       // 2048 items per block
constexpr int kScanBlock = kScanThreads * kScanItems;

__device__ __forceinline__ bool finite_d(double v) { return fabs(v) <= 1.7976931348623157e308; }

__global__ void k_bbox_partial(const double *__restrict__ pos, const double *__restrict__ w, int64_t n, double box,
                               double *__restrict__ part, int *__restrict__ flags)
{
    double lo[3] = {1.7976931348623157e308, 1.7976931348623157e308, 1.7976931348623157e308};
    double hi[3] = {-1.7976931348623157e308, -1.7976931348623157e308, -1.7976931348623157e308};
    int bad = 0, out = 0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double v = pos[a * n + i];
            if (!finite_d(v)) bad = 1;
            if (box > 0.0 && !(v >= 0.0 && v < box)) out = 1;
            lo[a] = fmin(lo[a], v);
            hi[a] = fmax(hi[a], v);
        }
        if (w && !finite_d(w[i])) bad = 1;
    }
    __shared__ double sh[6][kThreads];
#pragma unroll
    for (int a = 0; a < 3; ++a) { sh[a][threadIdx.x] = lo[a]; sh[3 + a][threadIdx.x] = hi[a]; }
    __syncthreads();
    for (int st = kThreads / 2; st > 0; st >>= 1) {
        if (threadIdx.x < st) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                sh[a][threadIdx.x] = fmin(sh[a][threadIdx.x], sh[a][threadIdx.x + st]);
                sh[3 + a][threadIdx.x] = fmax(sh[3 + a][threadIdx.x], sh[3 + a][threadIdx.x + st]);
            }
        }
        __syncthreads();
    }
    if (threadIdx.x < 6) part[blockIdx.x * 6 + threadIdx.x] = sh[threadIdx.x][0];
    if (bad) atomicOr(&flags[0], 1);
    if (out) atomicOr(&flags[1], 1);
}

__global__ void k_bbox_final(const double *__restrict__ part, int nblocks, double *__restrict__ bbox)
{
    const int a = threadIdx.x; // 6 threads
    if (a >= 6) return;
    double v = part[a];
    for (int b = 1; b < nblocks; ++b) v = a < 3 ? fmin(v, part[b * 6 + a]) : fmax(v, part[b * 6 + a]);
    bbox[a] = v;
}

// DESIGN.md R11:  i_a = min(nc_a - 1, (int)((x_a - org_a) * inv_a));  cid = (iz*ncy + iy)*ncx + ix
__device__ __forceinline__ int cell_coord(double x, double org, double inv, int nc)
{
    int v = (int)((x - org) * inv);
    v = v > nc - 1 ? nc - 1 : v;
    return v < 0 ? 0 : v;       // only below a caller-supplied bounding box (encore_compute_enqueue; flagged as a domain error)
}

__global__ void k_cell_ids(const double *__restrict__ pos, int64_t n, GridGeom g, int32_t *__restrict__ cid,
                           int *__restrict__ cell_count)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int ix = cell_coord(pos[i], g.org[0], g.inv[0], g.nc[0]);
    const int iy = cell_coord(pos[n + i], g.org[1], g.inv[1], g.nc[1]);
    const int iz = cell_coord(pos[2 * n + i], g.org[2], g.inv[2], g.nc[2]);
    const int c = (iz * g.nc[1] + iy) * g.nc[0] + ix;
    cid[i] = c;
    atomicAdd(&cell_count[c], 1);
}

// ---- exclusive scan (three small kernels; m <= 2048*2048) ------------------------------------------------
__device__ int block_exclusive_scan(int v, int *total)
{
    __shared__ int warp_sums[kScanThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, x, d);
        if (lane >= d) x += y;
    }
    if (lane == 31) warp_sums[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int s = lane < kScanThreads / 32 ? warp_sums[lane] : 0;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, s, d);
            if (lane >= d) s += y;
        }
        if (lane < kScanThreads / 32) warp_sums[lane] = s;
    }
    __syncthreads();
    const int base = wid > 0 ? warp_sums[wid - 1] : 0;
    *total = warp_sums[kScanThreads / 32 - 1];
    __syncthreads();
    return base + x - v;
}

__global__ void k_scan_blocks(const int *__restrict__ in, int *__restrict__ out, int m, int *__restrict__ block_tot)
{
    const int base = blockIdx.x * kScanBlock + threadIdx.x * kScanItems;
    int v[kScanItems], s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { v[k] = base + k < m ? in[base + k] : 0; s += v[k]; }
    int tot;
    int ex = block_exclusive_scan(s, &tot);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { if (base + k < m) out[base + k] = ex; ex += v[k]; }
    if (threadIdx.x == 0) block_tot[blockIdx.x] = tot;
}

__global__ void k_scan_totals(int *__restrict__ block_tot, int nblocks, int *__restrict__ grand)
{
    // single block; nblocks <= 2048
    const int base = threadIdx.x * kScanItems;
    int v[kScanItems], s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { v[k] = base + k < nblocks ? block_tot[base + k] : 0; s += v[k]; }
    int tot;
    int ex = block_exclusive_scan(s, &tot);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { if (base + k < nblocks) block_tot[base + k] = ex; ex += v[k]; }
    if (threadIdx.x == 0) *grand = tot;
}

__global__ void k_scan_add(int *__restrict__ out, int m, const int *__restrict__ block_tot)
{
    const int i = blockIdx.x * kScanBlock + threadIdx.x;
    const int add = block_tot[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        const int j = i + k * kScanThreads;
        if (j < m) out[j] += add;
    }
}

// ---- scatter + rank + gather -----------------------------------------------------------------------------
__global__ void k_scatter(int64_t n, const int32_t *__restrict__ cid, const int *__restrict__ cell_start,
                          int *__restrict__ cell_fill, int *__restrict__ tmp_idx)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int c = cid[i];
    const int slot = cell_start[c] + atomicAdd(&cell_fill[c], 1);
    tmp_idx[slot] = (int)i;
}

// Cells with more particles than this are put in order by k_sort_big_cells; smaller ones by the counting loop of k_rank_gather.
constexpr int kRankLoopMax = 64;
constexpr int kBigSortThreads = 1024;

// Sorts a[0..len) ascending with the CTA's threads: a bitonic network whose merges all run in the same direction (the first
// step of each stage compares mirror images, i with block_end - 1 - i, the others i with i + j), so that elements beyond len
// act as +infinity without being stored - a compare-exchange whose upper partner is >= len is simply skipped.
// O(len log^2 len) compare-exchanges in global memory (L2-resident), __syncthreads between steps.
__device__ void sort_segment_ascending(int *__restrict__ a, int len)
{
    int P = 1;
    while (P < len) P <<= 1;
    const int half = P >> 1;
    for (int k = 2; k <= P; k <<= 1) {
        const int hk = k >> 1;
        for (int t = threadIdx.x; t < half; t += blockDim.x) {
            const int blk = t / hk, off = t - blk * hk;
            const int i = blk * k + off, q = blk * k + k - 1 - off;
            if (q < len) {
                const int x = a[i], y = a[q];
                if (x > y) { a[i] = y; a[q] = x; }
            }
        }
        __syncthreads();
        for (int j = hk >> 1; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < half; t += blockDim.x) {
                const int i = (t / j) * 2 * j + (t % j), q = i + j;
                if (q < len) {
                    const int x = a[i], y = a[q];
                    if (x > y) { a[i] = y; a[q] = x; }
                }
            }
            __syncthreads();
        }
    }
}

// A dense clump in a coarse cell would make the counting loop of k_rank_gather quadratic in the cell's occupancy.  CTAs sweep the
// cell table (1024 cells at a time); a cell holding more than kRankLoopMax particles has its slice of tmp_idx sorted by original
// index, by the whole CTA.  After that a slot of such a cell IS its rank.  On ordinary inputs (c1..c5: <= 40 per cell) this
// kernel reads cell_start once and sorts nothing.  No list of big cells, no extra buffer, nothing read back.
__global__ void __launch_bounds__(kBigSortThreads) k_sort_big_cells(const int *__restrict__ cell_start, int ncell, int *__restrict__ tmp_idx)
{
    __shared__ int big[kBigSortThreads];
    __shared__ int nbig;
    for (int base = blockIdx.x * kBigSortThreads; base < ncell; base += gridDim.x * kBigSortThreads) {
        if (threadIdx.x == 0) nbig = 0;
        __syncthreads();
        const int c = base + threadIdx.x;
        if (c < ncell && cell_start[c + 1] - cell_start[c] > kRankLoopMax) big[atomicAdd(&nbig, 1)] = c;
        __syncthreads();
        const int nb = nbig;
        for (int k = 0; k < nb; ++k) {      // the order of `big` is arbitrary; every cell is sorted on its own, the result is not
            const int b = cell_start[big[k]];
            sort_segment_ascending(tmp_idx + b, cell_start[big[k] + 1] - b);
        }
        __syncthreads();
    }
}

// Each particle finds its rank inside its cell by counting smaller original indices: the arrival order of the
// scatter's atomics does not survive.  Cells hold a handful of particles, so this is O(n * occupancy); cells above
// kRankLoopMax were sorted by k_sort_big_cells and a slot there is already the rank.
__global__ void k_rank_gather(int64_t n, const double *__restrict__ pos, const double *__restrict__ w,
                              const int32_t *__restrict__ cid, const int *__restrict__ cell_start,
                              const int *__restrict__ tmp_idx, int *__restrict__ sorted_idx,
                              double4 *__restrict__ pos4)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= n) return;
    const int i = tmp_idx[s];
    const int c = cid[i];
    const int b = cell_start[c], e = cell_start[c + 1];
    int rank = (int)s - b;
    if (e - b <= kRankLoopMax) {
        rank = 0;
        for (int q = b; q < e; ++q) rank += tmp_idx[q] < i;
    }
    const int dst = b + rank;
    sorted_idx[dst] = i;
    pos4[dst] = make_double4(pos[i], pos[n + i], pos[2 * n + i], w ? w[i] : 1.0);
}

__global__ void k_pencil_groups(const int *__restrict__ cell_start, GridGeom g, int *__restrict__ groups)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= g.npencil) return;
    const int cnt = cell_start[(p + 1) * g.nc[0]] - cell_start[p * g.nc[0]];
    groups[p] = (cnt + ENCORE_GROUP - 1) / ENCORE_GROUP;
}

// encore_compute_enqueue: the caller's bounding box must hold every particle (flags[1] otherwise)
__global__ void k_bbox_check(const double *__restrict__ bbox, double lx, double ly, double lz, double hx, double hy, double hz,
                             int *__restrict__ flags)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        const bool ok = bbox[0] >= lx && bbox[1] >= ly && bbox[2] >= lz && bbox[3] <= hx && bbox[4] <= hy && bbox[5] <= hz;
        if (!ok) flags[1] = 1;
    }
}

// fp32-harmonics variant: candidate records of 16 instead of 32 bytes (the gather of k_harm is bound by L1 bytes)
__global__ void k_make_pos4f(const double4 *__restrict__ pos4, int64_t count, double cx, double cy, double cz, float4 *__restrict__ out)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= count) return;
    const double4 p = pos4[i];
    out[i] = make_float4((float)(p.x - cx), (float)(p.y - cy), (float)(p.z - cz), (float)p.w);
}

__global__ void k_set_particle(double4 *dst, double x, double y, double z, double w)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) *dst = make_double4(x, y, z, w);
}

} // namespace

cudaError_t launch_make_pos4f(const double4 *pos4, int64_t count, const double ctr[3], float4 *pos4f, cudaStream_t s, int *launches)
{
    k_make_pos4f<<<(unsigned)((count + kThreads - 1) / kThreads), kThreads, 0, s>>>(pos4, count, ctr[0], ctr[1], ctr[2], pos4f);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_set_particle(double4 *dst, double x, double y, double z, double w, cudaStream_t s, int *launches)
{
    k_set_particle<<<1, 32, 0, s>>>(dst, x, y, z, w);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_bbox_check(const double *bbox_dev, const double lo[3], const double hi[3], int *flags, cudaStream_t s, int *launches)
{
    k_bbox_check<<<1, 32, 0, s>>>(bbox_dev, lo[0], lo[1], lo[2], hi[0], hi[1], hi[2], flags);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_bbox_validate(const double *pos, const double *w, int64_t n, double box, double *bbox_tmp,
                                 double *bbox_out, int *flags, cudaStream_t s, int *launches)
{
    int nblocks = (int)((n + kThreads - 1) / kThreads);
    if (nblocks > 592) nblocks = 592; // 4 x 148
    cudaError_t e = cudaMemsetAsync(flags, 0, 2 * sizeof(int), s);
    if (e != cudaSuccess) return e;
    k_bbox_partial<<<nblocks, kThreads, 0, s>>>(pos, w, n, box, bbox_tmp, flags);
    k_bbox_final<<<1, 32, 0, s>>>(bbox_tmp, nblocks, bbox_out);
    *launches += 2;
    return cudaGetLastError();
}

cudaError_t launch_cell_ids(const double *pos, int64_t n, GridGeom g, int32_t *cid, int *cell_count,
                            cudaStream_t s, int *launches)
{
    cudaError_t e = cudaMemsetAsync(cell_count, 0, sizeof(int) * (size_t)g.ncell, s);
    if (e != cudaSuccess) return e;
    k_cell_ids<<<(unsigned)((n + kThreads - 1) / kThreads), kThreads, 0, s>>>(pos, n, g, cid, cell_count);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_exclusive_scan(const int *in, int *out, int m, int *tmp, cudaStream_t s, int *launches)
{
    const int nblocks = (m + kScanBlock - 1) / kScanBlock;
    if (nblocks > kScanBlock) return cudaErrorInvalidValue;
    k_scan_blocks<<<nblocks, kScanThreads, 0, s>>>(in, out, m, tmp);
    k_scan_totals<<<1, kScanThreads, 0, s>>>(tmp, nblocks, out + m);
    k_scan_add<<<nblocks, kScanThreads, 0, s>>>(out, m, tmp);
    *launches += 3;
    return cudaGetLastError();
}

cudaError_t launch_sort_gather(const double *pos, const double *w, int64_t n, const int32_t *cid,
                               const int *cell_start, int ncell, int *cell_fill, int *tmp_idx, int *sorted_idx,
                               double4 *pos4, cudaStream_t s, int *launches)
{
    const unsigned nb = (unsigned)((n + kThreads - 1) / kThreads);
    k_scatter<<<nb, kThreads, 0, s>>>(n, cid, cell_start, cell_fill, tmp_idx);
    const int sweep = std::max(1, std::min(296, (ncell + kBigSortThreads - 1) / kBigSortThreads));   // at most 2 CTAs per SM
    k_sort_big_cells<<<sweep, kBigSortThreads, 0, s>>>(cell_start, ncell, tmp_idx);
    k_rank_gather<<<nb, kThreads, 0, s>>>(n, pos, w, cid, cell_start, tmp_idx, sorted_idx, pos4);
    *launches += 3;
    return cudaGetLastError();
}

cudaError_t launch_pencil_groups(const int *cell_start, GridGeom g, int *groups_per_pencil, cudaStream_t s,
                                 int *launches)
{
    k_pencil_groups<<<(g.npencil + kThreads - 1) / kThreads, kThreads, 0, s>>>(cell_start, g, groups_per_pencil);
    *launches += 1;
    return cudaGetLastError();
}
