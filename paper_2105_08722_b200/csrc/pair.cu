// pair.cu — steps a3 (neighbour sweep + radial binning) and a4 (a_lm accumulation) of the ENCORE hot path.
//
//   a^b_lm(s_i) = (1/v_b) sum_{j != i} w_j Y_lm((r_j - s_i)^) Theta^b(|r_j - s_i|)          eq. 35
//
// The paper does this on the CPU, histogramming Cartesian monomials with AVX, eight secondaries at a time
// (Alg. 2) and has no GPU version of it.  Design here:
// the work is split by resource profile into two kernels around "groups" of 32 consecutive cell-sorted
// primaries of one (iy,iz) pencil (lane = primary everywhere):
//   k_fill  (a3, integer/fp32, few registers): ONE WARP per group.  Candidates = contiguous runs of the sorted
//     array (one or two per neighbouring pencil, x-range culled against the group's cell range), cut into WORDS of
//     32 consecutive sorted particles.  A word is read lane = candidate, made relative to primary 0 (periodic image)
//     in fp32 and culled against the bounding box of the group's primaries; the survivors are broadcast from shared
//     memory and every lane (= primary) tests them.  A first fp32 evaluation decides every pair whose radius is
//     farther than a proven error margin from all bin edges; the rest (~1e-4) is decided in fp64 exactly as
//     DESIGN.md R8-R10 fix it (r^2 = fma(dz,dz,fma(dy,dy,dx*dx)) against e_b^2), so the binning is bit-exact.  The
//     result of a word is one 32-bit acceptance mask per (bin, primary); for every bin with any bit set the warp
//     writes ONE coalesced 128-byte ROW (32 masks, lane = primary) plus a one-word descriptor (first sorted index |
//     image codes << 26) to the row stream of (group, bin), which sits at a fixed place (capacity = words of the
//     group): no allocation, no lane-private list state, no atomics.
//   k_harm  (a4, fp64, ~166 registers): one warp per (group, bin).  The rows are staged into shared memory with
//     cp.async (two chunks of 16 rows in flight); every lane pushes its non-empty masks into a lane-private queue of
//     (mask, descriptor) records in shared memory and walks their set bits, gathering the candidate four pairs ahead
//     with one 256-bit load.  The (lmax+1)^2 real accumulators of a^b_lm(s_i) stay in REGISTERS: no atomics, no
//     cross-lane reductions, summation order = candidate order -> deterministic.  Per pair: unit vector (fp32 rsqrt
//     seed + one third-order fp64 step), w (x+iy)^m by complex recurrence, powers of z, one FMA per component into
//     S_{m,k} = sum w z^k (x+iy)^m; the monic associated-Legendre polynomials p_lm(z) and the normalisation
//     (-1)^m N_lm k_lm / v_b are applied once per (primary, bin) in the epilogue (table ycoef).  The number of set
//     bits a lane walked is n_i(b), the per-(primary, bin) pair count (an integer output of the path).
//     Items are ordered heaviest bin first so the grid drains evenly.
#include "device.cuh"

#include <algorithm>
#include <climits>
#include <mutex>
#include <type_traits>

namespace {

#ifndef ENCORE_HARM_DEPTH
#define ENCORE_HARM_DEPTH 4
#endif
#ifndef ENCORE_HARM_DEPTH_FAT
#define ENCORE_HARM_DEPTH_FAT 4
#endif
#ifndef ENCORE_HARM_FAT
#define ENCORE_HARM_FAT 44      // passes with more accumulators run at 8 warps/SM and 255 registers
#endif
#ifndef ENCORE_HARM_WARPS
#define ENCORE_HARM_WARPS 4
#endif
constexpr int kHarmWarps = ENCORE_HARM_WARPS;       // k_harm: independent warps (items) per CTA
#ifndef ENCORE_HARM_QUEUE
#define ENCORE_HARM_QUEUE 32
#endif
constexpr int kQueue = ENCORE_HARM_QUEUE;           // k_harm: (mask, descriptor) records queued per lane (power of two)
constexpr int kQueueF32 = 16;                       // fp32-harmonics variant: its fp64 accumulators take the shared memory (3 CTAs per SM)
constexpr int kStageRows = 8;                       // k_harm: rows per cp.async chunk (two chunks in flight)
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kNoHit = 254u;
constexpr unsigned kIdxMask = 0x3ffffffu;
constexpr float kMagic = 12582912.f;          // 1.5 * 2^23: (x + kMagic) - kMagic = round-to-nearest-integer(x)
constexpr int kMagicBits = 0x4B400000;

__host__ __device__ constexpr int ncomp_range(int lmax, int mlo, int mhi)
{
    int n = 0;
    for (int m = mlo; m <= mhi; ++m) n += (lmax - m + 1) * (m ? 2 : 1);
    return n;
}

__device__ __forceinline__ int cell_coord(double x, double org, double inv, int nc)
{
    int v = (int)((x - org) * inv);
    v = v > nc - 1 ? nc - 1 : v;
    return v < 0 ? 0 : v;
}

// acc[] order: m ascending, k ascending, (re, im): S_{m,k} = sum w z^k (x+iy)^m, k = 0..LMAX-m.
// Same number of accumulators as the a_lm themselves ((LMAX+1)^2 reals over all m) and one FMA each per pair; the
// Legendre polynomials p_lm(z) are applied once per (primary, bin) in the epilogue through the table ycoef
// (tables.cpp): 4 multiplies for the powers of z replace the 2 operations per (l,m) of a recurrence in every pair.
// T = double: the fp64 path.  T = float: the fp32-harmonics variant: same operations
// in fp32 into fp32 chunk sums that k_harm adds to the fp64 accumulators every 16 pairs.
// T = float: the (re, im) accumulators of an m > 0 component are adjacent, so one packed fp32x2 operation of sm_100
// (FFMA2 / FMUL2, each element the IEEE round-to-nearest scalar operation) updates both and the complex recurrence takes two
// instead of four instructions: 48 instead of 72 fp32 instructions per pair at lmax = 5.
template <int LMAX, int MLO, int MHI>
__device__ __forceinline__ void accumulate_f32(float (&acc)[ncomp_range(LMAX, MLO, MHI)], float x, float y, float z, float w)
{
    float zp[LMAX + 1];
    zp[0] = 1.f;
#pragma unroll
    for (int k = 1; k <= LMAX - MLO; ++k) zp[k] = k == 1 ? z : zp[k - 1] * z;
    const float2 xy = make_float2(x, y), myx = make_float2(-y, x);
    float2 cs = make_float2(w, 0.f);        // w (x + i y)^m
    int k = 0;
#pragma unroll
    for (int m = 0; m <= MHI; ++m) {
        if (m == 1) cs = __fmul2_rn(make_float2(w, w), xy);
        if (m > 1) cs = __ffma2_rn(make_float2(cs.x, cs.x), xy, __fmul2_rn(make_float2(cs.y, cs.y), myx));
        if (m >= MLO) {
#pragma unroll
            for (int q = 0; q <= LMAX - m; ++q) {
                if (m == 0) { acc[k] = q == 0 ? acc[k] + cs.x : fmaf(zp[q], cs.x, acc[k]); k += 1; }
                else {
                    float2 t = make_float2(acc[k], acc[k + 1]);
                    t = q == 0 ? __fadd2_rn(t, cs) : __ffma2_rn(make_float2(zp[q], zp[q]), cs, t);
                    acc[k] = t.x; acc[k + 1] = t.y;
                    k += 2;
                }
            }
        }
    }
}

template <int LMAX, int MLO, int MHI, class T>
__device__ __forceinline__ void accumulate(T (&acc)[ncomp_range(LMAX, MLO, MHI)], T x, T y, T z, T w)
{
    T zp[LMAX + 1];
    zp[0] = T(1);
#pragma unroll
    for (int k = 1; k <= LMAX - MLO; ++k) zp[k] = k == 1 ? z : zp[k - 1] * z;
    T c = w, s = T(0); // w (x + i y)^m
    int k = 0;
#pragma unroll
    for (int m = 0; m <= MHI; ++m) {
        if (m == 1) { c = w * x; s = w * y; }
        if (m > 1) {
            const T cn = fma(c, x, -(s * y));
            const T sn = fma(c, y, s * x);
            c = cn; s = sn;
        }
        if (m >= MLO) {
#pragma unroll
            for (int q = 0; q <= LMAX - m; ++q) {
                if (q == 0) { acc[k] += c; if (m) acc[k + 1] += s; }
                else { acc[k] = fma(zp[q], c, acc[k]); if (m) acc[k + 1] = fma(zp[q], s, acc[k + 1]); }
                k += m ? 2 : 1;
            }
        }
    }
}

// 1/sqrt(a) to full double precision from the hardware seed y0 = rsqrt.approx.f64 (MUFU.RSQ64H: works on the upper
// word of the double, relative error below 2^-20) and ONE third-order step: with e = 1 - a y0^2,
// a^-1/2 = y0 (1 - e)^-1/2 = y0 (1 + e/2 + 3e^2/8 + 5e^3/16 + ...), truncation 5/16 |e|^3 < 2^-58.
// 5 fp64 operations and no conversions.  The seed flushes subnormals and has no special cases: k_harm checks the
// edges of the item's bin once (every pair of the item has its r^2 between them) and takes the library routine for
// bins that reach down to 0 or beyond 1e290.
__device__ __forceinline__ double rsqrt_pair(double a)
{
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(a));
    const double t = a * y0;
    const double e = fma(-t, y0, 1.0);
    const double p = fma(0.375, e, 0.5);
    return fma(y0, e * p, y0);
}

template <bool PERIODIC>
__device__ __forceinline__ double sep(double xj, double xi, double box, double half)
{
    double d = xj - xi; // DESIGN.md R7, R10
    if (PERIODIC) {
        if (d > half) d -= box;
        else if (d < -half) d += box;
    }
    return d;
}

// ---- the group of a warp ---------------------------------------------------------------------------------
struct Group {
    int first, cnt;      // sorted index of primary 0, number of primaries (1..32)
    int py, pz;          // pencil
    int gx0, gx1;        // x-cell range of the members
    double ext[3];       // bound on |x_i - x_primary0| per axis (cell geometry + 1 cell of slack)
    bool fast;           // periodic only: the image of a candidate is the same for every member
};

template <bool PERIODIC>
__device__ __forceinline__ Group locate_group(const PairArgs &a, int g)
{
    const GridGeom &G = a.geom;
    Group gr;
    const int ncx = G.nc[0], ncy = G.nc[1];
    const int p = find_pencil_of_group(a.group_start, G.npencil, g);
    const int pstart = a.cell_start[p * ncx], pend = a.cell_start[(p + 1) * ncx];
    gr.first = pstart + ENCORE_GROUP * (g - a.group_start[p]);
    gr.cnt = min(ENCORE_GROUP, pend - gr.first);
    gr.py = p % ncy; gr.pz = p / ncy;
    gr.gx0 = cell_coord(a.pos4[gr.first].x, G.org[0], G.inv[0], ncx);
    gr.gx1 = cell_coord(a.pos4[gr.first + gr.cnt - 1].x, G.org[0], G.inv[0], ncx);
    gr.ext[0] = (double)(gr.gx1 - gr.gx0 + 2) / G.inv[0];
    gr.ext[1] = 2.0 / G.inv[1];
    gr.ext[2] = 2.0 / G.inv[2];
    // r_max + extent < L/2: an accepted pair's minimal image is then fixed by the candidate's image relative to
    // primary 0, so it can travel with the list entry
    gr.fast = !PERIODIC || (a.rmax + fmax(gr.ext[0], fmax(gr.ext[1], gr.ext[2])) < G.half * (1.0 - 1e-9));
    return gr;
}

// ---- candidate ranges of a group (one warp): one or two runs of the sorted array per neighbouring pencil -----
// A run is cut into words of 32 consecutive sorted particles (the last word of a run may be partial).
// STORE: rng_start[r] = first sorted index of run r, rng_len[r] = its length, rng_woff[r] = words before run r
// (rng_woff[nr] = words of the group).  Returns the number of words W of the group.  *wide is set when a candidate
// x-range covers the whole periodic axis (then no image is common to a run and the group takes the exact path).
template <bool PERIODIC, bool STORE>
__device__ __forceinline__ int build_ranges(const PairArgs &a, const Group &gr, int lane, int *rng_start, int *rng_len,
                                            int *rng_woff, int *nr_out, bool *wide)
{
    const GridGeom &G = a.geom;
    const int ncx = G.nc[0], ncy = G.nc[1], ncz = G.nc[2];
    int Ry = (int)floor(a.rmax * G.inv[1] + 1e-6) + 1, Rz = (int)floor(a.rmax * G.inv[2] + 1e-6) + 1;
    if (!PERIODIC) { Ry = min(Ry, ncy - 1); Rz = min(Rz, ncz - 1); } // nothing beyond the grid
    const bool full_y = PERIODIC && (2 * Ry + 1 >= ncy), full_z = PERIODIC && (2 * Rz + 1 >= ncz);
    const int wy = full_y ? ncy : 2 * Ry + 1, wz = full_z ? ncz : 2 * Rz + 1;
    const int nyz = wy * wz; // host guarantees 2*nyz <= nr_cap
    const double rmax2 = a.rmax * a.rmax;
    int mine = 0;
    bool covers = full_y || full_z;
    for (int r = lane; r < nyz; r += 32) {
        const int iy = r % wy, iz = r / wy;
        int cy, cz, dyc, dzc;
        bool ok = true;
        if (full_y) { cy = iy; const int d = abs(cy - gr.py); dyc = min(d, ncy - d); }
        else {
            cy = gr.py - Ry + iy; dyc = abs(iy - Ry);
            if (PERIODIC) cy = (cy + ncy) % ncy; else ok = ok && cy >= 0 && cy < ncy;
        }
        if (full_z) { cz = iz; const int d = abs(cz - gr.pz); dzc = min(d, ncz - d); }
        else {
            cz = gr.pz - Rz + iz; dzc = abs(iz - Rz);
            if (PERIODIC) cz = (cz + ncz) % ncz; else ok = ok && cz >= 0 && cz < ncz;
        }
        int s0 = 0, l0 = 0, s1 = 0, l1 = 0;
        if (ok) {
            // smallest possible transverse separation between the two pencils (cells are 1/inv wide)
            const double ty = (double)max(dyc - 1, 0) / G.inv[1] * (1.0 - 1e-9);
            const double tz = (double)max(dzc - 1, 0) / G.inv[2] * (1.0 - 1e-9);
            const double t2 = ty * ty + tz * tz;
            if (t2 < rmax2) {
                const int rx = (int)floor(sqrt(rmax2 - t2) * G.inv[0] + 1e-6) + 1;
                int lo = gr.gx0 - rx, hi = gr.gx1 + rx; // inclusive x-cell range
                const int row = (cz * ncy + cy) * ncx;
                if (PERIODIC) {
                    if (hi - lo + 1 >= ncx) { lo = 0; hi = ncx - 1; covers = true; }
                    if (lo < 0) {
                        s0 = a.cell_start[row + lo + ncx]; l0 = a.cell_start[row + ncx] - s0;
                        s1 = a.cell_start[row]; l1 = a.cell_start[row + hi + 1] - s1;
                    } else if (hi >= ncx) {
                        s0 = a.cell_start[row + lo]; l0 = a.cell_start[row + ncx] - s0;
                        s1 = a.cell_start[row]; l1 = a.cell_start[row + hi - ncx + 1] - s1;
                    } else {
                        s0 = a.cell_start[row + lo]; l0 = a.cell_start[row + hi + 1] - s0;
                    }
                } else {
                    lo = max(lo, 0); hi = min(hi, ncx - 1);
                    s0 = a.cell_start[row + lo]; l0 = a.cell_start[row + hi + 1] - s0;
                }
            }
        }
        mine += ((l0 + 31) >> 5) + ((l1 + 31) >> 5);
        if (STORE) {
            rng_start[2 * r] = s0; rng_len[2 * r] = l0; rng_woff[2 * r + 1] = (l0 + 31) >> 5; // words parked in [.+1], scanned below
            rng_start[2 * r + 1] = s1; rng_len[2 * r + 1] = l1; rng_woff[2 * r + 2] = (l1 + 31) >> 5;
        }
    }
    const int nr = 2 * nyz;
    *nr_out = nr;
    *wide = __any_sync(kFull, covers);
    if (!STORE) return __reduce_add_sync(kFull, mine);
    __syncwarp();
    { // inclusive scan of the word counts into offsets
        const int per = (nr + 31) / 32;
        const int b0 = lane * per, b1 = min(nr, b0 + per);
        int sum = 0;
        for (int r = b0; r < b1; ++r) sum += rng_woff[r + 1];
        int x = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { int y = __shfl_up_sync(kFull, x, d); if (lane >= d) x += y; }
        int run = x - sum;
        for (int r = b0; r < b1; ++r) { const int len = rng_woff[r + 1]; run += len; rng_woff[r + 1] = run; }
        if (lane == 0) rng_woff[0] = 0;
    }
    __syncwarp();
    return rng_woff[nr];
}

// exact decision, the operations of DESIGN.md R8-R10 (the oracle's): returns the bin or kNoHit
template <bool PERIODIC>
__device__ __noinline__ unsigned classify_exact(const double4 &cj, const double *sp, int i, const double *e2, int nb,
                                                   double box, double half, float rmin_f, float invw_f)
{
    const double dx = sep<PERIODIC>(cj.x, sp[i], box, half);
    const double dy = sep<PERIODIC>(cj.y, sp[32 + i], box, half);
    const double dz = sep<PERIODIC>(cj.z, sp[64 + i], box, half);
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    if (!(r2 > 0.0 && r2 >= e2[0] && r2 < e2[nb])) return kNoHit; // DESIGN.md R8
    int b = (int)((sqrtf((float)r2) - rmin_f) * invw_f);
    b = max(0, min(nb - 1, b));
    while (r2 < e2[b]) --b;               // DESIGN.md R9: the decision is on squares, fp64
    while (!(r2 < e2[b + 1])) ++b;
    return (unsigned)b;
}

// per group: number of candidate words (row capacity of each of its bins; sizes the super-steps on the host)
template <bool PERIODIC>
__global__ void __launch_bounds__(128) k_group_bound(PairArgs a)
{
    const int g = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (g >= a.ngroups) return;
    if (g >= a.group_start[a.geom.npencil]) { if (lane == 0) { a.gbound[g] = 0; a.gwide[g] = 0; } return; }
    const Group gr = locate_group<PERIODIC>(a, g);
    int nr;
    bool wide;
    const int W = build_ranges<PERIODIC, false>(a, gr, lane, nullptr, nullptr, nullptr, &nr, &wide);
    if (lane == 0) { a.gbound[g] = W; a.gwide[g] = wide ? 1 : 0; }
}

// ==========================================================================================================
// k_fill: a3.  One warp (= one CTA) per group.
// ==========================================================================================================
// dynamic shared memory: cand[36] float4 | sp[96] double | e2[nb+1] double | masks[nb+1][32] u32 |
//                        rng_start[nr_cap] | rng_len[nr_cap] | rng_woff[nr_cap+1]
__host__ __device__ inline size_t fill_smem_bytes(int nb, int nr_cap)
{
    return 36 * 16 + 96 * 8 + (size_t)((nb + 2) & ~1) * 8 + (size_t)(nb + 1) * 32 * 4 + (size_t)(3 * nr_cap + 4) * 4;
}

template <bool PERIODIC>
__global__ void __launch_bounds__(32) k_fill(PairArgs a, int g0, int g1, int nr_cap)
{
    const int g = g0 + blockIdx.x;
    const GridGeom &G = a.geom;
    if (g >= g1 || g >= a.group_start[G.npencil]) return;
    const int lane = threadIdx.x;
    const int nb = a.bins.nbins;

    extern __shared__ __align__(16) unsigned char fill_smem[];
    float4 *cand = reinterpret_cast<float4 *>(fill_smem);
    double *sp = reinterpret_cast<double *>(cand + 36);
    double *e2 = sp + 96;
    unsigned *masks = reinterpret_cast<unsigned *>(e2 + ((nb + 2) & ~1)); // row nb takes the bits of rejected candidates
    int *rng_start = reinterpret_cast<int *>(masks + (nb + 1) * 32);
    int *rng_len = rng_start + nr_cap;
    int *rng_woff = rng_len + nr_cap;

    if (a.rows_cap_words && (size_t)(a.gprefix[g + 1] - a.gprefix[g0]) > a.rows_cap_words) {
        // encore_compute_enqueue: the rows of this group would not fit the reservation of the last encore_compute
        if (lane < nb) a.rowcnt[(size_t)g * nb + lane] = 0;
        if (lane == 0) atomicOr(a.err_flag, 2);
        return;
    }
    const Group gr = locate_group<PERIODIC>(a, g);
    const int first = gr.first, cnt = gr.cnt;
    const double4 ctr = a.pos4[first];
    const double4 mine = a.pos4[first + (lane < cnt ? lane : 0)];
    sp[lane] = mine.x; sp[32 + lane] = mine.y; sp[64 + lane] = mine.z;
    a.gweights[(size_t)g * 32 + lane] = lane < cnt ? mine.w : 0.0;
    for (int b = lane; b <= nb; b += 32) e2[b] = a.bins.e2[b];   // nb + 1 edges: 33 at ENCORE_MAX_BINS
    for (int b = 0; b < nb; ++b) masks[b * 32 + lane] = 0u;
    // this lane's primary, relative to primary 0, fp32 (lanes beyond the group sit far away: never a hit)
    const float pxf = lane < cnt ? (float)(mine.x - ctr.x) : -1e18f, pyf = (float)(mine.y - ctr.y), pzf = (float)(mine.z - ctr.z);

    int nr;
    bool wide;
    const int nwords = build_ranges<PERIODIC, true>(a, gr, lane, rng_start, rng_len, rng_woff, &nr, &wide);

    // fp32 screening constants: the bin coordinate u = (r - r_min)/width computed in fp32 is within
    // du = [2^-18 (r + r_min) + 2^-19 E^2 / r] / width + 2^-20 |u| of the exact one (E^2 = sum of squared group
    // extents).  For r <= 2 r_max the r-dependent part is bounded by the constant duc; beyond, u - du >= N_r trivially.
    // The loop works with uh = u - 1/2: round-to-nearest(uh) = floor(u) away from the edges, and the pair is surely
    // inside bin floor(u) iff |uh - rn(uh)| <= 1/2 - du.
    const float rmin_f = a.bins.rmin_f, invw_f = a.bins.invw_f;
    const float c0h = -rmin_f * invw_f - 0.5f;
    const float nb_f = (float)nb;
    const float duc = 3.814697265625e-06f * invw_f * (2.f * (float)a.rmax + rmin_f) + 9.5367431640625e-07f * (2.f * nb_f + 2.f);
    const float kB = 1.9073486328125e-06f * invw_f *
                     (float)(gr.ext[0] * gr.ext[0] + gr.ext[1] * gr.ext[1] + gr.ext[2] * gr.ext[2]);
    const float thr0 = 0.5f - duc;
    // a common periodic image per run needs r_max + extent < L/2 and no run covering a whole axis
    const bool fast = gr.fast && !wide;

    // bounding box of the group's primaries (same fp32 values the tests use) and the cull radius: r_max plus the
    // fp32 rounding of the coordinates involved (<= 2^-23 (extent + r_max) per axis), with a safety factor
    float blo[3], bhi[3];
    {
        const bool act = lane < cnt;
        const float v[3] = {act ? pxf : 0.f, act ? pyf : 0.f, act ? pzf : 0.f}; // primary 0 sits at the origin
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
            float lo = v[ax], hi = v[ax];
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                lo = fminf(lo, __shfl_xor_sync(kFull, lo, d));
                hi = fmaxf(hi, __shfl_xor_sync(kFull, hi, d));
            }
            blo[ax] = lo; bhi[ax] = hi;
        }
    }
    const double rcut = (a.rmax + 9.5367431640625e-07 * (gr.ext[0] + gr.ext[1] + gr.ext[2] + a.rmax)) * (1.0 + 1e-6);
    const float cut2 = (float)(rcut * rcut * (1.0 + 1e-6));

    // row streams of this group: bin b owns rows [b * nwords, (b+1) * nwords) behind the group's base
    const size_t wbase = (size_t)(a.gprefix[g] - a.gprefix[g0]) * (size_t)nb;
    unsigned *rows_g = a.rows + wbase * 32;
    unsigned *desc_g = a.rowdesc + wbase;
    int rowcnt = 0;                     // lane b holds the number of rows written for bin b
    const unsigned lt_mask = (1u << lane) - 1u;
    unsigned long long kept = 0ull;

    // words are read one ahead: lane = candidate
    int run = 0; // rng_woff[run] <= w < rng_woff[run + 1] once advanced (runs without words are stepped over)
    auto load_word = [&](int w, double4 &cj, int &jbase, bool &valid) {
        valid = false; jbase = 0;
        if (w < nwords) {
            while (rng_woff[run + 1] <= w) ++run; // w < nwords = rng_woff[nr] bounds the walk
            const int k0 = (w - rng_woff[run]) << 5;
            jbase = rng_start[run] + k0;
            valid = k0 + lane < rng_len[run];
            if (valid) cj = a.pos4[jbase + lane];
        }
    };
    double4 cjA = make_double4(0, 0, 0, 0), cjB = cjA;
    int jbA = 0, jbB = 0;
    bool vA = false, vB = false;
    load_word(0, cjA, jbA, vA);
    for (int w = 0; w < nwords; ++w) {
        load_word(w + 1, cjB, jbB, vB); // in flight during the tests below
        // ---- stage the word: fp64 -> relative to primary 0 (periodic image) -> fp32, bounding-box cull ----
        float4 cf = make_float4(1e18f, 1e18f, 1e18f, 0.f);
        unsigned code = 0x15u; // image codes (1,1,1): the consumer subtracts {-L, 0, +L}[code] per axis from x_i
        bool keep = false;
        if (vA) {
            double rx = cjA.x - ctr.x, ry = cjA.y - ctr.y, rz = cjA.z - ctr.z;
            unsigned kx = 1, ky = 1, kz = 1;
            if (PERIODIC) {
                if (rx > G.half) { rx -= G.box; kx = 2; } else if (rx < -G.half) { rx += G.box; kx = 0; }
                if (ry > G.half) { ry -= G.box; ky = 2; } else if (ry < -G.half) { ry += G.box; ky = 0; }
                if (rz > G.half) { rz -= G.box; kz = 2; } else if (rz < -G.half) { rz += G.box; kz = 0; }
            }
            code = kx | (ky << 2) | (kz << 4);
            cf = make_float4((float)rx, (float)ry, (float)rz, 0.f);
            const float ex = fmaxf(fmaxf(blo[0] - cf.x, cf.x - bhi[0]), 0.f);
            const float ey = fmaxf(fmaxf(blo[1] - cf.y, cf.y - bhi[1]), 0.f);
            const float ez = fmaxf(fmaxf(blo[2] - cf.z, cf.z - bhi[2]), 0.f);
            keep = !fast || fmaf(ez, ez, fmaf(ey, ey, ex * ex)) <= cut2; // wide groups (exact path) keep everything
        }
        const unsigned km = __ballot_sync(kFull, keep);
        const int jbase = jbA;
        cjA = cjB; jbA = jbB; vA = vB;
        if (km == 0u) continue;         // no candidate of the word is within reach of the group
        const unsigned wcode = __shfl_sync(kFull, code, 0); // lane 0 of a word is always a candidate
        if (PERIODIC && fast && __any_sync(kFull, keep && code != wcode)) { // excluded by DESIGN.md §5.3
            if (lane == 0) atomicOr(a.err_flag, 1);
        }
        // survivors compacted to the front of cand[], two per 32-byte slot as {x0,x1,y0,y1 | z0,z1,pos0,pos1} (pos =
        // position in the word) so that a pair of candidates feeds the packed fp32x2 instructions of sm_100; padded
        // with never-hit fillers to a multiple of four
        const int nk = __popc(km);
        float *candf = reinterpret_cast<float *>(cand);
        if (keep) {
            const int k = __popc(km & lt_mask);
            float *slot = candf + (k >> 1) * 8 + (k & 1);
            slot[0] = cf.x; slot[2] = cf.y; slot[4] = cf.z; slot[6] = __int_as_float(lane);
        }
        if (lane < 4) {
            const int k = nk + lane;
            float *slot = candf + (k >> 1) * 8 + (k & 1);
            slot[0] = 1e18f; slot[2] = 1e18f; slot[4] = 1e18f; slot[6] = __int_as_float(0);
        }
        __syncwarp();
        kept += (unsigned long long)nk;
        if (fast) {
            const float2 npx = make_float2(-pxf, -pxf), npy = make_float2(-pyf, -pyf), npz = make_float2(-pzf, -pzf);
            const float2 invw2 = make_float2(invw_f, invw_f), c0h2 = make_float2(c0h, c0h), nkB2 = make_float2(-kB, -kB);
            const float2 thr02 = make_float2(thr0, thr0), mag2 = make_float2(kMagic, kMagic), nmag2 = make_float2(-kMagic, -kMagic);
            const float2 neg1 = make_float2(-1.f, -1.f);
#pragma unroll 1
            for (int q0 = 0; q0 < nk; q0 += 4) {
                // two packed pairs = four independent tests (instruction-level parallelism); every operation is the
                // IEEE round-to-nearest fp32 operation of the scalar formulation, two lanes at a time
                unsigned codeb[4], bitv[4];
                int cpos[4];
                bool ok[4], am[4];
#pragma unroll
                for (int pp = 0; pp < 2; ++pp) {
                    const float4 qa = cand[(q0 >> 1) * 2 + pp * 2], qb = cand[(q0 >> 1) * 2 + pp * 2 + 1];
                    const float2 dx = __fadd2_rn(make_float2(qa.x, qa.y), npx), dy = __fadd2_rn(make_float2(qa.z, qa.w), npy);
                    const float2 dz = __fadd2_rn(make_float2(qb.x, qb.y), npz);
                    float2 t = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
                    t.x = fmaxf(t.x, 1e-30f); t.y = fmaxf(t.y, 1e-30f); // t = 0: r = 0 -> exact path
                    float2 rinv;
                    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv.x) : "f"(t.x));
                    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv.y) : "f"(t.y));
                    const float2 uh = __ffma2_rn(__fmul2_rn(t, rinv), invw2, c0h2);
                    const float2 thr = __ffma2_rn(nkB2, rinv, thr02);
                    const float2 v = __fadd2_rn(uh, mag2);
                    const float2 fr = __ffma2_rn(__fadd2_rn(v, nmag2), neg1, uh); // uh - (v - kMagic), exact products
                    const float vv[2] = {v.x, v.y}, ff[2] = {fr.x, fr.y}, tt[2] = {thr.x, thr.y};
                    const float ww[2] = {qb.z, qb.w};
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int cc = pp * 2 + e;
                        const bool sure = fabsf(ff[e]) <= tt[e];         // farther than du from every bin edge
                        // v in [kMagic, kMagic + nb) <=> uh rounds into 0..nb-1 (float bits are monotonic)
                        codeb[cc] = (unsigned)(__float_as_int(vv[e]) - kMagicBits);
                        ok[cc] = sure && codeb[cc] < (unsigned)nb;
                        am[cc] = !sure;                                  // ~2 du of all pairs, in range or not
                        cpos[cc] = __float_as_int(ww[e]);
                        bitv[cc] = 1u << cpos[cc];
                    }
                }
                if (!__any_sync(kFull, am[0] | am[1] | am[2] | am[3])) {
                    // branch-free: a rejected candidate sets its bit in the spare row nb
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) atomicOr(&masks[(ok[cc] ? codeb[cc] : (unsigned)nb) * 32 + lane], bitv[cc]);
                } else {
                    // some pair is within the error margin of a bin edge (~1e-4 of the pairs): exact decision
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) {
                        if (ok[cc]) atomicOr(&masks[codeb[cc] * 32 + lane], bitv[cc]);
                        else if (am[cc] && codeb[cc] + 1u < (unsigned)nb + 2u && q0 + cc < nk) {
                            const unsigned cx = classify_exact<PERIODIC>(a.pos4[jbase + cpos[cc]], sp, lane, e2, nb, G.box, G.half, rmin_f, invw_f);
                            if (cx != kNoHit) atomicOr(&masks[cx * 32 + lane], bitv[cc]);
                        }
                    }
                }
            }
        } else {
            // group too wide for a common image: every pair is decided exactly
            unsigned rem = km;
            while (rem) {
                const int c = __ffs(rem) - 1;
                rem &= rem - 1u;
                if (lane < cnt) {
                    const unsigned cx = classify_exact<PERIODIC>(a.pos4[jbase + c], sp, lane, e2, nb, G.box, G.half, rmin_f, invw_f);
                    if (cx != kNoHit) masks[cx * 32 + lane] |= 1u << c;
                }
            }
        }
        // ---- one coalesced row per bin that has any bit set --------------------------------------------------------
        const unsigned desc = (unsigned)jbase | (wcode << 26);
        for (int b = 0; b < nb; ++b) {
            const unsigned m = masks[b * 32 + lane];
            if (__any_sync(kFull, m != 0u)) {
                const int k = __shfl_sync(kFull, rowcnt, b);
                const size_t ro = (size_t)b * nwords + k;
                __stcs(rows_g + ro * 32 + lane, m);
                if (lane == 0) __stcs(desc_g + ro, desc);
                if (lane == b) ++rowcnt;
                masks[b * 32 + lane] = 0u;
            }
        }
        __syncwarp(); // every lane is done with cand[] before the next word overwrites it
    }
    if (lane < nb) a.rowcnt[(size_t)g * nb + lane] = rowcnt;
    if (lane == 0) atomicAdd(a.cand_pairs, kept * (unsigned long long)cnt);
}

// ==========================================================================================================
// k_harm: a4.  One warp per item (group, bin): every lane walks the set bits of its column of the item's rows,
// a_lm accumulates in registers.
// ==========================================================================================================
struct Raw { double2 xy, zw; };

// One 256-bit load per candidate (LDG.E.256, sm_100): the gather is one 32-byte sector per lane, and the L1 tag stage
// handles one sector per cycle, so two 128-bit loads of the same sector cost twice the L1 time.
__device__ __forceinline__ Raw gather(const double4 *__restrict__ pos4, unsigned idx)
{
    Raw r;
    const double4 *q = pos4 + idx;
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.xy.x), "=d"(r.xy.y), "=d"(r.zw.x), "=d"(r.zw.y) : "l"(q));
    return r;
}

__device__ __forceinline__ void cp_async4(unsigned *smem_dst, const unsigned *gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async16(unsigned *smem_dst, const unsigned *gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// MODE 0: open geometry; 1: periodic, image carried by the row descriptor; 2: periodic, image decided per pair
// mtab (MODE 1): shared memory [axis][image code][thread] = x_i + {-L, 0, +L}: x_j - (x_i -/+ L) is the minimal image
// D: candidates gathered ahead of the one being accumulated.  Returns the number of pairs this lane accumulated.
// q: this warp's record queue [kQueue][32] of (mask, descriptor); stm: row staging [2][kStageRows][32];
// std_: descriptors [2][kStageRows].
// padent: entry of the padding particle pos4[n] (weight 0, far from everything): a lane with nothing left adds exact zeros.
// CAREFUL: the bin reaches outside fp32's comfortable range for r^2 (r_min = 0, or extreme units): library rsqrt.
struct HarmStats { unsigned steps; };

// GF (fp32-harmonics variant only): the candidates are gathered from pos4f, 16-byte fp32 records relative to the centre of
// the box (half the L1 bytes of the gather, no conversions), the separation is formed in fp32; mef = this primary in the
// same coordinates, mtab then holds floats.
template <int LMAX, int MLO, int MHI, int MODE, int D, bool CAREFUL, bool F32, bool GF = false>
__device__ __forceinline__ unsigned harm_rows(double (&acc)[ncomp_range(LMAX, MLO, MHI)], const unsigned *__restrict__ rows,
                                              const unsigned *__restrict__ rdesc, int nrows, bool active, uint2 *q,
                                              unsigned *stm, unsigned *std_, const double4 *__restrict__ pos4,
                                              const double4 &me, const double *mtab, double box, double half, int lane,
                                              unsigned padent, HarmStats &st, const float4 *__restrict__ pos4f = nullptr,
                                              float3 mef = make_float3(0.f, 0.f, 0.f), double *sacc = nullptr)
{
    static_assert(!GF || (F32 && !CAREFUL), "fp32 candidate records belong to the fp32-harmonics variant");
    static_assert(D >= 1 && D <= 4 && 4 % D == 0, "four steps per loop trip use the D gather slots in turn");
    // ---- rows -> shared memory: a ring of 2 chunks of kStageRows rows, both in flight (every chunk slot commits one
    // cp.async group, empty or not).  A chunk is kStageRows * 128 contiguous bytes: 16 bytes per lane and copy.
    auto issue_chunk = [&](int c) {
        const int r0 = c * kStageRows;
        if (r0 < nrows) {
            const int nr = min(kStageRows, nrows - r0);
            unsigned *dst = stm + (c & 1) * kStageRows * 32;
            const unsigned *src = rows + (size_t)r0 * 32;
#pragma unroll
            for (int j = 0; j < kStageRows / 4; ++j) {
                const int w = j * 128 + lane * 4;              // word offset inside the chunk; row = w / 32
                if ((w >> 5) < nr) cp_async16(dst + w, src + w);
            }
            if (lane < nr) cp_async4(std_ + (c & 1) * kStageRows + lane, rdesc + r0 + lane);
        }
        cp_async_commit();
    };
    issue_chunk(0);
    issue_chunk(1);
    int rows_done = 0;
    // lane-private queue cursors as byte offsets into the lane's column of q (stride 256 bytes per record)
    constexpr int QN = F32 ? kQueueF32 : kQueue;
    constexpr unsigned kQBytes = QN * 256u;
    unsigned head = 0u, tail = 0u, level = 0u;
    char *const qcol = reinterpret_cast<char *>(q + lane);
    int avail = 0;                      // pairs queued and not yet generated (bits of cur + bits of the queued masks)
    unsigned npairs = 0u;
    unsigned cur = 0u, dsc = 0u;        // record being walked: remaining bits, descriptor
    bool drained = false;
    // push rows while every lane has room for one more record; returns the number of steps to run next (0: finished)
    auto refill = [&]() -> int {
        int room = QN - __reduce_max_sync(kFull, (int)level);
        while (room > 0 && rows_done < nrows) {
            const int k0 = rows_done & (kStageRows - 1);
            if (k0 == 0) { cp_async_wait<1>(); __syncwarp(); }
            const int nr = min(min(room, nrows - rows_done), kStageRows - k0);
            const unsigned *ps = stm + (rows_done & (2 * kStageRows - 1)) * 32 + lane;
            const unsigned *pd = std_ + (rows_done & (2 * kStageRows - 1));
            for (int i = 0; i < nr; ++i) {
                const unsigned m = ps[i * 32];
                const unsigned d = pd[i];
                if (m) {
                    *reinterpret_cast<uint2 *>(qcol + tail) = make_uint2(m, d);
                    tail = (tail + 256u) & (kQBytes - 1u);
                    ++level;
                    const int pc = __popc(m);
                    avail += pc; npairs += (unsigned)pc;
                }
            }
            rows_done += nr; room -= nr;
            if ((rows_done & (kStageRows - 1)) == 0) { __syncwarp(); issue_chunk(rows_done / kStageRows + 1); }
        }
        int s;
        if (rows_done < nrows) { // a starving lane waits for rows: run while every active lane has pairs (at least 4 steps)
            s = __reduce_min_sync(kFull, active ? avail : INT_MAX);
            s = s >= 4 ? (s & ~3) : 4;
        } else {
            s = __reduce_max_sync(kFull, avail);
            if (s > 0) s = (s + 3) & ~3;
            else if (drained) s = 0;
            else { drained = true; s = 4; } // the last D gathers are still in flight
        }
#ifdef ENCORE_HARM_STATS
        st.steps += (unsigned)s;
#endif
        return s;
    };
    // next pair of this lane as an entry: sorted index | image codes << 26 (padent: nothing left)
    auto gen = [&]() -> unsigned {
        if (cur == 0u && level != 0u) {
            const uint2 rec = *reinterpret_cast<const uint2 *>(qcol + head);
            cur = rec.x; dsc = rec.y;
            head = (head + 256u) & (kQBytes - 1u);
            --level;
        }
        const bool pad = cur == 0u;
        const unsigned bit = (unsigned)(__ffs((int)cur) - 1);
        cur &= cur - 1u;
        if (!pad) --avail;
        return pad ? padent : dsc + bit; // the word's first index + bit stays below 2^26
    };

    int S = refill();
    if (S == 0 || (drained && S == 4)) { // no pair in this item
        cp_async_wait<0>();
#ifdef ENCORE_HARM_STATS
        st.steps = 0u;
#endif
        return 0u;
    }
    using RawT = std::conditional_t<GF, float4, Raw>;
    RawT r[D];
    unsigned ent[D];
    auto fetch = [&](unsigned idx) -> RawT {
        if constexpr (GF) return __ldg(pos4f + idx);
        else return gather(pos4, idx);
    };
#pragma unroll
    for (int d = 0; d < D; ++d) {
        ent[d] = gen();
        r[d] = fetch(ent[d] & kIdxMask);
    }
    // F32: fp32 chunk sums, added every sixteen loop trips (64 pairs) to the fp64 accumulators, which sit in shared memory
    // (sacc, this thread's column, stride = threads of the CTA): in registers they held the kernel at 219 registers and
    // 8 warps per SM
    constexpr int NACCF = F32 ? ncomp_range(LMAX, MLO, MHI) : 1;
    float facc[NACCF];
#pragma unroll
    for (int k = 0; k < NACCF; ++k) facc[k] = 0.f;
    int trips = 0;
    auto flush_f32 = [&]() {
        if constexpr (F32) {
#pragma unroll
            for (int k = 0; k < NACCF; ++k) { sacc[k * (kHarmWarps * 32)] += (double)facc[k]; facc[k] = 0.f; }
        }
    };
    // MODE 1: byte address of this thread's column of mtab; the image code of an axis selects one of three rows
    const char *const mcol = reinterpret_cast<const char *>(mtab);
    constexpr unsigned kRowB = kHarmWarps * 32 * 8;   // bytes per mtab row (power of two: 1024 at 4 warps)
    static_assert((kRowB & (kRowB - 1)) == 0, "mtab rows are selected by or-ing the code into the address");
    do {
        for (int s = 0; s < S; s += 4) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                // everything that reads slot u first, so that the next gather can land in the same registers
                if constexpr (GF) {
                    float fx, fy, fz;
                    constexpr unsigned kRowF = kRowB / 2;       // bytes per row of the float table
                    if (MODE == 1) {
                        const unsigned c0 = ent[u % D];
                        fx = r[u % D].x - *reinterpret_cast<const float *>(mcol + (((c0 >> 26) & 3u) * kRowF));
                        fy = r[u % D].y - *reinterpret_cast<const float *>(mcol + 4 * kRowF + (((c0 >> 28) & 3u) * kRowF));
                        fz = r[u % D].z - *reinterpret_cast<const float *>(mcol + 8 * kRowF + ((c0 >> 30) * kRowF));
                    } else {
                        fx = r[u % D].x - mef.x; fy = r[u % D].y - mef.y; fz = r[u % D].z - mef.z;
                        if (MODE == 2) {
                            const float bf = (float)box, hf = (float)half;
                            if (fx > hf) fx -= bf; else if (fx < -hf) fx += bf;
                            if (fy > hf) fy -= bf; else if (fy < -hf) fy += bf;
                            if (fz > hf) fz -= bf; else if (fz < -hf) fz += bf;
                        }
                    }
                    const float wf = r[u % D].w;
                    ent[u % D] = gen();
                    r[u % D] = fetch(ent[u % D] & kIdxMask);
                    const float r2f = fmaxf(fmaf(fz, fz, fmaf(fy, fy, fx * fx)), 1e-30f);
                    float y0;
                    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(r2f));
                    const float h = 0.5f * y0;
                    const float rinvf = fmaf(h, fmaf(-r2f * y0, y0, 1.f), y0); // one Newton step: ~1 ulp
                    accumulate_f32<LMAX, MLO, MHI>(facc, fx * rinvf, fy * rinvf, fz * rinvf, wf);
                } else {
                double dx, dy, dz;
                if (MODE == 1) {
                    const unsigned c0 = ent[u % D];
                    // rows 0..2 = x, 4..6 = y, 8..10 = z (a fourth, unused row per axis keeps the stride a power of two)
                    dx = r[u % D].xy.x - *reinterpret_cast<const double *>(mcol + (((c0 >> 26) & 3u) * kRowB));
                    dy = r[u % D].xy.y - *reinterpret_cast<const double *>(mcol + 4 * kRowB + (((c0 >> 28) & 3u) * kRowB));
                    dz = r[u % D].zw.x - *reinterpret_cast<const double *>(mcol + 8 * kRowB + ((c0 >> 30) * kRowB));
                } else {
                    dx = sep<MODE == 2>(r[u % D].xy.x, me.x, box, half);
                    dy = sep<MODE == 2>(r[u % D].xy.y, me.y, box, half);
                    dz = sep<MODE == 2>(r[u % D].zw.x, me.z, box, half);
                }
                const double wj = r[u % D].zw.y;
                ent[u % D] = gen();
                r[u % D] = fetch(ent[u % D] & kIdxMask); // D candidates ahead
                if constexpr (F32) {
                    // fp32 harmonics: the separation is formed in fp64 (positions are large, separations small) and
                    // rounded once; unit vector, powers and (x+iy)^m in fp32.  CAREFUL bins keep the fp64 normalisation.
                    float fx, fy, fz;
                    if (CAREFUL) {
                        const double rinv = rsqrt(fma(dz, dz, fma(dy, dy, dx * dx)));
                        fx = (float)(dx * rinv); fy = (float)(dy * rinv); fz = (float)(dz * rinv);
                    } else {
                        fx = (float)dx; fy = (float)dy; fz = (float)dz;
                        const float r2f = fmaf(fz, fz, fmaf(fy, fy, fx * fx));
                        float y0;
                        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(r2f));
                        const float h = 0.5f * y0;
                        const float rinvf = fmaf(h, fmaf(-r2f * y0, y0, 1.f), y0); // one Newton step: ~1 ulp
                        fx *= rinvf; fy *= rinvf; fz *= rinvf;
                    }
                    accumulate<LMAX, MLO, MHI, float>(facc, fx, fy, fz, (float)wj);
                } else {
                    const double r2s = fma(dz, dz, fma(dy, dy, dx * dx));
                    const double rinv = CAREFUL ? rsqrt(r2s) : rsqrt_pair(r2s);
                    accumulate<LMAX, MLO, MHI, double>(acc, dx * rinv, dy * rinv, dz * rinv, wj);
                }
                }
            }
            if (F32 && ++trips == 16) { flush_f32(); trips = 0; }
        }
        S = refill();
    } while (S > 0);
    flush_f32();
    cp_async_wait<0>();
    return npairs;
}

// dynamic shared memory of k_harm per CTA: mtab[12][threads] double | queue[warps][kQueue][32] uint2 |
//                                          stage[warps][2][kStageRows][32] u32 | stage descriptors[warps][2][kStageRows] u32
__host__ __device__ constexpr size_t harm_smem_bytes(bool periodic, bool f32 = false)
{
    return (periodic ? (size_t)12 * kHarmWarps * 32 * 8 : 0) + (size_t)kHarmWarps * (f32 ? kQueueF32 : kQueue) * 32 * 8 +
           (size_t)kHarmWarps * 2 * kStageRows * 32 * 4 + (size_t)kHarmWarps * 2 * kStageRows * 4;
}

// F32: the fp32-harmonics variant (ENCORE_FP32_HARMONICS): weighted harmonics in fp32, fp64 accumulation of 64-pair
// chunk sums; the pair list (binning) is the fp64-exact one of k_fill either way.
template <int LMAX, int MLO, int MHI, bool PERIODIC, bool F32>
__global__ void __launch_bounds__(kHarmWarps * 32, F32 ? 3 : (ncomp_range(LMAX, MLO, MHI) > ENCORE_HARM_FAT ? 2 : 3)) k_harm(PairArgs a, int g0, int g1, int write_counts)
{
    constexpr int NACC = ncomp_range(LMAX, MLO, MHI), D = F32 ? 2 : (NACC > ENCORE_HARM_FAT ? ENCORE_HARM_DEPTH_FAT : ENCORE_HARM_DEPTH);
    extern __shared__ __align__(16) unsigned char harm_smem[];
    double *mtab = reinterpret_cast<double *>(harm_smem);
    uint2 *s_q = reinterpret_cast<uint2 *>(harm_smem + (PERIODIC ? (size_t)12 * kHarmWarps * 32 * 8 : 0));
    constexpr int QN = F32 ? kQueueF32 : kQueue;
    unsigned *s_stm = reinterpret_cast<unsigned *>(s_q + kHarmWarps * QN * 32);
    unsigned *s_std = s_stm + kHarmWarps * 2 * kStageRows * 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ng = g1 - g0, nb = a.bins.nbins;
    const int item = blockIdx.x * kHarmWarps + warp;
    if (item >= ng * nb) return;
    const int bin = a.bin_order[item / ng], g = g0 + item % ng;
    if (g >= a.group_start[a.geom.npencil]) return;    // (g1 is an upper bound when the group count was not read back)
    const Group gr = locate_group<PERIODIC>(a, g);
    const bool active = lane < gr.cnt;
    const double4 me = a.pos4[gr.first + (active ? lane : 0)];
    const size_t col = ((size_t)g * nb + bin) * 32 + lane;
    // the row stream of (g, bin): see k_fill
    const int nwords = a.gprefix[g + 1] - a.gprefix[g];
    const size_t ro = (size_t)(a.gprefix[g] - a.gprefix[g0]) * (size_t)nb + (size_t)bin * nwords;
    const unsigned *rows = a.rows + ro * 32;
    const unsigned *rdesc = a.rowdesc + ro;
    const int nrows = a.rowcnt[(size_t)g * nb + bin];
    // the exact path of k_fill (no common image per run) is taken under the same condition there
    bool fast = gr.fast;
    if (PERIODIC && fast) fast = !a.gwide[g];
    // padding entry: particle n of pos4 (weight 0, far away), image codes (1,1,1) = no shift
    const unsigned padent = (unsigned)a.npart | (0x15u << 26);
    // r^2 of every pair of this item lies in [e2[bin], e2[bin+1]) up to rounding; the padding particle is a few box sizes away
    const bool careful = !(a.bins.e2[bin] > 1e-290 && a.bins.e2[bin + 1] < 1e290 && a.pad_r2max < 1e290);
    uint2 *q = s_q + warp * QN * 32;
    unsigned *stm = s_stm + warp * 2 * kStageRows * 32, *std_ = s_std + warp * 2 * kStageRows;

    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    unsigned np;
    HarmStats st{0u};
    // F32: the fp64 accumulators of this thread are a column of shared memory behind the other regions
    double *sacc = reinterpret_cast<double *>(harm_smem + harm_smem_bytes(PERIODIC, F32)) + threadIdx.x;
    if constexpr (F32) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) sacc[k * (kHarmWarps * 32)] = 0.0;
    }
    // fp32-harmonics variant: 16-byte fp32 candidate records for the bins fp32 coordinates resolve (api.cu: gf_min_r2)
    const bool gf = F32 && !careful && a.pos4f != nullptr && a.bins.e2[bin] >= a.gf_min_r2;
    const float3 mef = make_float3((float)(me.x - a.ctr[0]), (float)(me.y - a.ctr[1]), (float)(me.z - a.ctr[2]));
    if (!PERIODIC) {
        if constexpr (F32) {
            if (gf) np = harm_rows<LMAX, MLO, MHI, 0, D, false, true, true>(acc, rows, rdesc, nrows, active, q, stm, std_, a.pos4, me, nullptr, 0.0, 0.0, lane, padent, st, a.pos4f, mef, sacc);
        }
        if (!gf) {
            if (careful) np = harm_rows<LMAX, MLO, MHI, 0, D, true, F32>(acc, rows, rdesc, nrows, active, q, stm, std_, a.pos4, me, nullptr, 0.0, 0.0, lane, padent, st, nullptr, mef, sacc);
            else np = harm_rows<LMAX, MLO, MHI, 0, D, false, F32>(acc, rows, rdesc, nrows, active, q, stm, std_, a.pos4, me, nullptr, 0.0, 0.0, lane, padent, st, nullptr, mef, sacc);
        }
    } else if (fast) {
        const double L = a.geom.box;
        constexpr int R = kHarmWarps * 32;
        if (gf) {
            float *mt = reinterpret_cast<float *>(mtab) + threadIdx.x;
            const double x = me.x - a.ctr[0], y = me.y - a.ctr[1], z = me.z - a.ctr[2];
            mt[0 * R] = (float)(x - L); mt[1 * R] = (float)x; mt[2 * R] = (float)(x + L);
            mt[4 * R] = (float)(y - L); mt[5 * R] = (float)y; mt[6 * R] = (float)(y + L);
            mt[8 * R] = (float)(z - L); mt[9 * R] = (float)z; mt[10 * R] = (float)(z + L);
            __syncwarp();
            if constexpr (F32)
                np = harm_rows<LMAX, MLO, MHI, 1, D, false, true, true>(acc, rows, rdesc, nrows, active, q, stm, std_, a.pos4, me, reinterpret_cast<const double *>(mt), L, a.geom.half, lane, padent, st, a.pos4f, mef, sacc);
        } else {
            double *mt = mtab + threadIdx.x;
            mt[0 * R] = me.x - L; mt[1 * R] = me.x; mt[2 * R] = me.x + L;
            mt[4 * R] = me.y - L; mt[5 * R] = me.y; mt[6 * R] = me.y + L;
            mt[8 * R] = me.z - L; mt[9 * R] = me.z; mt[10 * R] = me.z + L;
            __syncwarp();
            if (careful) np = harm_rows<LMAX, MLO, MHI, 1, D, true, F32>(acc, rows, rdesc, nrows, active, q, stm, std_, a.pos4, me, mt, L, a.geom.half, lane, padent, st, nullptr, mef, sacc);
            else np = harm_rows<LMAX, MLO, MHI, 1, D, false, F32>(acc, rows, rdesc, nrows, active, q, stm, std_, a.pos4, me, mt, L, a.geom.half, lane, padent, st, nullptr, mef, sacc);
        }
    } else {
        if constexpr (F32) {
            if (gf) np = harm_rows<LMAX, MLO, MHI, 2, D, false, true, true>(acc, rows, rdesc, nrows, active, q, stm, std_, a.pos4, me, nullptr, a.geom.box, a.geom.half, lane, padent, st, a.pos4f, mef, sacc);
        }
        if (!gf) np = harm_rows<LMAX, MLO, MHI, 2, D, true, F32>(acc, rows, rdesc, nrows, active, q, stm, std_, a.pos4, me, nullptr, a.geom.box, a.geom.half, lane, padent, st, nullptr, mef, sacc);
    }
    if constexpr (F32) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) acc[k] = sacc[k * (kHarmWarps * 32)];
    }
    if (write_counts) {
        a.counts[col] = np;     // n_i(b); every m-range pass walks the same bits, the first one reports
#ifdef ENCORE_HARM_STATS
        // diagnostics (build with -DENCORE_HARM_STATS): lock-step pair steps executed and the most pairs any lane of the
        // item had; their ratio is the lane utilisation of this kernel
        const unsigned mx = __reduce_max_sync(kFull, np);
        if (lane == 0) { atomicAdd(a.cand_pairs + 1, (unsigned long long)st.steps); atomicAdd(a.cand_pairs + 2, (unsigned long long)mx); }
#endif
    }

    // epilogue: a_lm = (1/v_b) sum_k ycoef[c][k] S_{m,k}, k = l-m, l-m-2, ... (p_lm has the parity of l-m)
    const double vinv = a.bins.vinv[bin];
    double *out = a.alm + (size_t)g * a.ncomp * nb * 32 + (size_t)bin * 32 + lane;
    int base = 0;
#pragma unroll
    for (int m = MLO; m <= MHI; ++m) {
        const int st2 = m ? 2 : 1;
#pragma unroll
        for (int l = m; l <= LMAX; ++l) {
            const int cre = m == 0 ? l * l : l * l + 2 * m - 1;
            const double *yc = a.ycoef + (size_t)cre * (LMAX + 1);
            double sr = 0.0, si = 0.0;
#pragma unroll
            for (int qq = (l - m) & 1; qq <= l - m; qq += 2) {
                const double cf = __ldg(yc + qq);
                sr = fma(cf, acc[base + qq * st2], sr);
                if (m) si = fma(cf, acc[base + qq * st2 + 1], si);
            }
            out[(size_t)cre * nb * 32] = active ? sr * vinv : 0.0;
            if (m) out[(size_t)(cre + 1) * nb * 32] = active ? si * vinv : 0.0;
        }
        base += (LMAX - m + 1) * st2;
    }
}

template <int LMAX, int MLO, int MHI, bool F32>
cudaError_t launch_harm_t(const PairArgs &a, int g0, int g1, int write_counts, cudaStream_t s, int *launches)
{
    const int nitems = (g1 - g0) * a.bins.nbins;
    const int grid = (nitems + kHarmWarps - 1) / kHarmWarps;
    // F32: the fp64 accumulators live in shared memory, one column per thread
    constexpr size_t kAccBytes = F32 ? (size_t)ncomp_range(LMAX, MLO, MHI) * kHarmWarps * 32 * sizeof(double) : 0;
    // the opt-in shared-memory limit is a per-kernel, per-DEVICE attribute: set once per instantiation and device
    static PerDeviceOnce once;
    const cudaError_t attr_err = once.run([] {
        cudaError_t e = cudaFuncSetAttribute(k_harm<LMAX, MLO, MHI, true, F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(harm_smem_bytes(true, F32) + kAccBytes));
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_harm<LMAX, MLO, MHI, false, F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(harm_smem_bytes(false, F32) + kAccBytes));
        return e;
    });
    if (attr_err != cudaSuccess) return attr_err;
    if (a.geom.periodic) k_harm<LMAX, MLO, MHI, true, F32><<<grid, kHarmWarps * 32, harm_smem_bytes(true, F32) + kAccBytes, s>>>(a, g0, g1, write_counts);
    else k_harm<LMAX, MLO, MHI, false, F32><<<grid, kHarmWarps * 32, harm_smem_bytes(false, F32) + kAccBytes, s>>>(a, g0, g1, write_counts);
    *launches += 1;
    return cudaGetLastError();
}

template <int LMAX, int MLO, int MHI>
cudaError_t launch_harm(const PairArgs &a, int g0, int g1, int write_counts, cudaStream_t s, int *launches)
{
    return a.fp32_harmonics ? launch_harm_t<LMAX, MLO, MHI, true>(a, g0, g1, write_counts, s, launches)
                            : launch_harm_t<LMAX, MLO, MHI, false>(a, g0, g1, write_counts, s, launches);
}

} // namespace

int pair_stage_supported(int lmax, int nbins)
{
    return lmax >= 0 && lmax <= ENCORE_MAX_LMAX && nbins >= 1 && nbins <= ENCORE_MAX_BINS;
}

size_t pair_fill_smem_bytes(int nbins, int nr_cap) { return fill_smem_bytes(nbins, nr_cap); }

cudaError_t launch_pair_bounds(const PairArgs &a, cudaStream_t s, int *launches)
{
    if (a.ngroups <= 0) return cudaSuccess;
    if (a.geom.periodic) k_group_bound<true><<<(a.ngroups + 3) / 4, 128, 0, s>>>(a);
    else k_group_bound<false><<<(a.ngroups + 3) / 4, 128, 0, s>>>(a);
    *launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return launch_exclusive_scan(a.gbound, a.gprefix, a.ngroups, a.scan_tmp, s, launches);
}

#define HARM_PASS(L, A, B)                                                      \
    {                                                                           \
        cudaError_t e = launch_harm<L, A, B>(a, g0, g1, (A) == 0, s, launches); \
        if (e != cudaSuccess) return e;                                         \
    }

// m-ranges per lmax.  Every pass walks the rows and gathers the candidates again (the L1 data pipe is ~70 % busy),
// so fewer, fatter passes win: up to 44 accumulators run at 168 registers and 12 warps/SM, 45-65 at 255 registers and
// 8 warps/SM (c2, lmax 10: four passes 46.3 ms, three 40.1 ms, two 37.1 ms for the pair stage).
cudaError_t launch_pair_fill(const PairArgs &a, int g0, int g1, int nr_cap, cudaStream_t s, int *launches)
{
    const int ng = g1 - g0, nb = a.bins.nbins;
    if (ng <= 0) return cudaSuccess;
    // the opt-in shared-memory limit is a per-kernel, per-DEVICE attribute: set it once per device, to the most any plan asks for
    static PerDeviceOnce once;
    const cudaError_t attr_err = once.run([] {
        cudaError_t e = cudaFuncSetAttribute(k_fill<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fill<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        return e;
    });
    if (attr_err != cudaSuccess) return attr_err;
    const size_t smem = fill_smem_bytes(nb, nr_cap);
    if (a.geom.periodic) k_fill<true><<<ng, 32, smem, s>>>(a, g0, g1, nr_cap);
    else k_fill<false><<<ng, 32, smem, s>>>(a, g0, g1, nr_cap);
    *launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_pair_harmonics(const PairArgs &a, int g0, int g1, cudaStream_t s, int *launches)
{
    if (g1 - g0 <= 0) return cudaSuccess;
    switch (a.lmax) {
    case 0: HARM_PASS(0, 0, 0) break;
    case 1: HARM_PASS(1, 0, 1) break;
    case 2: HARM_PASS(2, 0, 2) break;
    case 3: HARM_PASS(3, 0, 3) break;
    case 4: HARM_PASS(4, 0, 4) break;
    case 5: HARM_PASS(5, 0, 5) break;
    case 6: HARM_PASS(6, 0, 6) break;
    case 7: HARM_PASS(7, 0, 7) break;
    case 8: HARM_PASS(8, 0, 2) HARM_PASS(8, 3, 8) break;
    case 9: HARM_PASS(9, 0, 3) HARM_PASS(9, 4, 9) break;
    case 10: HARM_PASS(10, 0, 3) HARM_PASS(10, 4, 10) break;
    default: return cudaErrorInvalidValue;
    }
    return cudaSuccess;
}
