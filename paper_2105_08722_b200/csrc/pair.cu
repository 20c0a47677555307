// pair.cu — steps a3 (neighbour sweep + radial binning) and a4 (a_lm accumulation) of the ENCORE hot path.
//
//   a^b_lm(s_i) = (1/v_b) sum_{j != i} w_j Y_lm((r_j - s_i)^) Theta^b(|r_j - s_i|)          eq. 35
//
// The paper does this on the CPU, histogramming Cartesian monomials with AVX, eight secondaries at a time
// (Alg. 2) and has no GPU version of it.  Design here:
// the work is split by resource profile into two kernels around "groups" of 32 consecutive cell-sorted
// primaries of one (iy,iz) pencil (lane = primary everywhere):
//   k_fill  (a3, integer/fp32, few registers): ONE WARP per group.  Candidates = contiguous runs of the sorted
//     array (one or two per neighbouring pencil, x-range culled against the group's cell range), read 32 at a time,
//     made relative to primary 0 in fp32, culled against the bounding box of the group's primaries and compacted
//     into a ring in shared memory, from where they are broadcast to the lanes.  A first fp32 evaluation
//     decides every pair whose radius is farther than a proven error margin from all bin edges; the rest (~1e-4)
//     is decided in fp64 exactly as DESIGN.md R8-R10 fix it (r^2 = fma(dz,dz,fma(dy,dy,dx*dx)) against e_b^2), so
//     counts are bit-exact.  An accepted pair is appended, in candidate order, to the list of (primary, bin):
//     lane-private cursors and one 4-entry block per (bin, lane) in shared memory, written 16 bytes at a time
//     into 256-byte pages of a pool in HBM; pages of one list are chained through page_next[].
//     The final cursors are n_i(b), the per-(primary, bin) pair counts (an integer output of the path).
//   k_harm  (a4, fp64, ~166 registers): one warp per (group, bin); every lane streams its own list, gathers the
//     candidates two rows ahead, and keeps the (lmax+1)^2 real accumulators of a^b_lm(s_i) in REGISTERS: no
//     atomics, no cross-lane reductions, summation order = candidate order -> deterministic.  Per pair: unit
//     vector (fp32 rsqrt seed + one third-order fp64 step), w (x+iy)^m by complex recurrence, powers of z, one FMA
//     per component into S_{m,k} = sum w z^k (x+iy)^m; the monic associated-Legendre polynomials p_lm(z) and the
//     normalisation (-1)^m N_lm k_lm / v_b are applied once per (primary, bin) in the epilogue (table ycoef).
//     Items are ordered heaviest bin first so the grid drains evenly.
#include "device.cuh"

#include <algorithm>
#include <climits>

namespace {

constexpr int kRing = 4;            // k_fill: one block of 4 entries (16 bytes) per (bin, lane); see the append/flush notes
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
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kNoHit = 254u;
constexpr unsigned kPadEntry = 0xffffffffu;
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
    return v > nc - 1 ? nc - 1 : v;
}

// acc[] order: m ascending, k ascending, (re, im): S_{m,k} = sum w z^k (x+iy)^m, k = 0..LMAX-m.
// Same number of accumulators as the a_lm themselves ((LMAX+1)^2 reals over all m) and one FMA each per pair; the
// Legendre polynomials p_lm(z) are applied once per (primary, bin) in the epilogue through the table ycoef
// (tables.cpp): 4 multiplies for the powers of z replace the 2 operations per (l,m) of a recurrence in every pair.
template <int LMAX, int MLO, int MHI>
__device__ __forceinline__ void accumulate(double (&acc)[ncomp_range(LMAX, MLO, MHI)], double x, double y, double z,
                                           double w)
{
    double zp[LMAX + 1];
    zp[0] = 1.0;
#pragma unroll
    for (int k = 1; k <= LMAX - MLO; ++k) zp[k] = k == 1 ? z : zp[k - 1] * z;
    double c = w, s = 0.0; // w (x + i y)^m
    int k = 0;
#pragma unroll
    for (int m = 0; m <= MHI; ++m) {
        if (m == 1) { c = w * x; s = w * y; }
        if (m > 1) {
            const double cn = fma(c, x, -(s * y));
            const double sn = fma(c, y, s * x);
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

// 1/sqrt(a) to full double precision from the fp32 approximation y0 (relative error <= 2^-21.4 including the
// rounding of a to fp32) and ONE third-order step: with e = 1 - a y0^2, a^-1/2 = y0 (1 - e)^-1/2 =
// y0 (1 + e/2 + 3e^2/8 + 5e^3/16 + ...), truncation 5/16 |e|^3 < 2^-62.  5 fp64 operations instead of the
// library routine's ~10; arguments outside fp32's comfortable range take the library path.
__device__ __forceinline__ double rsqrt_pair(double a)
{
    const float af = __double2float_rn(a);
    if (!(af > 1e-30f && af < 1e30f)) return rsqrt(a);
    float yf;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(yf) : "f"(af));
    const double y0 = (double)yf;
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
// STORE: rng_start[r] = first sorted index of run r, rng_off[r] = candidates before run r (rng_off[nr] = total).
// Returns the number of candidates T of the group.
template <bool PERIODIC, bool STORE>
__device__ __forceinline__ int build_ranges(const PairArgs &a, const Group &gr, int lane, int *rng_start, int *rng_off,
                                            int *nr_out)
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
                    if (hi - lo + 1 >= ncx) { lo = 0; hi = ncx - 1; }
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
        mine += l0 + l1;
        if (STORE) {
            rng_start[2 * r] = s0; rng_off[2 * r + 1] = l0;       // lengths parked in rng_off[.+1], scanned below
            rng_start[2 * r + 1] = s1; rng_off[2 * r + 2] = l1;
        }
    }
    const int nr = 2 * nyz;
    *nr_out = nr;
    if (!STORE) return __reduce_add_sync(kFull, mine);
    __syncwarp();
    { // inclusive scan of the lengths into offsets
        const int per = (nr + 31) / 32;
        const int b0 = lane * per, b1 = min(nr, b0 + per);
        int sum = 0;
        for (int r = b0; r < b1; ++r) sum += rng_off[r + 1];
        int x = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { int y = __shfl_up_sync(kFull, x, d); if (lane >= d) x += y; }
        int run = x - sum;
        for (int r = b0; r < b1; ++r) { const int len = rng_off[r + 1]; run += len; rng_off[r + 1] = run; }
        if (lane == 0) rng_off[0] = 0;
    }
    __syncwarp();
    return rng_off[nr];
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

// upper bound on the pool slabs a group can take (see k_fill: a slab yields >= kSlabPages-31 usable pages)
__device__ __forceinline__ int slab_bound(long long cand, int cnt, int nb)
{
    const long long need = (cand * cnt) / ENCORE_PAGE_WORDS + (long long)cnt * nb;
    const long long slabs = need / (ENCORE_SLAB_PAGES - 31) + 1;
    return (int)(slabs > INT_MAX ? INT_MAX : slabs);
}

// per group: candidates T and the slab bound (sizes the super-steps on the host)
template <bool PERIODIC>
__global__ void __launch_bounds__(128) k_group_bound(PairArgs a)
{
    const int g = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (g >= a.ngroups) return;
    if (g >= a.group_start[a.geom.npencil]) { if (lane == 0) a.gbound[g] = 0; return; }
    const Group gr = locate_group<PERIODIC>(a, g);
    int nr;
    const int T = build_ranges<PERIODIC, false>(a, gr, lane, nullptr, nullptr, &nr);
    if (lane == 0) a.gbound[g] = slab_bound(T, gr.cnt, a.bins.nbins);
}

// ==========================================================================================================
// k_fill: a3.  One warp (= one CTA) per group.
// ==========================================================================================================
// dynamic shared memory: cand[64] float4 | sp[96] double | e2[nb+1] double | ring[nb][32][4] u32 |
//                        cursor[nb][32] u32 | pagecur[nb][32] int | rng_start[nr_cap] | rng_off[nr_cap+1]
__host__ __device__ inline size_t fill_smem_bytes(int nb, int nr_cap)
{
    return 2 * 32 * 16 + 96 * 8 + (size_t)((nb + 2) & ~1) * 8 + (size_t)nb * kRing * 32 * 4 + (size_t)nb * 32 * 4 * 2 +
           (size_t)(2 * nr_cap + 4) * 4;
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
    double *sp = reinterpret_cast<double *>(cand + 64);
    double *e2 = sp + 96;
    unsigned *ring = reinterpret_cast<unsigned *>(e2 + ((nb + 2) & ~1));
    unsigned *cursor = ring + nb * kRing * 32;
    int *pagecur = reinterpret_cast<int *>(cursor + nb * 32);
    int *rng_start = pagecur + nb * 32;
    int *rng_off = rng_start + nr_cap;

    const Group gr = locate_group<PERIODIC>(a, g);
    const int first = gr.first, cnt = gr.cnt;
    const double4 ctr = a.pos4[first];
    const double4 mine = a.pos4[first + (lane < cnt ? lane : 0)];
    sp[lane] = mine.x; sp[32 + lane] = mine.y; sp[64 + lane] = mine.z;
    a.gweights[(size_t)g * 32 + lane] = lane < cnt ? mine.w : 0.0;
    if (lane <= nb) e2[lane] = a.bins.e2[lane];
    for (int b = 0; b < nb; ++b) cursor[b * 32 + lane] = 0u;
    // this lane's primary, relative to primary 0, fp32 (lanes beyond the group sit far away: never a hit)
    const float pxf = lane < cnt ? (float)(mine.x - ctr.x) : -1e18f, pyf = (float)(mine.y - ctr.y), pzf = (float)(mine.z - ctr.z);

    int nr;
    const int T = build_ranges<PERIODIC, true>(a, gr, lane, rng_start, rng_off, &nr);

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
    const float uh_hi = nb_f - 0.5f;
    const bool fast = gr.fast;

    // ---- list state -----------------------------------------------------------------------------------------
    // blocks of 4 completed but not yet written: (block index << 5) | bin.  The tests run two candidates between
    // flushes and a lane appends at most once per candidate, so at most two blocks (of two different bins) complete
    // in between: two slots.  If the first append completes a block and the second goes to the same bin, the entry
    // waits in a register (ovf_entry) and becomes entry 0 of the block once that has been written: the ring is a
    // single block per (bin, lane) - 5 kB for 10 bins instead of 10 kB, which is what sets the warps per SM.
    int pendA = -1, pendB = -1;
    bool ovf = false;
    unsigned ovf_entry = 0u;
    int slab_next = 0, slab_end = 0; // pages of the pool owned by this warp (uniform)
    const unsigned lt_mask = (1u << lane) - 1u;

    // all lanes call; lanes with a pending block write it (4 entries, 16 bytes) to their page.
    // ring layout [bin][lane][4]: the flush is one conflict-free 16-byte shared-memory load
    auto flush_block = [&](int &pend, bool with_ovf) {
        const bool act = pend >= 0;
        const int b = pend & 31, kb = pend >> 5;
        const bool newpage = act && (kb & 15) == 0;
        const unsigned nm = __ballot_sync(kFull, newpage);
        if (nm) {
            const int nn = __popc(nm);
            if (slab_next + nn > slab_end) { // the rest of the old slab (< 32 pages) is dropped: see slab_bound
                unsigned base = 0;
                if (lane == 0) base = atomicAdd(a.pool_cursor, (unsigned)ENCORE_SLAB_PAGES);
                base = __shfl_sync(kFull, base, 0);
                if (base + ENCORE_SLAB_PAGES > a.pool_pages) { // excluded by the host's step bounds; stay in bounds
                    if (lane == 0) *a.err_flag = 1;
                    base = 0;
                }
                slab_next = (int)base; slab_end = (int)base + ENCORE_SLAB_PAGES;
            }
            if (newpage) {
                const int pg = slab_next + __popc(nm & lt_mask);
                if (kb == 0) a.first_page[((size_t)g * nb + b) * 32 + lane] = pg;
                else a.page_next[pagecur[b * 32 + lane]] = pg;
                pagecur[b * 32 + lane] = pg;
            }
            slab_next += nn;
        }
        if (act) {
            unsigned *blk = ring + ((b << 5) + lane) * 4;
            const uint4 v = *reinterpret_cast<const uint4 *>(blk);
            __stcs(reinterpret_cast<uint4 *>(a.pool + (size_t)pagecur[b * 32 + lane] * ENCORE_PAGE_WORDS + ((kb & 15) << 2)), v);
            if (with_ovf && ovf) blk[0] = ovf_entry;
        }
        pend = -1;
    };
    auto flush_all = [&]() {
        if (__any_sync(kFull, pendA >= 0)) {
            flush_block(pendA, true);
            ovf = false;
            if (__any_sync(kFull, pendB >= 0)) flush_block(pendB, false);
        }
    };
    // `second`: an append may have happened since the last flush (then pendA may hold this bin's full block)
    auto append = [&](unsigned code, unsigned entry, bool second) {
        unsigned *cp = cursor + code * 32 + lane;
        const unsigned pos = *cp;
        *cp = pos + 1u;
        if (second && pendA >= 0 && (unsigned)(pendA & 31) == code) { ovf = true; ovf_entry = entry; } // pos & 3 == 0
        else {
            ring[((code << 5) + lane) * 4 + (pos & 3u)] = entry;
            if ((pos & 3u) == 3u) {
                const int v = (int)(((pos >> 2) << 5) | code);
                if (pendA < 0) pendA = v; else pendB = v;
            }
        }
    };

    // ---- candidate queue ------------------------------------------------------------------------------------------
    // Candidates are read a word (32) at a time, lane = candidate: fp64 -> relative to primary 0 (periodic image) ->
    // fp32, then culled against the group's bounding box (distance to the box > r_max: no primary of the group can
    // accept it) and the survivors are compacted into a 64-entry ring in shared memory (.w = list entry).  The pair
    // tests below always run on 32 queued candidates, so their cost follows the culled candidate count.
    // a lane asks for s = lane, 32 + lane, 64 + lane, ...: its run index only moves forward
    int run_lo = 0; // rng_off[run_lo] <= s < rng_off[run_lo + 1] once advanced (empty runs are stepped over)
    auto load_cand = [&](int s, double4 &cj, unsigned &j) {
        j = kPadEntry;
        if (s < T) {
            while (rng_off[run_lo + 1] <= s) ++run_lo; // s < T = rng_off[nr] bounds the walk
            j = (unsigned)(rng_start[run_lo] + (s - rng_off[run_lo]));
            cj = a.pos4[j];
        }
    };
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
    int qh = 0, qn = 0; // ring head and fill level (uniform)
    unsigned long long kept = 0ull;
    auto stage = [&](const double4 &cj, unsigned j) {
        float4 cf = make_float4(0.f, 0.f, 0.f, 0.f);
        bool keep = false;
        if (j != kPadEntry) {
            double rx = cj.x - ctr.x, ry = cj.y - ctr.y, rz = cj.z - ctr.z;
            unsigned kx = 1, ky = 1, kz = 1;  // image code: the list consumer subtracts {-L, 0, +L}[code] from x_i
            if (PERIODIC) {
                if (rx > G.half) { rx -= G.box; kx = 2; } else if (rx < -G.half) { rx += G.box; kx = 0; }
                if (ry > G.half) { ry -= G.box; ky = 2; } else if (ry < -G.half) { ry += G.box; ky = 0; }
                if (rz > G.half) { rz -= G.box; kz = 2; } else if (rz < -G.half) { rz += G.box; kz = 0; }
            }
            cf = make_float4((float)rx, (float)ry, (float)rz, __uint_as_float(j | (kx << 26) | (ky << 28) | (kz << 30)));
            const float ex = fmaxf(fmaxf(blo[0] - cf.x, cf.x - bhi[0]), 0.f);
            const float ey = fmaxf(fmaxf(blo[1] - cf.y, cf.y - bhi[1]), 0.f);
            const float ez = fmaxf(fmaxf(blo[2] - cf.z, cf.z - bhi[2]), 0.f);
            keep = !fast || fmaf(ez, ez, fmaf(ey, ey, ex * ex)) <= cut2; // wide groups (exact path) keep everything
        }
        const unsigned km = __ballot_sync(kFull, keep);
        if (keep) cand[(qh + qn + __popc(km & lt_mask)) & 63] = cf;
        qn += __popc(km);
        kept += (unsigned long long)__popc(km);
    };

    const int nwords = (T + 31) >> 5;
    int wnext = 0; // next word to stage; cjA holds it, cjB the one after
    double4 cjA = make_double4(0, 0, 0, 0), cjB = cjA;
    unsigned jA = kPadEntry, jB = kPadEntry;
    load_cand(lane, cjA, jA);
    load_cand(32 + lane, cjB, jB);
    for (;;) {
        while (qn < 32 && wnext < nwords) {
            stage(cjA, jA);
            cjA = cjB; jA = jB;
            ++wnext;
            load_cand((wnext + 1) * 32 + lane, cjB, jB); // two words ahead: in flight during the tests below
        }
        if (qn == 0) break;
        const int nvalid = min(qn, 32);
        if (lane >= nvalid) cand[(qh + lane) & 63] = make_float4(1e18f, 1e18f, 1e18f, __uint_as_float(kPadEntry)); // never a hit
        __syncwarp();
        if (fast) {
#pragma unroll 1
            for (int c4 = 0; c4 < 32; c4 += 4) {
                // four independent tests first (instruction-level parallelism), then the appends in candidate order
                unsigned ent[4], code[4];
                bool ok[4], am[4];
#pragma unroll
                for (int cc = 0; cc < 4; ++cc) {
                    const float4 q = cand[(qh + c4 + cc) & 63];
                    const float dx = q.x - pxf, dy = q.y - pyf, dz = q.z - pzf;
                    const float t = fmaxf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)), 1e-30f); // t = 0: r = 0 -> exact path
                    float rinv;
                    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(t));
                    const float uh = fmaf(t * rinv, invw_f, c0h);
                    const float thr = fmaf(-kB, rinv, thr0);
                    const float v = uh + kMagic;
                    const float fr = uh - (v - kMagic);
                    const bool sure = fabsf(fr) <= thr;              // farther than du from every bin edge
                    // v in [kMagic, kMagic + nb) <=> uh rounds into 0..nb-1 (float bits are monotonic)
                    code[cc] = (unsigned)(__float_as_int(v) - kMagicBits);
                    ok[cc] = sure && code[cc] < (unsigned)nb;
                    am[cc] = !sure;                                  // ~2 du of all pairs, in range or not
                    ent[cc] = __float_as_uint(q.w);
                }
                if (!__any_sync(kFull, am[0] | am[1] | am[2] | am[3])) {
                    if (ok[0]) append(code[0], ent[0], false);
                    if (ok[1]) append(code[1], ent[1], true);
                    flush_all();
                    if (ok[2]) append(code[2], ent[2], false);
                    if (ok[3]) append(code[3], ent[3], true);
                    flush_all();
                } else {
                    // some pair is within the error margin of a bin edge (~1e-4 of the pairs): exact decision
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) {
                        if (ok[cc]) append(code[cc], ent[cc], cc & 1);
                        else if (am[cc] && code[cc] + 1u < (unsigned)nb + 2u && ent[cc] != kPadEntry) {
                            const unsigned cx = classify_exact<PERIODIC>(a.pos4[ent[cc] & kIdxMask], sp, lane, e2, nb, G.box, G.half, rmin_f, invw_f);
                            if (cx != kNoHit) append(cx, ent[cc], cc & 1);
                        }
                        if (cc & 1) flush_all();
                    }
                }
            }
        } else {
            // group too wide for a common image: every pair is decided exactly
            for (int c = 0; c < nvalid; ++c) {
                const unsigned e = __float_as_uint(cand[(qh + c) & 63].w);
                if (lane < cnt) {
                    const unsigned code = classify_exact<PERIODIC>(a.pos4[e & kIdxMask], sp, lane, e2, nb, G.box, G.half, rmin_f, invw_f);
                    if (code != kNoHit) append(code, e, false);
                }
                flush_all();
            }
        }
        qh = (qh + 32) & 63;
        qn -= nvalid;
        __syncwarp();
    }
    if (lane == 0) atomicAdd(a.cand_pairs, kept * (unsigned long long)cnt);

    // close the open block of every (bin, lane): pad it to 4 entries, flush, and complete the last group of 8
    // (k_harm reads 8 entries at a time); cursors are n_i(b)
    for (int b = 0; b < nb; ++b) {
        const unsigned k = cursor[b * 32 + lane];
        a.counts[((size_t)g * nb + b) * 32 + lane] = k;
        unsigned *blk = ring + ((b << 5) + lane) * 4;
        unsigned nblk4 = k >> 2;
        if (k & 3u) {
            for (unsigned q = k & 3u; q < 4u; ++q) blk[q] = kPadEntry;
            pendA = (int)((nblk4 << 5) | (unsigned)b);
            ++nblk4;
        }
        flush_all();
        if (nblk4 & 1u) {
            for (unsigned q = 0; q < 4u; ++q) blk[q] = kPadEntry;
            pendA = (int)((nblk4 << 5) | (unsigned)b);
        }
        flush_all();
    }
}

// ==========================================================================================================
// k_harm: a4.  One warp per item (group, bin): every lane streams its list, a_lm accumulates in registers.
// ==========================================================================================================
struct Raw { double2 xy, zw; };

// One 256-bit load per candidate (LDG.E.256, sm_100): the gather is one 32-byte sector per lane, and the L1 tag stage
// handles one sector per cycle, so two 128-bit loads of the same sector cost twice the L1 time (the v4 kernel sat at
// 80 % L1 throughput with the FP64 pipe at 60 %).
__device__ __forceinline__ Raw gather(const double4 *__restrict__ pos4, unsigned e)
{
    Raw r;
    // a padding entry reads particle 0 (always valid memory); its contribution is cancelled by weight 0 below
    const double4 *q = pos4 + (e == kPadEntry ? 0u : (e & kIdxMask));
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.xy.x), "=d"(r.xy.y), "=d"(r.zw.x), "=d"(r.zw.y) : "l"(q));
    return r;
}

// MODE 0: open geometry; 1: periodic, image carried by the entry; 2: periodic, image decided per pair
// mtab (MODE 1): shared memory [axis][image code][thread] = x_i + {-L, 0, +L}: x_j - (x_i -/+ L) is the minimal image
// D: candidates gathered ahead of the one being accumulated (2 at 12 warps/SM, 4 in the fat passes at 8 warps/SM)
template <int LMAX, int MLO, int MHI, int MODE, int D>
__device__ __forceinline__ void harm_rows(double (&acc)[ncomp_range(LMAX, MLO, MHI)], const unsigned *__restrict__ pool,
                                          const int *__restrict__ page_next, int page, int nblk_lane, int nblk,
                                          const double4 *__restrict__ pos4, const double4 &me, const double *mtab,
                                          double box, double half)
{
    const uint4 padv = make_uint4(kPadEntry, kPadEntry, kPadEntry, kPadEntry);
    uint4 q0 = padv, q1 = padv;
    int nextp = 0;
    if (nblk_lane > 0) {
        const uint4 *p = reinterpret_cast<const uint4 *>(pool + (size_t)page * ENCORE_PAGE_WORDS);
        q0 = __ldcg(p); q1 = __ldcg(p + 1);
        if (nblk_lane > 8) nextp = page_next[page];
    }
    Raw r[D];
    {
        const unsigned e0[4] = {q0.x, q0.y, q0.z, q0.w};
#pragma unroll
        for (int d = 0; d < D; ++d) r[d] = gather(pos4, e0[d]);
    }
    for (int kb = 0; kb < nblk; ++kb) {
        uint4 n0 = padv, n1 = padv; // entries of block kb+1
        if (kb + 1 < nblk_lane) {
            const bool turn = ((kb + 1) & 7) == 0;
            if (turn) page = nextp;
            const uint4 *p = reinterpret_cast<const uint4 *>(pool + (size_t)page * ENCORE_PAGE_WORDS + (((kb + 1) & 7) << 3));
            n0 = __ldcg(p); n1 = __ldcg(p + 1);
            if (turn && kb + 9 < nblk_lane) nextp = page_next[page];
        }
        const unsigned e[12] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w, n0.x, n0.y, n0.z, n0.w};
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const Raw r0 = r[u % D];
            r[u % D] = gather(pos4, e[u + D]); // D candidates ahead
            const unsigned en = e[u];
            double dx, dy, dz;
            if (MODE == 1) {
                const unsigned kx = (en >> 26) & 3u, ky = (en >> 28) & 3u, kz = en >> 30;
                dx = r0.xy.x - mtab[(0 * 3 + kx) * (kHarmWarps * 32)];
                dy = r0.xy.y - mtab[(1 * 3 + ky) * (kHarmWarps * 32)];
                dz = r0.zw.x - mtab[(2 * 3 + (kz > 2u ? 1u : kz)) * (kHarmWarps * 32)];
            } else {
                dx = sep<MODE == 2>(r0.xy.x, me.x, box, half);
                dy = sep<MODE == 2>(r0.xy.y, me.y, box, half);
                dz = sep<MODE == 2>(r0.zw.x, me.z, box, half);
            }
            const bool pad = en == kPadEntry;
            if (pad) { dx = 1.0; dy = 0.0; dz = 0.0; }
            const double wj = pad ? 0.0 : r0.zw.y;
            const double r2s = fma(dz, dz, fma(dy, dy, dx * dx));
            const double rinv = rsqrt_pair(r2s);
            accumulate<LMAX, MLO, MHI>(acc, dx * rinv, dy * rinv, dz * rinv, wj);
        }
        q0 = n0; q1 = n1;
    }
}

template <int LMAX, int MLO, int MHI, bool PERIODIC>
__global__ void __launch_bounds__(kHarmWarps * 32, ncomp_range(LMAX, MLO, MHI) > ENCORE_HARM_FAT ? 2 : 3) k_harm(PairArgs a, int g0, int g1)
{
    constexpr int NACC = ncomp_range(LMAX, MLO, MHI), D = NACC > ENCORE_HARM_FAT ? ENCORE_HARM_DEPTH_FAT : ENCORE_HARM_DEPTH;
    __shared__ double mtab[PERIODIC ? 9 * kHarmWarps * 32 : 1];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ng = g1 - g0, nb = a.bins.nbins;
    const int item = blockIdx.x * kHarmWarps + warp;
    if (item >= ng * nb) return;
    const int bin = a.bin_order[item / ng], g = g0 + item % ng;
    const Group gr = locate_group<PERIODIC>(a, g);
    const bool active = lane < gr.cnt;
    const double4 me = a.pos4[gr.first + (active ? lane : 0)];
    const size_t col = ((size_t)g * nb + bin) * 32 + lane;
    const unsigned n_mine = active ? a.counts[col] : 0u;
    const int nblk_lane = (int)((n_mine + 7u) >> 3);
    const int nblk = __reduce_max_sync(kFull, nblk_lane);
    const int page = nblk_lane > 0 ? a.first_page[col] : 0;

    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    if (!PERIODIC) harm_rows<LMAX, MLO, MHI, 0, D>(acc, a.pool, a.page_next, page, nblk_lane, nblk, a.pos4, me, nullptr, 0.0, 0.0);
    else if (gr.fast) {
        double *mt = mtab + threadIdx.x;
        const double L = a.geom.box;
        mt[0 * kHarmWarps * 32] = me.x - L; mt[1 * kHarmWarps * 32] = me.x; mt[2 * kHarmWarps * 32] = me.x + L;
        mt[3 * kHarmWarps * 32] = me.y - L; mt[4 * kHarmWarps * 32] = me.y; mt[5 * kHarmWarps * 32] = me.y + L;
        mt[6 * kHarmWarps * 32] = me.z - L; mt[7 * kHarmWarps * 32] = me.z; mt[8 * kHarmWarps * 32] = me.z + L;
        __syncwarp();
        harm_rows<LMAX, MLO, MHI, 1, D>(acc, a.pool, a.page_next, page, nblk_lane, nblk, a.pos4, me, mt, L, a.geom.half);
    } else harm_rows<LMAX, MLO, MHI, 2, D>(acc, a.pool, a.page_next, page, nblk_lane, nblk, a.pos4, me, nullptr, a.geom.box, a.geom.half);

    // epilogue: a_lm = (1/v_b) sum_k ycoef[c][k] S_{m,k}, k = l-m, l-m-2, ... (p_lm has the parity of l-m)
    const double vinv = a.bins.vinv[bin];
    double *out = a.alm + (size_t)g * a.ncomp * nb * 32 + (size_t)bin * 32 + lane;
    int base = 0;
#pragma unroll
    for (int m = MLO; m <= MHI; ++m) {
        const int st = m ? 2 : 1;
#pragma unroll
        for (int l = m; l <= LMAX; ++l) {
            const int cre = m == 0 ? l * l : l * l + 2 * m - 1;
            const double *yc = a.ycoef + (size_t)cre * (LMAX + 1);
            double sr = 0.0, si = 0.0;
#pragma unroll
            for (int q = (l - m) & 1; q <= l - m; q += 2) {
                const double cf = __ldg(yc + q);
                sr = fma(cf, acc[base + q * st], sr);
                if (m) si = fma(cf, acc[base + q * st + 1], si);
            }
            out[(size_t)cre * nb * 32] = active ? sr * vinv : 0.0;
            if (m) out[(size_t)(cre + 1) * nb * 32] = active ? si * vinv : 0.0;
        }
        base += (LMAX - m + 1) * st;
    }
}

template <int LMAX, int MLO, int MHI>
cudaError_t launch_harm(const PairArgs &a, int g0, int g1, cudaStream_t s, int *launches)
{
    const int nitems = (g1 - g0) * a.bins.nbins;
    const int grid = (nitems + kHarmWarps - 1) / kHarmWarps;
    if (a.geom.periodic) k_harm<LMAX, MLO, MHI, true><<<grid, kHarmWarps * 32, 0, s>>>(a, g0, g1);
    else k_harm<LMAX, MLO, MHI, false><<<grid, kHarmWarps * 32, 0, s>>>(a, g0, g1);
    *launches += 1;
    return cudaGetLastError();
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

#define HARM_PASS(L, A, B)                                              \
    {                                                                   \
        cudaError_t e = launch_harm<L, A, B>(a, g0, g1, s, launches);   \
        if (e != cudaSuccess) return e;                                 \
    }

// m-ranges per lmax.  Every pass re-reads the lists and gathers the candidates again (the L1 data pipe is ~70 % busy),
// so fewer, fatter passes win: up to 44 accumulators run at 168 registers and 12 warps/SM, 45-65 at 255 registers and
// 8 warps/SM (c2, lmax 10: four passes 46.3 ms, three 40.1 ms, two 37.1 ms for the pair stage).
cudaError_t launch_pair_fill_harmonics(const PairArgs &a, int g0, int g1, int nr_cap, cudaStream_t s, int *launches)
{
    const int ng = g1 - g0, nb = a.bins.nbins;
    if (ng <= 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(a.pool_cursor, 0, sizeof(unsigned), s);
    if (e != cudaSuccess) return e;
    const size_t smem = fill_smem_bytes(nb, nr_cap);
    if (a.geom.periodic) {
        e = cudaFuncSetAttribute(k_fill<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        k_fill<true><<<ng, 32, smem, s>>>(a, g0, g1, nr_cap);
    } else {
        e = cudaFuncSetAttribute(k_fill<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        k_fill<false><<<ng, 32, smem, s>>>(a, g0, g1, nr_cap);
    }
    *launches += 1;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
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
