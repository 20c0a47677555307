// pair.cu — steps a3 (neighbour sweep + radial binning) and a4 (a_lm accumulation) of the ENCORE hot path.
//
//   a^b_lm(s_i) = (1/v_b) sum_{j != i} w_j Y_lm((r_j - s_i)^) Theta^b(|r_j - s_i|)          eq. 35
//
// The paper does this on the CPU, histogramming Cartesian monomials with AVX, eight secondaries at a time
// (Alg. 2) and has no GPU version of it.  Design here:
// the work is split by resource profile into three kernels around "groups" of 32 consecutive cell-sorted
// primaries of one (iy,iz) pencil (lane = primary everywhere):
//   k_bin<COUNT>  (a3, integer/fp32, few registers, high occupancy): candidates = contiguous runs of the sorted
//     array (one per neighbouring pencil, x-range culled against the group's cell range); lane = candidate, loop
//     over the 32 primaries.  A first fp32 evaluation on coordinates relative to the group decides every pair
//     whose radius is farther than a proven error margin from all bin edges; the rest (~1e-4) is decided in fp64
//     exactly as DESIGN.md R8-R10 fix it (r^2 = fma(dz,dz,fma(dy,dy,dx*dx)) against e_b^2), so counts are
//     bit-exact.  __match_any_sync turns the 32 codes of a warp step into one hit mask per (primary, bin).
//     Output: n_i(b), the per-(primary, bin) pair counts (an integer output of the path), which also size
//   k_bin<FILL>   (a3 again, same tests): thread (i,b) pops the set bits of its masks, in candidate order, into
//     the candidate list of item (group, b) in HBM: rows of 32 lanes, 4 bytes per accepted pair.
//   k_harm        (a4, fp64, ~140 registers): one warp per item streams its rows (coalesced), gathers the
//     candidates, and thread (i,b) keeps the (lmax+1)^2 real accumulators of a^b_lm(s_i) in REGISTERS: no
//     atomics, no cross-lane reductions, summation order = candidate order -> deterministic.  Per pair: unit
//     vector, w (x+iy)^m by complex recurrence, monic associated-Legendre polynomials
//     p_lm(z) = z p_{l-1,m} - gamma_lm p_{l-2,m}, one FMA per component; normalisation (-1)^m N_lm k_lm / v_b once
//     per (primary, bin) in the epilogue.  Items are ordered heaviest bin first so the grid drains evenly.
#include "device.cuh"

#include <algorithm>
#include <climits>

namespace {

constexpr int kBinWarps = 8;        // k_bin: warps per CTA
constexpr int kCandPerThread = 2;   // k_bin: candidates per thread and chunk
constexpr int kNWord = kBinWarps * kCandPerThread;      // 32-candidate words per chunk
constexpr int kChunk = kNWord * 32;
constexpr int kMaxRanges = 1024;
constexpr int kHarmWarps = 4;       // k_harm: independent warps (items) per CTA
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kNoHit = 254u;
constexpr unsigned kPadEntry = 0xffffffffu;
constexpr unsigned kIdxMask = 0x3ffffffu;

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

// acc[] order: m ascending, l ascending, (re, im)
template <int LMAX, int MLO, int MHI>
__device__ __forceinline__ void accumulate(double (&acc)[ncomp_range(LMAX, MLO, MHI)], double x, double y, double z,
                                           double w)
{
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
            double pm2 = 1.0, pm1 = z;
#pragma unroll
            for (int l = m; l <= LMAX; ++l) {
                double p;
                if (l == m) p = 1.0;
                else if (l == m + 1) p = z;
                else {
                    // monic recurrence: gamma_lm = ((l-1)^2 - m^2) / (4 (l-1)^2 - 1)
                    const double gam = (double)((l - 1) * (l - 1) - m * m) / (double)(4 * (l - 1) * (l - 1) - 1);
                    p = fma(z, pm1, -(gam * pm2));
                    pm2 = pm1; pm1 = p;
                }
                if (l == m) { acc[k] += c; if (m) acc[k + 1] += s; }
                else { acc[k] = fma(p, c, acc[k]); if (m) acc[k + 1] = fma(p, s, acc[k + 1]); }
                k += m ? 2 : 1;
            }
        }
    }
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

// ---- the group of a CTA / warp ---------------------------------------------------------------------------
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

// ==========================================================================================================
// k_bin: a3.  COUNT: counts[g][b][lane].  FILL: candidate lists.
// ==========================================================================================================
struct BinSmem {
    double sp[96];                 // [3][32] primary positions (exact)
    double e2[ENCORE_MAX_BINS + 2];
    float4 cand4[kChunk];          // candidates of the chunk relative to primary 0, fp32
    int rng_start[kMaxRanges];
    int rng_off[kMaxRanges + 4];
    unsigned jidx[kChunk];         // sorted index | image codes << 26
};

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

template <bool PERIODIC, bool FILL>
__global__ void __launch_bounds__(kBinWarps * 32) k_bin(PairArgs a, int g0, int g1)
{
    const int g = g0 + blockIdx.x;
    const GridGeom &G = a.geom;
    if (g >= g1 || g >= a.group_start[G.npencil]) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nb = a.bins.nbins;
    constexpr int nthreads = kBinWarps * 32;

    __shared__ BinSmem S;
    extern __shared__ __align__(16) unsigned hm[]; // FILL: [nb][kNWord][32] hit masks of the current chunk

    const Group gr = locate_group<PERIODIC>(a, g);
    const int first = gr.first, cnt = gr.cnt;
    const double4 ctr = a.pos4[first];
    if (warp == 0) {
        const double4 me = a.pos4[first + (lane < cnt ? lane : 0)];
        S.sp[lane] = me.x; S.sp[32 + lane] = me.y; S.sp[64 + lane] = me.z;
        if (!FILL) a.gweights[(size_t)g * 32 + lane] = lane < cnt ? me.w : 0.0;
    }
    if (tid <= nb) S.e2[tid] = a.bins.e2[tid];
    // this lane's primary, relative to primary 0, fp32 (lanes beyond the group sit far away: never a hit)
    const double4 mine = a.pos4[first + (lane < cnt ? lane : 0)];
    const float pxf = lane < cnt ? (float)(mine.x - ctr.x) : -1e18f, pyf = (float)(mine.y - ctr.y), pzf = (float)(mine.z - ctr.z);
    // COUNT: per-warp private counters [warp][bin][lane] in dynamic shared memory
    int *wcnt = reinterpret_cast<int *>(hm) + warp * nb * 32;
    if (!FILL) for (int b = 0; b < nb; ++b) wcnt[b * 32 + lane] = 0;

    // ---- candidate ranges: one or two runs of the sorted array per neighbouring pencil ------------------
    const int ncx = G.nc[0], ncy = G.nc[1], ncz = G.nc[2];
    int Ry = (int)floor(a.rmax * G.inv[1] + 1e-6) + 1, Rz = (int)floor(a.rmax * G.inv[2] + 1e-6) + 1;
    if (!PERIODIC) { Ry = min(Ry, ncy - 1); Rz = min(Rz, ncz - 1); } // nothing beyond the grid
    const bool full_y = PERIODIC && (2 * Ry + 1 >= ncy), full_z = PERIODIC && (2 * Rz + 1 >= ncz);
    const int wy = full_y ? ncy : 2 * Ry + 1, wz = full_z ? ncz : 2 * Rz + 1;
    const int nyz = wy * wz; // host guarantees 2*nyz <= kMaxRanges
    const double rmax2 = a.rmax * a.rmax;
    for (int r = tid; r < nyz; r += nthreads) {
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
        S.rng_start[2 * r] = s0; S.rng_off[2 * r + 1] = l0;       // lengths parked in rng_off[.+1], scanned below
        S.rng_start[2 * r + 1] = s1; S.rng_off[2 * r + 2] = l1;
    }
    __syncthreads();
    const int nr = 2 * nyz;
    if (warp == 0) { // inclusive scan of the lengths into offsets
        const int per = (nr + 31) / 32;
        const int b0 = lane * per, b1 = min(nr, b0 + per);
        int sum = 0;
        for (int r = b0; r < b1; ++r) sum += S.rng_off[r + 1];
        int x = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { int y = __shfl_up_sync(kFull, x, d); if (lane >= d) x += y; }
        int run = x - sum;
        for (int r = b0; r < b1; ++r) { const int len = S.rng_off[r + 1]; run += len; S.rng_off[r + 1] = run; }
        if (lane == 0) S.rng_off[0] = 0;
    }
    __syncthreads();
    const int T = S.rng_off[nr];
    const int nchunks = (T + kChunk - 1) / kChunk;
    if (!FILL && tid == 0) atomicAdd(a.cand_pairs, (unsigned long long)T * (unsigned long long)cnt);

    // fp32 screening constants: the bin coordinate u = (r - r_min)/width computed in fp32 is within
    // du = [2^-18 (r + r_min) + 2^-19 E^2 / r] / width + 2^-20 |u| of the exact one (E^2 = sum of squared group
    // extents).  For r <= 2 r_max the r-dependent part is bounded by the constant duc; beyond, u - du >= N_r trivially.
    const float rmin_f = a.bins.rmin_f, invw_f = a.bins.invw_f;
    const float c0 = -rmin_f * invw_f;
    const float nb_f = (float)nb;
    const float duc = 3.814697265625e-06f * invw_f * (2.f * (float)a.rmax + rmin_f) + 9.5367431640625e-07f * (2.f * nb_f + 2.f);
    const float kB = 1.9073486328125e-06f * invw_f *
                     (float)(gr.ext[0] * gr.ext[0] + gr.ext[1] * gr.ext[1] + gr.ext[2] * gr.ext[2]);
    const bool fast = gr.fast;

    // FILL: list cursor of (primary lane, bin) for the bins this thread owns: b = warp, warp + 8, ...
    // list layout of an item: blocks of 8 rows, [block][lane][8] (a lane's 8 entries are one 32-byte sector)
    constexpr int kOwn = (ENCORE_MAX_BINS + kBinWarps - 1) / kBinWarps;
    int kk[kOwn];
    size_t base[kOwn];
    int rows[kOwn];
    unsigned *stg = hm + nb * kNWord * 32; // [nb][8][32] staging of the open block of every (bin, lane)
    if (FILL) {
        const int ng = g1 - g0;
#pragma unroll
        for (int sI = 0; sI < kOwn; ++sI) {
            const int b = warp + sI * kBinWarps;
            kk[sI] = 0; base[sI] = 0; rows[sI] = 0;
            if (b < nb) {
                int rank = 0;
                for (int q = 0; q < nb; ++q) if (a.bin_order[q] == b) rank = q;
                const int item = rank * ng + (g - g0);
                base[sI] = (size_t)a.item_off[item] * 32 + (size_t)lane * 8;
                rows[sI] = a.item_rows[item];
            }
        }
    }
    auto flush_block = [&](int b, size_t dst) { // stg[b][0..7][lane] -> 32 bytes at list[dst]
        const unsigned *sp = stg + (b * 8) * 32 + lane;
        const uint4 v0 = make_uint4(sp[0], sp[32], sp[64], sp[96]);
        const uint4 v1 = make_uint4(sp[128], sp[160], sp[192], sp[224]);
        uint4 *d = reinterpret_cast<uint4 *>(a.list + dst);
        __stcs(d, v0);
        __stcs(d + 1, v1);
    };

    for (int ch = 0; ch < nchunks; ++ch) {
        // -- phase A: every warp stages two words of 32 candidates (fp32, relative to primary 0) and then walks
        //    through them with lane = primary: the bin of (primary lane, candidate c) lands in lane-private state,
        //    a hit mask per (bin, word) in FILL and a counter per bin in COUNT; no votes, no atomics -------------
#pragma unroll 1
        for (int u = 0; u < kCandPerThread; ++u) {
            const int wd = u * kBinWarps + warp;   // word of this chunk handled by this warp
            const int slot = wd * 32 + lane;
            const int s = ch * kChunk + slot;
            float4 cf = make_float4(1e18f, 1e18f, 1e18f, 0.f); // beyond the candidate list: never a hit
            unsigned packed = kPadEntry;
            if (s < T) {
                int lo = 0, hi = nr; // rng_off[lo] <= s < rng_off[hi]
                while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (S.rng_off[mid] <= s) lo = mid; else hi = mid; }
                const unsigned j = (unsigned)(S.rng_start[lo] + (s - S.rng_off[lo]));
                const double4 cj = a.pos4[j];
                double rx = cj.x - ctr.x, ry = cj.y - ctr.y, rz = cj.z - ctr.z;
                unsigned kx = 1, ky = 1, kz = 1;  // image code: the list consumer adds {+L, 0, -L}[code] to x_j
                if (PERIODIC) {
                    if (rx > G.half) { rx -= G.box; kx = 2; } else if (rx < -G.half) { rx += G.box; kx = 0; }
                    if (ry > G.half) { ry -= G.box; ky = 2; } else if (ry < -G.half) { ry += G.box; ky = 0; }
                    if (rz > G.half) { rz -= G.box; kz = 2; } else if (rz < -G.half) { rz += G.box; kz = 0; }
                }
                cf = make_float4((float)rx, (float)ry, (float)rz, 0.f);
                packed = j | (kx << 26) | (ky << 28) | (kz << 30);
            }
            S.cand4[slot] = cf;
            S.jidx[slot] = packed;
            if (FILL) for (int b = 0; b < nb; ++b) hm[(b * kNWord + wd) * 32 + lane] = 0u;
            __syncwarp();
            const int nvalid = min(32, T - (ch * kChunk + wd * 32)); // candidates of this word (<= 0: none)
            if (lane < cnt) {
                unsigned amb = 0u; // candidates whose pair with this primary needs the exact fp64 decision
                if (fast) {
#pragma unroll 8
                    for (int c = 0; c < 32; ++c) {
                        const float4 q = S.cand4[wd * 32 + c];
                        const float dx = q.x - pxf, dy = q.y - pyf, dz = q.z - pzf;
                        const float t = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                        float rinv;
                        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(t));
                        const float uu = fmaf(t * rinv, invw_f, c0);    // NaN for t == 0 -> exact path
                        const float du = fmaf(kB, rinv, duc);
                        const float fl = floorf(uu);
                        const float fr = uu - fl;
                        const bool sure = fr >= du && fr <= 1.f - du;   // farther than du from every bin edge
                        if (!sure && !(uu < -du) && !(uu >= nb_f + du)) amb |= 1u << c;
                        if (sure && uu >= 0.f && uu < nb_f) {
                            const int code = (int)fl;
                            if (FILL) hm[(code * kNWord + wd) * 32 + lane] |= 1u << c;
                            else wcnt[code * 32 + lane] += 1;
                        }
                    }
                } else if (nvalid > 0) amb = nvalid >= 32 ? 0xffffffffu : ((1u << nvalid) - 1u);
                // near a bin edge (~1e-4 of the pairs), or a group too wide for a common image: exact decision
                while (amb) {
                    const int c = __ffs(amb) - 1;
                    amb &= amb - 1;
                    const unsigned j = S.jidx[wd * 32 + c] & kIdxMask;
                    if (j == (unsigned)(first + lane)) continue;
                    const unsigned code = classify_exact<PERIODIC>(a.pos4[j], S.sp, lane, S.e2, nb, G.box, G.half, rmin_f, invw_f);
                    if (code != kNoHit) {
                        if (FILL) hm[(code * kNWord + wd) * 32 + lane] |= 1u << c;
                        else wcnt[code * 32 + lane] += 1;
                    }
                }
            }
        }
        if (FILL) {
            __syncthreads();
            // -- phase B: thread (lane = primary, bin) appends its hits, in candidate order, to its list -------
            if (lane < cnt) {
#pragma unroll
                for (int sI = 0; sI < kOwn; ++sI) {
                    const int b = warp + sI * kBinWarps;
                    if (b < nb) {
                        for (int q = 0; q < kNWord; ++q) {
                            unsigned m = hm[(b * kNWord + q) * 32 + lane];
                            while (m) {
                                const int c = __ffs(m) - 1;
                                m &= m - 1;
                                stg[(b * 8 + (kk[sI] & 7)) * 32 + lane] = S.jidx[q * 32 + c];
                                ++kk[sI];
                                if ((kk[sI] & 7) == 0) flush_block(b, base[sI] + (size_t)(kk[sI] / 8 - 1) * 256);
                            }
                        }
                    }
                }
            }
            __syncthreads();
        }
    }

    if (FILL) {
        // close the open block of every lane and pad the rest of its column
#pragma unroll
        for (int sI = 0; sI < kOwn; ++sI) {
            const int b = warp + sI * kBinWarps;
            if (b < nb) {
                int k = lane < cnt ? kk[sI] : 0;
                if (k & 7) {
                    for (int q = k & 7; q < 8; ++q) stg[(b * 8 + q) * 32 + lane] = kPadEntry;
                    flush_block(b, base[sI] + (size_t)(k / 8) * 256);
                    k = (k + 7) & ~7;
                }
                const uint4 padv = make_uint4(kPadEntry, kPadEntry, kPadEntry, kPadEntry);
                for (; k < rows[sI]; k += 8) {
                    uint4 *d = reinterpret_cast<uint4 *>(a.list + base[sI] + (size_t)(k / 8) * 256);
                    __stcs(d, padv);
                    __stcs(d + 1, padv);
                }
            }
        }
    } else {
        __syncthreads();
        const int *all = reinterpret_cast<const int *>(hm);
        for (int k = tid; k < nb * 32; k += nthreads) {
            int tot = 0;
#pragma unroll
            for (int w = 0; w < kBinWarps; ++w) tot += all[w * nb * 32 + k];
            a.counts[(size_t)g * nb * 32 + k] = (uint32_t)tot;
        }
    }
}

// rows needed by a group: sum over bins of the largest per-lane count
__global__ void k_group_rows(PairArgs a)
{
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= a.ngroups) return;
    const int lane = threadIdx.x & 31, nb = a.bins.nbins;
    int tot = 0;
    if (g < a.group_start[a.geom.npencil])
        for (int b = 0; b < nb; ++b) tot += ((int)__reduce_max_sync(kFull, a.counts[((size_t)g * nb + b) * 32 + lane]) + 7) & ~7;
    if (lane == 0) a.grows[g] = tot;
}

// rows of the items of super-step [g0,g1): item = rank(b) * (g1-g0) + (g-g0)
__global__ void k_item_rows(PairArgs a, int g0, int g1)
{
    const int ng = g1 - g0, nb = a.bins.nbins;
    const int item = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (item >= ng * nb) return;
    const int lane = threadIdx.x & 31;
    const int b = a.bin_order[item / ng], g = g0 + item % ng;
    const unsigned m = __reduce_max_sync(kFull, a.counts[((size_t)g * nb + b) * 32 + lane]);
    if (lane == 0) a.item_rows[item] = ((int)m + 7) & ~7; // whole blocks of 8 rows
}

// ==========================================================================================================
// k_harm: a4.  One warp per item (group, bin): stream the rows, accumulate a_lm in registers.
// ==========================================================================================================
// MODE 0: open geometry; 1: periodic, image carried by the entry; 2: periodic, image decided per pair
template <int MODE>
__device__ __forceinline__ double4 fetch(const double4 *__restrict__ pos4, unsigned e, const double4 &pad, double box)
{
    if (e == kPadEntry) return pad;
    const double2 *q = reinterpret_cast<const double2 *>(pos4 + (e & kIdxMask));
    const double2 xy = __ldg(q), zw = __ldg(q + 1);
    double4 p = make_double4(xy.x, xy.y, zw.x, zw.y);
    if (MODE == 1) { // x_j + {+L, 0, -L}[code]
        const unsigned kx = (e >> 26) & 3u, ky = (e >> 28) & 3u, kz = e >> 30;
        p.x += kx == 1u ? 0.0 : (kx == 0u ? box : -box);
        p.y += ky == 1u ? 0.0 : (ky == 0u ? box : -box);
        p.z += kz == 1u ? 0.0 : (kz == 0u ? box : -box);
    }
    return p;
}

template <int LMAX, int MLO, int MHI, int MODE>
__device__ __forceinline__ void harm_rows(double (&acc)[ncomp_range(LMAX, MLO, MHI)], const uint4 *__restrict__ col,
                                          int nblk, const double4 *__restrict__ pos4, const double4 &me, double box, double half)
{
    // col: this lane's two uint4 of block 0; block kb is 64 uint4 further (32 lanes x 2)
    const double4 pad = make_double4(me.x + 1.0, me.y, me.z, 0.0); // padding entry: unit separation, weight 0
    const uint4 padv = make_uint4(kPadEntry, kPadEntry, kPadEntry, kPadEntry);
    uint4 q0 = nblk > 0 ? __ldcs(col) : padv, q1 = nblk > 0 ? __ldcs(col + 1) : padv;
    double4 p0 = fetch<MODE>(pos4, q0.x, pad, box);
    for (int kb = 0; kb < nblk; ++kb) {
        const unsigned e[8] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w};
        if (kb + 1 < nblk) { q0 = __ldcs(col + (size_t)(kb + 1) * 64); q1 = __ldcs(col + (size_t)(kb + 1) * 64 + 1); }
        else { q0 = padv; q1 = padv; }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const double4 p1 = fetch<MODE>(pos4, u < 7 ? e[u + 1] : q0.x, pad, box); // next candidate, one step ahead
            const double dx = sep<MODE == 2>(p0.x, me.x, box, half);
            const double dy = sep<MODE == 2>(p0.y, me.y, box, half);
            const double dz = sep<MODE == 2>(p0.z, me.z, box, half);
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            const double rinv = rsqrt(r2);
            accumulate<LMAX, MLO, MHI>(acc, dx * rinv, dy * rinv, dz * rinv, p0.w);
            p0 = p1;
        }
    }
}

template <int LMAX, int MLO, int MHI, bool PERIODIC>
__global__ void __launch_bounds__(kHarmWarps * 32) k_harm(PairArgs a, int g0, int g1)
{
    constexpr int NACC = ncomp_range(LMAX, MLO, MHI);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ng = g1 - g0, nb = a.bins.nbins;
    const int item = blockIdx.x * kHarmWarps + warp;
    if (item >= ng * nb) return;
    const int bin = a.bin_order[item / ng], g = g0 + item % ng;
    const int rows = a.item_rows[item] >> 3; // blocks of 8 rows
    const uint4 *col = reinterpret_cast<const uint4 *>(a.list + (size_t)a.item_off[item] * 32) + lane * 2;
    const Group gr = locate_group<PERIODIC>(a, g);
    const bool active = lane < gr.cnt;
    const double4 me = a.pos4[gr.first + (active ? lane : 0)];

    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    if (!PERIODIC) harm_rows<LMAX, MLO, MHI, 0>(acc, col, rows, a.pos4, me, a.geom.box, a.geom.half);
    else if (gr.fast) harm_rows<LMAX, MLO, MHI, 1>(acc, col, rows, a.pos4, me, a.geom.box, a.geom.half);
    else harm_rows<LMAX, MLO, MHI, 2>(acc, col, rows, a.pos4, me, a.geom.box, a.geom.half);

    const double vinv = a.bins.vinv[bin];
    double *out = a.alm + (size_t)g * a.ncomp * nb * 32 + (size_t)bin * 32 + lane;
    int k = 0;
#pragma unroll
    for (int m = MLO; m <= MHI; ++m) {
#pragma unroll
        for (int l = m; l <= LMAX; ++l) {
            const int cre = m == 0 ? l * l : l * l + 2 * m - 1;
            out[(size_t)cre * nb * 32] = active ? acc[k] * (a.ynorm[cre] * vinv) : 0.0;
            if (m) out[(size_t)(cre + 1) * nb * 32] = active ? acc[k + 1] * (a.ynorm[cre + 1] * vinv) : 0.0;
            k += m ? 2 : 1;
        }
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

cudaError_t launch_pair_count(const PairArgs &a, cudaStream_t s, int *launches)
{
    if (a.ngroups <= 0) return cudaSuccess;
    const size_t cnt_bytes = (size_t)kBinWarps * a.bins.nbins * 32 * sizeof(int);
    if (a.geom.periodic) k_bin<true, false><<<a.ngroups, kBinWarps * 32, cnt_bytes, s>>>(a, 0, a.ngroups);
    else k_bin<false, false><<<a.ngroups, kBinWarps * 32, cnt_bytes, s>>>(a, 0, a.ngroups);
    k_group_rows<<<(a.ngroups + 7) / 8, 256, 0, s>>>(a);
    *launches += 2;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return launch_exclusive_scan(a.grows, a.gprefix, a.ngroups, a.scan_tmp, s, launches);
}

#define HARM_PASS(L, A, B)                                              \
    {                                                                   \
        cudaError_t e = launch_harm<L, A, B>(a, g0, g1, s, launches);   \
        if (e != cudaSuccess) return e;                                 \
    }

// m-ranges per lmax keep the register-resident accumulators of one pass at <= 36 doubles
cudaError_t launch_pair_fill_harmonics(const PairArgs &a, int g0, int g1, cudaStream_t s, int *launches)
{
    const int ng = g1 - g0, nb = a.bins.nbins;
    if (ng <= 0) return cudaSuccess;
    const int nitems = ng * nb;
    k_item_rows<<<(nitems + 7) / 8, 256, 0, s>>>(a, g0, g1);
    *launches += 1;
    cudaError_t e = launch_exclusive_scan(a.item_rows, a.item_off, nitems, a.scan_tmp, s, launches);
    if (e != cudaSuccess) return e;
    const size_t hm_bytes = (size_t)nb * (kNWord + 8) * 32 * sizeof(unsigned); // hit masks + staging blocks
    if (a.geom.periodic) {
        e = cudaFuncSetAttribute(k_bin<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)hm_bytes);
        if (e != cudaSuccess) return e;
        k_bin<true, true><<<ng, kBinWarps * 32, hm_bytes, s>>>(a, g0, g1);
    } else {
        e = cudaFuncSetAttribute(k_bin<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)hm_bytes);
        if (e != cudaSuccess) return e;
        k_bin<false, true><<<ng, kBinWarps * 32, hm_bytes, s>>>(a, g0, g1);
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
    case 6: HARM_PASS(6, 0, 2) HARM_PASS(6, 3, 6) break;
    case 7: HARM_PASS(7, 0, 1) HARM_PASS(7, 2, 3) HARM_PASS(7, 4, 7) break;
    case 8: HARM_PASS(8, 0, 1) HARM_PASS(8, 2, 3) HARM_PASS(8, 4, 8) break;
    case 9: HARM_PASS(9, 0, 1) HARM_PASS(9, 2, 3) HARM_PASS(9, 4, 5) HARM_PASS(9, 6, 9) break;
    case 10: HARM_PASS(10, 0, 1) HARM_PASS(10, 2, 3) HARM_PASS(10, 4, 5) HARM_PASS(10, 6, 10) break;
    default: return cudaErrorInvalidValue;
    }
    return cudaSuccess;
}
