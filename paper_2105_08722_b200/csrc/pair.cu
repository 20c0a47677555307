// pair.cu — steps a3 (neighbour sweep + radial binning) and a4 (a_lm accumulation) of the ENCORE hot path.
//
//   a^b_lm(s_i) = (1/v_b) sum_{j != i} w_j Y_lm((r_j - s_i)^) Theta^b(|r_j - s_i|)          eq. 35
//
// The paper does this on the CPU, histogramming Cartesian monomials with AVX, eight secondaries at a time
// (Alg. 2) and has no GPU version of it.  Design here:
//   * one CTA per group of 32 consecutive cell-sorted primaries of one (iy,iz) pencil; lane = primary,
//     warp = radial bin, so thread (i,b) owns the (lmax+1)^2 real accumulators of a^b_lm(s_i) in REGISTERS:
//     no atomics, no cross-lane reductions, summation order fixed by the candidate order -> deterministic;
//   * candidates = contiguous runs of the sorted array (one per neighbouring pencil, x-range culled against the
//     group's cell range), streamed in chunks of one candidate per thread;
//   * phase A: every thread tests its candidate against the 32 primaries in fp64 exactly as DESIGN.md R8-R10
//     fix it (r^2 = fma(dz,dz,fma(dy,dy,dx*dx)), compare with e_b^2) and writes a one-byte bin code;
//   * phase B: thread (i,b) scans row i of the code table for its bin, appends the hits to a private ring in
//     shared memory and consumes them in lock-step with the other lanes of its warp (all lanes work on the same
//     bin, so their queues fill at the same rate); per hit: unit vector, w (x+iy)^m by complex recurrence,
//     monic associated-Legendre polynomials p_lm(z) = z p_{l-1,m} - gamma_lm p_{l-2,m}, one FMA per component.
//   Normalisation (-1)^m N_lm k_lm / v_b is applied once per (primary, bin) in the epilogue.
#include "device.cuh"

#include <climits>

namespace {

constexpr int kCap = 64;          // ring slots per consumer thread
constexpr int kMaxWarps = 12;     // bins handled per pass
constexpr int kMaxRanges = 1024;
constexpr int kMinBatch = 4;      // do not start a lock-step consume for fewer entries than this
constexpr unsigned kFull = 0xffffffffu;

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

struct Smem {
    double *sp;           // [3][32] primary positions
    double *e2;           // [40] squared bin edges
    int *rng_start;       // [kMaxRanges]
    int *rng_off;         // [kMaxRanges+1]
    unsigned *jidx;       // [C]
    unsigned char *codes; // [32][C+16]
    unsigned *ring;       // [kCap][nthreads]
};

template <int LMAX, int MLO, int MHI, bool PERIODIC>
__global__ void __launch_bounds__(kMaxWarps * 32, 1) k_pair(PairArgs a, int bin0, int nw)
{
    constexpr int NACC = ncomp_range(LMAX, MLO, MHI);
    const int g = blockIdx.x;
    const GridGeom &G = a.geom;
    if (g >= a.group_start[G.npencil]) return;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthreads = nw * 32, C = nthreads, rowlen = C + 16;
    const int bin = bin0 + warp;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem S;
    S.sp = reinterpret_cast<double *>(smem_raw);
    S.e2 = S.sp + 96;
    S.rng_start = reinterpret_cast<int *>(S.sp + 136);
    S.rng_off = S.rng_start + kMaxRanges;
    S.jidx = reinterpret_cast<unsigned *>(S.rng_off + kMaxRanges + 4);
    S.codes = reinterpret_cast<unsigned char *>(S.jidx + C);
    S.ring = reinterpret_cast<unsigned *>(S.codes + 32 * rowlen);

    // ---- the group ------------------------------------------------------------------------------------
    const int ncx = G.nc[0], ncy = G.nc[1], ncz = G.nc[2];
    const int p = find_pencil_of_group(a.group_start, G.npencil, g);
    const int pstart = a.cell_start[p * ncx], pend = a.cell_start[(p + 1) * ncx];
    const int first = pstart + ENCORE_GROUP * (g - a.group_start[p]);
    const int cnt = min(ENCORE_GROUP, pend - first);
    const bool active = lane < cnt;
    const double4 me = a.pos4[first + (active ? lane : 0)];
    if (warp == 0) { S.sp[lane] = me.x; S.sp[32 + lane] = me.y; S.sp[64 + lane] = me.z; }
    if (tid <= a.bins.nbins) S.e2[tid] = a.bins.e2[tid];
    const int gx0 = cell_coord(a.pos4[first].x, G.org[0], G.inv[0], ncx);
    const int gx1 = cell_coord(a.pos4[first + cnt - 1].x, G.org[0], G.inv[0], ncx);
    const int py = p % ncy, pz = p / ncy;

    // ---- candidate ranges: one or two runs of the sorted array per neighbouring pencil ------------------
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
        if (full_y) { cy = iy; const int d = abs(cy - py); dyc = min(d, ncy - d); }
        else {
            cy = py - Ry + iy; dyc = abs(iy - Ry);
            if (PERIODIC) cy = (cy + ncy) % ncy; else ok = ok && cy >= 0 && cy < ncy;
        }
        if (full_z) { cz = iz; const int d = abs(cz - pz); dzc = min(d, ncz - d); }
        else {
            cz = pz - Rz + iz; dzc = abs(iz - Rz);
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
                int lo = gx0 - rx, hi = gx1 + rx; // inclusive x-cell range
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
    const int nchunks = (T + C - 1) / C;
    if (MLO == 0 && bin0 == 0 && tid == 0) atomicAdd(a.cand_pairs, (unsigned long long)T * (unsigned long long)cnt);

    // ---- stream the candidates -----------------------------------------------------------------------
    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    unsigned count = 0;
    int head = 0, tail = 0;
    const unsigned pat = 0x01010101u * (unsigned)bin;
    const int nq = C / 16;
    const uint4 *row = reinterpret_cast<const uint4 *>(S.codes + lane * rowlen);
    const int nb = a.bins.nbins;
    const double e2lo = a.bins.e2[0], e2hi = a.bins.e2[nb];

    for (int ch = 0; ch < nchunks; ++ch) {
        // -- phase A: bin code of (primary i, this thread's candidate) for all i ---------------------------
        {
            const int s = ch * C + tid;
            const bool valid = s < T;
            double4 cj = make_double4(0, 0, 0, 0);
            unsigned j = 0;
            if (valid) {
                int lo = 0, hi = nr; // rng_off[lo] <= s < rng_off[hi]
                while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (S.rng_off[mid] <= s) lo = mid; else hi = mid; }
                j = (unsigned)(S.rng_start[lo] + (s - S.rng_off[lo]));
                cj = a.pos4[j];
                S.jidx[tid] = j;
            }
            for (int i = 0; i < cnt; ++i) {
                unsigned char code = 255;
                if (valid && j != (unsigned)(first + i)) {
                    const double dx = sep<PERIODIC>(cj.x, S.sp[i], G.box, G.half);
                    const double dy = sep<PERIODIC>(cj.y, S.sp[32 + i], G.box, G.half);
                    const double dz = sep<PERIODIC>(cj.z, S.sp[64 + i], G.box, G.half);
                    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    if (r2 > 0.0 && r2 >= e2lo && r2 < e2hi) { // DESIGN.md R8
                        int b = (int)((sqrtf((float)r2) - a.bins.rmin_f) * a.bins.invw_f);
                        b = max(0, min(nb - 1, b));
                        while (r2 < S.e2[b]) --b;               // DESIGN.md R9: the decision is on squares, fp64
                        while (!(r2 < S.e2[b + 1])) ++b;
                        code = (unsigned char)b;
                    }
                }
                S.codes[i * rowlen + tid] = code;
            }
        }
        __syncthreads();

        // -- phase B: gather my bin's hits into my ring, consume in lock-step with my warp -------------
        const bool last = ch == nchunks - 1;
        int q = 0;
        for (;;) {
            if (active) {
                while (q < nq && tail - head <= kCap - 16) {
                    const uint4 v = row[q];
                    const unsigned wds[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                    for (int wi = 0; wi < 4; ++wi) {
                        unsigned m = __vcmpeq4(wds[wi], pat);
                        while (m) {
                            const int byte = (__ffs(m) - 1) >> 3;
                            S.ring[(tail & (kCap - 1)) * nthreads + tid] = S.jidx[q * 16 + wi * 4 + byte];
                            ++tail;
                            m &= ~(0xffu << (8 * byte));
                        }
                    }
                    ++q;
                }
            }
            const bool done = !active || q == nq;
            const bool alldone = __all_sync(kFull, done);
            const int avail = tail - head;
            const int K = __reduce_min_sync(kFull, active ? avail : INT_MAX);
            int n;
            if (!active) n = 0;
            else if (alldone) n = last ? avail : (K >= kMinBatch ? K : 0);
            else n = max(K, avail - kCap / 2);
            const int nmax = __reduce_max_sync(kFull, n);
            if (nmax > 0) {
                double4 nxt;
                if (0 < n) nxt = a.pos4[S.ring[(head & (kCap - 1)) * nthreads + tid]];
                else nxt = make_double4(me.x + 1.0, me.y, me.z, 0.0);
                for (int k = 0; k < nmax; ++k) {
                    const double4 cj = nxt;
                    if (k + 1 < nmax) {
                        if (k + 1 < n) nxt = a.pos4[S.ring[((head + k + 1) & (kCap - 1)) * nthreads + tid]];
                        else nxt = make_double4(me.x + 1.0, me.y, me.z, 0.0); // padding entry: weight 0
                    }
                    const double dx = sep<PERIODIC>(cj.x, me.x, G.box, G.half);
                    const double dy = sep<PERIODIC>(cj.y, me.y, G.box, G.half);
                    const double dz = sep<PERIODIC>(cj.z, me.z, G.box, G.half);
                    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    const double rinv = rsqrt(r2);
                    accumulate<LMAX, MLO, MHI>(acc, dx * rinv, dy * rinv, dz * rinv, cj.w);
                }
                head += n;
                count += (unsigned)n;
            }
            if (alldone) break;
        }
        __syncthreads();
    }

    // ---- epilogue: normalise and store the tile column of (primary lane, bin) --------------------------
    if (bin < nb) {
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
        if (MLO == 0) a.counts[((size_t)g * nb + bin) * 32 + lane] = active ? count : 0u;
    }
}

size_t pair_smem_bytes(int nw)
{
    const int C = nw * 32;
    return 136 * sizeof(double) + (2 * kMaxRanges + 4) * sizeof(int) + (size_t)C * 4 + 32 * (size_t)(C + 16) +
           (size_t)kCap * C * 4;
}

template <int LMAX, int MLO, int MHI>
cudaError_t launch_one(const PairArgs &a, cudaStream_t s, int *launches)
{
    const int nb = a.bins.nbins;
    for (int bin0 = 0; bin0 < nb; bin0 += kMaxWarps) {
        const int nw = min(kMaxWarps, nb - bin0);
        const size_t smem = pair_smem_bytes(nw);
        cudaError_t e;
        if (a.geom.periodic) {
            e = cudaFuncSetAttribute(k_pair<LMAX, MLO, MHI, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            k_pair<LMAX, MLO, MHI, true><<<a.ngroups_max, nw * 32, smem, s>>>(a, bin0, nw);
        } else {
            e = cudaFuncSetAttribute(k_pair<LMAX, MLO, MHI, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            k_pair<LMAX, MLO, MHI, false><<<a.ngroups_max, nw * 32, smem, s>>>(a, bin0, nw);
        }
        *launches += 1;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

} // namespace

int pair_stage_supported(int lmax, int nbins)
{
    return lmax >= 0 && lmax <= ENCORE_MAX_LMAX && nbins >= 1 && nbins <= ENCORE_MAX_BINS;
}

#define PAIR_PASS(L, A, B)                                              \
    {                                                                   \
        cudaError_t e = launch_one<L, A, B>(a, s, launches);            \
        if (e != cudaSuccess) return e;                                 \
    }

// m-ranges per lmax keep the register-resident accumulators of one pass at <= 36 doubles
cudaError_t launch_pair_stage(const PairArgs &a, cudaStream_t s, int *launches)
{
    switch (a.lmax) {
    case 0: PAIR_PASS(0, 0, 0) break;
    case 1: PAIR_PASS(1, 0, 1) break;
    case 2: PAIR_PASS(2, 0, 2) break;
    case 3: PAIR_PASS(3, 0, 3) break;
    case 4: PAIR_PASS(4, 0, 4) break;
    case 5: PAIR_PASS(5, 0, 5) break;
    case 6: PAIR_PASS(6, 0, 2) PAIR_PASS(6, 3, 6) break;
    case 7: PAIR_PASS(7, 0, 1) PAIR_PASS(7, 2, 3) PAIR_PASS(7, 4, 7) break;
    case 8: PAIR_PASS(8, 0, 1) PAIR_PASS(8, 2, 3) PAIR_PASS(8, 4, 8) break;
    case 9: PAIR_PASS(9, 0, 1) PAIR_PASS(9, 2, 3) PAIR_PASS(9, 4, 5) PAIR_PASS(9, 6, 9) break;
    case 10: PAIR_PASS(10, 0, 1) PAIR_PASS(10, 2, 3) PAIR_PASS(10, 4, 5) PAIR_PASS(10, 6, 10) break;
    default: return cudaErrorInvalidValue;
    }
    return cudaSuccess;
}
