// contract6.cu — step a5 for N = 6, factorised through the two intermediates of eq. 5:
//
//   H^B_Lam(i) = sum_{M >= 0} Re[ T_M(b1,b2,b3) R45_M(b4,b5) ]
//   U_m(b1,b2)    = sum_{m1+m2=m} (l1 l2 l12; m1 m2 -m) a~1 a~2                                       m = 0 .. l12
//   T_M(b1,b2,b3) = f_M sum_{m12+m3=M} (-1)^{l12-m12} (l12 l3 l123; m12 m3 -M) U~_{m12}(b1,b2) a~3(b3)
//   R45_M(b4,b5)  = sum_{m4+m5=-M} (l123 l4 l5; M m4 m5) a~4 a~5
//
// with f_M = sqrt((2 l12+1)(2 l123+1)) (-1)^{l123-M} (2 - delta_M0) and U~_{-m} = (-1)^{l1+l2+l12+m} conj(U_m): the terms M and
// -M of the full sum are E(Lam) times each other's conjugates (App. B), which gives the half-sum.  The literal eq. 44 kernel
// evaluates every (term, bin tuple) product of five factors; here a coupled pair serves all third bins and a coupled triple
// all (b4, b5): ~12 times fewer fp64 operations at lmax = 2, 8 bins.
//
// Two warps per multiplet split the quintuples by the THIRD bin (b3 <= T, b3 > T; T balances the quintuple counts), lane =
// primary.  Per group of 32 primaries a warp (i) evaluates U_m for its pairs (b2 < its largest b3) and all m into a scratch
// area of shared memory (the T terms index U by m12, a run-time index, so it cannot stay in registers), (ii) per M: T for its
// triples and R45 for the pairs above its smallest b3 in registers, then the products into partial sums that stay in
// registers over all groups of the CTA's chunk (as k_contract4/5).  The a_lm tiles arrive through the TMA tile pipeline.
#include "contract_tile.cuh"

#include <algorithm>
#include <mutex>
#include <vector>

namespace {

constexpr int kWarps6 = 8;      // work units (multiplet, warp role) per CTA (255 registers)

__host__ __device__ constexpr int tup6(int nb, int b3) { return c2(b3) * c2(nb - 1 - b3); }   // quintuples with third bin b3
// third bins 2 .. T go to warp 0, T+1 .. NB-3 to warp 1
__host__ __device__ constexpr int t6(int nb)
{
    int best = 2, cost = 1 << 30;
    for (int t = 2; t <= nb - 3; ++t) {
        int a = 0, b = 0;
        for (int b3 = 2; b3 <= nb - 3; ++b3) (b3 <= t ? a : b) += tup6(nb, b3);
        const int m = a > b ? a : b;
        if (m < cost) { cost = m; best = t; }
    }
    return best;
}
// Up to 8 bins: two warp roles per multiplet, third bins 2..T and T+1..NB-3.  9 and 10 bins (126 / 252 quintuples): contiguous
// ranges grown greedily while partial sums + T + R45 + the pre-weighted operands of a term stay under 110 doubles
// (4 and 6 roles).
__host__ __device__ constexpr int regs6(int nb, int lo, int hi)
{
    int acc = 0, nt = 0;
    for (int b = lo; b <= hi; ++b) { acc += tup6(nb, b); nt += c2(b); }
    int ny = nb - 2 - lo;
    if (hi - lo + 1 > ny) ny = hi - lo + 1;
    if (hi - 1 > ny) ny = hi - 1;
    return acc + 2 * nt + 2 * c2(nb - 1 - lo) + 4 * ny;
}
constexpr int kMaxRoles6 = 8;
struct Part6 { int n; int lo[kMaxRoles6], hi[kMaxRoles6]; };
__host__ __device__ constexpr Part6 make_part6(int nb)
{
    Part6 p{};
    for (int w = 0; w < kMaxRoles6; ++w) { p.lo[w] = 3; p.hi[w] = 2; }
    if (nb <= 8) {
        p.n = 2;
        p.lo[0] = 2; p.hi[0] = t6(nb); p.lo[1] = t6(nb) + 1; p.hi[1] = nb - 3;
        return p;
    }
    int lo = 2, w = 0;
    while (lo <= nb - 3 && w < kMaxRoles6) {
        int hi = lo;
        while (hi + 1 <= nb - 3 && regs6(nb, lo, hi + 1) <= 110) ++hi;
        p.lo[w] = lo; p.hi[w] = hi;
        lo = hi + 1; ++w;
    }
    p.n = w;
    return p;
}
__host__ __device__ constexpr int nw6(int nb) { return make_part6(nb).n; }
__host__ __device__ constexpr int lo6(int nb, int w) { return make_part6(nb).lo[w]; }
__host__ __device__ constexpr int hi6(int nb, int w) { return make_part6(nb).hi[w]; }

// index spaces of a warp whose third bins are LO..HI
__host__ __device__ constexpr int npu6(int hi) { return hi >= 2 ? c2(hi) : 0; }                       // pairs b1 < b2 <= HI-1
__host__ __device__ constexpr int pu6(int b1, int b2) { return c2(b2) + b1; }
__host__ __device__ constexpr int nt6(int lo, int hi) { int s = 0; for (int b = lo; b <= hi; ++b) s += c2(b); return s; }
__host__ __device__ constexpr int tt6(int lo, int b1, int b2, int b3) { return nt6(lo, b3 - 1) + c2(b2) + b1; }
__host__ __device__ constexpr int npr6(int nb, int lo) { return c2(nb - 1 - lo); }                   // pairs LO+1 <= b4 < b5 <= NB-1
__host__ __device__ constexpr int pr6(int nb, int lo, int b4, int b5)
{
    int s = 0;
    for (int b = lo + 1; b < b4; ++b) s += nb - 1 - b;
    return s + (b5 - b4 - 1);
}
__host__ __device__ constexpr int nacc6(int nb, int lo, int hi) { int s = 0; for (int b = lo; b <= hi; ++b) s += tup6(nb, b); return s > 0 ? s : 1; }
__host__ __device__ constexpr int ai6(int nb, int lo, int b1, int b2, int b3, int b4, int b5)
{
    int s = 0;
    for (int b = lo; b < b3; ++b) s += tup6(nb, b);
    return s + pr6(nb, b3, b4, b5) * c2(b3) + c2(b2) + b1;
}
// doubles of U scratch of warp role w of a multiplet with intermediate l12: [component 2m, 2m+1][pair][lane]
__host__ __device__ constexpr int scratch6(int nb, int w, int l12) { return (l12 + 1) * 2 * npu6(hi6(nb, w)) * 32; }

struct SlotU6 { __host__ __device__ constexpr int operator()(int x, int y) const { return pu6(x, y); } };
template <int NB, int LO>
struct SlotR6 { __host__ __device__ constexpr int operator()(int x, int y) const { return pr6(NB, LO, x, y); } };

// Z(x,y) += sum_t [wrr r_x r_y + wii i_x i_y] + i [wri r_x i_y + wir i_x r_y] for x in X0..X1, y in max(x+1,Y0)..Y1, every operand
// read once per term; SLOT(x, y) is the register slot
template <int NB, int X0, int X1, int Y0, int Y1, class Slot, int NZ>
__device__ __forceinline__ void pair_sums6(double (&zr)[NZ], double (&zi)[NZ], const PairTerm *terms, int t0, int t1, const double *pa,
                                           const double *pb)
{
    constexpr int rs = NB * 32, NY = Y1 - Y0 + 1;
    if constexpr (NY > 0 && X1 >= X0) {
#pragma unroll 1
        for (int t = t0; t < t1; ++t) {
            const PairTerm T = terms[t];
            double u[NY], v[NY], sx[NY], w[NY];
            const double *br = pb + T.ib_re * rs, *bi = pb + T.ib_im * rs;
            static_for<Y0, Y1 + 1>([&](auto Yc) {
                constexpr int y = decltype(Yc)::value;
                const double ry = br[y * 32], iy = bi[y * 32];
                u[y - Y0] = T.wrr * ry; v[y - Y0] = T.wii * iy; sx[y - Y0] = T.wri * iy; w[y - Y0] = T.wir * ry;
            });
            const double *ar = pa + T.ia_re * rs, *ai = pa + T.ia_im * rs;
            static_for<X0, X1 + 1>([&](auto Xc) {
                constexpr int x = decltype(Xc)::value;
                const double rx = ar[x * 32], ix = ai[x * 32];
                static_for<(x + 1 > Y0 ? x + 1 : Y0), Y1 + 1>([&](auto Yc) {
                    constexpr int y = decltype(Yc)::value;
                    constexpr int k = Slot{}(x, y);
                    zr[k] = fma(u[y - Y0], rx, fma(v[y - Y0], ix, zr[k]));
                    zi[k] = fma(sx[y - Y0], rx, fma(w[y - Y0], ix, zi[k]));
                });
            });
        }
    }
}

template <int NB, int LO, int HI, int NACC>
__device__ __forceinline__ void task6(double (&acc)[NACC], const Lam6 &L, const PairTerm *terms, double *scr, const double *p1, const double *p2,
                                      const double *p3, const double *p4, const double *p5, double wi)
{
    if constexpr (LO <= HI && HI <= NB - 3) {
        constexpr int NPU = npu6(HI), NT = nt6(LO, HI), NPR = npr6(NB, LO), NB3 = HI - LO + 1, rs = NB * 32;
        // (i) U_m(b1,b2), b1 < b2 <= HI-1, m = 0 .. l12 -> scratch [2m | 2m+1][pair][lane]
        for (int m = 0; m <= L.l12; ++m) {
            double zr[NPU], zi[NPU];
#pragma unroll
            for (int k = 0; k < NPU; ++k) { zr[k] = 0.0; zi[k] = 0.0; }
            pair_sums6<NB, 0, HI - 2, 1, HI - 1, SlotU6>(zr, zi, terms, L.ubeg[m], L.ubeg[m + 1], p1, p2);
            double *dr = scr + (2 * m) * NPU * 32, *di = dr + NPU * 32;
#pragma unroll
            for (int k = 0; k < NPU; ++k) { dr[k * 32] = zr[k]; di[k * 32] = zi[k]; }
        }
        __syncwarp();
        for (int M = 0; M <= L.l123; ++M) {
            // (ii) T_M(b1,b2,b3), b3 in LO..HI: the a~3 side of a term is pre-weighted, the U pairs are streamed from the scratch
            double tr[NT], ti[NT];
#pragma unroll
            for (int k = 0; k < NT; ++k) { tr[k] = 0.0; ti[k] = 0.0; }
            const int t1 = L.tbeg[M + 1];
#pragma unroll 1
            for (int t = L.tbeg[M]; t < t1; ++t) {
                const PairTerm T = terms[t];
                double u[NB3], v[NB3], sx[NB3], w[NB3];
                const double *br = p3 + T.ib_re * rs, *bi = p3 + T.ib_im * rs;
                static_for<LO, HI + 1>([&](auto B3) {
                    constexpr int b3 = decltype(B3)::value;
                    const double r3 = br[b3 * 32], i3 = bi[b3 * 32];
                    u[b3 - LO] = T.wrr * r3; v[b3 - LO] = T.wii * i3; sx[b3 - LO] = T.wri * i3; w[b3 - LO] = T.wir * r3;
                });
                const double *ur = scr + T.ia_re * NPU * 32, *ui = scr + T.ia_im * NPU * 32;
                static_for<1, HI>([&](auto B2) {
                    constexpr int b2 = decltype(B2)::value;
                    static_for<0, b2>([&](auto B1) {
                        constexpr int b1 = decltype(B1)::value;
                        const double Ur = ur[pu6(b1, b2) * 32], Ui = ui[pu6(b1, b2) * 32];
                        static_for<(b2 + 1 > LO ? b2 + 1 : LO), HI + 1>([&](auto B3) {
                            constexpr int b3 = decltype(B3)::value, k = tt6(LO, b1, b2, b3);
                            tr[k] = fma(u[b3 - LO], Ur, fma(v[b3 - LO], Ui, tr[k]));
                            ti[k] = fma(sx[b3 - LO], Ur, fma(w[b3 - LO], Ui, ti[k]));
                        });
                    });
                });
            }
            const double wti = L.odd ? wi : -wi;    // even: Re[T R] = Tr Rr - Ti Ri;  odd: Im[T R] = Tr Ri + Ti Rr (App. B)
#pragma unroll
            for (int k = 0; k < NT; ++k) { tr[k] *= wi; ti[k] *= wti; }
            // R45_M(b4,b5), LO+1 <= b4 < b5
            double rr[NPR], ri[NPR];
#pragma unroll
            for (int k = 0; k < NPR; ++k) { rr[k] = 0.0; ri[k] = 0.0; }
            pair_sums6<NB, LO + 1, NB - 2, LO + 2, NB - 1, SlotR6<NB, LO>>(rr, ri, terms, L.rbeg[M], L.rbeg[M + 1], p4, p5);
            if (L.odd) {
#pragma unroll
                for (int k = 0; k < NPR; ++k) { const double x = rr[k]; rr[k] = ri[k]; ri[k] = x; }
            }
            static_for<LO, HI + 1>([&](auto B3) {
                constexpr int b3 = decltype(B3)::value;
                static_for<b3 + 1, NB - 1>([&](auto B4) {
                    constexpr int b4 = decltype(B4)::value;
                    static_for<b4 + 1, NB>([&](auto B5) {
                        constexpr int b5 = decltype(B5)::value, k = pr6(NB, LO, b4, b5);
                        static_for<1, b3>([&](auto B2) {
                            constexpr int b2 = decltype(B2)::value;
                            static_for<0, b2>([&](auto B1) {
                                constexpr int b1 = decltype(B1)::value;
                                constexpr int o = ai6(NB, LO, b1, b2, b3, b4, b5), q = tt6(LO, b1, b2, b3);
                                acc[o] = fma(tr[q], rr[k], fma(ti[q], ri[k], acc[o]));
                            });
                        });
                    });
                });
            });
        }
        __syncwarp();   // every lane is done with the scratch before the next group rewrites it
    }
}

template <int NB, int LO, int HI, int NACC>
__device__ __forceinline__ void flush6(const double (&acc)[NACC], const int *tuple_index, double *out, int lane)
{
    static_for<LO, HI + 1>([&](auto B3) {
        constexpr int b3 = decltype(B3)::value;
        static_for<b3 + 1, NB - 1>([&](auto B4) {
            constexpr int b4 = decltype(B4)::value;
            static_for<b4 + 1, NB>([&](auto B5) {
                constexpr int b5 = decltype(B5)::value;
                static_for<1, b3>([&](auto B2) {
                    constexpr int b2 = decltype(B2)::value;
                    static_for<0, b2>([&](auto B1) {
                        constexpr int b1 = decltype(B1)::value;
                        const double v = warp_sum(acc[ai6(NB, LO, b1, b2, b3, b4, b5)]);
                        if (lane == 0) out[tuple_index[(((b1 * NB + b2) * NB + b3) * NB + b4) * NB + b5]] = v;
                    });
                });
            });
        });
    });
}

template <int NB, int W>
__device__ __forceinline__ void warp6(const ContractArgs &a, const CtaPlan &C, const TilePipe &tp, bool have, const Lam6 &L, int iL, int toff, int soff)
{
    constexpr int LO = lo6(NB, W), HI = hi6(NB, W), NACC = nacc6(NB, LO, HI);
    const int lane = threadIdx.x & 31;
    const int o1 = C.off[L.l1] + lane, o2 = C.off[L.l2] + lane, o3 = C.off[L.l3] + lane, o4 = C.off[L.l4] + lane, o5 = C.off[L.l5] + lane;
    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    for_each_group_tile<true>(a, C, tp, [&](int t, int g) {
        if (!have) return;
        const double wi = a.gweights[(size_t)g * 32 + lane];
        task6<NB, LO, HI, NACC>(acc, L, reinterpret_cast<const PairTerm *>(smem_c + toff) - L.ubeg[0], smem_c + soff + lane, smem_c + t + o1, smem_c + t + o2, smem_c + t + o3, smem_c + t + o4,
                                smem_c + t + o5, wi);
    });
    if (!have) return;
    double *out = a.partial + ((size_t)blockIdx.x * a.nLam + iL) * a.nB;
    if constexpr (LO <= HI) flush6<NB, LO, HI, NACC>(acc, a.tuple_index, out, lane);
}

template <int NB, int W>
__device__ __forceinline__ void dispatch6(int role, const ContractArgs &a, const CtaPlan &C, const TilePipe &tp, bool have, const Lam6 &L, int iL, int toff, int soff)
{
    if (role == W) warp6<NB, W>(a, C, tp, have, L, iL, toff, soff);
    else if constexpr (W + 1 < nw6(NB)) dispatch6<NB, W + 1>(role, a, C, tp, have, L, iL, toff, soff);
}

// A CTA holds 8 work units (multiplet, warp role), dealt by decreasing cost so that the warps of a CTA - which advance tile
// by tile together - carry about the same work.  shared memory: [nbuf tile buffers][4 mbarriers (+pad)][term lists of the 8 warps][U scratch of the 8 warps]
template <int NB>
__global__ void __launch_bounds__(kWarps6 * 32, 1) k_contract6(ContractArgs a)
{
    __shared__ CtaPlan C;
    if (threadIdx.x < sizeof(CtaPlan) / sizeof(int)) reinterpret_cast<int *>(&C)[threadIdx.x] = reinterpret_cast<const int *>(a.ctas + blockIdx.y)[threadIdx.x];
    __syncthreads();
    const int warp = threadIdx.x >> 5;
    const int unit = C.lam[warp];
    const bool have = unit >= 0;
    const int iL = have ? unit >> 3 : 0, role = have ? unit & 7 : 0;
    const Lam6 L = a.lam6[iL];
    const TilePipe tp = make_pipe(C);
    const int toff = tp.bar + kBarDoubles + warp * 6 * a.max_terms;           // every warp stages the term lists of its multiplet
    const int soff = tp.bar + kBarDoubles + kWarps6 * 6 * a.max_terms + C.scr[warp];
    if (have) stage_terms(toff, a.pair_terms + L.ubeg[0], L.nterms, threadIdx.x & 31);
    __syncthreads();
    dispatch6<NB, 0>(role, a, C, tp, have, L, iL, toff, soff);
}

constexpr size_t kSmemLimit6 = 224 * 1024;

template <int NB>
cudaError_t launch6(const ContractArgs &a, cudaStream_t s)
{
    static PerDeviceOnce once;
    const cudaError_t attr_err = once.run([] { return cudaFuncSetAttribute(k_contract6<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemLimit6); });
    if (attr_err != cudaSuccess) return attr_err;
    k_contract6<NB><<<dim3(a.nchunk, a.ncta), kWarps6 * 32, a.cta_smem, s>>>(a);
    return cudaGetLastError();
}

} // namespace

int contraction6_supported(int nbins, int lmax) { return nbins >= 5 && nbins <= 10 && lmax >= 0 && lmax <= 4; }

// fp64 instructions of one group of unit (multiplet q, warp role w), the cost the units are sorted and packed by
static double unit_cost6(int nb, const Lam6 &q, int w)
{
    const int lo = lo6(nb, w), hi = hi6(nb, w);
    if (lo > hi || hi > nb - 3) return 0.0;
    const double npu = npu6(hi), nt = nt6(lo, hi), npr = npr6(nb, lo), nb3 = hi - lo + 1;
    double tup = 0;
    for (int b = lo; b <= hi; ++b) tup += tup6(nb, b);
    const double nu = q.ubeg[q.l12 + 1] - q.ubeg[0], ntt = q.tbeg[q.l123 + 1] - q.tbeg[0], nr = q.rbeg[q.l123 + 1] - q.rbeg[0], nM = q.l123 + 1;
    return nu * (4.0 * (hi - 1) + 4.0 * npu + 6.0) + ntt * (4.0 * nb3 + 4.0 * nt + 2.0 * npu + 6.0) + nr * (4.0 * (nb - 2 - lo) + 4.0 * npr + 6.0) +
           nM * (2.0 * tup + 2.0 * nt + 30.0) + 2.0 * npu * (q.l12 + 1);
}

// Deal the work units (multiplet, warp role), heaviest first, to CTAs of 8 warps while the l-blocks of all their multiplets
// and the U scratch of the warps fit the shared memory; returns the dynamic shared memory of the launch (0: the factorised
// kernel does not cover this plan).
size_t contraction_plan_ctas6(const HostTables &T, std::vector<CtaPlan> &ctas)
{
    ctas.clear();
    if (T.order != 6 || !contraction6_supported(T.nbins, T.lmax) || T.lam6.empty()) return 0;
    const int nb = T.nbins, nL = T.nLam();
    const size_t blk = (size_t)nb * 32 * sizeof(double);
    auto scratch_doubles = [&](int w, int l12) {
        switch (nb) {
        case 5: return scratch6(5, w, l12);
        case 6: return scratch6(6, w, l12);
        case 7: return scratch6(7, w, l12);
        case 8: return scratch6(8, w, l12);
        case 9: return scratch6(9, w, l12);
        default: return scratch6(10, w, l12);
        }
    };
    auto tile_bytes = [&](unsigned mask) {
        size_t b = 0;
        for (int l = 0; l <= T.lmax; ++l) if (mask >> l & 1u) b += (size_t)(2 * l + 1) * blk;
        return b;
    };
    size_t max_terms = 1;
    for (const Lam6 &q : T.lam6) max_terms = std::max<size_t>(max_terms, (size_t)q.nterms);
    const size_t fixed = kBarDoubles * sizeof(double) + (size_t)kWarps6 * max_terms * sizeof(PairTerm);
    std::vector<std::pair<double, int>> units;
    for (int iL = 0; iL < nL; ++iL)
        for (int w = 0; w < nw6(nb); ++w) {
            const double c = unit_cost6(nb, T.lam6[iL], w);
            if (c > 0.0) units.push_back({c, 8 * iL + w});
        }
    std::stable_sort(units.begin(), units.end(), [](const std::pair<double, int> &x, const std::pair<double, int> &y) { return x.first > y.first; });
    std::vector<unsigned> masks;
    std::vector<size_t> scr;
    int fill = kWarps6;
    for (const auto &u : units) {
        const Lam6 &q = T.lam6[u.second >> 3];
        const unsigned m = (1u << q.l1) | (1u << q.l2) | (1u << q.l3) | (1u << q.l4) | (1u << q.l5);
        const size_t s = (size_t)scratch_doubles(u.second & 7, q.l12) * sizeof(double);
        if (tile_bytes(m) + fixed + s > kSmemLimit6) { ctas.clear(); return 0; }
        if (fill == kWarps6 || tile_bytes(masks.back() | m) + fixed + scr.back() + s > kSmemLimit6) {
            CtaPlan c{};
            for (int j = 0; j < 12; ++j) c.lam[j] = -1;
            ctas.push_back(c);
            masks.push_back(0u);
            scr.push_back(0);
            fill = 0;
        }
        ctas.back().scr[fill] = (int)(scr.back() / sizeof(double));
        ctas.back().lam[fill++] = u.second;
        masks.back() |= m;
        scr.back() += s;
    }
    size_t smem = 0;
    for (size_t i = 0; i < ctas.size(); ++i) {
        CtaPlan &c = ctas[i];
        int off = 0;
        c.nblk = 0;
        for (int l = 0; l <= ENCORE_MAX_LMAX; ++l) {
            c.off[l] = -1;
            if (l <= T.lmax && (masks[i] >> l & 1u)) { c.bl[c.nblk++] = l; c.off[l] = off; off += (2 * l + 1) * nb * 32; }
        }
        c.tile = off;
        const size_t tb = (size_t)off * sizeof(double), extra = fixed + scr[i];
        c.nbuf = 1;     // as many tile buffers as fit, up to 4 (contract_tile.cuh)
        for (int nbf = 2; nbf <= kMaxTileBufs; ++nbf) if (nbf * tb + extra <= kSmemLimit6) c.nbuf = nbf;
        smem = std::max(smem, c.nbuf * tb + extra);
    }
    return smem;
}

// executed fp64 flops per primary of k_contract6 (FMA = 2)
double contraction6_flops(const HostTables &T)
{
    const int nb = T.nbins;
    double ex = 0.0;
    for (int w = 0; w < nw6(nb); ++w) {
        const int lo = lo6(nb, w), hi = hi6(nb, w);
        if (lo > hi || hi > nb - 3) continue;
        const double npu = npu6(hi), nt = nt6(lo, hi), npr = npr6(nb, lo), nb3 = hi - lo + 1;
        double tup = 0;
        for (int b = lo; b <= hi; ++b) tup += tup6(nb, b);
        for (const Lam6 &q : T.lam6) {
            const double nu = q.ubeg[q.l12 + 1] - q.ubeg[0], ntt = q.tbeg[q.l123 + 1] - q.tbeg[0], nr = q.rbeg[q.l123 + 1] - q.rbeg[0], nM = q.l123 + 1;
            ex += nu * (4.0 * (hi - 1) + 8.0 * npu);            // U: 4 multiplies per second bin, 4 FMA per pair
            ex += ntt * (4.0 * nb3 + 8.0 * nt) + nM * 2.0 * nt;  // T: 4 multiplies per third bin, 4 FMA per triple; times w_i
            ex += nr * (4.0 * (nb - 2 - lo) + 8.0 * npr);        // R45
            ex += nM * 4.0 * tup;                                // products
        }
    }
    return ex;
}

cudaError_t launch_contract6(const ContractArgs &a, cudaStream_t s)
{
    switch (a.nbins) {
    case 5: return launch6<5>(a, s);
    case 6: return launch6<6>(a, s);
    case 7: return launch6<7>(a, s);
    case 8: return launch6<8>(a, s);
    case 9: return launch6<9>(a, s);
    case 10: return launch6<10>(a, s);
    }
    return cudaErrorInvalidValue;
}
