// contract.cu — steps a5 (per-primary coupling contraction) and a6 (deterministic reduction over primaries).
//
//   H^B_Lam(i) = sum_{M, m_{N-1} >= 0} 2 S(m_{N-1}) E(Lam) C^Lam_M Re[ prod_k a~^{b_k}_{l_k m_k}(s_i) ]      eq. 44
//   zeta^B_Lam = (1/V) sum_i w_i H^B_Lam(i)                                                                 eq. 34
//
// The paper's CUDA kernels take one thread per (Lam,B) ("GPU-a") or per (Lam,B,M) with atomics ("GPU-b"), are
// launched once per primary and get their a_lm from the CPU.  Here the a_lm tiles of all
// primaries are already in HBM in [group][component][bin][lane] order, so a warp works on 32 primaries at once
// (lane = primary: uniform control flow, fully coalesced operand loads), and the sum over primaries is a fixed
// shuffle tree per warp, a fixed-order sum over groups per segment and a fixed-order sum over segments: no atomics.
#include "contract_tile.cuh"

#include <algorithm>
#include <mutex>
#include <type_traits>
#include <vector>

namespace {

constexpr int kWarps = 8;
// Generic kernel, any N in {3,..,6}: one warp per output (Lam,B) at a time, terms looped (literal eq. 44), complex products in registers.
// One CTA per group of 32 primaries; its a_lm tile ([component][bin][lane], contiguous) is first copied to shared memory
// when it fits (STAGED), otherwise read through the caches.  The term records carry row offsets and the conjugation sign
// as a multiplier (DevTerm), the number of factors NM = N - 1 is a template parameter: the inner loop is two loads, one
// multiply and a complex product per factor, and the partial products of the leading factors a term shares with its
// predecessor (terms are in lexicographic order of their m's) are kept.
extern __shared__ __align__(128) double smem_generic[];
constexpr int kTermChunk = 128;     // terms of a multiplet staged in shared memory at a time (12 kB)

template <bool STAGED, int NM>
__global__ void __launch_bounds__(kWarps * 32) k_contract_generic(ContractArgs a)
{
    const int g = a.g_begin + blockIdx.x;
    if (g >= group_end(a)) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nb = a.nbins;
    const double wi = a.gweights[(size_t)g * 32 + lane];
    const size_t tile_len = (size_t)a.ncomp * nb * 32;
    const double *tbase = a.alm + (size_t)g * tile_len;
    // dynamic shared memory: [term chunk][tile, if staged]
    DevTerm *s_terms = reinterpret_cast<DevTerm *>(smem_generic);
    double *s_tile = smem_generic + kTermChunk * sizeof(DevTerm) / sizeof(double);
    if (STAGED) {
        const double2 *src = reinterpret_cast<const double2 *>(a.alm + (size_t)g * tile_len);
        double2 *dst = reinterpret_cast<double2 *>(s_tile);
        for (int i = threadIdx.x; i < (int)(tile_len / 2); i += kWarps * 32) dst[i] = src[i];
    }
    const int nout = a.nLam * a.nB;
    double *out = a.partial + (size_t)g * nout;

    // the CTA walks the multiplets; the terms of the current one sit in shared memory (a chunk at a time), the warps
    // share out its bin tuples.  out[o] is owned by one warp: a later chunk adds to what the first one wrote.
    for (int iL = blockIdx.y; iL < a.nLam; iL += gridDim.y) {    // (interleaved: heavy and light multiplets mix)
        const int t0 = a.term_start[iL], t1 = a.term_start[iL + 1];
        const bool odd = a.lam_parity[iL] != 0;   // parity-odd multiplet: zeta = i * sum W Im[prod] (App. B)
        for (int c0 = t0; c0 < t1 || c0 == t0; c0 += kTermChunk) {
            const int nt = min(t1, c0 + kTermChunk) - c0;
            __syncthreads();        // the previous chunk has been consumed (and, the first time, the tile is complete)
            {
                const double *src = reinterpret_cast<const double *>(a.terms + c0);
                double *dst = reinterpret_cast<double *>(s_terms);
                for (int i = threadIdx.x; i < nt * (int)(sizeof(DevTerm) / sizeof(double)); i += kWarps * 32) dst[i] = src[i];
            }
            __syncthreads();
            for (int iB = warp; iB < a.nB; iB += kWarps) {
                int fo[NM];                 // offset of row 0 of the tile at the bin of factor k (this lane's primary)
#pragma unroll
                for (int k = 0; k < NM; ++k) fo[k] = a.bin_tuples[iB * NM + k] * 32 + lane;
                double accr = 0.0, acci = 0.0;
                double pr[NM], pi[NM];      // partial products a~_0 .. a~_k of the current term
#pragma unroll
                for (int k = 0; k < NM; ++k) { pr[k] = 0.0; pi[k] = 0.0; }
                auto factor = [&](auto K, const DevTerm &tm) {
                    constexpr int k = decltype(K)::value;
                    const double re = STAGED ? s_tile[fo[k] + tm.off_re[k]] : tbase[fo[k] + tm.off_re[k]];
                    const double im = tm.tau[k] * (STAGED ? s_tile[fo[k] + tm.off_im[k]] : tbase[fo[k] + tm.off_im[k]]);
                    if constexpr (k == 0) { pr[0] = re; pi[0] = im; }
                    else {
                        pr[k] = fma(pr[k - 1], re, -(pi[k - 1] * im));
                        pi[k] = fma(pr[k - 1], im, pi[k - 1] * re);
                    }
                };
                for (int t = 0; t < nt; ++t) {
                    const DevTerm &tm = s_terms[t];
                    // the factors from tm.start on are new (warp-uniform); the first term of a chunk starts from scratch
                    switch (t == 0 ? 0 : tm.start) {
                    case 0: factor(std::integral_constant<int, 0>{}, tm); [[fallthrough]];
                    case 1: if constexpr (NM > 1) factor(std::integral_constant<int, 1>{}, tm); [[fallthrough]];
                    case 2: if constexpr (NM > 2) factor(std::integral_constant<int, 2>{}, tm); [[fallthrough]];
                    case 3: if constexpr (NM > 3) factor(std::integral_constant<int, 3>{}, tm); [[fallthrough]];
                    default: if constexpr (NM > 4) factor(std::integral_constant<int, 4>{}, tm);
                    }
                    accr = fma(tm.W, pr[NM - 1], accr); acci = fma(tm.W, pi[NM - 1], acci);
                }
                double acc = (odd ? acci : accr) * wi;
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(kFull, acc, d);
                const int o = iL * a.nB + iB;
                if (lane == 0) out[o] = c0 == t0 ? acc : out[o] + acc;
            }
        }
    }
}

template <int NM>
cudaError_t launch_generic(const ContractArgs &a, cudaStream_t s)
{
    const size_t tile_bytes = (size_t)a.ncomp * a.nbins * 32 * sizeof(double), term_bytes = kTermChunk * sizeof(DevTerm);
    static_assert(sizeof(DevTerm) % sizeof(double) == 0, "DevTerm is copied by doubles");
    // grid: (group, slice of the multiplet list); enough CTAs for ~8 waves of 148 SMs x 4 CTAs, so that the last wave is short
    const int ng = a.g_end - a.g_begin;
    const int slices = std::max(1, std::min(a.nLam, (8 * 148 * 4 + ng - 1) / ng));
    const dim3 grid(ng, slices);
    if (tile_bytes <= 96 * 1024) {   // at least two CTAs per SM
        static PerDeviceOnce once;
        const cudaError_t attr_err = once.run([] { return cudaFuncSetAttribute(k_contract_generic<true, NM>, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024); });
        if (attr_err != cudaSuccess) return attr_err;
        k_contract_generic<true, NM><<<grid, kWarps * 32, tile_bytes + term_bytes, s>>>(a);
    } else k_contract_generic<false, NM><<<grid, kWarps * 32, term_bytes, s>>>(a);
    return cudaGetLastError();
}

// a6, level 1: segment s sums its groups in index order.  level 2: sums the segments in index order, times 1/V.
__global__ void k_reduce_groups(ContractArgs a)
{
    const int nout = a.nLam * a.nB;
    const int o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= nout) return;
    // rows of `partial`: one per chunk (factorised kernels) or one per group of this call's range
    const int r0 = a.factorised ? 0 : a.g_begin, r1 = a.factorised ? a.nchunk : group_end(a);
    const int s = blockIdx.y;
    const int per = (r1 - r0 + a.nseg - 1) / a.nseg;
    const int g0 = r0 + s * per, g1 = min(r1, g0 + per);
    double sum = 0.0;
    for (int g = g0; g < g1; ++g) sum += a.partial[(size_t)g * nout + o];
    a.partial2[(size_t)s * nout + o] = sum;
}

__global__ void k_reduce_segments(ContractArgs a)
{
    const int nout = a.nLam * a.nB;
    const int o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= nout) return;
    double sum = 0.0;
    for (int s = 0; s < a.nseg; ++s) sum += a.partial2[(size_t)s * nout + o];
    a.zeta_out[o] = sum * a.vinv_total;
}


// ==========================================================================================================
// Factorised contraction.  lane = primary of a 32-group; the a_lm blocks a multiplet needs are
// staged in shared memory as [component][bin][lane]; every warp owns a fixed set of bin tuples of one multiplet
// and keeps their zeta partial sums in registers over all groups of its chunk.
// ==========================================================================================================
// ---- N = 3 ------------------------------------------------------------------------------------------------
// eq. 16 with a_{l,-m} = (-1)^m a*_lm:
//   H_l(b1,b2) = (-1)^l / sqrt(2l+1) [ a_l0(b1) a_l0(b2) + 2 sum_{m>0} Re(a_lm(b1) conj a_lm(b2)) ]
// i.e. a real dot product over the 2l+1 real components of the l-block.  One CTA per (l, chunk of groups), a warp per
// group in turn, lane = primary; the c2(NB) partial sums of the block stay in registers over the warp's groups.  The
// kernel reads every a_lm element exactly once (coalesced 256-byte rows): it is bound by HBM, not by arithmetic.
template <int NB>
__global__ void __launch_bounds__(128) k_contract3(ContractArgs a)
{
    constexpr int NP = c2(NB);
    __shared__ double red[4][NP];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = a.nLam - 1 - (int)blockIdx.x; // heaviest block first
    const int chunk = blockIdx.y;
    double acc[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) acc[p] = 0.0;
    const int g_end = group_end(a);
    for (int g = a.g_begin + chunk * 4 + warp; g < g_end; g += 4 * (int)gridDim.y) {
        const double wi = a.gweights[(size_t)g * 32 + lane];
        const double *tile = a.alm + ((size_t)g * a.ncomp + (size_t)l * l) * NB * 32 + lane;
        for (int c = 0; c <= 2 * l; ++c) {
            const double s = c == 0 ? wi : 2.0 * wi;
            double v[NB], sv[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) { v[b] = tile[((size_t)c * NB + b) * 32]; sv[b] = s * v[b]; }
#pragma unroll
            for (int b2 = 1; b2 < NB; ++b2)
#pragma unroll
                for (int b1 = 0; b1 < b2; ++b1) acc[c2(b2) + b1] = fma(sv[b1], v[b2], acc[c2(b2) + b1]);
        }
    }
    const double cl = ((l & 1) ? -1.0 : 1.0) / sqrt(2.0 * l + 1.0);
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const double t = warp_sum(acc[p]);
        if (lane == 0) red[warp][p] = t;
    }
    __syncthreads();
    double *out = a.partial + ((size_t)chunk * a.nLam + l) * a.nB;
    for (int p = threadIdx.x; p < NP; p += 128) {
        int b2 = 1;
        while (c2(b2 + 1) <= p) ++b2;
        const int b1 = p - c2(b2);
        out[a.tuple_index[b1 * NB + b2]] = cl * (((red[0][p] + red[1][p]) + red[2][p]) + red[3][p]); // fixed order
    }
}

template <int NB>
cudaError_t launch3(const ContractArgs &a, cudaStream_t s)
{
    k_contract3<NB><<<dim3(a.nLam, a.nchunk), 128, 0, s>>>(a);
    return cudaGetLastError();
}

// ---- N = 4 ------------------------------------------------------------------------------------------------
// The first bins b1 = 0 .. NB-3 of a multiplet are dealt to its NW warps in snake order (0,1,..,NW-1,NW-1,..,1,0,0,1,..):
// equal numbers of (b1,b2) pairs per warp.  A warp sweeps ALL its b1 together, so that an operand a~2(b2) or a3(b3)
// read from shared memory is used for every b1 below it: the kernel is bound by shared-memory wavefronts, and this
// cuts the operand loads per term from 2 + 2 (NB-2-b1) per b1 to 2 |set| + 2 (NB-2-min b1).
// acc layout: for the j-th b1 of the set, offset aoff(j), then [c2(b3-b1-1) + (b2-b1-1)] for b1 < b2 < b3.
struct Set4 {
    int n;          // number of b1 in the set
    int b1[8];      // ascending
    int goff[9];    // prefix sums of (NB-2-b1): G_{m3}(b1, b2) slots
    int aoff[9];    // prefix sums of c2(NB-1-b1): partial sums
};
__host__ __device__ constexpr Set4 make_set4(int nb, int nw, int w)
{
    Set4 s{};
    s.n = 0;
    s.goff[0] = 0; s.aoff[0] = 0;
    for (int p = 0; p < nb - 2; ++p) {
        const int r = p / nw, i = p % nw;
        const int owner = (r & 1) ? nw - 1 - i : i;
        if (owner == w) {
            s.b1[s.n] = p;
            s.goff[s.n + 1] = s.goff[s.n] + (nb - 2 - p);
            s.aoff[s.n + 1] = s.aoff[s.n] + c2(nb - 1 - p);
            ++s.n;
        }
    }
    return s;
}

template <int NB, int NW, int W>
__device__ __forceinline__ void task4(double (&acc)[make_set4(NB, NW, W).aoff[make_set4(NB, NW, W).n]], const Lam4 &L,
                                      int toff, int s1, int s2, int s3, double wi)
{
    constexpr Set4 S = make_set4(NB, NW, W);
    constexpr int NS = S.n, NG = S.goff[S.n], BMIN = S.b1[0];
    // s1, s2, s3: offsets (in doubles, lane included) of the l1, l2, l3 blocks inside smem_c; toff: of the term list
    constexpr int rs = NB * 32;
    const double *p1 = smem_c + s1, *p2 = smem_c + s2, *p3 = smem_c + s3;
    const PairTerm *terms = reinterpret_cast<const PairTerm *>(smem_c + toff) - L.tbeg[0];
    {   // m3 = 0: G_0 is real (even) or imaginary (odd) and a_{l3 0} is real: half terms, one real G, one FMA per triple
        double g0[NG];
#pragma unroll
        for (int k = 0; k < NG; ++k) g0[k] = 0.0;
        const int t1 = L.tbeg[1];
#pragma unroll 1
        for (int t = L.tbeg[0]; t < t1; ++t) {
            const PairTerm T = terms[t];
            double u[NS], v[NS];
            const double *ar = p1 + T.ia_re * rs, *ai = p1 + T.ia_im * rs;
            static_for<0, NS>([&](auto J) {
                constexpr int j = decltype(J)::value, b1 = make_set4(NB, NW, W).b1[j];
                u[j] = T.wrr * ar[b1 * 32]; v[j] = T.wii * ai[b1 * 32];
            });
            const double *qr = p2 + T.ib_re * rs, *qi = p2 + T.ib_im * rs;
            static_for<BMIN + 1, NB - 1>([&](auto B2) {
                constexpr int b2 = decltype(B2)::value;
                const double r2 = qr[b2 * 32], i2 = qi[b2 * 32];
                static_for<0, NS>([&](auto J) {
                    constexpr int j = decltype(J)::value, b1 = make_set4(NB, NW, W).b1[j];
                    if constexpr (b2 > b1) {
                        constexpr int k = make_set4(NB, NW, W).goff[j] + b2 - b1 - 1;
                        g0[k] = fma(u[j], r2, fma(v[j], i2, g0[k]));
                    }
                });
            });
        }
        static_for<BMIN + 2, NB>([&](auto B3) {
            constexpr int b3 = decltype(B3)::value;
            const double r3 = wi * p3[b3 * 32];
            static_for<0, NS>([&](auto J) {
                constexpr int j = decltype(J)::value, b1 = make_set4(NB, NW, W).b1[j];
                static_for<b1 + 1, b3>([&](auto B2) {
                    constexpr int b2 = decltype(B2)::value;
                    constexpr int k = make_set4(NB, NW, W).goff[j] + b2 - b1 - 1;
                    constexpr int o = make_set4(NB, NW, W).aoff[j] + c2(b3 - b1 - 1) + (b2 - b1 - 1);
                    acc[o] = fma(g0[k], r3, acc[o]);
                });
            });
        });
    }
    for (int m3 = 1; m3 <= L.l3; ++m3) {
        double gr[NG], gi[NG]; // G_{m3}(b1, b2)
#pragma unroll
        for (int k = 0; k < NG; ++k) { gr[k] = 0.0; gi[k] = 0.0; }
        const int t1 = L.tbeg[m3 + 1];
#pragma unroll 1
        for (int t = L.tbeg[m3]; t < t1; ++t) {
            const PairTerm T = terms[t];
            double u[NS], v[NS], sx[NS], w[NS];
            const double *ar = p1 + T.ia_re * rs, *ai = p1 + T.ia_im * rs;
            static_for<0, NS>([&](auto J) {
                constexpr int j = decltype(J)::value, b1 = make_set4(NB, NW, W).b1[j];
                const double r1 = ar[b1 * 32], i1 = ai[b1 * 32];
                u[j] = T.wrr * r1; v[j] = T.wii * i1; sx[j] = T.wri * r1; w[j] = T.wir * i1;
            });
            const double *qr = p2 + T.ib_re * rs, *qi = p2 + T.ib_im * rs;
            static_for<BMIN + 1, NB - 1>([&](auto B2) {
                constexpr int b2 = decltype(B2)::value;
                const double r2 = qr[b2 * 32], i2 = qi[b2 * 32];
                static_for<0, NS>([&](auto J) {
                    constexpr int j = decltype(J)::value, b1 = make_set4(NB, NW, W).b1[j];
                    if constexpr (b2 > b1) {
                        constexpr int k = make_set4(NB, NW, W).goff[j] + b2 - b1 - 1;
                        gr[k] = fma(u[j], r2, fma(v[j], i2, gr[k]));
                        gi[k] = fma(sx[j], i2, fma(w[j], r2, gi[k]));
                    }
                });
            });
        }
        const int cr = 2 * m3 - 1;
        const double *q3r = p3 + cr * rs, *q3i = p3 + (cr + 1) * rs;
        // even parity: Re[G a3] = Gr Re a3 - Gi Im a3;  odd parity: Im[G a3] = Gr Im a3 + Gi Re a3
        const double *pA = L.odd ? q3i : q3r, *pB = L.odd ? q3r : q3i;
        const double cA = wi, cB = L.odd ? wi : -wi;
        static_for<BMIN + 2, NB>([&](auto B3) {
            constexpr int b3 = decltype(B3)::value;
            const double r3 = cA * pA[b3 * 32], i3 = cB * pB[b3 * 32];
            static_for<0, NS>([&](auto J) {
                constexpr int j = decltype(J)::value, b1 = make_set4(NB, NW, W).b1[j];
                static_for<b1 + 1, b3>([&](auto B2) {
                    constexpr int b2 = decltype(B2)::value;
                    constexpr int k = make_set4(NB, NW, W).goff[j] + b2 - b1 - 1;
                    constexpr int o = make_set4(NB, NW, W).aoff[j] + c2(b3 - b1 - 1) + (b2 - b1 - 1);
                    acc[o] = fma(gr[k], r3, fma(gi[k], i3, acc[o]));
                });
            });
        });
    }
}

template <int NB, int NW, int W>
__device__ __forceinline__ void flush4(const double (&acc)[make_set4(NB, NW, W).aoff[make_set4(NB, NW, W).n]],
                                       const int *tuple_index, double *out, int lane)
{
    constexpr int NS = make_set4(NB, NW, W).n;
    static_for<0, NS>([&](auto J) {
        constexpr int j = decltype(J)::value, b1 = make_set4(NB, NW, W).b1[j];
        static_for<b1 + 2, NB>([&](auto B3) {
            constexpr int b3 = decltype(B3)::value;
            static_for<b1 + 1, b3>([&](auto B2) {
                constexpr int b2 = decltype(B2)::value;
                const double v = warp_sum(acc[make_set4(NB, NW, W).aoff[j] + c2(b3 - b1 - 1) + (b2 - b1 - 1)]);
                if (lane == 0) out[tuple_index[(b1 * NB + b2) * NB + b3]] = v;
            });
        });
    });
}

constexpr int kCtaWarps = 12;
#ifndef ENCORE_NW4_WIDE
#define ENCORE_NW4_WIDE 2     // N = 4, 9-10 bins: warps per multiplet (measured on c3: 4x3 19.4 ms, 3x3 15.0, 4x2 22.8, 2x4 10.9)
#define ENCORE_LPC4_WIDE 4    //                   multiplets per CTA
#endif

// warps per multiplet and multiplets per CTA for the N = 4 kernel
__host__ __device__ constexpr int nw4(int nb) { return nb >= 9 ? ENCORE_NW4_WIDE : (nb - 2 + 1) / 2; }
__host__ __device__ constexpr int lpc4(int nb) { return nb >= 9 ? ENCORE_LPC4_WIDE : kCtaWarps / nw4(nb); }

template <int NB, int NW, int W>
__device__ __forceinline__ void warp4(const ContractArgs &a, const CtaPlan &C, const TilePipe &tp, bool have, const Lam4 &L, int iL, int toff)
{
    constexpr Set4 S = make_set4(NB, NW, W);
    constexpr int NTOT = S.aoff[S.n];
    const int lane = threadIdx.x & 31;
    const int o1 = C.off[L.l1] + lane, o2 = C.off[L.l2] + lane, o3 = C.off[L.l3] + lane;
    double acc[NTOT];
#pragma unroll
    for (int k = 0; k < NTOT; ++k) acc[k] = 0.0;
    for_each_group_tile(a, C, tp, [&](int t, int g) {
        if (!have) return;
        const double wi = a.gweights[(size_t)g * 32 + lane];
        task4<NB, NW, W>(acc, L, toff, t + o1, t + o2, t + o3, wi);
    });
    if (!have) return;
    double *out = a.partial + ((size_t)blockIdx.x * a.nLam + iL) * a.nB;
    flush4<NB, NW, W>(acc, a.tuple_index, out, lane);
}

template <int NB, int NW, int W>
__device__ __forceinline__ void dispatch4(int w, const ContractArgs &a, const CtaPlan &C, const TilePipe &tp, bool have, const Lam4 &L, int iL, int toff)
{
    if (w == W) warp4<NB, NW, W>(a, C, tp, have, L, iL, toff);
    else if constexpr (W + 1 < NW) dispatch4<NB, NW, W + 1>(w, a, C, tp, have, L, iL, toff);
}

// LPC multiplets per CTA, each on NW warps
// registers: the file is split over the 4 SM sub-partitions (16384 each), so 9-12 warps cap a thread at 168 registers
// and up to 8 warps allow 255
template <int NB>
__global__ void __launch_bounds__(nw4(NB) * lpc4(NB) * 32, 1) k_contract4(ContractArgs a)
{
    constexpr int NW = nw4(NB);
    __shared__ CtaPlan C;
    if (threadIdx.x < sizeof(CtaPlan) / sizeof(int)) reinterpret_cast<int *>(&C)[threadIdx.x] = reinterpret_cast<const int *>(a.ctas + blockIdx.y)[threadIdx.x];
    __syncthreads();
    const int warp = threadIdx.x >> 5;
    const int iLs = C.lam[warp / NW];
    const bool have = iLs >= 0;
    const int iL = have ? iLs : 0;
    const Lam4 L = a.lam4[iL];
    const TilePipe tp = make_pipe(C);
    const int toff = tp.bar + kBarDoubles + (warp / NW) * 6 * a.max_terms; // this multiplet's term list in shared memory
    if (have && warp % NW == 0) stage_terms(toff, a.pair_terms + L.tbeg[0], L.nterms, threadIdx.x & 31);
    __syncthreads();
    dispatch4<NB, NW, 0>(warp % NW, a, C, tp, have, L, iL, toff);
}

// ---- N = 5 ------------------------------------------------------------------------------------------------
// H = sum_{M>=0} Re[ Y12_M(b1,b2) R34_M(b3,b4) ] over b1 < b2 < b3 < b4.  Two warps per multiplet split the tuples by
// the second bin: warp A takes b2 <= T, warp B takes b2 > T (T = t5(NB) balances the coupled-pair sums per warp).
//   warp A holds its few Y(b1,b2) (b2 <= T) and streams R(b3,.) one b3 at a time;
//   warp B holds its few R(b3,b4) (b3 >= T+2) and streams Y(.,b2) one b2 at a time.
// Every Y pair is computed once and an R pair at most twice (36 coupled-pair sums per M at 8 bins instead of the 50 of
// a split by b1), and both warps keep 35 partial sums at 8 bins.
__host__ __device__ constexpr int npairs_above(int nb, int b) { return c2(nb - 1 - b); } // pairs b < b3 < b4 <= nb-1
__host__ __device__ constexpr int work5(int nb, int t, int second)
{
    int y = 0;
    if (!second) { for (int b2 = 1; b2 <= t; ++b2) y += b2; return y + npairs_above(nb, 1); }
    for (int b2 = t + 1; b2 <= nb - 3; ++b2) y += b2;
    return y + (t + 1 <= nb - 3 ? npairs_above(nb, t + 1) : 0);
}
__host__ __device__ constexpr int t5(int nb)
{
    int best = 1, cost = 1 << 30;
    for (int t = 1; t <= nb - 3; ++t) {
        const int a = work5(nb, t, 0), b = work5(nb, t, 1), m = a > b ? a : b;
        if (m < cost) { cost = m; best = t; }
    }
    return best;
}
// partial sums of a warp whose second bins are lo..hi: [abase(b2) + pidx(b2; b3, b4) * b2 + b1]
__host__ __device__ constexpr int abase5(int nb, int lo, int b2)
{
    int s = 0;
    for (int b = lo; b < b2; ++b) s += b * npairs_above(nb, b);
    return s;
}
__host__ __device__ constexpr int pidx5(int nb, int b2, int b3, int b4)
{
    int s = 0;
    for (int b = b2 + 1; b < b3; ++b) s += nb - 1 - b;
    return s + (b4 - b3 - 1);
}
__host__ __device__ constexpr int aidx5(int nb, int lo, int b1, int b2, int b3, int b4)
{
    return abase5(nb, lo, b2) + pidx5(nb, b2, b3, b4) * b2 + b1;
}
__host__ __device__ constexpr int ntot5(int nb, int lo, int hi) { const int n = hi >= lo ? abase5(nb, lo, hi + 1) : 0; return n > 0 ? n : 1; }

// Coupled-pair sums  Z(x,y) += sum_t [wrr r_x r_y + wii i_x i_y] + i [wri r_x i_y + wir i_x r_y]  (PairTerm), first
// factor from block pa at bin x, second from block pb at bin y, for the terms [t0, t1).
// fixed first bin X, second bins Y0..Y1: zr[y - Y0]
template <int NB, int X, int Y0, int Y1, int NZ>
__device__ __forceinline__ void pairs_fixed_x(double (&zr)[NZ], double (&zi)[NZ], const PairTerm *terms, int t0, int t1,
                                              const double *pa, const double *pb)
{
    constexpr int rs = NB * 32;
#pragma unroll 1
    for (int t = t0; t < t1; ++t) {
        const PairTerm T = terms[t];
        const double rx = pa[T.ia_re * rs + X * 32], ix = pa[T.ia_im * rs + X * 32];
        const double u = T.wrr * rx, v = T.wii * ix, sx = T.wri * rx, w = T.wir * ix;
        const double *qr = pb + T.ib_re * rs, *qi = pb + T.ib_im * rs;
        static_for<Y0, Y1 + 1>([&](auto Yc) {
            constexpr int y = decltype(Yc)::value;
            const double ry = qr[y * 32], iy = qi[y * 32];
            zr[y - Y0] = fma(u, ry, fma(v, iy, zr[y - Y0]));
            zi[y - Y0] = fma(sx, iy, fma(w, ry, zi[y - Y0]));
        });
    }
}
// fixed second bin Y, first bins X0..X1: zr[x - X0]
template <int NB, int Y, int X0, int X1, int NZ>
__device__ __forceinline__ void pairs_fixed_y(double (&zr)[NZ], double (&zi)[NZ], const PairTerm *terms, int t0, int t1,
                                              const double *pa, const double *pb)
{
    constexpr int rs = NB * 32;
#pragma unroll 1
    for (int t = t0; t < t1; ++t) {
        const PairTerm T = terms[t];
        const double ry = pb[T.ib_re * rs + Y * 32], iy = pb[T.ib_im * rs + Y * 32];
        const double u = T.wrr * ry, v = T.wii * iy, sx = T.wri * iy, w = T.wir * ry;
        const double *qr = pa + T.ia_re * rs, *qi = pa + T.ia_im * rs;
        static_for<X0, X1 + 1>([&](auto Xc) {
            constexpr int x = decltype(Xc)::value;
            const double rx = qr[x * 32], ix = qi[x * 32];
            zr[x - X0] = fma(u, rx, fma(v, ix, zr[x - X0]));
            zi[x - X0] = fma(sx, rx, fma(w, ix, zi[x - X0]));
        });
    }
}
// block of pairs x in X0..X1, y in Y0..Y1, x < y, all swept together (each operand is read once per term);
// KIND 0: slot = c2(y) - c2(Y0) + x (pairs (b1,b2) by b2);  KIND 1: slot = sum_{b=X0}^{x-1} (NB-1-b) + y-x-1 (pairs (b3,b4) by b3)
template <int NB, int KIND, int X0, int Y0>
__host__ __device__ constexpr int slot5(int x, int y)
{
    if (KIND == 0) return c2(y) - c2(Y0) + x;
    int s = 0;
    for (int b = X0; b < x; ++b) s += NB - 1 - b;
    return s + (y - x - 1);
}
template <int NB, int KIND, int X0, int X1, int Y0, int Y1, int NZ>
__device__ __forceinline__ void pairs_block(double (&zr)[NZ], double (&zi)[NZ], const PairTerm *terms, int t0, int t1,
                                            const double *pa, const double *pb)
{
    constexpr int rs = NB * 32, NY = Y1 - Y0 + 1;
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
                constexpr int k = slot5<NB, KIND, X0, Y0>(x, y);
                zr[k] = fma(u[y - Y0], rx, fma(v[y - Y0], ix, zr[k]));
                zi[k] = fma(sx[y - Y0], rx, fma(w[y - Y0], ix, zi[k]));
            });
        });
    }
}

// M = 0 ("half terms", tables.cpp): the coupled pair is one real number,  Z(x,y) += wrr A[ia_re](x) B[ib_re](y) + wii A[ia_im](x) B[ib_im](y)
template <int NB, int KIND, int X0, int X1, int Y0, int Y1, int NZ>
__device__ __forceinline__ void pairs_block_half(double (&z)[NZ], const PairTerm *terms, int t0, int t1, const double *pa, const double *pb)
{
    constexpr int rs = NB * 32, NY = Y1 - Y0 + 1;
#pragma unroll 1
    for (int t = t0; t < t1; ++t) {
        const PairTerm T = terms[t];
        double u[NY], v[NY];
        const double *br = pb + T.ib_re * rs, *bi = pb + T.ib_im * rs;
        static_for<Y0, Y1 + 1>([&](auto Yc) {
            constexpr int y = decltype(Yc)::value;
            u[y - Y0] = T.wrr * br[y * 32]; v[y - Y0] = T.wii * bi[y * 32];
        });
        const double *ar = pa + T.ia_re * rs, *ai = pa + T.ia_im * rs;
        static_for<X0, X1 + 1>([&](auto Xc) {
            constexpr int x = decltype(Xc)::value;
            const double rx = ar[x * 32], ix = ai[x * 32];
            static_for<(x + 1 > Y0 ? x + 1 : Y0), Y1 + 1>([&](auto Yc) {
                constexpr int y = decltype(Yc)::value;
                constexpr int k = slot5<NB, KIND, X0, Y0>(x, y);
                z[k] = fma(u[y - Y0], rx, fma(v[y - Y0], ix, z[k]));
            });
        });
    }
}

// ---- how the second bins 1 .. NB-3 of a multiplet are dealt to its warps -----------------------------------
// Up to 8 bins: two warps, b2 <= T and b2 > T (T = t5(NB), measured on c5).  9 and 10 bins: consecutive ranges grown
// greedily while partial sums + held coupled pairs stay under 105 doubles (3 and 5 warps).
#ifndef ENCORE_REGS5
#define ENCORE_REGS5 105
#endif
constexpr int kRegs5 = ENCORE_REGS5;    // doubles a warp role of the N = 5 kernel may hold at 9-10 bins
__host__ __device__ constexpr int regs5(int nb, int lo, int hi)
{
    return ntot5(nb, lo, hi) + 2 * c2(nb - 1 - lo) + 2 * (c2(hi + 1) - c2(lo));
}
__host__ __device__ constexpr int hi5(int nb, int w);
__host__ __device__ constexpr int lo5(int nb, int w)
{
    if (nb <= 8) return w == 0 ? 1 : t5(nb) + 1;
    return w == 0 ? 1 : hi5(nb, w - 1) + 1;
}
__host__ __device__ constexpr int hi5(int nb, int w)
{
    if (nb <= 8) return w == 0 ? t5(nb) : nb - 3;
    const int lo = lo5(nb, w);
    int hi = lo;
    while (hi + 1 <= nb - 3 && regs5(nb, lo, hi + 1) <= kRegs5) ++hi;
    return hi;
}
__host__ __device__ constexpr int nw5(int nb)
{
    if (nb <= 8) return 2;
    int w = 0;
    while (hi5(nb, w) < nb - 3) ++w;
    return w + 1;
}
__host__ __device__ constexpr int lpc5(int nb) { return 8 / nw5(nb); } // multiplets per CTA: at most 8 warps, so that a thread may hold 255 registers

// A warp whose second bins are LO..HI: Y(b1,b2) of its pairs (b2 in LO..HI) and R(b3,b4) of the pairs above LO
// (b3 >= LO+1) are swept whole (every operand and every term read once per M) and held in registers, then the
// products of the warp's tuples are added.
template <int NB, int LO, int HI, int NTOT>
__device__ __forceinline__ void task5(double (&acc)[NTOT], const Lam5 &L, int toff, const double *p1, const double *p2,
                                      const double *p3, const double *p4, double wi)
{
    if constexpr (LO <= HI && HI <= NB - 3) {
        constexpr int NYH = c2(HI + 1) - c2(LO);   // pairs b1 < b2, LO <= b2 <= HI
        constexpr int NRH = c2(NB - 1 - LO);       // pairs LO+1 <= b3 < b4 <= NB-1
        const PairTerm *terms = reinterpret_cast<const PairTerm *>(smem_c + toff) - L.lbeg[0];
        {   // M = 0: Y12_0 and R34_0 are one real number each (half terms), H_0 = Ys Rs: one FMA per quadruple
            double ys[NYH];
#pragma unroll
            for (int k = 0; k < NYH; ++k) ys[k] = 0.0;
            pairs_block_half<NB, 0, 0, HI - 1, LO, HI, NYH>(ys, terms, L.lbeg[0], L.lbeg[1], p1, p2);
#pragma unroll
            for (int k = 0; k < NYH; ++k) ys[k] *= wi;
            double rs0[NRH];
#pragma unroll
            for (int k = 0; k < NRH; ++k) rs0[k] = 0.0;
            pairs_block_half<NB, 1, LO + 1, NB - 2, LO + 2, NB - 1, NRH>(rs0, terms, L.rbeg[0], L.rbeg[1], p3, p4);
            static_for<LO, HI + 1>([&](auto B2) {
                constexpr int b2 = decltype(B2)::value;
                static_for<b2 + 1, NB - 1>([&](auto B3) {
                    constexpr int b3 = decltype(B3)::value;
                    static_for<b3 + 1, NB>([&](auto B4) {
                        constexpr int b4 = decltype(B4)::value;
                        constexpr int k = slot5<NB, 1, LO + 1, LO + 2>(b3, b4);
                        static_for<0, b2>([&](auto B1) {
                            constexpr int b1 = decltype(B1)::value;
                            constexpr int o = aidx5(NB, LO, b1, b2, b3, b4), q = slot5<NB, 0, 0, LO>(b1, b2);
                            acc[o] = fma(ys[q], rs0[k], acc[o]);
                        });
                    });
                });
            });
        }
        for (int M = 1; M <= L.l12; ++M) {
            double yr[NYH], yi[NYH];
#pragma unroll
            for (int k = 0; k < NYH; ++k) { yr[k] = 0.0; yi[k] = 0.0; }
            pairs_block<NB, 0, 0, HI - 1, LO, HI, NYH>(yr, yi, terms, L.lbeg[M], L.lbeg[M + 1], p1, p2);
            const double wyi = L.odd ? wi : -wi;
#pragma unroll
            for (int k = 0; k < NYH; ++k) { yr[k] *= wi; yi[k] *= wyi; } // even: Re[Y R] = Yr Rr - Yi Ri; odd: Im[Y R] = Yr Ri + Yi Rr
            double rr[NRH], ri[NRH];
#pragma unroll
            for (int k = 0; k < NRH; ++k) { rr[k] = 0.0; ri[k] = 0.0; }
            pairs_block<NB, 1, LO + 1, NB - 2, LO + 2, NB - 1, NRH>(rr, ri, terms, L.rbeg[M], L.rbeg[M + 1], p3, p4);
            if (L.odd) {
#pragma unroll
                for (int k = 0; k < NRH; ++k) { const double x = rr[k]; rr[k] = ri[k]; ri[k] = x; }
            }
            static_for<LO, HI + 1>([&](auto B2) {
                constexpr int b2 = decltype(B2)::value;
                static_for<b2 + 1, NB - 1>([&](auto B3) {
                    constexpr int b3 = decltype(B3)::value;
                    static_for<b3 + 1, NB>([&](auto B4) {
                        constexpr int b4 = decltype(B4)::value;
                        constexpr int k = slot5<NB, 1, LO + 1, LO + 2>(b3, b4);
                        static_for<0, b2>([&](auto B1) {
                            constexpr int b1 = decltype(B1)::value;
                            constexpr int o = aidx5(NB, LO, b1, b2, b3, b4), q = slot5<NB, 0, 0, LO>(b1, b2);
                            acc[o] = fma(yr[q], rr[k], fma(yi[q], ri[k], acc[o]));
                        });
                    });
                });
            });
        }
    }
}

// one shuffle tree per tuple of a warp whose second bins are LO..HI
template <int NB, int LO, int HI, int NTOT>
__device__ __forceinline__ void flush5(const double (&acc)[NTOT], const int *tuple_index, double *out, int lane)
{
    static_for<LO, HI + 1>([&](auto B2) {
        constexpr int b2 = decltype(B2)::value;
        static_for<b2 + 1, NB - 1>([&](auto B3) {
            constexpr int b3 = decltype(B3)::value;
            static_for<b3 + 1, NB>([&](auto B4) {
                constexpr int b4 = decltype(B4)::value;
                static_for<0, b2>([&](auto B1) {
                    constexpr int b1 = decltype(B1)::value;
                    const double v = warp_sum(acc[aidx5(NB, LO, b1, b2, b3, b4)]);
                    if (lane == 0) out[tuple_index[((b1 * NB + b2) * NB + b3) * NB + b4]] = v;
                });
            });
        });
    });
}

template <int NB, int W>
__device__ __forceinline__ void warp5(const ContractArgs &a, const CtaPlan &C, const TilePipe &tp, bool have, const Lam5 &L, int iL, int toff)
{
    constexpr int LO = lo5(NB, W), HI = hi5(NB, W), NTOT = ntot5(NB, LO, HI);
    const int lane = threadIdx.x & 31;
    const int o1 = C.off[L.l1] + lane, o2 = C.off[L.l2] + lane, o3 = C.off[L.l3] + lane, o4 = C.off[L.l4] + lane;
    double acc[NTOT];
#pragma unroll
    for (int k = 0; k < NTOT; ++k) acc[k] = 0.0;
    for_each_group_tile(a, C, tp, [&](int t, int g) {
        if (!have) return;
        const double wi = a.gweights[(size_t)g * 32 + lane];
        task5<NB, LO, HI, NTOT>(acc, L, toff, smem_c + t + o1, smem_c + t + o2, smem_c + t + o3, smem_c + t + o4, wi);
    });
    if (!have) return;
    double *out = a.partial + ((size_t)blockIdx.x * a.nLam + iL) * a.nB;
    if constexpr (LO <= HI) flush5<NB, LO, HI, NTOT>(acc, a.tuple_index, out, lane);
}

template <int NB, int W>
__device__ __forceinline__ void dispatch5(int w, const ContractArgs &a, const CtaPlan &C, const TilePipe &tp, bool have, const Lam5 &L, int iL, int toff)
{
    if (w == W) warp5<NB, W>(a, C, tp, have, L, iL, toff);
    else if constexpr (W + 1 < nw5(NB)) dispatch5<NB, W + 1>(w, a, C, tp, have, L, iL, toff);
}

// Up to 8 bins: lpc5 = 4 multiplets per CTA on two warps each.  9 and 10 bins (3 / 5 warp roles per multiplet): the 8 warps of
// a CTA take (multiplet, role) units of up to four consecutive multiplets, so that no warp slot stays empty
// (C.lam[w] = 8 * multiplet + role, C.scr[w] = the term slot of that multiplet, C.lam[8 + s] = multiplet staged in slot s).
__host__ __device__ constexpr int cta_warps5(int nb) { return nb >= 9 ? 8 : nw5(nb) * lpc5(nb); }
template <int NB>
__global__ void __launch_bounds__(cta_warps5(NB) * 32, 1) k_contract5(ContractArgs a)
{
    constexpr int NW = nw5(NB);
    __shared__ CtaPlan C;
    if (threadIdx.x < sizeof(CtaPlan) / sizeof(int)) reinterpret_cast<int *>(&C)[threadIdx.x] = reinterpret_cast<const int *>(a.ctas + blockIdx.y)[threadIdx.x];
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if constexpr (NB >= 9) {
        const int unit = C.lam[warp];
        const bool have = unit >= 0;
        const int iL = have ? unit >> 3 : 0, role = have ? unit & 7 : 0;
        const Lam5 L = a.lam5[iL];
        const TilePipe tp = make_pipe(C);
        const int tbase = tp.bar + kBarDoubles;
        if (warp < 4 && C.lam[8 + warp] >= 0) {
            const Lam5 &S = a.lam5[C.lam[8 + warp]];
            stage_terms(tbase + warp * 6 * a.max_terms, a.pair_terms + S.lbeg[0], S.nterms, lane);
        }
        __syncthreads();
        dispatch5<NB, 0>(role, a, C, tp, have, L, iL, tbase + C.scr[warp] * 6 * a.max_terms);
    } else {
        const int iLs = C.lam[warp / NW];
        const bool have = iLs >= 0;
        const int iL = have ? iLs : 0;
        const Lam5 L = a.lam5[iL];
        const TilePipe tp = make_pipe(C);
        const int toff = tp.bar + kBarDoubles + (warp / NW) * 6 * a.max_terms; // left terms first, right terms behind them (host order)
        if (have && warp % NW == 0) stage_terms(toff, a.pair_terms + L.lbeg[0], L.nterms, lane);
        __syncthreads();
        dispatch5<NB, 0>(warp % NW, a, C, tp, have, L, iL, toff);
    }
}

// ---- host side: multiplets -> CTAs, l-blocks per CTA, shared memory ----------------------------------------------
static int lpc_of(int order, int nb) { return order == 4 ? lpc4(nb) : lpc5(nb); }
static_assert(kCtaWarps <= 12, "CtaPlan::lam has 12 slots");
static constexpr size_t kSmemLimit = 224 * 1024;

template <int NB>
cudaError_t launch4(const ContractArgs &a, cudaStream_t s)
{
    static PerDeviceOnce once;
    const cudaError_t attr_err = once.run([] { return cudaFuncSetAttribute(k_contract4<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemLimit); });
    if (attr_err != cudaSuccess) return attr_err;
    // x = chunk (dispatched fastest), y = CTA plan: the CTAs of the heaviest multiplets all start first and the light ones
    // fill the tail (with the plan index on x, a heavy CTA of the last chunk started late: 8.4 against 6.1 by the cost model)
    k_contract4<NB><<<dim3(a.nchunk, a.ncta), nw4(NB) * lpc4(NB) * 32, a.cta_smem, s>>>(a);
    return cudaGetLastError();
}

template <int NB>
cudaError_t launch5(const ContractArgs &a, cudaStream_t s)
{
    static PerDeviceOnce once;
    const cudaError_t attr_err = once.run([] { return cudaFuncSetAttribute(k_contract5<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemLimit); });
    if (attr_err != cudaSuccess) return attr_err;
    k_contract5<NB><<<dim3(a.nchunk, a.ncta), cta_warps5(NB) * 32, a.cta_smem, s>>>(a);
    return cudaGetLastError();
}

} // namespace

// Factorised kernels cover the bin counts whose per-warp partial sums fit in registers; anything else runs the generic
// kernel (one warp per (Lambda, B), literal eq. 44).
int contraction_split5(int nbins) { return t5(nbins); }
int contraction_warps5(int nbins) { return nw5(nbins); }
void contraction_range5(int nbins, int w, int *lo, int *hi) { *lo = lo5(nbins, w); *hi = hi5(nbins, w); }

int contraction_is_factorised(int order, int nbins, int lmax)
{
    if (order == 3) return nbins >= 2 && nbins <= 10;
    if (order == 4) return nbins >= 3 && nbins <= 10 && lmax <= ENCORE_MAX_LMAX;
    if (order == 5) return nbins >= 4 && nbins <= 10 && lmax <= 5;
    if (order == 6) return contraction6_supported(nbins, lmax);
    return 0;
}

// Deal the multiplets (heaviest first) to CTAs of lpc slots: a CTA takes the next multiplet while the l-blocks of all
// its multiplets still fit one tile buffer; two buffers whenever they fit.  Returns the dynamic shared memory the
// launch needs (0: a single multiplet does not fit).
size_t contraction_plan_ctas(const HostTables &T, std::vector<CtaPlan> &ctas)
{
    ctas.clear();
    if (T.order < 4) return 0;
    const int lpc = lpc_of(T.order, T.nbins), nL = T.nLam();
    size_t max_terms = 1;
    for (const Lam4 &q : T.lam4) max_terms = std::max<size_t>(max_terms, (size_t)q.nterms);
    for (const Lam5 &q : T.lam5) max_terms = std::max<size_t>(max_terms, (size_t)q.nterms);
    const size_t extra = kBarDoubles * sizeof(double) + sizeof(CtaPlan) + (size_t)lpc * max_terms * sizeof(PairTerm);
    const size_t blk = (size_t)T.nbins * 32 * sizeof(double); // bytes of one component of a tile
    auto ls_of = [&](int iL, int *l) {
        if (T.order == 4) { const Lam4 &q = T.lam4[iL]; l[0] = q.l1; l[1] = q.l2; l[2] = q.l3; return 3; }
        const Lam5 &q = T.lam5[iL]; l[0] = q.l1; l[1] = q.l2; l[2] = q.l3; l[3] = q.l4; return 4;
    };
    auto tile_bytes = [&](unsigned mask) {
        size_t b = 0;
        for (int l = 0; l <= T.lmax; ++l) if (mask >> l & 1u) b += (size_t)(2 * l + 1) * blk;
        return b;
    };
    std::vector<unsigned> masks;
    if (T.order == 5 && T.nbins >= 9) {
        // (multiplet, role) units of consecutive multiplets fill the 8 warps of a CTA; at most four multiplets (term slots)
        const int nw = nw5(T.nbins);
        const size_t extra5 = kBarDoubles * sizeof(double) + sizeof(CtaPlan) + (size_t)4 * max_terms * sizeof(PairTerm);
        int fillw = 8, nslots = 0;
        for (int k = 0; k < nL; ++k) {
            const int iL = T.lam_order[k];
            int l[4];
            const int nl = ls_of(iL, l);
            unsigned m = 0;
            for (int j = 0; j < nl; ++j) m |= 1u << l[j];
            if (tile_bytes(m) + extra5 > kSmemLimit) return 0;
            for (int role = 0; role < nw; ++role) {
                bool fresh = ctas.empty() || fillw == 8;
                if (!fresh) {
                    const bool staged = nslots > 0 && ctas.back().lam[8 + nslots - 1] == iL;
                    if ((!staged && nslots == 4) || tile_bytes(masks.back() | m) + extra5 > kSmemLimit) fresh = true;
                }
                if (fresh) {
                    CtaPlan c{};
                    for (int j = 0; j < 12; ++j) c.lam[j] = -1;
                    ctas.push_back(c);
                    masks.push_back(0u);
                    fillw = 0; nslots = 0;
                }
                CtaPlan &c = ctas.back();
                if (nslots == 0 || c.lam[8 + nslots - 1] != iL) c.lam[8 + nslots++] = iL;
                c.scr[fillw] = nslots - 1;
                c.lam[fillw++] = 8 * iL + role;
                masks.back() |= m;
            }
        }
        size_t smem5 = 0;
        for (size_t i = 0; i < ctas.size(); ++i) {
            CtaPlan &c = ctas[i];
            int off = 0;
            c.nblk = 0;
            for (int l = 0; l <= ENCORE_MAX_LMAX; ++l) {
                c.off[l] = -1;
                if (l <= T.lmax && (masks[i] >> l & 1u)) { c.bl[c.nblk++] = l; c.off[l] = off; off += (2 * l + 1) * T.nbins * 32; }
            }
            c.tile = off;
            const size_t tb = (size_t)off * sizeof(double);
            c.nbuf = 2 * tb + extra5 <= kSmemLimit ? 2 : 1;
            smem5 = std::max(smem5, c.nbuf * tb + extra5);
        }
        return smem5;
    }
    int fill = lpc;
    for (int k = 0; k < nL; ++k) {
        const int iL = T.lam_order[k];
        int l[4];
        const int nl = ls_of(iL, l);
        unsigned m = 0;
        for (int j = 0; j < nl; ++j) m |= 1u << l[j];
        if (tile_bytes(m) + extra > kSmemLimit) return 0;
        if (fill == lpc || tile_bytes(masks.back() | m) + extra > kSmemLimit) {
            CtaPlan c{};
            for (int j = 0; j < 12; ++j) c.lam[j] = -1;
            ctas.push_back(c);
            masks.push_back(0u);
            fill = 0;
        }
        ctas.back().lam[fill++] = iL;
        masks.back() |= m;
    }
    size_t smem = 0;
    for (size_t i = 0; i < ctas.size(); ++i) {
        CtaPlan &c = ctas[i];
        int off = 0;
        c.nblk = 0;
        for (int l = 0; l <= ENCORE_MAX_LMAX; ++l) {
            c.off[l] = -1;
            if (l <= T.lmax && (masks[i] >> l & 1u)) { c.bl[c.nblk++] = l; c.off[l] = off; off += (2 * l + 1) * T.nbins * 32; }
        }
        c.tile = off;
        const size_t tb = (size_t)off * sizeof(double);
        c.nbuf = 2 * tb + extra <= kSmemLimit ? 2 : 1;
        smem = std::max(smem, c.nbuf * tb + extra);
    }
    return smem;
}

cudaError_t launch_contraction(const ContractArgs &a, cudaStream_t s, int *launches)
{
    *launches += 1;
    if (!a.factorised) {
        if (a.g_end <= a.g_begin) return cudaSuccess;
        switch (a.order) {
        case 3: return launch_generic<2>(a, s);
        case 4: return launch_generic<3>(a, s);
        case 5: return launch_generic<4>(a, s);
        case 6: return launch_generic<5>(a, s);
        }
        return cudaErrorInvalidValue;
    }
    // every (multiplet, tuple) of a chunk row is written by exactly one warp; no initialisation needed
    if (a.order == 3) {
        switch (a.nbins) {
        case 2: return launch3<2>(a, s);
        case 3: return launch3<3>(a, s);
        case 4: return launch3<4>(a, s);
        case 5: return launch3<5>(a, s);
        case 6: return launch3<6>(a, s);
        case 7: return launch3<7>(a, s);
        case 8: return launch3<8>(a, s);
        case 9: return launch3<9>(a, s);
        case 10: return launch3<10>(a, s);
        }
    } else if (a.order == 4) {
        switch (a.nbins) {
        case 3: return launch4<3>(a, s);
        case 4: return launch4<4>(a, s);
        case 5: return launch4<5>(a, s);
        case 6: return launch4<6>(a, s);
        case 7: return launch4<7>(a, s);
        case 8: return launch4<8>(a, s);
        case 9: return launch4<9>(a, s);
        case 10: return launch4<10>(a, s);
        }
    } else if (a.order == 6) {
        return launch_contract6(a, s);
    } else if (a.order == 5) {
        switch (a.nbins) {
        case 4: return launch5<4>(a, s);
        case 5: return launch5<5>(a, s);
        case 6: return launch5<6>(a, s);
        case 7: return launch5<7>(a, s);
        case 8: return launch5<8>(a, s);
        case 9: return launch5<9>(a, s);
        case 10: return launch5<10>(a, s);
        }
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_reduction(const ContractArgs &a, cudaStream_t s, int *launches)
{
    const int nout = a.nLam * a.nB;
    dim3 grid1((nout + 127) / 128, a.nseg);
    k_reduce_groups<<<grid1, 128, 0, s>>>(a);
    k_reduce_segments<<<(nout + 127) / 128, 128, 0, s>>>(a);
    *launches += 2;
    return cudaGetLastError();
}
