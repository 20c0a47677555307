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
#include "device.cuh"

namespace {

constexpr int kWarps = 8;
constexpr unsigned kFull = 0xffffffffu;

// Generic kernel, any N in {3,4,5}: one warp per output (Lam,B), terms looped, complex products in registers.
__global__ void __launch_bounds__(kWarps * 32) k_contract_generic(ContractArgs a)
{
    const int g = blockIdx.x;
    const GridGeom &G = a.geom;
    if (g >= a.group_start[G.npencil]) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nb = a.nbins, nm = a.order - 1;
    const int p = find_pencil_of_group(a.group_start, G.npencil, g);
    const int pstart = a.cell_start[p * G.nc[0]], pend = a.cell_start[(p + 1) * G.nc[0]];
    const int first = pstart + ENCORE_GROUP * (g - a.group_start[p]);
    const int cnt = min(ENCORE_GROUP, pend - first);
    const double wi = lane < cnt ? a.pos4[first + lane].w : 0.0;
    const double *tile = a.alm + (size_t)g * a.ncomp * nb * 32 + lane;
    const int nout = a.nLam * a.nB;
    double *out = a.partial + (size_t)g * nout;

    for (int o = warp; o < nout; o += kWarps) {
        const int iL = o / a.nB, iB = o - iL * a.nB;
        int boff[4];
        for (int k = 0; k < nm; ++k) boff[k] = a.bin_tuples[iB * nm + k] * 32;
        double acc = 0.0;
        const int t1 = a.term_start[iL + 1];
        for (int t = a.term_start[iL]; t < t1; ++t) {
            const DevTerm tm = a.terms[t];
            double pr = tm.W, pi = 0.0;
            for (int k = 0; k < nm; ++k) {
                const double re = tile[(size_t)tm.re[k] * nb * 32 + boff[k]];
                const double im = tm.im[k] >= 0 ? (double)tm.tau[k] * tile[(size_t)tm.im[k] * nb * 32 + boff[k]] : 0.0;
                const double nr = pr * re - pi * im;
                const double ni = pr * im + pi * re;
                pr = nr; pi = ni;
            }
            acc += pr;
        }
        acc *= wi;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(kFull, acc, d);
        if (lane == 0) out[o] = acc;
    }
}

// a6, level 1: segment s sums its groups in index order.  level 2: sums the segments in index order, times 1/V.
__global__ void k_reduce_groups(ContractArgs a)
{
    const int nout = a.nLam * a.nB;
    const int o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= nout) return;
    const int ngroups = a.group_start[a.geom.npencil];
    const int s = blockIdx.y;
    const int per = (ngroups + a.nseg - 1) / a.nseg;
    const int g0 = s * per, g1 = min(ngroups, g0 + per);
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

} // namespace

cudaError_t launch_contraction(const ContractArgs &a, cudaStream_t s, int *launches)
{
    k_contract_generic<<<a.ngroups_max, kWarps * 32, 0, s>>>(a);
    *launches += 1;
    return cudaGetLastError();
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
