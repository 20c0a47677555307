// contract_tile.cuh — pieces shared by the factorised contraction kernels (contract.cu, contract6.cu): the dynamic
// shared-memory window, compile-time loops, and the TMA tile pipeline that streams the a_lm tile of one 32-primary
// group after the other into shared memory.
#pragma once
#include "device.cuh"

#include <type_traits>

namespace {

constexpr unsigned kFull = 0xffffffffu;

// one past the last group of this call: a.g_end, or (encore_compute_enqueue) the device-side group count it bounds
__device__ __forceinline__ int group_end(const ContractArgs &a)
{
    return a.ngroups_dev ? min(a.g_end, *a.ngroups_dev) : a.g_end;
}

extern __shared__ __align__(128) double smem_c[]; // dynamic shared memory of the factorised kernels

__host__ __device__ constexpr int c2(int n) { return n * (n - 1) / 2; }
__host__ __device__ constexpr int c3(int n) { return n * (n - 1) * (n - 2) / 6; }

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(kFull, v, d);
    return v;
}


// compile-time loop: f(std::integral_constant<int, I>) for I = A .. B-1 (indices into Set4 must be constant expressions)
template <int A, int B, class F>
__device__ __forceinline__ void static_for(F &&f)
{
    if constexpr (A < B) {
        f(std::integral_constant<int, A>{});
        static_for<A + 1, B>(f);
    }
}

// ---- tile pipeline: the a_lm tile of a group ([component][bin][lane], contiguous in HBM) is brought into shared
// memory by one TMA bulk copy (cp.async.bulk + mbarrier complete_tx), double-buffered so that group k+1 streams in
// while group k is contracted.  All warps of the CTA run the same loop (same number of barriers).
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void bulk_copy(double *dst, const double *src, unsigned bytes, unsigned long long *bar)
{
    // (the tx-count field of an mbarrier holds 2^20-1 bytes; the staged blocks of a group are < 256 kB)
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

constexpr int kMaxTileBufs = 8;                 // tile buffers of the ring (k_contract6: as many as fit; N = 4, 5: two)
constexpr int kBarDoubles = 2 * kMaxTileBufs;   // shared memory of the mbarriers, in doubles

struct TilePipe {
    int buf[kMaxTileBufs];   // offsets into smem_c (doubles)
    int bar;                 // offset of the mbarriers: full[kMaxTileBufs], empty[kMaxTileBufs]
    unsigned bytes;          // bytes of the staged l-blocks of one group
    int nbuf;
};

// Calls body(tile_in_smem, g) for the groups g = g_begin + blockIdx.x, + gridDim.x, ... < g_end (the chunk of this CTA).  Only the l-blocks the
// CTA's multiplets need (CtaPlan) are copied: one bulk copy per block, all completing on the buffer's mbarrier.
// RING: the plan may ask for 3-4 buffers (k_contract6; the N = 4, 5 plans stay at two: their heavy tiles leave no room and a
// third copy of their fully unrolled bodies costs more than the light CTAs gain).
template <bool RING = false, class Body>
__device__ __forceinline__ void for_each_group_tile(const ContractArgs &a, const CtaPlan &C, const TilePipe &tp, Body body)
{
    const int ngroups = group_end(a);
    const size_t tile = (size_t)a.ncomp * a.nbins * 32;
    const int stride = gridDim.x;
    const bool issuer = threadIdx.x == 0;
    const int rs = a.nbins * 32;
    int g = a.g_begin + blockIdx.x;
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(smem_c + tp.bar);
    auto load = [&](int buf, int gg) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&bar[buf])), "r"(tp.bytes) : "memory");
        const double *src = a.alm + (size_t)gg * tile;
        for (int j = 0; j < C.nblk; ++j) {
            const int l = C.bl[j];
            bulk_copy(smem_c + tp.buf[buf] + C.off[l], src + (size_t)l * l * rs, (unsigned)((2 * l + 1) * rs * sizeof(double)), &bar[buf]);
        }
    };
    if (RING && tp.nbuf > 2) {
        // a ring of 3-8 buffers: "full" barriers carry the copies, "empty" barriers (one arrival per warp) say that every warp
        // is done with a buffer.  Tile k + nbuf - 1 is requested while tile k is contracted (light CTAs finish a tile faster
        // than a copy takes to arrive: one tile of look-ahead left them waiting for data).  Only the issuing thread waits for
        // the other warps (before it refills the buffer they used one tile ago); nobody else waits on anything but data, so
        // the warps drift by up to a tile instead of meeting at a CTA barrier after every group.
        const int nbuf = tp.nbuf;
        unsigned long long *empty = bar + kMaxTileBufs;
        const int lane = threadIdx.x & 31;
        if (issuer)
            for (int j = 0; j < nbuf - 1 && g + j * stride < ngroups; ++j) load(j, g + j * stride);
        int st = 0, use = 0;                            // tile k sits in buffer st = k % nbuf, as that buffer's use-th tile
        for (int k = 0; g < ngroups; ++k, g += stride) {
            if (issuer && g + (nbuf - 1) * stride < ngroups) {
                const int sb = st == 0 ? nbuf - 1 : st - 1;     // (k + nbuf - 1) % nbuf: the buffer of tile k - 1
                const int ub = st == 0 ? use : use + 1;         // (k + nbuf - 1) / nbuf
                if (ub >= 1) mbar_wait(&empty[sb], (unsigned)((ub - 1) & 1));
                load(sb, g + (nbuf - 1) * stride);
            }
            mbar_wait(&bar[st], (unsigned)(use & 1));
            body(tp.buf[st], g);
            __syncwarp();
            if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&empty[st])) : "memory");
            if (++st == nbuf) { st = 0; ++use; }
        }
        return;
    }
    if (issuer && g < ngroups) load(0, g);
    if (tp.nbuf == 2) {
        // two buffers (the tiles of the heavy CTAs are too large for more): the same scheme with one tile of look-ahead
        unsigned long long *empty = bar + kMaxTileBufs;
        const int lane = threadIdx.x & 31;
        for (int k = 0; g < ngroups; ++k, g += stride) {
            const int st = k & 1;
            if (issuer && g + stride < ngroups) {
                const int use = (k + 1) >> 1;              // tile k+1 is the use-th tile of buffer st^1
                if (use >= 1) mbar_wait(&empty[st ^ 1], (unsigned)((use - 1) & 1));
                load(st ^ 1, g + stride);
            }
            mbar_wait(&bar[st], (unsigned)((k >> 1) & 1));
            body(tp.buf[st], g);
            __syncwarp();
            if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&empty[st])) : "memory");
        }
        return;
    }
    for (int k = 0; g < ngroups; ++k, g += stride) {
        mbar_wait(&bar[0], (unsigned)(k & 1));
        body(tp.buf[0], g);
        __syncthreads(); // every warp is done with the buffer before it is refilled
        if (issuer && g + stride < ngroups) load(0, g + stride);
    }
}

// shared memory: [nbuf tile buffers][2 x 8 mbarriers = kBarDoubles doubles][term lists of the CTA's multiplets]
__device__ __forceinline__ TilePipe make_pipe(const CtaPlan &C)
{
    TilePipe tp;
    for (int i = 0; i < kMaxTileBufs; ++i) tp.buf[i] = i < C.nbuf ? i * C.tile : 0;
    tp.bar = C.nbuf * C.tile;
    tp.bytes = (unsigned)(C.tile * sizeof(double));
    tp.nbuf = C.nbuf;
    if (threadIdx.x == 0) {
        unsigned long long *bar = reinterpret_cast<unsigned long long *>(smem_c + tp.bar);
        for (int i = 0; i < kMaxTileBufs; ++i) {
            mbar_init(&bar[i], 1);                                  // "full": the issuing thread's expect_tx arrival
            mbar_init(&bar[kMaxTileBufs + i], blockDim.x / 32);     // "empty": one arrival per warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    return tp; // the caller's __syncthreads (after it has copied its term list) publishes the barriers
}

// copy `n` terms starting at `src` to smem_c + off (one warp), 6 doubles per term
__device__ __forceinline__ void stage_terms(int off, const PairTerm *src, int n, int lane)
{
    const double *s = reinterpret_cast<const double *>(src);
    for (int k = lane; k < 6 * n; k += 32) smem_c[off + k] = s[k];
}
} // namespace
