// device.cuh — structures passed to the CUDA stages and their launch entry points.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <mutex>

#include "common.h"

// Set-up that CUDA keeps per DEVICE (cudaFuncSetAttribute acts on the current device only): run f once on every device
// a kernel is launched on, not once per process - a process may hold plans on several GPUs (encore.h binds a plan to the
// device current at its first compute).  Costs one cudaGetDevice and an uncontended lock per launch.  A failure is not
// remembered: the next launch tries again.
struct PerDeviceOnce {
    std::mutex mu;
    unsigned long long done[4] = {0, 0, 0, 0};   // bit d: device d is set up (devices >= 256: set up at every launch)
    template <class F> cudaError_t run(F f)
    {
        int dev = -1;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        const bool tracked = dev >= 0 && dev < 256;
        std::lock_guard<std::mutex> lock(mu);
        if (tracked && (done[dev >> 6] >> (dev & 63) & 1ull)) return cudaSuccess;
        e = f();
        if (e == cudaSuccess && tracked) done[dev >> 6] |= 1ull << (dev & 63);
        return e;
    }
};

// Uniform grid (R11): per axis a, cell size ~ r_max / sub[a]; x is the fast (fine) axis so that a
// "pencil" (iy,iz) is one contiguous run of the cell-sorted particle array.
struct GridGeom {
    double org[3];
    double inv[3];      // cells per unit length
    int nc[3];
    int sub[3];
    int periodic;
    double box, half;
    int ncell, npencil;
};

struct DevTerm {        // device image of HostTerm for the literal eq. 44 kernel (96 bytes)
    int off_re[5];      // offset (doubles) of the real-part row of factor k inside a tile: component * nbins * 32
    int off_im[5];      // same for the imaginary part (m = 0: the real-part row, with tau = 0)
    double tau[5];      // +1, -1 (conjugated factor) or 0 (m = 0: no imaginary part)
    double W;
    int start;          // first factor that differs from the previous term of the multiplet (terms are in lexicographic
    int pad;            // order of m_1 .. m_{N-2}): the partial products of the factors before it are reused
};

struct BinTable {       // passed by value (kernel parameter space -> constant bank)
    int nbins;
    float rmin_f, invw_f;       // fp32 first guess of the bin; the decision itself is fp64 on e2[]
    double e2[ENCORE_MAX_BINS + 1];
    double vinv[ENCORE_MAX_BINS];
};

// ---- grid.cu --------------------------------------------------------------------------------------------
// bbox[0..5] = min xyz, max xyz; flags[0] != 0 if a coordinate/weight is non-finite, flags[1] != 0 if a
// periodic coordinate is outside [0, box)
cudaError_t launch_bbox_validate(const double *pos, const double *w, int64_t n, double box, double *bbox_tmp,
                                 double *bbox_out, int *flags, cudaStream_t s, int *launches);
cudaError_t launch_set_particle(double4 *dst, double x, double y, double z, double w, cudaStream_t s, int *launches);
cudaError_t launch_bbox_check(const double *bbox_dev, const double lo[3], const double hi[3], int *flags, cudaStream_t s, int *launches);
cudaError_t launch_cell_ids(const double *pos, int64_t n, GridGeom g, int32_t *cid, int *cell_count,
                            cudaStream_t s, int *launches);
// exclusive scan of `in[0..m)` into `out[0..m]` (out[m] = total); tmp needs (m/2048+2) ints; m <= 2048*2048
cudaError_t launch_exclusive_scan(const int *in, int *out, int m, int *tmp, cudaStream_t s, int *launches);
cudaError_t launch_sort_gather(const double *pos, const double *w, int64_t n, const int32_t *cid,
                               const int *cell_start, int ncell, int *cell_fill, int *tmp_idx, int *sorted_idx,
                               double4 *pos4, cudaStream_t s, int *launches);
cudaError_t launch_make_pos4f(const double4 *pos4, int64_t count, const double ctr[3], float4 *pos4f, cudaStream_t s, int *launches);
cudaError_t launch_pencil_groups(const int *cell_start, GridGeom g, int *groups_per_pencil, cudaStream_t s,
                                 int *launches);

// ---- pair.cu --------------------------------------------------------------------------------------------
struct PairArgs {
    const double4 *pos4;        // cell-sorted {x,y,z,w}; entry [npart] is the padding particle (weight 0, far away)
    int npart;
    double pad_r2max;           // bound on the squared distance of the padding particle from any particle
    const int *cell_start;      // [ncell+1]
    const int *group_start;     // [npencil+1]; group_start[npencil] = number of groups
    GridGeom geom;
    BinTable bins;
    double rmax;
    int lmax, ncomp;
    int fp32_harmonics;         // ENCORE_FP32_HARMONICS: k_harm evaluates the weighted harmonics in fp32 (fp64 accumulation)
    const float4 *pos4f;        // ENCORE_FP32_HARMONICS: {x - c, y - c, z - c, w} of pos4 rounded to fp32 (c = ctr: box / bounding-box centre)
    double ctr[3];
    double gf_min_r2;           // bins whose lower edge^2 is at least this gather pos4f (16 B per candidate) instead of pos4
    const double *ynorm;        // [ncomp] device
    const double *ycoef;        // [ncomp][lmax+1] device: Y_lm = sum_k ycoef[c][k] z^k (x+iy)^m
    double *alm;                // [ngroups][ncomp][nbins][32]
    uint32_t *counts;           // [ngroups][nbins][32]  accepted pairs per (primary, bin): integer output of a3
    unsigned long long *cand_pairs; // candidate pairs tested (diagnostic)
    double *gweights;           // [ngroups][32] weight of (group, lane), 0 for empty lanes
    int ngroups;                // upper bound n/32 + npencil + 1 before the bounds are read back; exact afterwards
    // acceptance-mask rows: per (group, bin) a stream of 128-byte rows, one 32-bit mask per primary,
    // each row covering one word of 32 consecutive sorted candidates named by its descriptor
    int *gbound;                // [ngroups]   candidate words of a group = row capacity of each of its bins
    int *gprefix;               // [ngroups+1] exclusive scan of gbound
    int *gwide;                 // [ngroups]   1: a candidate run covers a whole periodic axis (exact path, no common image)
    int *scan_tmp;
    unsigned *rows;             // [(gprefix[g]-gprefix[g0]) * nbins + bin * words(g) + k][32] masks, lane = primary
    unsigned *rowdesc;          // same index: first sorted index of the word | image codes << 26
    int *rowcnt;                // [ngroups][nbins] rows written
    int *err_flag;              // bit 0: a word's candidates disagreed on the periodic image (excluded by DESIGN.md §5.3);
                                // bit 1: the row reservation is too small for this input (encore_compute_enqueue only)
    size_t rows_cap_words;      // candidate words the row buffers hold; 0: sized from the word counts on the host (not checked)
    int bin_order[ENCORE_MAX_BINS]; // bins by decreasing shell volume (work per item)
};
// per-group word counts -> gbound, gprefix, gwide (device).  The caller reads gprefix back, sizes the row buffer, and
// calls launch_pair_fill then launch_pair_harmonics once per super-step [g0, g1); nr_cap >= number of candidate runs of a group.
cudaError_t launch_pair_bounds(const PairArgs &a, cudaStream_t s, int *launches);
cudaError_t launch_pair_fill(const PairArgs &a, int g0, int g1, int nr_cap, cudaStream_t s, int *launches);
cudaError_t launch_pair_harmonics(const PairArgs &a, int g0, int g1, cudaStream_t s, int *launches);
size_t pair_fill_smem_bytes(int nbins, int nr_cap);
int pair_stage_supported(int lmax, int nbins);

// ---- contract.cu ----------------------------------------------------------------------------------------
struct ContractArgs {
    int order, nbins, ncomp, nLam, nB;
    const DevTerm *terms;       // device
    const int *term_start;      // device [nLam+1]
    const int *bin_tuples;      // device [nB][order-1]
    const double *alm;
    const double *gweights;     // [ngroups][32] weight of the primary (group, lane), 0 for empty lanes
    double *partial;            // [ngroups_max][nout]
    double *partial2;           // [nseg][nout]
    int nseg;
    double vinv_total;          // 1/V
    double *zeta_out;
    int ngroups_max;
    int g_begin, g_end;         // groups of this call (all of them, or one shard's contiguous range)
    const int *ngroups_dev;     // encore_compute_enqueue: the group count lives on the device and g_end is an upper bound; else NULL
    // factorised kernels (N = 4, 5)
    const PairTerm *pair_terms; // device
    const Lam4 *lam4;           // device [nLam]
    const Lam5 *lam5;           // device [nLam]
    const Lam6 *lam6;           // device [nLam] (factorised N = 6 only)
    const int *lam_order;       // device [nLam], heaviest first
    const int *lam_parity;      // device [nLam]: 1 = parity-odd multiplet (the stored value is Im zeta)
    const int *tuple_index;     // device [nbins^(N-1)]: index of the ordered tuple in bin_tuples, -1 if not ordered
    int lmax;
    int max_terms;              // largest number of coupled-pair terms of one multiplet
    const CtaPlan *ctas;        // device [ncta]: multiplets and staged l-blocks of every CTA of the factorised N = 4, 5 kernels
    int ncta;
    size_t cta_smem;            // dynamic shared memory of that launch
    int nchunk;                 // partial has nchunk rows when the factorised kernels ran (ngroups rows otherwise)
    int factorised;             // set by launch_contraction
};
int contraction_is_factorised(int order, int nbins, int lmax);
int contraction_split5(int nbins);   // N = 5, up to 8 bins: second bins <= this go to the first warp of a multiplet
int contraction_warps5(int nbins);   // N = 5: warps per multiplet
void contraction_range5(int nbins, int w, int *lo, int *hi); // N = 5: second bins lo..hi of warp w
// multiplets -> CTAs of the factorised N = 4, 5 kernels; returns the dynamic shared memory of the launch (0: does not fit)
size_t contraction_plan_ctas(const HostTables &T, std::vector<CtaPlan> &ctas);
cudaError_t launch_contraction(const ContractArgs &a, cudaStream_t s, int *launches);
// factorised N = 6 (contract6.cu): shapes covered, host plan (dynamic shared memory, 0: not covered), executed flops, launch
int contraction6_supported(int nbins, int lmax);
size_t contraction_plan_ctas6(const HostTables &T, std::vector<CtaPlan> &ctas);
double contraction6_flops(const HostTables &T);
cudaError_t launch_contract6(const ContractArgs &a, cudaStream_t s);
cudaError_t launch_reduction(const ContractArgs &a, cudaStream_t s, int *launches);

// ---- edge.cu -------------------------------------------------------------------------------------------
// T: [n][n][n] E G tensor; Nraw, Rraw: [n][nB] raw multiplets; A: [nB][n][n], rhs: [nB][n] scratch; zeta: [n][nB]
cudaError_t launch_edge_correct(const double *T, const double *Nraw, const double *Rraw, int n, int nB, double *A, double *rhs,
                                double *zeta, cudaStream_t s);
// same kernels with A and rhs in the library's fixed file-scope device array (no allocation; sizes checked by the caller)
cudaError_t launch_edge_correct_noalloc(const double *T, const double *Nraw, const double *Rraw, int n, int nB, double *zeta,
                                        cudaStream_t s);

// ---- mesh.cu (gridded estimator, eq. 36) ------------------------------------------------------------------
cudaError_t launch_mesh_alm(const double *delta, int G, double box, int lmax, int nb, const double *e2, const double *vinv,
                            const double *ycoef_dev, void *fd, void *kern, double *alm, double *gweights, int fft_plan1, int fft_planb,
                            int batch, cudaStream_t s, int *launches, int *fft_error);
int mesh_fft_plan_create(int G, int batch, cudaStream_t s, int *plan_out);
int mesh_fft_plan_set_stream(int plan, cudaStream_t s);
void mesh_fft_plan_destroy(int plan);

// ---- diag.cu --------------------------------------------------------------------------------------------
cudaError_t launch_sum_bin_counts(const uint32_t *counts, const int *group_start, int npencil, int nbins,
                                  unsigned long long *out, int ngroups_max, cudaStream_t s);
cudaError_t launch_export_primary_counts(const uint32_t *counts, const int32_t *cid, const int *sorted_idx,
                                         const int *cell_start, const int *group_start, GridGeom g, int nbins,
                                         int64_t n, uint32_t *out, cudaStream_t s);
cudaError_t launch_export_alm(const double *alm, const int32_t *cid, const int *sorted_idx, const int *cell_start,
                              const int *group_start, GridGeom g, int nbins, int lmax, int64_t n, int64_t i,
                              double *out_dev, cudaStream_t s);
cudaError_t launch_fp64_peak(double *sink, int iters, cudaStream_t s);
cudaError_t launch_dmma_peak(double *sink, int iters, cudaStream_t s);   // 148 * 8 CTAs x 8 warps x iters x 32 MMAs (m8n8k4, 256 FMA each)

// locate the group of cell-sorted slot `s` (shared by diag and contraction kernels)
__device__ __forceinline__ int find_pencil_of_group(const int *group_start, int npencil, int g)
{
    int lo = 0, hi = npencil; // invariant: group_start[lo] <= g < group_start[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (group_start[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}
