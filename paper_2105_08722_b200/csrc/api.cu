// api.cu — the C ABI of include/encore.h: plan life-cycle, the encore_compute pipeline, diagnostics.
#include "../../include/encore.h"
#include "device.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

namespace {

thread_local int g_last_cuda = 0;

struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
    cudaError_t ensure(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e == cudaSuccess) cap = bytes;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
    template <class T> T *as() const { return static_cast<T *>(p); }
};

} // namespace

struct encore_plan_s {
    HostTables T;
    bool uploaded = false;
    DevBuf d_terms, d_term_start, d_bin_tuples, d_ynorm, d_ycoef, d_pair_terms, d_lam4, d_lam5, d_lam6, d_lam_order, d_lam_parity, d_tuple_index, d_ctas, gweights;
    std::vector<CtaPlan> ctas;      // factorised N = 4, 5 kernels: multiplets and staged l-blocks per CTA
    size_t cta_smem = 0;
    bool force_generic = false;
    bool fp32_harmonics = false;    // ENCORE_FP32_HARMONICS
    int nchunk_override = 0;        // option "nchunk"
    // scratch
    DevBuf cid, cell_count, cell_fill, cell_start, scan_tmp, tmp_idx, sorted_idx, pos4, groups, group_start;
    DevBuf alm, counts, partial, partial2, bbox_tmp, bbox, flags, cand, bincounts, alm_export;
    DevBuf io_pos, io_w, io_zeta, pos4f;
    DevBuf gbound, gprefix, gwide, rows, rowdesc, rowcnt, errflag;
    DevBuf mesh_fd, mesh_kern;          // gridded estimator: F[delta h^3] and the kernel / a_lm field being transformed
    int mesh_fft = -1, mesh_fftb = -1, mesh_G = 0, mesh_batch = 0;   // cuFFT plans for one and for mesh_batch G^3 fields
    DevBuf d_gaunt, edge_A, edge_rhs;   // edge correction: E G tensor, per-tuple matrices and right-hand sides
    bool gaunt_ready = false;
    int *h_gprefix = nullptr;   // pinned
    size_t h_gprefix_cap = 0;
    size_t list_budget_bytes = (size_t)32 << 30;
    bool list_budget_set = false;   // option "list_mb" given: use it as is
    int pair_steps = 0;
    double *pinned = nullptr; // 16 doubles: bbox[6], flags as 2 ints in [6], internal-error flag as int in [7], padding particle [8..11]
    // state of the last compute
    bool have = false;
    bool have_grid = false;   // the last compute was encore_compute_grid: stream / launch count / timers are valid, particle diagnostics are not
    int64_t n = 0;
    GridGeom geom{};
    int ngroups_max = 0;
    int g_begin = 0, g_end = 0, ngroups = 0;  // groups the last compute covered (a shard's range, or all) of how many
    cudaStream_t stream = nullptr;
    bool timing = false;
    std::vector<cudaEvent_t> ev;    // event pool (timing only); ev[i] closes an interval of kind ev_kind[i]
    std::vector<int> ev_kind;
    size_t ev_used = 0;
    float ms[5] = {0, 0, 0, 0, 0};
    int launches = 0;
    int sub_yz_override = 0, sub_x_override = 0;
};

namespace {

#define CU(call)                                     \
    do {                                             \
        cudaError_t e__ = (call);                    \
        if (e__ != cudaSuccess) {                    \
            g_last_cuda = (int)e__;                  \
            return e__ == cudaErrorMemoryAllocation ? ENCORE_EALLOC : ENCORE_ECUDA; \
        }                                            \
    } while (0)

// literal eq. 44 kernel: first factor of term t that differs from term t-1 of the same multiplet (the terms are in
// lexicographic order of m_1 .. m_{N-2}; the partial products of the factors before it are reused).  The last factor
// always differs: m_{N-1} = -(m_1 + .. + m_{N-2}).
int term_prefix_start(const HostTables &T, int t)
{
    int k = 0;
    while (k < T.order - 2 && T.terms[t].re[k] == T.terms[t - 1].re[k] && T.terms[t].im[k] == T.terms[t - 1].im[k] &&
           T.terms[t].tau[k] == T.terms[t - 1].tau[k]) ++k;
    return k;
}

int upload_tables(encore_plan_s *P, cudaStream_t s)
{
    if (P->uploaded) return ENCORE_OK;
    const HostTables &T = P->T;
    std::vector<DevTerm> dt(T.terms.size());
    for (size_t i = 0; i < dt.size(); ++i) {
        for (int k = 0; k < 5; ++k) {
            const int rs = T.nbins * 32;
            dt[i].off_re[k] = T.terms[i].re[k] * rs;
            dt[i].off_im[k] = (T.terms[i].im[k] >= 0 ? T.terms[i].im[k] : T.terms[i].re[k]) * rs;
            dt[i].tau[k] = T.terms[i].im[k] >= 0 ? (double)T.terms[i].tau[k] : 0.0;
        }
        dt[i].W = T.terms[i].W;
        dt[i].start = 0; dt[i].pad = 0;
    }
    for (int iL = 0; iL < T.nLam(); ++iL)
        for (int t = T.term_start[iL] + 1; t < T.term_start[iL + 1]; ++t) dt[t].start = term_prefix_start(T, t);
    CU(P->d_terms.ensure(sizeof(DevTerm) * std::max<size_t>(1, dt.size())));
    CU(P->d_term_start.ensure(sizeof(int) * T.term_start.size()));
    CU(P->d_bin_tuples.ensure(sizeof(int) * T.bin_tuples.size()));
    CU(P->d_ynorm.ensure(sizeof(double) * T.ynorm.size()));
    CU(P->d_ycoef.ensure(sizeof(double) * T.ycoef.size()));
    CU(cudaMemcpyAsync(P->d_terms.p, dt.data(), sizeof(DevTerm) * dt.size(), cudaMemcpyHostToDevice, s));
    CU(cudaMemcpyAsync(P->d_term_start.p, T.term_start.data(), sizeof(int) * T.term_start.size(), cudaMemcpyHostToDevice, s));
    CU(cudaMemcpyAsync(P->d_bin_tuples.p, T.bin_tuples.data(), sizeof(int) * T.bin_tuples.size(), cudaMemcpyHostToDevice, s));
    CU(cudaMemcpyAsync(P->d_ynorm.p, T.ynorm.data(), sizeof(double) * T.ynorm.size(), cudaMemcpyHostToDevice, s));
    CU(cudaMemcpyAsync(P->d_ycoef.p, T.ycoef.data(), sizeof(double) * T.ycoef.size(), cudaMemcpyHostToDevice, s));
    {   // factorised-contraction tables
        const int nm = T.order - 1, nb = T.nbins;
        size_t cells = 1;
        if (contraction_is_factorised(T.order, nb, T.lmax)) // (tuple -> output index) is only read by the factorised kernels
            for (int k = 0; k < nm; ++k) cells *= (size_t)nb;
        std::vector<int> tix(cells, -1);
        for (int iB = 0; cells > 1 && iB < T.nB(); ++iB) {
            size_t key = 0;
            for (int k = 0; k < nm; ++k) key = key * nb + (size_t)T.bin_tuples[(size_t)iB * nm + k];
            tix[key] = iB;
        }
        CU(P->d_pair_terms.ensure(sizeof(PairTerm) * std::max<size_t>(1, T.pair_terms.size())));
        CU(P->d_lam4.ensure(sizeof(Lam4) * std::max<size_t>(1, T.lam4.size())));
        CU(P->d_lam5.ensure(sizeof(Lam5) * std::max<size_t>(1, T.lam5.size())));
        CU(P->d_lam6.ensure(sizeof(Lam6) * std::max<size_t>(1, T.lam6.size())));
        CU(cudaMemcpyAsync(P->d_lam6.p, T.lam6.data(), sizeof(Lam6) * T.lam6.size(), cudaMemcpyHostToDevice, s));
        CU(P->d_lam_order.ensure(sizeof(int) * std::max<size_t>(1, T.lam_order.size())));
        CU(P->d_lam_parity.ensure(sizeof(int) * std::max<size_t>(1, T.parity.size())));
        CU(cudaMemcpyAsync(P->d_lam_parity.p, T.parity.data(), sizeof(int) * T.parity.size(), cudaMemcpyHostToDevice, s));
        CU(P->d_tuple_index.ensure(sizeof(int) * cells));
        CU(P->d_ctas.ensure(sizeof(CtaPlan) * std::max<size_t>(1, P->ctas.size())));
        CU(cudaMemcpyAsync(P->d_ctas.p, P->ctas.data(), sizeof(CtaPlan) * P->ctas.size(), cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(P->d_pair_terms.p, T.pair_terms.data(), sizeof(PairTerm) * T.pair_terms.size(), cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(P->d_lam4.p, T.lam4.data(), sizeof(Lam4) * T.lam4.size(), cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(P->d_lam5.p, T.lam5.data(), sizeof(Lam5) * T.lam5.size(), cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(P->d_lam_order.p, T.lam_order.data(), sizeof(int) * T.lam_order.size(), cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(P->d_tuple_index.p, tix.data(), sizeof(int) * cells, cudaMemcpyHostToDevice, s));
        CU(cudaStreamSynchronize(s));
    }
    CU(cudaStreamSynchronize(s)); // the staging vectors die at return
    CU(cudaMallocHost((void **)&P->pinned, 16 * sizeof(double)));
    P->uploaded = true;
    return ENCORE_OK;
}

// DESIGN.md R11.  Per axis: h_a = r_max / sub_a, nc_a = max(1, floor(ext_a / h_a)), inv_a = nc_a / ext_a.
// sub_y = sub_z chosen so that a pencil cross-section holds ~32 particles per pencil-width of length;
// x is subdivided 4x finer (x-ranges of candidate pencils are culled at that granularity).
bool choose_geometry(const encore_plan_s *P, int64_t n, const double lo[3], const double hi[3], GridGeom &G)
{
    const HostTables &T = P->T;
    double ext[3];
    G.periodic = T.box > 0.0;
    G.box = T.box; G.half = 0.5 * T.box;
    for (int a = 0; a < 3; ++a) {
        if (G.periodic) { G.org[a] = 0.0; ext[a] = T.box; }
        else { G.org[a] = lo[a]; ext[a] = hi[a] - lo[a]; }
    }
    double vol = 1.0;
    for (int a = 0; a < 3; ++a) vol *= std::max(ext[a], T.rmax);
    const double rho = (double)n / vol;
    const double h_target = std::cbrt((double)ENCORE_GROUP / rho);
    int syz = (int)std::lround(T.rmax / h_target);
    syz = std::max(1, std::min(8, syz));
    if (P->sub_yz_override > 0) syz = std::min(8, P->sub_yz_override);
    int sx = 4 * syz;
    if (P->sub_x_override > 0) sx = P->sub_x_override;
    double cells = 0.0;
    for (;;) {
        G.sub[0] = sx; G.sub[1] = syz; G.sub[2] = syz;
        cells = 1.0;
        for (int a = 0; a < 3; ++a) {
            const double h = T.rmax / (double)G.sub[a];
            const double q = std::floor(ext[a] / h);
            G.nc[a] = q < 1.0 ? 1 : (q > 1e9 ? 1000000000 : (int)q);
            G.inv[a] = ext[a] > 0.0 ? (double)G.nc[a] / ext[a] : 1.0;
            // an axis thinner than one cell (nc = 1, e.g. a planar catalogue with noise in z): every particle is in
            // cell 0 whatever inv is; keep inv <= 1/h so that r_max * inv stays a small number of cells
            if (G.nc[a] == 1 && G.inv[a] > 1.0 / h) G.inv[a] = 1.0 / h;
            cells *= (double)G.nc[a];
        }
        if (cells <= 4.0e6 || sx == 1) break;
        sx = std::max(1, sx / 2);
    }
    if (cells > 4.0e6) return false;    // box / r_max beyond what the cell tables are sized for
    G.ncell = G.nc[0] * G.nc[1] * G.nc[2];
    G.npencil = G.nc[1] * G.nc[2];
    return true;
}

// interval kinds of encore_get_kernel_ms
enum { K_GRID = 0, K_SORT, K_BOUNDS, K_FILL, K_HARM, K_CONTRACT, K_REDUCE, K_COUNT, K_START = -1 };

// timing only: record an event that closes an interval of kind `kind` (K_START opens the first one)
int mark(encore_plan_s *P, int kind, cudaStream_t s)
{
    if (!P->timing) return ENCORE_OK;
    if (kind == K_START) P->ev_used = 0;
    if (P->ev_used == P->ev.size()) {
        cudaEvent_t e;
        CU(cudaEventCreate(&e));
        P->ev.push_back(e);
        P->ev_kind.push_back(0);
    }
    P->ev_kind[P->ev_used] = kind;
    CU(cudaEventRecord(P->ev[P->ev_used++], s));
    return ENCORE_OK;
}

#define TRY(call) do { int r__ = (call); if (r__ != ENCORE_OK) return r__; } while (0)

// steps a5 + a6 on a_lm tiles [group][component][bin][lane] with primary weights gweights[group][lane]
int contract_and_reduce(encore_plan_s *P, const double *alm, const double *gweights, int g_begin, int g_end, int ngmax, bool factorised,
                        int nchunk, double *zeta_out, cudaStream_t s, const int *ngroups_dev = nullptr)
{
    const HostTables &T = P->T;
    ContractArgs ca{};
    ca.order = T.order; ca.nbins = T.nbins; ca.ncomp = T.ncomp; ca.nLam = T.nLam(); ca.nB = T.nB();
    ca.terms = P->d_terms.as<DevTerm>();
    ca.term_start = P->d_term_start.as<int>();
    ca.bin_tuples = P->d_bin_tuples.as<int>();
    ca.alm = alm; ca.gweights = gweights;
    ca.partial = P->partial.as<double>();
    ca.partial2 = P->partial2.as<double>();
    ca.nseg = 64;
    ca.vinv_total = T.box > 0.0 ? 1.0 / (T.box * T.box * T.box) : 1.0; // DESIGN.md R12
    ca.zeta_out = zeta_out;
    ca.ngroups_max = ngmax;
    ca.g_begin = g_begin; ca.g_end = g_end;
    ca.ngroups_dev = ngroups_dev;
    ca.pair_terms = P->d_pair_terms.as<PairTerm>();
    ca.lam4 = P->d_lam4.as<Lam4>();
    ca.lam5 = P->d_lam5.as<Lam5>();
    ca.lam6 = P->d_lam6.as<Lam6>();
    ca.lam_order = P->d_lam_order.as<int>();
    ca.lam_parity = P->d_lam_parity.as<int>();
    ca.tuple_index = P->d_tuple_index.as<int>();
    ca.lmax = T.lmax;
    ca.max_terms = 1;
    for (const Lam4 &q : T.lam4) ca.max_terms = std::max(ca.max_terms, q.nterms);
    for (const Lam5 &q : T.lam5) ca.max_terms = std::max(ca.max_terms, q.nterms);
    for (const Lam6 &q : T.lam6) ca.max_terms = std::max(ca.max_terms, q.nterms);
    ca.ctas = P->d_ctas.as<CtaPlan>();
    ca.ncta = (int)P->ctas.size();
    ca.cta_smem = P->cta_smem;
    ca.nchunk = nchunk;
    ca.factorised = factorised ? 1 : 0;
    CU(launch_contraction(ca, s, &P->launches));
    TRY(mark(P, K_CONTRACT, s));
    CU(launch_reduction(ca, s, &P->launches));
    TRY(mark(P, K_REDUCE, s));
    return ENCORE_OK;
}

// chunks of groups per multiplet slot of the factorised kernels: the grid (slots x chunks CTAs, one per SM) should fill whole waves
int choose_nchunk(const encore_plan_s *P, bool factorised)
{
    int nchunk = 32;
    if (P->nchunk_override > 0) return P->nchunk_override;
    if (factorised) {
        int sms = 148, dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const int slots = P->T.order == 3 ? P->T.nLam() : (int)P->ctas.size();
        double best = 0.0;
        for (int c = 28; c <= 40; ++c) {
            const int ctas = slots * c, waves = (ctas + sms - 1) / sms;
            const double eff = (double)ctas / ((double)waves * sms) - 1e-4 * std::abs(c - 32);
            if (eff > best) { best = eff; nchunk = c; }
        }
    }
    return nchunk;
}

// shard/nshards: the primaries are cut into nshards contiguous ranges of cell-sorted groups with equal pair-stage
// work bounds; this call evaluates the sums over the primaries of range `shard` only (1 of 1 = everything).
//
// enqueue = true (encore_compute_enqueue): nothing is read back and nothing is allocated, so the call can be captured into
// a CUDA graph.  The grid geometry comes from the caller's bounding box `ubox` (open geometry; lo[3], hi[3]), the group
// count stays on the device (kernels are launched for the upper bound ngmax and clamp), the row reservation of the
// plan is used as it is (k_fill flags a group whose rows would not fit), validation flags travel with the status word.
int compute_device(encore_plan_s *P, const double *pos, const double *w, int64_t n, double *zeta_out, cudaStream_t s,
                   int shard = 0, int nshards = 1, const double *ubox = nullptr, bool enqueue = false)
{
    const HostTables &T = P->T;
    P->have = false;
    P->have_grid = false;
    P->launches = 0;
    if (enqueue && !P->uploaded) return ENCORE_ESTATE;
    TRY(upload_tables(P, s));
// scratch: grown on demand, or (enqueue) only checked against what the plan already owns
#define ENS(buf, bytes)                                                      \
    do {                                                                     \
        if (enqueue) { if ((size_t)(bytes) > (buf).cap) return ENCORE_ECAPACITY; } \
        else CU((buf).ensure(bytes));                                        \
    } while (0)

    // ---- validation + bounding box (one small device->host read) ------------------------------------------
    ENS(P->bbox_tmp, sizeof(double) * 6 * 592);
    ENS(P->bbox, sizeof(double) * 8);
    ENS(P->flags, sizeof(int) * 2);
    CU(launch_bbox_validate(pos, w, n, T.box, P->bbox_tmp.as<double>(), P->bbox.as<double>(), P->flags.as<int>(), s, &P->launches));
    double bb[6] = {0, 0, 0, 0, 0, 0};  // bounding box the grid is built on (open geometry)
    if (!enqueue) {
        CU(cudaMemcpyAsync(P->pinned, P->bbox.p, 6 * sizeof(double), cudaMemcpyDeviceToHost, s));
        CU(cudaMemcpyAsync(P->pinned + 6, P->flags.p, 2 * sizeof(int), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        int fl[2];
        std::memcpy(fl, P->pinned + 6, sizeof(fl));
        if (fl[0] || fl[1]) return ENCORE_EDOMAIN;
        std::memcpy(bb, P->pinned, sizeof(bb));
    } else if (!(T.box > 0.0)) {
        std::memcpy(bb, ubox, sizeof(bb));
        CU(launch_bbox_check(P->bbox.as<double>(), bb, bb + 3, P->flags.as<int>(), s, &P->launches));
    }
    GridGeom G;
    if (!choose_geometry(P, n, bb, bb + 3, G)) return ENCORE_EUNSUPPORTED;
    int nr_cap;
    {
        // inv <= sub / r_max (choose_geometry), so these are at most sub + 1 cells
        int Ry = (int)std::floor(std::min(T.rmax * G.inv[1], 1e6) + 1e-6) + 1, Rz = (int)std::floor(std::min(T.rmax * G.inv[2], 1e6) + 1e-6) + 1;
        if (!G.periodic) { Ry = std::min(Ry, G.nc[1] - 1); Rz = std::min(Rz, G.nc[2] - 1); }
        const int wy = std::min(2 * Ry + 1, G.periodic ? G.nc[1] : 2 * Ry + 1);
        const int wz = std::min(2 * Rz + 1, G.periodic ? G.nc[2] : 2 * Rz + 1);
        nr_cap = 2 * wy * wz;   // candidate runs of a group (k_fill keeps their table in shared memory)
        if (pair_fill_smem_bytes(T.nbins, nr_cap) > 200 * 1024) return ENCORE_EUNSUPPORTED;
    }
    const int ngmax = (int)(n / ENCORE_GROUP) + G.npencil + 1;
    if (ngmax > 2048 * 2048) return ENCORE_EUNSUPPORTED;   // (the three-kernel scan of the per-group word counts)
    const int nb = T.nbins, ncomp = T.ncomp;
    const size_t nout = (size_t)T.nLam() * T.nB();
    const int nseg = 64;   // (contract_and_reduce uses the same count)

    // ---- scratch ----------------------------------------------------------------------------------------------
    ENS(P->cid, sizeof(int32_t) * n);
    ENS(P->cell_count, sizeof(int) * (size_t)G.ncell);
    ENS(P->cell_fill, sizeof(int) * (size_t)G.ncell);
    ENS(P->cell_start, sizeof(int) * ((size_t)G.ncell + 1));
    ENS(P->scan_tmp, sizeof(int) * (std::max<size_t>(std::max<size_t>((size_t)G.ncell, (size_t)ngmax), 4000000) / 2048 + 8));
    ENS(P->tmp_idx, sizeof(int) * n);
    ENS(P->sorted_idx, sizeof(int) * n);
    ENS(P->pos4, sizeof(double4) * ((size_t)n + 1));   // + the padding particle
    ENS(P->groups, sizeof(int) * (size_t)G.npencil);
    ENS(P->group_start, sizeof(int) * ((size_t)G.npencil + 1));
    ENS(P->alm, sizeof(double) * (size_t)ngmax * ncomp * nb * 32);
    ENS(P->counts, sizeof(uint32_t) * (size_t)ngmax * nb * 32);
    const bool factorised = !P->force_generic && contraction_is_factorised(T.order, nb, T.lmax) && (T.order == 3 || P->cta_smem > 0);
    const int nchunk = choose_nchunk(P, factorised);
    ENS(P->partial, sizeof(double) * (size_t)(factorised ? nchunk : ngmax) * nout);
    ENS(P->gweights, sizeof(double) * (size_t)ngmax * 32);
    ENS(P->partial2, sizeof(double) * (size_t)nseg * nout);
    ENS(P->cand, 3 * sizeof(unsigned long long));   // candidate pairs, k_harm steps, k_harm ideal steps

    TRY(mark(P, K_START, s));
    // ---- a1: cell ids + histogram -----------------------------------------------------------------------------
    CU(launch_cell_ids(pos, n, G, P->cid.as<int32_t>(), P->cell_count.as<int>(), s, &P->launches));
    TRY(mark(P, K_GRID, s));
    // ---- a2: counting sort by cell, gather to AoS, groups of 32 per pencil ----------------------------------
    CU(launch_exclusive_scan(P->cell_count.as<int>(), P->cell_start.as<int>(), G.ncell, P->scan_tmp.as<int>(), s, &P->launches));
    CU(cudaMemsetAsync(P->cell_fill.p, 0, sizeof(int) * (size_t)G.ncell, s));
    CU(launch_sort_gather(pos, w, n, P->cid.as<int32_t>(), P->cell_start.as<int>(), G.ncell, P->cell_fill.as<int>(), P->tmp_idx.as<int>(),
                          P->sorted_idx.as<int>(), P->pos4.as<double4>(), s, &P->launches));
    CU(launch_pencil_groups(P->cell_start.as<int>(), G, P->groups.as<int>(), s, &P->launches));
    CU(launch_exclusive_scan(P->groups.as<int>(), P->group_start.as<int>(), G.npencil, P->scan_tmp.as<int>(), s, &P->launches));
    TRY(mark(P, K_SORT, s));
    // ---- a3 + a4: pair stage -----------------------------------------------------------------------------------
    PairArgs pa{};
    pa.pos4 = P->pos4.as<double4>();
    pa.npart = (int)n;
    {   // padding particle pos4[n]: weight 0, a few box sizes away from everything (k_harm's idle lanes add exact zeros)
        double far[3], r2 = 0.0;
        for (int a = 0; a < 3; ++a) {
            if (G.periodic) { far[a] = 3.0 * T.box; r2 += 9.0 * T.box * T.box; }
            else {
                const double ext = bb[3 + a] - bb[a];
                const double emax = std::max(std::max(bb[3] - bb[0], bb[4] - bb[1]), bb[5] - bb[2]);
                const double off = 2.0 * (emax + T.rmax);
                far[a] = bb[3 + a] + off;
                r2 += (ext + off) * (ext + off);
            }
        }
        pa.pad_r2max = r2;
        CU(launch_set_particle(P->pos4.as<double4>() + n, far[0], far[1], far[2], 0.0, s, &P->launches));
        if (P->fp32_harmonics) {
            // 16-byte candidate records relative to the centre of the box / bounding box; used for the bins whose lower edge
            // is at least 2^-10 of the largest such coordinate (fp32 then resolves every accepted separation to < 2^-13)
            double cmax = 0.0;
            for (int a = 0; a < 3; ++a) {
                pa.ctr[a] = G.periodic ? 0.5 * T.box : 0.5 * (bb[a] + bb[3 + a]);
                cmax = std::max(cmax, G.periodic ? 0.5 * T.box : 0.5 * (bb[3 + a] - bb[a]));
            }
            pa.gf_min_r2 = (cmax / 1024.0) * (cmax / 1024.0);
            ENS(P->pos4f, sizeof(float4) * ((size_t)n + 1));
            pa.pos4f = P->pos4f.as<float4>();
            CU(launch_make_pos4f(P->pos4.as<double4>(), n + 1, pa.ctr, P->pos4f.as<float4>(), s, &P->launches));
        }
    }
    pa.cell_start = P->cell_start.as<int>();
    pa.group_start = P->group_start.as<int>();
    pa.geom = G;
    pa.bins.nbins = nb;
    pa.bins.rmin_f = (float)T.rmin;
    pa.bins.invw_f = (float)((double)nb / (T.rmax - T.rmin));
    for (int b = 0; b <= nb; ++b) pa.bins.e2[b] = T.edges2[b];
    for (int b = 0; b < nb; ++b) pa.bins.vinv[b] = T.vinv[b];
    for (int b = 0; b < nb; ++b) pa.bin_order[b] = b;
    std::sort(pa.bin_order, pa.bin_order + nb, [&](int x, int y) { return T.vinv[x] != T.vinv[y] ? T.vinv[x] < T.vinv[y] : x < y; });
    pa.rmax = T.rmax;
    pa.lmax = T.lmax; pa.ncomp = ncomp;
    pa.fp32_harmonics = P->fp32_harmonics ? 1 : 0;
    pa.ynorm = P->d_ynorm.as<double>();
    pa.ycoef = P->d_ycoef.as<double>();
    pa.alm = P->alm.as<double>();
    pa.counts = P->counts.as<uint32_t>();
    pa.cand_pairs = P->cand.as<unsigned long long>();
    pa.gweights = P->gweights.as<double>();
    pa.ngroups = ngmax;
    ENS(P->gbound, sizeof(int) * (size_t)ngmax);
    ENS(P->gprefix, sizeof(int) * ((size_t)ngmax + 2));
    ENS(P->gwide, sizeof(int) * (size_t)ngmax);
    ENS(P->rowcnt, sizeof(int) * (size_t)ngmax * nb);
    ENS(P->errflag, sizeof(int));
    pa.gbound = P->gbound.as<int>();
    pa.gprefix = P->gprefix.as<int>();
    pa.gwide = P->gwide.as<int>();
    pa.scan_tmp = P->scan_tmp.as<int>();
    pa.rowcnt = P->rowcnt.as<int>();
    pa.err_flag = P->errflag.as<int>();
    if (!enqueue && P->h_gprefix_cap < (size_t)ngmax + 2) {
        if (P->h_gprefix) cudaFreeHost(P->h_gprefix);
        P->h_gprefix = nullptr; P->h_gprefix_cap = 0;
        CU(cudaMallocHost((void **)&P->h_gprefix, sizeof(int) * ((size_t)ngmax + 2)));
        P->h_gprefix_cap = (size_t)ngmax + 2;
    }
    int g_begin = 0, g_end = 0, ngroups_total = 0;
    CU(cudaMemsetAsync(P->cand.p, 0, 3 * sizeof(unsigned long long), s));
    CU(cudaMemsetAsync(P->errflag.p, 0, sizeof(int), s));
    CU(launch_pair_bounds(pa, s, &P->launches));
    if (enqueue) {
        // no read-back: one step over the upper bound of the group count with the rows the plan already owns
        const size_t cap_words = std::min(P->rows.cap / ((size_t)nb * 32 * sizeof(unsigned)), P->rowdesc.cap / ((size_t)nb * sizeof(unsigned)));
        if (cap_words == 0) return ENCORE_ECAPACITY;
        TRY(mark(P, K_BOUNDS, s));
        pa.rows = P->rows.as<unsigned>();
        pa.rowdesc = P->rowdesc.as<unsigned>();
        pa.rows_cap_words = cap_words;
        g_begin = 0; g_end = ngmax; ngroups_total = ngmax;
        P->pair_steps = 1;
        CU(launch_pair_fill(pa, 0, ngmax, nr_cap, s, &P->launches));
        TRY(mark(P, K_FILL, s));
        CU(launch_pair_harmonics(pa, 0, ngmax, s, &P->launches));
        TRY(mark(P, K_HARM, s));
    } else {
    // second small device->host read: candidate words per group (prefix) and the number of groups -> super-steps
    CU(cudaMemcpyAsync(P->h_gprefix, P->gprefix.p, sizeof(int) * ((size_t)ngmax + 1), cudaMemcpyDeviceToHost, s));
    CU(cudaMemcpyAsync(P->h_gprefix + ngmax + 1, P->group_start.as<int>() + G.npencil, sizeof(int), cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    TRY(mark(P, K_BOUNDS, s));
    {
        const int ngroups = P->h_gprefix[ngmax + 1];
        const int *gp = P->h_gprefix;
        // a word of a group owns one 128-byte row and one descriptor in each of the nb bin streams
        const size_t word_bytes = (size_t)nb * (32 + 1) * sizeof(unsigned);
        const size_t total_words = (size_t)gp[ngroups];
        // byte budget of the rows of one super-step: option "list_mb" if set, else 32 GB, or - when the rows do not fit
        // that - half of what the device has free (counting the buffer this plan already owns), between 4 GB and
        // 96 GB: fewer, longer steps are faster (every step ends with a partly filled last wave)
        size_t budget_bytes = P->list_budget_bytes;
        if (!P->list_budget_set && total_words * word_bytes > budget_bytes) {
            size_t free_b = 0, total_b = 0;
            if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
                const size_t avail = free_b + P->rows.cap + P->rowdesc.cap;
                budget_bytes = std::min<size_t>(std::max<size_t>(avail / 2, (size_t)4 << 30), (size_t)96 << 30);
            }
        }
        const size_t budget_words = std::max<size_t>(budget_bytes / word_bytes, 1);
        size_t max_group_words = 0;
        for (int g = 0; g < ngroups; ++g) max_group_words = std::max(max_group_words, (size_t)(gp[g + 1] - gp[g]));
        const size_t cap_words = std::max(std::min(total_words, budget_words), std::max<size_t>(max_group_words, 1));
        // reserved: an eighth more than this catalogue needs when the budget allows, so that encore_compute_enqueue can
        // replay the plan on other catalogues of the same size and clustering (a reservation is never shrunk)
        const size_t reserve_words = std::max(cap_words, std::min(budget_words, total_words + total_words / 8));
        if (P->rows.cap < cap_words * nb * 32 * sizeof(unsigned) || P->rowdesc.cap < cap_words * nb * sizeof(unsigned)) {
            CU(P->rows.ensure(reserve_words * nb * 32 * sizeof(unsigned)));
            CU(P->rowdesc.ensure(reserve_words * nb * sizeof(unsigned)));
        }
        pa.rows = P->rows.as<unsigned>();
        pa.rowdesc = P->rowdesc.as<unsigned>();
        pa.ngroups = ngroups;
        ngroups_total = ngroups;
        P->pair_steps = 0;
        // shard k takes the groups [cut(k), cut(k+1)), cut(k) = first g with gp[g] >= total * k / nshards
        auto cut = [&](int k) {
            if (k <= 0) return 0;
            if (k >= nshards) return ngroups;
            const long long want = ((long long)total_words * k + nshards - 1) / nshards;
            return (int)(std::lower_bound(gp, gp + ngroups + 1, want, [](int v, long long t) { return (long long)v < t; }) - gp);
        };
        g_begin = cut(shard); g_end = std::max(g_begin, std::min(ngroups, cut(shard + 1)));
        if (nshards > 1) CU(cudaMemsetAsync(P->counts.p, 0, sizeof(uint32_t) * (size_t)ngroups * nb * 32, s));
        // super-steps of whole groups, evenly sized (a short last step would run at a few percent occupancy)
        const size_t range_words = (size_t)(gp[g_end] - gp[g_begin]);
        const size_t nsteps = std::max<size_t>((range_words + cap_words - 1) / cap_words, 1);
        const size_t step_words = std::min(cap_words, std::max((range_words + nsteps - 1) / nsteps, std::max<size_t>(max_group_words, 1)));
        int g0 = g_begin;
        while (g0 < g_end) {
            int g1 = g0 + 1;
            while (g1 < g_end && (size_t)(gp[g1 + 1] - gp[g0]) <= step_words) ++g1;
            CU(launch_pair_fill(pa, g0, g1, nr_cap, s, &P->launches));
            TRY(mark(P, K_FILL, s));
            CU(launch_pair_harmonics(pa, g0, g1, s, &P->launches));
            TRY(mark(P, K_HARM, s));
            ++P->pair_steps;
            g0 = g1;
        }
    }
    }
    if (enqueue) CU(cudaMemcpyAsync(P->pinned + 6, P->flags.p, 2 * sizeof(int), cudaMemcpyDeviceToHost, s)); // validation flags
    // internal-consistency flag of the pair stage, read by whoever synchronises next (encore_get_status, the getters)
    CU(cudaMemcpyAsync(reinterpret_cast<int *>(P->pinned + 7), P->errflag.p, sizeof(int), cudaMemcpyDeviceToHost, s));
    // ---- a5: contraction, a6: reduction ------------------------------------------------------------------------
    TRY(contract_and_reduce(P, pa.alm, pa.gweights, g_begin, g_end, ngmax, factorised, nchunk, zeta_out, s,
                            enqueue ? P->group_start.as<int>() + G.npencil : nullptr));
#undef ENS

    P->have = true; P->n = n; P->geom = G; P->ngroups_max = ngmax; P->stream = s;
    P->g_begin = g_begin; P->g_end = g_end; P->ngroups = ngroups_total;
    return ENCORE_OK;
}

} // namespace

extern "C" {

int encore_plan(encore_plan_t **plan_out, int npcf_order, double r_min, double r_max, int nbins, int lmax, double box_size)
{
    return encore_plan_flags(plan_out, npcf_order, r_min, r_max, nbins, lmax, box_size, 0u);
}

int encore_plan_flags(encore_plan_t **plan_out, int npcf_order, double r_min, double r_max, int nbins, int lmax, double box_size,
                      unsigned flags)
{
    if (flags & ~(unsigned)(ENCORE_ALLPARITY | ENCORE_FP32_HARMONICS)) return plan_out ? (*plan_out = nullptr, ENCORE_EINVAL) : ENCORE_EINVAL;
    if (!plan_out) return ENCORE_EINVAL;
    *plan_out = nullptr;
    if (npcf_order < 3 || npcf_order > ENCORE_MAX_ORDER) return ENCORE_EINVAL;
    if (!(r_min >= 0.0) || !(r_max > r_min) || !std::isfinite(r_max)) return ENCORE_EINVAL;
    if (nbins < npcf_order - 1 || nbins > ENCORE_MAX_BINS) return ENCORE_EINVAL;
    if (lmax < 0 || !std::isfinite(box_size) || box_size < 0.0) return ENCORE_EINVAL;
    if (box_size > 0.0 && r_max > 0.5 * box_size) return ENCORE_EINVAL;
    if (lmax > ENCORE_MAX_LMAX) return ENCORE_EUNSUPPORTED;
    encore_plan_s *P = new (std::nothrow) encore_plan_s();
    if (!P) return ENCORE_EALLOC;
    try {   // everything that grows a std::vector stays inside: nothing may throw across the C ABI
        encore_build_tables(P->T, npcf_order, r_min, r_max, nbins, lmax, box_size, (flags & ENCORE_ALLPARITY) ? 1 : 0);
        if (npcf_order >= 4 && npcf_order <= 5 && contraction_is_factorised(npcf_order, nbins, lmax)) P->cta_smem = contraction_plan_ctas(P->T, P->ctas);
        if (npcf_order == 6 && contraction_is_factorised(npcf_order, nbins, lmax)) P->cta_smem = contraction_plan_ctas6(P->T, P->ctas);
    } catch (...) {
        delete P;
        return ENCORE_EALLOC;
    }
    P->fp32_harmonics = (flags & ENCORE_FP32_HARMONICS) != 0;
    *plan_out = P;
    return ENCORE_OK;
}

int encore_compute(encore_plan_t *P, const double *positions, const double *weights, int64_t n, double *zeta_out, void *cuda_stream)
{
    if (!P || !positions || !zeta_out || n < 1 || n >= (int64_t(1) << 26)) return ENCORE_EINVAL;
    return compute_device(P, positions, weights, n, zeta_out, static_cast<cudaStream_t>(cuda_stream));
}

int encore_compute_shard(encore_plan_t *P, const double *positions, const double *weights, int64_t n, int shard, int nshards,
                         double *zeta_partial_out, void *cuda_stream)
{
    if (!P || !positions || !zeta_partial_out || n < 1 || n >= (int64_t(1) << 26)) return ENCORE_EINVAL;
    if (nshards < 1 || shard < 0 || shard >= nshards) return ENCORE_EINVAL;
    return compute_device(P, positions, weights, n, zeta_partial_out, static_cast<cudaStream_t>(cuda_stream), shard, nshards);
}

int encore_compute_enqueue(encore_plan_t *P, const double *positions, const double *weights, int64_t n, const double *bbox_lo,
                           const double *bbox_hi, double *zeta_out, void *cuda_stream)
{
    if (!P || !positions || !zeta_out || n < 1 || n >= (int64_t(1) << 26)) return ENCORE_EINVAL;
    double ub[6] = {0, 0, 0, 0, 0, 0};
    if (!(P->T.box > 0.0)) {
        if (!bbox_lo || !bbox_hi) return ENCORE_EINVAL;
        for (int a = 0; a < 3; ++a) {
            if (!std::isfinite(bbox_lo[a]) || !std::isfinite(bbox_hi[a]) || bbox_hi[a] < bbox_lo[a]) return ENCORE_EINVAL;
            ub[a] = bbox_lo[a]; ub[3 + a] = bbox_hi[a];
        }
    }
    return compute_device(P, positions, weights, n, zeta_out, static_cast<cudaStream_t>(cuda_stream), 0, 1, ub, true);
}

int encore_query_grid(const encore_plan_t *P, int64_t n, const double *bbox_lo, const double *bbox_hi, int nc[3], int sub[3])
{
    if (!P || !nc || !sub || n < 1) return ENCORE_EINVAL;
    double lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    if (!(P->T.box > 0.0)) {
        if (!bbox_lo || !bbox_hi) return ENCORE_EINVAL;
        for (int a = 0; a < 3; ++a) { lo[a] = bbox_lo[a]; hi[a] = bbox_hi[a]; }
    }
    GridGeom G;
    if (!choose_geometry(P, n, lo, hi, G)) return ENCORE_EUNSUPPORTED;
    for (int a = 0; a < 3; ++a) { nc[a] = G.nc[a]; sub[a] = G.sub[a]; }
    return ENCORE_OK;
}

int encore_set_option(encore_plan_t *P, const char *key, long long value)
{
    if (!P || !key) return ENCORE_EINVAL;
    const std::string k(key);
    if (k == "list_mb") {           // byte budget of the acceptance-mask rows of one pair-stage super-step, in MiB; 0: default
        if (value < 0) return ENCORE_EINVAL;
        P->list_budget_set = value > 0;
        P->list_budget_bytes = value > 0 ? (size_t)value << 20 : (size_t)32 << 30;
    } else if (k == "sub_yz") {     // grid subdivision S_y = S_z (cell size r_max / S); 0: automatic
        if (value < 0 || value > 8) return ENCORE_EINVAL;
        P->sub_yz_override = (int)value;
    } else if (k == "sub_x") {      // grid subdivision S_x; 0: 4 S_y
        if (value < 0 || value > 32) return ENCORE_EINVAL;
        P->sub_x_override = (int)value;
    } else if (k == "nchunk") {     // chunks of groups per CTA column of the factorised contraction kernels; 0: automatic
        if (value < 0 || value > 1024) return ENCORE_EINVAL;
        P->nchunk_override = (int)value;
    } else if (k == "generic_contract") { // 1: run the literal eq. 44 kernel instead of the factorised ones
        if (value < 0 || value > 1) return ENCORE_EINVAL;
        P->force_generic = value != 0;
    } else return ENCORE_EINVAL;
    return ENCORE_OK;
}

int encore_get_status(const encore_plan_t *P)
{
    if (!P) return ENCORE_EINVAL;
    if (P->have_grid) {           // gridded estimator: no device-side checks to report, the call is the synchronisation point
        CU(cudaStreamSynchronize(P->stream));
        return ENCORE_OK;
    }
    if (!P->have) return ENCORE_ESTATE;
    CU(cudaStreamSynchronize(P->stream));
    int f = 0, fl[2];
    std::memcpy(&f, P->pinned + 7, sizeof(int));
    std::memcpy(fl, P->pinned + 6, sizeof(fl));   // validation flags (encore_compute reports them itself; encore_compute_enqueue cannot)
    if (fl[0] || fl[1]) return ENCORE_EDOMAIN;
    if (f & 2) return ENCORE_ECAPACITY;
    return f ? ENCORE_EINTERNAL : ENCORE_OK;
}

int encore_compute_grid(encore_plan_t *P, const double *delta, int G, double *zeta_out, void *cuda_stream)
{
    if (!P || !delta || !zeta_out || G < 2 || G > 1024) return ENCORE_EINVAL;
    const HostTables &T = P->T;
    if (!(T.box > 0.0)) return ENCORE_EINVAL;     // the mesh is periodic
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    P->have = false;
    P->have_grid = false;
    P->launches = 0;
    TRY(upload_tables(P, s));
    const size_t ncell = (size_t)G * G * G, npad = (ncell + 31) / 32 * 32;
    const int ngroups = (int)(npad / 32), nb = T.nbins, ncomp = T.ncomp;
    const size_t nout = (size_t)T.nLam() * T.nB();
    const bool factorised = !P->force_generic && contraction_is_factorised(T.order, nb, T.lmax) && (T.order == 3 || P->cta_smem > 0);
    const int nchunk = choose_nchunk(P, factorised);
    // (l, m >= 0) fields per FFT batch: all of them if they fit 2 GiB of scratch
    const int nlm = (T.lmax + 1) * (T.lmax + 2) / 2;
    const int batch = (int)std::max<size_t>(1, std::min<size_t>((size_t)nlm, ((size_t)2 << 30) / (ncell * 2 * sizeof(double))));
    CU(P->mesh_fd.ensure(sizeof(double) * 2 * ncell));
    CU(P->mesh_kern.ensure(sizeof(double) * 2 * ncell * (size_t)batch));
    CU(P->alm.ensure(sizeof(double) * (size_t)ngroups * ncomp * nb * 32));
    CU(P->gweights.ensure(sizeof(double) * npad));
    CU(P->partial.ensure(sizeof(double) * (size_t)(factorised ? nchunk : ngroups) * nout));
    CU(P->partial2.ensure(sizeof(double) * (size_t)64 * nout));
    if (P->mesh_fft < 0 || P->mesh_G != G || P->mesh_batch != batch) {
        if (P->mesh_fft >= 0) mesh_fft_plan_destroy(P->mesh_fft);
        if (P->mesh_fftb >= 0) mesh_fft_plan_destroy(P->mesh_fftb);
        P->mesh_fft = P->mesh_fftb = -1;
        if (mesh_fft_plan_create(G, 1, s, &P->mesh_fft) != 0) return ENCORE_EALLOC;
        if (mesh_fft_plan_create(G, batch, s, &P->mesh_fftb) != 0) return ENCORE_EALLOC;
        P->mesh_G = G; P->mesh_batch = batch;
    } else if (mesh_fft_plan_set_stream(P->mesh_fft, s) != 0 || mesh_fft_plan_set_stream(P->mesh_fftb, s) != 0) return ENCORE_ECUDA;
    TRY(mark(P, K_START, s));
    int fft_error = 0;
    CU(launch_mesh_alm(delta, G, T.box, T.lmax, nb, T.edges2.data(), T.vinv.data(), P->d_ycoef.as<double>(), P->mesh_fd.p, P->mesh_kern.p,
                       P->alm.as<double>(), P->gweights.as<double>(), P->mesh_fft, P->mesh_fftb, batch, s, &P->launches, &fft_error));
    if (fft_error) return ENCORE_ECUDA;
    TRY(mark(P, K_HARM, s));
    TRY(contract_and_reduce(P, P->alm.as<double>(), P->gweights.as<double>(), 0, ngroups, ngroups, factorised, nchunk, zeta_out, s));
    P->stream = s;
    P->have_grid = true;
    return ENCORE_OK;
}

int encore_edge_correct(encore_plan_t *P, const double *n_raw, const double *r_raw, double *zeta_out, void *cuda_stream)
{
    if (!P || !n_raw || !r_raw || !zeta_out) return ENCORE_EINVAL;
    const HostTables &T = P->T;
    const size_t n = (size_t)T.nLam(), nB = (size_t)T.nB();
    if (T.order > 5 || n > 256) return ENCORE_EUNSUPPORTED;   // App. A gives N = 3, 4, 5; the dense E G tensor holds n^3 doubles
    for (int k = 0; k < T.width; ++k) if (T.multiplets[k] != 0) return ENCORE_EUNSUPPORTED; // row 0 must be Lambda = 0
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (!P->gaunt_ready) {
        std::vector<double> G;
        try {
            if (encore_build_gaunt_tensor(T, G) != 0) return ENCORE_EUNSUPPORTED;
        } catch (...) {
            return ENCORE_EALLOC;
        }
        CU(P->d_gaunt.ensure(sizeof(double) * G.size()));
        CU(cudaMemcpyAsync(P->d_gaunt.p, G.data(), sizeof(double) * G.size(), cudaMemcpyHostToDevice, s));
        CU(cudaStreamSynchronize(s)); // the staging vector dies at return
        P->gaunt_ready = true;
    }
    CU(P->edge_A.ensure(sizeof(double) * nB * n * n));
    CU(P->edge_rhs.ensure(sizeof(double) * nB * n));
    CU(launch_edge_correct(P->d_gaunt.as<double>(), n_raw, r_raw, (int)n, (int)nB, P->edge_A.as<double>(), P->edge_rhs.as<double>(), zeta_out, s));
    return ENCORE_OK;
}

// Edge correction for callers that may not allocate device memory (see include/encore.h): no plan, no cudaMalloc / cudaFree;
// the scratch is the fixed device array in edge.cu.  Sizes beyond it are refused here, before anything touches the GPU.
int encore_edge_correct_noalloc(const double *gaunt, const double *n_raw, const double *r_raw, int n_lambda, int n_b,
                                double *zeta_out, void *cuda_stream)
{
    if (!gaunt || !n_raw || !r_raw || !zeta_out || n_lambda < 1 || n_b < 1) return ENCORE_EINVAL;
    const unsigned long long need = (unsigned long long)n_b * (unsigned long long)n_lambda * ((unsigned long long)n_lambda + 1ull);
    if (need > (unsigned long long)ENCORE_EDGE_NOALLOC_MAX_DOUBLES) return ENCORE_ETOOBIG;
    CU(launch_edge_correct_noalloc(gaunt, n_raw, r_raw, n_lambda, n_b, zeta_out, static_cast<cudaStream_t>(cuda_stream)));
    return ENCORE_OK;
}

int encore_get_contraction_layout(const encore_plan_t *P, int out[4])
{
    if (!P || !out) return ENCORE_EINVAL;
    const HostTables &T = P->T;
    const bool factorised = !P->force_generic && contraction_is_factorised(T.order, T.nbins, T.lmax) && (T.order == 3 || P->cta_smem > 0);
    out[0] = factorised ? T.order : 0;
    out[1] = factorised ? (int)P->ctas.size() : 0;
    out[2] = out[3] = 0;
    if (factorised && !P->ctas.empty()) {
        out[2] = out[3] = P->ctas[0].nbuf;
        for (const CtaPlan &c : P->ctas) { out[2] = std::min(out[2], c.nbuf); out[3] = std::max(out[3], c.nbuf); }
    }
    return ENCORE_OK;
}

int encore_get_gaunt_tensor(const encore_plan_t *P, double *out)
{
    if (!P || !out) return ENCORE_EINVAL;
    if (P->T.order > 5 || P->T.nLam() > 256) return ENCORE_EUNSUPPORTED;
    std::vector<double> G;
    try {
        if (encore_build_gaunt_tensor(P->T, G) != 0) return ENCORE_EUNSUPPORTED;
    } catch (...) {
        return ENCORE_EALLOC;
    }
    std::memcpy(out, G.data(), sizeof(double) * G.size());
    return ENCORE_OK;
}

int encore_get_pair_steps(const encore_plan_t *P)
{
    if (!P) return ENCORE_EINVAL;
    if (!P->have) return ENCORE_ESTATE;
    return P->pair_steps;
}

int encore_get_multiplet_parity(const encore_plan_t *P, int *out)
{
    if (!P || !out) return ENCORE_EINVAL;
    for (size_t i = 0; i < P->T.parity.size(); ++i) out[i] = P->T.parity[i];
    return ENCORE_OK;
}

int encore_get_shard_groups(const encore_plan_t *P, int out[3])
{
    if (!P || !out) return ENCORE_EINVAL;
    if (!P->have) return ENCORE_ESTATE;
    out[0] = P->g_begin; out[1] = P->g_end; out[2] = P->ngroups;
    return ENCORE_OK;
}

int encore_compute_host(encore_plan_t *P, const double *positions, const double *weights, int64_t n, double *zeta_out)
{
    if (!P || !positions || !zeta_out || n < 1 || n >= (int64_t(1) << 26)) return ENCORE_EINVAL;
    const size_t nout = (size_t)encore_zeta_len(P);
    CU(P->io_pos.ensure(sizeof(double) * 3 * (size_t)n));
    if (weights) CU(P->io_w.ensure(sizeof(double) * (size_t)n));
    CU(P->io_zeta.ensure(sizeof(double) * nout));
    cudaStream_t s = nullptr;
    CU(cudaMemcpyAsync(P->io_pos.p, positions, sizeof(double) * 3 * (size_t)n, cudaMemcpyHostToDevice, s));
    if (weights) CU(cudaMemcpyAsync(P->io_w.p, weights, sizeof(double) * (size_t)n, cudaMemcpyHostToDevice, s));
    TRY(compute_device(P, P->io_pos.as<double>(), weights ? P->io_w.as<double>() : nullptr, n, P->io_zeta.as<double>(), s));
    CU(cudaMemcpyAsync(zeta_out, P->io_zeta.p, sizeof(double) * nout, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    return encore_get_status(P);
}

int encore_destroy(encore_plan_t *P)
{
    if (!P) return ENCORE_EINVAL;
    DevBuf *bufs[] = {&P->d_terms, &P->d_term_start, &P->d_bin_tuples, &P->d_ynorm, &P->d_ycoef, &P->d_pair_terms, &P->d_lam4, &P->d_lam5, &P->d_lam6,
                      &P->d_lam_order, &P->d_lam_parity, &P->d_tuple_index, &P->d_ctas, &P->gweights, &P->cid, &P->cell_count, &P->cell_fill,
                      &P->cell_start, &P->scan_tmp, &P->tmp_idx, &P->sorted_idx, &P->pos4, &P->groups, &P->group_start,
                      &P->alm, &P->counts, &P->partial, &P->partial2, &P->bbox_tmp, &P->bbox, &P->flags, &P->cand,
                      &P->bincounts, &P->alm_export, &P->io_pos, &P->io_w, &P->io_zeta, &P->pos4f, &P->gbound, &P->gprefix, &P->gwide,
                      &P->rows, &P->rowdesc, &P->rowcnt, &P->errflag, &P->d_gaunt, &P->edge_A, &P->edge_rhs, &P->mesh_fd, &P->mesh_kern};
    for (DevBuf *b : bufs) b->release();
    if (P->pinned) cudaFreeHost(P->pinned);
    if (P->h_gprefix) cudaFreeHost(P->h_gprefix);
    for (cudaEvent_t e : P->ev) cudaEventDestroy(e);
    if (P->mesh_fft >= 0) mesh_fft_plan_destroy(P->mesh_fft);
    if (P->mesh_fftb >= 0) mesh_fft_plan_destroy(P->mesh_fftb);
    delete P;
    return ENCORE_OK;
}

int64_t encore_zeta_len(const encore_plan_t *P) { return P ? (int64_t)P->T.nLam() * P->T.nB() : ENCORE_EINVAL; }
int encore_num_multiplets(const encore_plan_t *P) { return P ? P->T.nLam() : ENCORE_EINVAL; }
int encore_num_bin_tuples(const encore_plan_t *P) { return P ? P->T.nB() : ENCORE_EINVAL; }
int64_t encore_num_terms(const encore_plan_t *P) { return P ? (int64_t)P->T.terms.size() : ENCORE_EINVAL; }

int encore_get_multiplets(const encore_plan_t *P, int *out)
{
    if (!P || !out) return ENCORE_EINVAL;
    std::memcpy(out, P->T.multiplets.data(), sizeof(int) * P->T.multiplets.size());
    return ENCORE_OK;
}

int encore_get_bin_tuples(const encore_plan_t *P, int *out)
{
    if (!P || !out) return ENCORE_EINVAL;
    std::memcpy(out, P->T.bin_tuples.data(), sizeof(int) * P->T.bin_tuples.size());
    return ENCORE_OK;
}

int encore_get_bin_edges(const encore_plan_t *P, double *out)
{
    if (!P || !out) return ENCORE_EINVAL;
    std::memcpy(out, P->T.edges.data(), sizeof(double) * P->T.edges.size());
    return ENCORE_OK;
}

int encore_contraction_flops(const encore_plan_t *P, double *executed, double *canonical)
{
    if (!P) return ENCORE_EINVAL;
    const HostTables &T = P->T;
    const double evals = (double)T.terms.size() * (double)T.nB();
    const int N = T.order, nb = T.nbins;
    // literal eq. 44 kernel: per term and bin tuple, one multiply (conjugation sign) + one complex multiply (2 mul + 2 FMA)
    // for every factor that differs from the previous term's (the first factor: the sign multiply only), 2 FMA for W
    double ex = 0.0;
    for (int iL = 0; iL < T.nLam(); ++iL)
        for (int t = T.term_start[iL]; t < T.term_start[iL + 1]; ++t) {
            const int start = t == T.term_start[iL] ? 0 : term_prefix_start(T, t);
            ex += (start == 0 ? 1.0 + 7.0 * (N - 2) : 7.0 * (N - 1 - start)) + 4.0;
        }
    ex *= (double)T.nB();
    if (!P->force_generic && contraction_is_factorised(N, nb, T.lmax) && (N == 3 || P->cta_smem > 0)) {
        // executed by the factorised kernels, fused multiply-add = 2
        ex = 0.0;
        auto c2 = [](int n) { return n * (n - 1) / 2; };
        if (N == 3) { // per real component: nb scalings + one FMA per bin pair
            ex = (double)T.ncomp * (nb + 2.0 * (nb * (nb - 1) / 2));
        } else if (N == 6) {
            ex = contraction6_flops(T);
        } else if (N == 4) {
            for (const Lam4 &q : T.lam4)
                for (int b1 = 0; b1 + 2 < nb; ++b1) {
                    const int nb2 = nb - 1 - b1;
                    const double n0 = q.tbeg[1] - q.tbeg[0], nr = q.tbeg[q.l3 + 1] - q.tbeg[1];
                    ex += n0 * (2.0 + 4.0 * (nb2 - 1));                                       // G_0: 2 mul + 2 FMA per upper bin
                    ex += nr * (4.0 + 8.0 * (nb2 - 1));                                       // G_{m3>0}: 4 mul + 4 FMA per upper bin
                    ex += 1.0 * (nb2 - 1) + 2.0 * nb2 * (nb2 - 1) / 2;                        // G_0 a3: 1 FMA per triple
                    ex += (double)q.l3 * (2.0 * (nb2 - 1) + 4.0 * nb2 * (nb2 - 1) / 2);       // Re[G a3]: 2 FMA per triple
                }
        } else {
            // warp w of a multiplet takes the second bins lo..hi (contract.cu): Y(b1, b2 in lo..hi) and R(b3 > lo, b4);
            // 4 multiplies per pre-weighted operand, 4 FMA per pair and term, 2 FMA per tuple and M
            const int nw = contraction_warps5(nb);
            for (int w = 0; w < nw; ++w) {
                int lo, hi;
                contraction_range5(nb, w, &lo, &hi);
                if (lo > hi || hi > nb - 3) continue;
                const double nyh = c2(hi + 1) - c2(lo), nrh = c2(nb - 1 - lo);
                double tup = 0;
                for (int b2 = lo; b2 <= hi; ++b2) tup += (double)b2 * c2(nb - 1 - b2);
                for (const Lam5 &q : T.lam5) {
                    const double nl = q.lbeg[q.l12 + 1] - q.lbeg[1], nr = q.rbeg[q.l12 + 1] - q.rbeg[1], nM = q.l12; // M >= 1
                    ex += nl * (4.0 * (hi - lo + 1) + 8.0 * nyh) + nM * 2.0 * nyh;   // Y block, times w_i
                    ex += nr * (4.0 * (nb - 2 - lo) + 8.0 * nrh);                    // R block
                    ex += nM * 4.0 * tup;                                            // Re[Y R]
                    const double hl = q.lbeg[1] - q.lbeg[0], hr = q.rbeg[1] - q.rbeg[0];   // M = 0: half terms, real pairs
                    ex += hl * (2.0 * (hi - lo + 1) + 4.0 * nyh) + nyh + hr * (2.0 * (nb - 2 - lo) + 4.0 * nrh) + 2.0 * tup;
                }
            }
        }
    }
    if (executed) *executed = ex;
    if (canonical) *canonical = evals * (6.0 * (N - 3) + 5.0);   // 5 / 11 / 17 / 23 flop per term evaluation for N = 3..6
    return ENCORE_OK;
}

int encore_get_grid(const encore_plan_t *P, int nc[3], int sub[3])
{
    if (!P || !nc || !sub) return ENCORE_EINVAL;
    if (!P->have) return ENCORE_ESTATE;
    for (int a = 0; a < 3; ++a) { nc[a] = P->geom.nc[a]; sub[a] = P->geom.sub[a]; }
    return ENCORE_OK;
}

int encore_get_cell_ids(const encore_plan_t *P, int32_t *out)
{
    if (!P || !out) return ENCORE_EINVAL;
    if (!P->have) return ENCORE_ESTATE;
    CU(cudaMemcpyAsync(out, P->cid.p, sizeof(int32_t) * (size_t)P->n, cudaMemcpyDeviceToDevice, P->stream));
    CU(cudaStreamSynchronize(P->stream));
    return ENCORE_OK;
}

int encore_get_bin_counts(const encore_plan_t *Pc, uint64_t *counts, uint64_t *pairs_total)
{
    encore_plan_t *P = const_cast<encore_plan_t *>(Pc);
    if (!P || !counts) return ENCORE_EINVAL;
    if (!P->have) return ENCORE_ESTATE;
    const int nb = P->T.nbins;
    CU(P->bincounts.ensure(sizeof(unsigned long long) * ENCORE_MAX_BINS));
    CU(launch_sum_bin_counts(P->counts.as<uint32_t>(), P->group_start.as<int>(), P->geom.npencil, nb,
                             P->bincounts.as<unsigned long long>(), P->ngroups_max, P->stream));
    unsigned long long h[ENCORE_MAX_BINS];
    CU(cudaMemcpyAsync(h, P->bincounts.p, sizeof(unsigned long long) * nb, cudaMemcpyDeviceToHost, P->stream));
    CU(cudaStreamSynchronize(P->stream));
    uint64_t tot = 0;
    for (int b = 0; b < nb; ++b) { counts[b] = h[b]; tot += h[b]; }
    if (pairs_total) *pairs_total = tot;
    return ENCORE_OK;
}

int encore_get_primary_counts(const encore_plan_t *P, uint32_t *out)
{
    if (!P || !out) return ENCORE_EINVAL;
    if (!P->have) return ENCORE_ESTATE;
    CU(launch_export_primary_counts(P->counts.as<uint32_t>(), P->cid.as<int32_t>(), P->sorted_idx.as<int>(), P->cell_start.as<int>(),
                                    P->group_start.as<int>(), P->geom, P->T.nbins, P->n, out, P->stream));
    CU(cudaStreamSynchronize(P->stream));
    return ENCORE_OK;
}

int encore_get_alm(const encore_plan_t *Pc, int64_t i, double *out)
{
    encore_plan_t *P = const_cast<encore_plan_t *>(Pc);
    if (!P || !out) return ENCORE_EINVAL;
    if (!P->have) return ENCORE_ESTATE;
    if (i < 0 || i >= P->n) return ENCORE_EINVAL;
    const int lmax = P->T.lmax, nb = P->T.nbins;
    const size_t cnt = (size_t)nb * (lmax + 1) * (lmax + 2);
    CU(P->alm_export.ensure(sizeof(double) * cnt));
    CU(launch_export_alm(P->alm.as<double>(), P->cid.as<int32_t>(), P->sorted_idx.as<int>(), P->cell_start.as<int>(),
                         P->group_start.as<int>(), P->geom, nb, lmax, P->n, i, P->alm_export.as<double>(), P->stream));
    CU(cudaMemcpyAsync(out, P->alm_export.p, sizeof(double) * cnt, cudaMemcpyDeviceToHost, P->stream));
    CU(cudaStreamSynchronize(P->stream));
    return ENCORE_OK;
}

int encore_get_kernel_ms(const encore_plan_t *Pc, float ms[7])
{
    encore_plan_t *P = const_cast<encore_plan_t *>(Pc);
    if (!P || !ms) return ENCORE_EINVAL;
    if (!P->timing || P->ev_used < 2) return ENCORE_ESTATE;   // (also valid after encore_compute_grid: [4] = the FFT stage)
    CU(cudaEventSynchronize(P->ev[P->ev_used - 1]));
    for (int k = 0; k < K_COUNT; ++k) ms[k] = 0.f;
    for (size_t i = 1; i < P->ev_used; ++i) {
        float t = 0.f;
        CU(cudaEventElapsedTime(&t, P->ev[i - 1], P->ev[i]));
        ms[P->ev_kind[i]] += t;
    }
    return ENCORE_OK;
}

int encore_get_stage_ms(const encore_plan_t *Pc, float ms[5])
{
    float k[K_COUNT];
    const int rc = encore_get_kernel_ms(Pc, k);
    if (rc != ENCORE_OK) return rc;
    ms[0] = k[K_GRID]; ms[1] = k[K_SORT]; ms[2] = k[K_BOUNDS] + k[K_FILL] + k[K_HARM]; ms[3] = k[K_CONTRACT]; ms[4] = k[K_REDUCE];
    return ENCORE_OK;
}

int encore_set_timing(encore_plan_t *P, int enabled)
{
    if (!P) return ENCORE_EINVAL;
    P->timing = enabled != 0;
    return ENCORE_OK;
}

int encore_get_launch_count(const encore_plan_t *P)
{
    if (!P) return ENCORE_EINVAL;
    return (P->have || P->have_grid) ? P->launches : ENCORE_ESTATE;
}

int encore_get_candidate_pairs(const encore_plan_t *P, uint64_t *out)
{
    if (!P || !out) return ENCORE_EINVAL;
    if (!P->have) return ENCORE_ESTATE;
    unsigned long long h = 0;
    CU(cudaMemcpyAsync(&h, P->cand.p, sizeof(h), cudaMemcpyDeviceToHost, P->stream));
    CU(cudaStreamSynchronize(P->stream));
    *out = h;
    return ENCORE_OK;
}

int encore_get_harm_steps(const encore_plan_t *P, uint64_t *executed, uint64_t *ideal)
{
    if (!P || !executed || !ideal) return ENCORE_EINVAL;
    if (!P->have) return ENCORE_ESTATE;
    unsigned long long h[3] = {0, 0, 0};
    CU(cudaMemcpyAsync(h, P->cand.p, sizeof(h), cudaMemcpyDeviceToHost, P->stream));
    CU(cudaStreamSynchronize(P->stream));
    *executed = h[1]; *ideal = h[2];
    return ENCORE_OK;
}

int encore_measure_fp64_peak(double *flops_per_s, void *cuda_stream)
{
    if (!flops_per_s) return ENCORE_EINVAL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    double *sink = nullptr;
    CU(cudaMalloc((void **)&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    const int iters = 4096;
    CU(launch_fp64_peak(sink, 256, s)); // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        CU(cudaEventRecord(e0, s));
        CU(launch_fp64_peak(sink, iters, s));
        CU(cudaEventRecord(e1, s));
        CU(cudaEventSynchronize(e1));
        float ms = 0;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    const double fmas = 148.0 * 4 * 512 * (double)iters * 16 * 8;
    *flops_per_s = 2.0 * fmas / (best * 1e-3);
    return ENCORE_OK;
}

int encore_measure_dmma_peak(double *flops_per_s, void *cuda_stream)
{
    if (!flops_per_s) return ENCORE_EINVAL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    double *sink = nullptr;
    CU(cudaMalloc((void **)&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    const int iters = 1024;
    CU(launch_dmma_peak(sink, 64, s)); // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        CU(cudaEventRecord(e0, s));
        CU(launch_dmma_peak(sink, iters, s));
        CU(cudaEventRecord(e1, s));
        CU(cudaEventSynchronize(e1));
        float ms = 0;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    const double fmas = 148.0 * 8 * 8 * (double)iters * 32 * 256;   // CTAs x warps x iterations x MMAs per iteration x FMA per MMA
    *flops_per_s = 2.0 * fmas / (best * 1e-3);
    return ENCORE_OK;
}

const char *encore_strerror(int status)
{
    switch (status) {
    case ENCORE_OK: return "ok";
    case ENCORE_EINVAL: return "invalid argument";
    case ENCORE_EDOMAIN: return "input outside the domain (non-finite value, or periodic coordinate outside [0, box))";
    case ENCORE_EALLOC: return "allocation failed";
    case ENCORE_ECUDA: return cudaGetErrorString((cudaError_t)g_last_cuda);
    case ENCORE_ESTATE: return "no successful encore_compute to report on (or timing disabled)";
    case ENCORE_EUNSUPPORTED: return "configuration not covered by this build's kernels";
    case ENCORE_EINTERNAL: return "internal consistency check of the pair stage failed (please report)";
    case ENCORE_ECAPACITY: return "encore_compute_enqueue: the plan's scratch (sized by its last encore_compute) is too small for this input";
    case ENCORE_ETOOBIG: return "encore_edge_correct_noalloc: n_b * n_lambda * (n_lambda + 1) exceeds ENCORE_EDGE_NOALLOC_MAX_DOUBLES, the library's fixed scratch array";
    default: return "unknown status";
    }
}

int encore_last_cuda_error(void) { return g_last_cuda; }

} // extern "C"
