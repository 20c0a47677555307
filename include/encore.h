/*
 * encore.h — C ABI of the B200-native hot path of ENCORE's O(N_g^2) NPCF estimator
 * (arxiv 2105.08722; citations are PAPER.md line + equation / algorithm).
 *
 * What one encore_compute() evaluates, entirely on the GPU (sm_100a), fp64 throughout:
 *
 *   a^b_lm(s_i) = (1/v_b) sum_{j != i} w_j Y_lm( (r_j - s_i)^ ) Theta^b(|r_j - s_i|)        eq. 35
 *   zeta^B_Lam  = (1/V) sum_i w_i sum_M E(Lam) C^Lam_M prod_k a^{b_k}_{l_k m_k}(s_i)          eq. 34
 *
 * for N = 3, 4, 5, 6 (Lam = {l}, {l1 l2 l3}, {l1 l2 (l12) l3 l4}, {l1 l2 (l12) l3 (l123) l4 l5}; eqs. 16, 18, 5/20 —
 * PAPER.md:135, :145, :69, :157),
 * even-parity multiplets (real zeta) and, with ENCORE_ALLPARITY, the parity-odd ones too (imaginary zeta,
 * stored as Im zeta), ordered distinct bins b_1 < .. < b_{N-1},
 * using the half-sum m_{N-1} >= 0 of eq. 44.  Steps:
 *   a1 cell assignment, a2 counting sort by cell, a3 neighbour sweep + radial binning, a4 a_lm accumulation,
 *   a5 per-primary coupling contraction, a6 deterministic fp64 reduction over primaries.
 *
 * Conventions fixed here (DESIGN.md §3 lists every reading of the paper):
 *   - separation r_j - s_i (eq. 35); periodic minimal image per axis when box_size > 0, which requires
 *     r_max <= box_size/2 and coordinates in [0, box_size);
 *   - half-open bins e_b <= r < e_{b+1}, e_b = r_min + b (r_max - r_min)/nbins, decided on r^2 =
 *     fma(dz,dz,fma(dy,dy,dx*dx)); pairs with r^2 == 0 or j == i are skipped;
 *   - Y_lm with the Condon-Shortley phase; v_b = 4 pi/3 (e_{b+1}^3 - e_b^3); V = box_size^3, or 1 when open;
 *   - zeta_out[iLam * n_B + iB]; Lam in nested ascending loops, last index fastest (order of PAPER.md:622 and
 *     Alg. 3); B lexicographic, last index fastest (Alg. 3 l.9-13).
 *
 * Pointers marked DEVICE are CUDA device pointers valid on the current device; HOST are ordinary host
 * pointers.  The caller owns every buffer it passes.  The plan owns its tables and scratch (grown on demand
 * and reused across calls).  One plan must not be used from two host threads at once; distinct plans may.
 *
 * Every function returning int returns ENCORE_OK (0) or a negative ENCORE_E* code; nothing throws or aborts
 * across this boundary.  After an error the contents of output buffers are unspecified.
 * There is no CPU fallback: without a usable CUDA device encore_compute() returns ENCORE_ECUDA.
 */
#ifndef ENCORE_H
#define ENCORE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct encore_plan_s encore_plan_t; /* opaque */

enum {
    ENCORE_OK = 0,
    ENCORE_EINVAL = -1,   /* bad argument (order, bins, lmax, radii, box, n, NULL pointer) */
    ENCORE_EDOMAIN = -2,  /* non-finite coordinate / weight, or periodic coordinate outside [0, box) */
    ENCORE_EALLOC = -3,   /* host or device allocation failed */
    ENCORE_ECUDA = -4,    /* a CUDA call failed; encore_last_cuda_error() has the cudaError_t */
    ENCORE_ESTATE = -5,   /* diagnostic getter called before a successful encore_compute */
    ENCORE_EUNSUPPORTED = -6, /* valid problem outside what this build's kernels cover (see encore_plan) */
    ENCORE_EINTERNAL = -7, /* a device-side consistency check failed; results must not be used (encore_get_status) */
    ENCORE_ECAPACITY = -8, /* encore_compute_enqueue: the plan's scratch, sized by its last encore_compute, is too small */
    ENCORE_ETOOBIG = -9    /* encore_edge_correct_noalloc: the problem needs more than the library's fixed scratch array holds */
};

/* Build a plan: the Lambda / B / M tables with weights 2 S(m_{N-1}) E(Lam) C^Lam_M (eq. 44, PAPER.md:428-430;
 * S(0) = 1/2, else 1), bin edges, 1/v_b, Y_lm normalisations.  Host work only; device tables are uploaded by the
 * first encore_compute on the then-current device.
 *   npcf_order  N in {3,4,5,6}  (N = 6: Lam = {l1 l2 (l12) l3 (l123) l4 l5}, eq. 5 with two intermediates)
 *   r_min,r_max 0 <= r_min < r_max
 *   nbins       N_r >= N-1 and <= 32
 *   lmax        0..10 (ENCORE_EUNSUPPORTED above).  The factorised contraction kernels cover N=3, nbins <= 10;
 *               N=4, nbins <= 10; N=5, nbins <= 10 and lmax <= 5; N=6, 5 <= nbins <= 10 and lmax <= 4; other shapes run the
 *               literal eq. 44 kernel (one warp per (Lam, B) at a time)
 *   box_size    > 0: periodic cube [0,L)^3 (PERIODIC mode), needs r_max <= L/2;  0: open geometry
 */
int encore_plan(encore_plan_t **plan_out, int npcf_order, double r_min, double r_max, int nbins, int lmax,
                double box_size);

/* encore_plan with mode flags.  ENCORE_ALLPARITY (the paper's ALLPARITY mode): the multiplet list
 * also holds the parity-odd multiplets (odd sum of the principal l's; 111 instead of 69 for N=4, lmax=5).
 * Their zeta is purely imaginary (eq. 8): zeta_out holds Re zeta for even and Im zeta for odd multiplets,
 *   Im zeta = (1/V) sum_i w_i sum_{M, m_{N-1} >= 0} 2 S(m_{N-1}) E(Lam) C^Lam_M Im[prod_k a~]   (App. B),
 * with separations r_j - s_i as in eq. 35 (the sign of odd multiplets depends on it).  Unknown flags: ENCORE_EINVAL. */
#define ENCORE_ALLPARITY 1u
/* ENCORE_FP32_HARMONICS (the paper's reduced-precision modes): step a4 evaluates
 * the unit vector, its powers and w (x+iy)^m of every pair in fp32 and adds fp32 chunk sums of 64 pairs to the fp64 a_lm
 * accumulators.  For the bins fp32 resolves (lower edge >= 2^-10 of the largest coordinate measured from the centre of
 * the box / bounding box) candidates are gathered as 16-byte fp32 records {x, y, z, w} relative to that centre and the
 * separation is an fp32 subtraction: its components are off by <= 2^-24 of that largest coordinate, i.e. < 2^-13 r.  For the
 * inner bins the separation is formed in fp64 and rounded once (2^-24 r).  These errors are independent from pair to pair
 * and average down over the thousands of pairs of a bin; with the <= 64 x 2^-24 of a chunk sum they give the ~1e-6 below.  Cell ids,
 * the radial binning and therefore every pair count stay those of the fp64 path (bit-exact); contraction and reduction
 * stay fp64.  A separate, separately reported path: zeta agrees with the fp64 result to ~1e-6 of max|zeta| (tests bound
 * it by 1e-5), not to 1e-9. */
#define ENCORE_FP32_HARMONICS 2u
int encore_plan_flags(encore_plan_t **plan_out, int npcf_order, double r_min, double r_max, int nbins, int lmax,
                      double box_size, unsigned flags);

/* Run steps a1..a6 on `cuda_stream` (a cudaStream_t cast to void*, NULL = default stream).
 *   positions DEVICE, SoA x[n] y[n] z[n] (3n doubles), read-only
 *   weights   DEVICE, n doubles, or NULL for unit weights (negative weights allowed: D-R fields)
 *   n         1 <= n < 2^26
 *   zeta_out  DEVICE, encore_zeta_len(plan) doubles, written
 * Work is enqueued on the stream; the call returns after at most two small device->host reads it needs for
 * sizing (the bounding box in open geometry, the group count).  zeta_out is valid once the stream has drained.
 * Inputs are validated on the device (ENCORE_EDOMAIN is reported by this call). */
int encore_compute(encore_plan_t *plan, const double *positions, const double *weights, int64_t n,
                   double *zeta_out, void *cuda_stream);

/* Enqueue-only variant of encore_compute ("enqueues on cuda_stream and returns without synchronising"):
 * no device->host read, no allocation, no host synchronisation, so the call can be captured into a CUDA graph and replayed
 * on new catalogues of the same size.  It needs a previous successful encore_compute / encore_compute_host on this plan
 * (tables uploaded, scratch and the pair stage's row reservation sized): ENCORE_ESTATE before that.
 *   bbox_lo, bbox_hi  HOST, 3 doubles each: a box holding every particle (open geometry; ignored, may be NULL, when the
 *                     plan is periodic).  The grid is built on THIS box (reading R11), so cell ids follow it; zeta, the
 *                     pair counts and a_lm do not depend on it.
 * What encore_compute decides on the host is decided on the device instead: kernels are launched for the upper bound
 * n/32 + pencils + 1 of the group count and clamp to the count on the device; the pair stage runs as ONE step inside the
 * plan's row reservation.  Returns ENCORE_ECAPACITY at once when a scratch array would have to grow (larger n, or a box
 * with more cells); everything that can only be seen on the device is reported by the next encore_get_status:
 * ENCORE_EDOMAIN (non-finite input, coordinate outside [0, box) or outside the given box), ENCORE_ECAPACITY (this
 * catalogue needs more rows than the reservation holds: run encore_compute once, it re-sizes), ENCORE_EINTERNAL.
 * After such a status zeta_out is unspecified.  Per-kernel timing (encore_set_timing) must be off while capturing. */
int encore_compute_enqueue(encore_plan_t *plan, const double *positions, const double *weights, int64_t n,
                           const double *bbox_lo, const double *bbox_hi, double *zeta_out, void *cuda_stream);

/* Same, with HOST buffers: copies positions/weights to the device, computes, copies zeta back and
 * synchronises.  This is the end-to-end entry bench.py times as `e2e`. */
int encore_compute_host(encore_plan_t *plan, const double *positions, const double *weights, int64_t n,
                        double *zeta_out);

/* Multi-GPU sharding over primaries (the paper's only parallel loop).
 * Every rank holds the whole catalogue and calls this with the same inputs and its own `shard` in [0, nshards):
 * the cell-sorted primaries are cut into nshards contiguous ranges of groups with equal pair-stage work bounds and
 * the call evaluates eq. 34's sum over the primaries of range `shard` only, INCLUDING the 1/V factor, into
 * zeta_partial_out (DEVICE, encore_zeta_len doubles).  The sum of the nshards partial vectors, taken in shard
 * order, is the estimator; that sum is the caller's one collective (paper_2105_08722_b200.sharded does it with an
 * all-gather and a fixed-order sum, bit-identical on every rank).  Diagnostics after this call (bin counts, primary
 * counts, a_lm tiles) cover the shard's primaries only; counts of other primaries read 0.
 * nshards = 1 is encore_compute.  Errors as encore_compute, plus ENCORE_EINVAL for shard outside [0, nshards). */
int encore_compute_shard(encore_plan_t *plan, const double *positions, const double *weights, int64_t n, int shard,
                         int nshards, double *zeta_partial_out, void *cuda_stream);
/* Gridded estimator (eq. 36): the multiplets of a density field given on a periodic
 * mesh.  The plan must be periodic (box_size > 0); delta DEVICE, G^3 doubles, delta[(ix G + iy) G + iz] = value at the cell
 * centre ((ix,iy,iz) + 1/2) h, h = box_size / G.  Discretised on the mesh (int dr -> h^3 sum over cells)
 *   a^b_lm(s) = (1/v_b) sum_{cells x != s} delta(x) h^3 Y_lm((x - s)^) Theta^b(|x - s|)        (eq. 36 evaluated with FFTs)
 *   zeta^B_Lam = (1/V) sum_{cells s} delta(s) h^3 sum_M E(Lam) C^Lam_M prod_k a^{b_k}_{l_k m_k}(s)  (steps i-iii)
 * i.e. eq. 34/35 for particles at the cell centres with weights delta h^3; separations are (integer offset) h, minimal
 * image, binned on r^2 like the particle path.  zeta_out DEVICE as for encore_compute.  Scratch: one complex G^3 field, one per (l, m >= 0) of a batch (all of them when they fit 2 GiB) and
 * the a_lm array of all cells, (lmax+1)^2 nbins G^3 doubles (the memory cost the paper warns of, PAPER.md fn. 5).  Uses cuFFT.
 * Enqueued on cuda_stream without host synchronisation once the scratch exists.  2 <= G <= 1024. */
int encore_compute_grid(encore_plan_t *plan, const double *delta, int G, double *zeta_out, void *cuda_stream);

/* Edge correction of raw multiplets (eqs. 38-42).  n_raw = the plan's multiplets of the
 * data-minus-random field (an encore_compute on D - R), r_raw = those of the random field (an encore_compute on R with
 * positive weights), both DEVICE [n_Lambda][n_B] as encore_compute writes them.  Per bin tuple B:
 *   f_Lam' = R_Lam' / R_0,  M_{Lam Lam''} = sum_Lam' f_Lam' E(Lam'') G^{Lam Lam' Lam''}  (generalised Gaunt integrals, eq. 15,
 *   from App. A's closed forms with 3-j and 9-j symbols),  solve  sum_Lam zeta_Lam M_{Lam Lam''} = N_Lam'' / R_0   (eq. 41/42)
 * by LU with partial pivoting, one CTA per B; zeta_out DEVICE [n_Lambda][n_B] (may not alias the inputs).  The basis is
 * truncated to the plan's multiplet list, as the paper truncates at lmax.  Enqueued on cuda_stream; the first call builds
 * the E G tensor on the host (n_Lambda^3 doubles) and synchronises once.  N = 3, 4, 5 and n_Lambda <= 256
 * (ENCORE_EUNSUPPORTED otherwise: N = 6 has no closed form in the paper).  R_0 = 0 or a singular M give non-finite output. */
int encore_edge_correct(encore_plan_t *plan, const double *n_raw, const double *r_raw, double *zeta_out, void *cuda_stream);
/* host query (no GPU needed): the tensor encore_edge_correct uses, out[(i n + j) n + k] = E(Lam_k) G^{Lam_i Lam_j Lam_k}, n = n_Lambda.
 * ENCORE_ALLPARITY plans: rows of parity-odd multiplets hold imaginary parts (coefficient = i x stored value) in n_raw, r_raw
 * and zeta_out alike; eqs. 40-42 relate the complex coefficients, so the entries with Lam_i and Lam_j BOTH odd (they feed an
 * even Lam_k) carry the extra factor i x i = -1 in this tensor.  With it the real system on stored values is eq. 41 exactly. */
int encore_get_gaunt_tensor(const encore_plan_t *plan, double *out /* HOST n_Lambda^3 */);

/* Edge correction for callers that must not allocate device memory.
 *
 * Who this is for: encore_edge_correct keeps its per-bin-tuple matrices in plan-owned buffers that it cudaMallocs (and
 * grows) on demand.  Some hosts cannot accept that: a serving or training process that has handed all of HBM to its own
 * pool allocator (a cudaMalloc there fails, or breaks the pool's accounting), a job running under a fixed device-memory
 * quota, and latency-bound loops in which cudaMalloc / cudaFree are unwelcome because they take driver-wide locks and
 * cudaFree waits for the whole device, stalling unrelated streams.  This entry point calls no cudaMalloc, no cudaFree and
 * no library routine that allocates; it needs no plan on the device.  The caller passes every input and the output:
 *   gaunt     DEVICE, n_lambda^3 doubles: the tensor of encore_get_gaunt_tensor (a host query), copied to the device by the caller
 *   n_raw     DEVICE [n_lambda][n_b], raw multiplets of the D - R field      (as for encore_edge_correct)
 *   r_raw     DEVICE [n_lambda][n_b], raw multiplets of the random field; row 0 must be Lambda = 0
 *   zeta_out  DEVICE [n_lambda][n_b], written; may not alias an input
 * The result is that of encore_edge_correct on the same inputs (same kernels, same order of operations).
 *
 * The scratch (n_b matrices of n_lambda^2 doubles and n_b right-hand sides) lives in ONE fixed array compiled into the
 * library, ENCORE_EDGE_NOALLOC_MAX_DOUBLES doubles (8 MiB) of device memory that every GPU which loads the library keeps
 * until the process exits.  Limit:  n_b * n_lambda * (n_lambda + 1) <= ENCORE_EDGE_NOALLOC_MAX_DOUBLES  (the c3/c4 shape,
 * 69 multiplets x 120 bin tuples, needs 579 600); anything larger is refused with ENCORE_ETOOBIG before any GPU work,
 * n_lambda < 1 or n_b < 1 or a NULL pointer with ENCORE_EINVAL.
 *
 * First call on a device: it looks up the array's address on the current device (cudaGetSymbolAddress) and remembers it
 * per device; make that first call, with the device current, before starting any stream capture.  Later calls only launch
 * the two kernels on cuda_stream and return without synchronising.
 * Sharing: every call on a device uses the same array.  The part a call uses is overwritten in full before it is read, so
 * nothing left behind by an earlier call (of any shape) can reach the result and nothing needs clearing; but two calls
 * whose kernels can overlap on the GPU - different streams, or two host threads - race on it and give garbage.  Keep all
 * calls of a device on one stream, or order them with events. */
#define ENCORE_EDGE_NOALLOC_MAX_DOUBLES 1048576
int encore_edge_correct_noalloc(const double *gaunt, const double *n_raw, const double *r_raw, int n_lambda, int n_b,
                                double *zeta_out, void *cuda_stream);

/* Plan options (host call, takes effect at the next encore_compute).  No behaviour is read from the environment.
 *   "list_mb"          byte budget, in MiB, of the pair stage's acceptance-mask rows per super-step (0 = default:
 *                      32 GiB, or half of the free device memory within 4-96 GiB when the rows need more)
 *   "sub_yz", "sub_x"  grid subdivisions S_y = S_z and S_x of reading R11 (cell size r_max / S; 0 = automatic:
 *                      S_y = clamp(round(r_max / (32 / density)^(1/3)), 1, 8), S_x = 4 S_y halved until <= 4e6 cells)
 *   "nchunk"           chunks of primaries per multiplet group in the factorised contraction kernels (grid = nchunk x CTA
 *                      columns; 0 = automatic)
 *   "generic_contract" 1: contract with the literal eq. 44 kernel (one warp per (Lambda, B)) instead of the
 *                      factorised kernels
 * Unknown key or value out of range: ENCORE_EINVAL. */
int encore_set_option(encore_plan_t *plan, const char *key, long long value);
/* Synchronises the last compute's stream and reports its device-side status: ENCORE_OK, or ENCORE_EINTERNAL if the
 * pair stage's consistency check (one periodic image per candidate word) failed; after
 * encore_compute_enqueue also ENCORE_EDOMAIN / ENCORE_ECAPACITY (see there).  encore_compute_host returns this status itself.
 * After encore_compute_grid it synchronises that call's stream and returns ENCORE_OK (the gridded path has no device-side
 * checks); encore_get_launch_count and the timers are valid then, the particle diagnostics return ENCORE_ESTATE.
 * The stream it waits on is the one the compute was ENQUEUED on: after replaying a CUDA graph captured around
 * encore_compute_enqueue, synchronise the replay stream yourself before calling this. */
int encore_get_status(const encore_plan_t *plan);
/* super-steps the pair stage of the last compute took: the acceptance-mask rows of a step stay under the byte budget
 * (option "list_mb"), whole groups per step, steps of equal size.  >= 1, or a status < 0. */
int encore_get_pair_steps(const encore_plan_t *plan);
/* groups of the last compute: out = {first group, one past the last group, number of groups} (HOST) */
int encore_get_shard_groups(const encore_plan_t *plan, int out[3]);

int encore_destroy(encore_plan_t *plan);

/* ---- host queries (valid right after encore_plan, no GPU needed) ---- */
int64_t encore_zeta_len(const encore_plan_t *plan);        /* n_Lambda * n_B */
int encore_num_multiplets(const encore_plan_t *plan);      /* n_Lambda (69 for N=4,lmax=5; 204 for N=5,lmax=3) */
int encore_num_bin_tuples(const encore_plan_t *plan);      /* n_B = C(nbins, N-1) */
int64_t encore_num_terms(const encore_plan_t *plan);       /* non-zero (Lam, M) with m_{N-1} >= 0 (1126 for N=4,lmax=5) */
int encore_get_multiplets(const encore_plan_t *plan, int *out /* HOST [n_Lambda][2N-5] */);
int encore_get_bin_tuples(const encore_plan_t *plan, int *out /* HOST [n_B][N-1] */);
int encore_get_multiplet_parity(const encore_plan_t *plan, int *out /* HOST [n_Lambda]: 0 even (Re zeta stored), 1 odd (Im zeta) */);
int encore_get_bin_edges(const encore_plan_t *plan, double *out /* HOST [nbins+1] */);
/* flop counts per primary of the contraction as executed (fused multiply-add = 2) and by the canonical
 * "Algorithm 3 literal" model of SURVEY.md §8(d) (5/11/17 flop per term evaluation for N=3/4/5) */
int encore_contraction_flops(const encore_plan_t *plan, double *executed, double *canonical);

/* How the contraction (step a5) of this plan is laid out - a host query for tests and benchmarks, so that they can tell
 * which kernel and which tile pipeline a shape runs on.  out = { order of the factorised kernel (3, 4, 5, 6) or 0 when the
 * literal eq. 44 kernel is used,  number of CTA work plans (0 for N = 3 and the literal kernel),  smallest and largest
 * number of a_lm tile buffers over those CTAs: 1 = one buffer refilled between tiles, 2 = double buffer, 3..8 = ring }. */
int encore_get_contraction_layout(const encore_plan_t *plan, int out[4] /* HOST */);

/* The grid a compute would build for n particles in the box [bbox_lo, bbox_hi] (open geometry; ignored when the plan is
 * periodic): cells per axis and subdivisions S_a of reading R11 / DESIGN.md §4.1.  Host arithmetic only, no GPU needed. */
int encore_query_grid(const encore_plan_t *plan, int64_t n, const double *bbox_lo, const double *bbox_hi, int nc[3] /* HOST */,
                      int sub[3] /* HOST */);

/* ---- diagnostics of the last successful encore_compute (each synchronises the compute stream) ---- */
/* grid geometry chosen for that input: cells per axis, subdivisions S_a with cell size r_max/S_a (reading R11) */
int encore_get_grid(const encore_plan_t *plan, int nc[3] /* HOST */, int sub[3] /* HOST */);
int encore_get_cell_ids(const encore_plan_t *plan, int32_t *out /* DEVICE [n], input order */);
int encore_get_bin_counts(const encore_plan_t *plan, uint64_t *counts /* HOST [nbins] */,
                          uint64_t *pairs_total /* HOST, may be NULL */);
int encore_get_primary_counts(const encore_plan_t *plan, uint32_t *out /* DEVICE [n][nbins], input order */);
/* a^b_lm of input-order primary i: HOST [nbins][(lmax+1)(lmax+2)/2][2] (re,im), (l,m>=0) at l(l+1)/2+m */
int encore_get_alm(const encore_plan_t *plan, int64_t i, double *out);
/* stage times of that call in ms: [0] grid (cell ids + histogram), [1] sort (scan, scatter, rank, gather, groups),
 * [2] pair (a3+a4), [3] contraction (a5), [4] reduction (a6).  Only measured when timing is enabled. */
int encore_get_stage_ms(const encore_plan_t *plan, float ms[5]);
/* per-kernel times of that call in ms, summed over the pair-stage super-steps: [0] grid (bounding box, cell ids),
 * [1] sort, [2] k_group_bound + scan + the host read of the word counts, [3] k_fill, [4] k_harm (all passes),
 * [5] contraction kernel, [6] reduction.  Only measured when timing is enabled. */
int encore_get_kernel_ms(const encore_plan_t *plan, float ms[7]);
int encore_set_timing(encore_plan_t *plan, int enabled);   /* record per-stage CUDA events (default off) */
/* number of kernel launches the last encore_compute enqueued */
int encore_get_launch_count(const encore_plan_t *plan);
/* candidate pairs tested in step a3 by the last compute (>= accepted pairs), for the rejected-pair flop term */
int encore_get_candidate_pairs(const encore_plan_t *plan, uint64_t *out /* HOST */);

/* lane utilisation of step a4 in the last compute: k_harm walks the pairs of 32 primaries in lock step, one warp per
 * (group of 32 primaries, bin); `executed` = lock-step pair steps summed over warps, `ideal` = sum over warps of the
 * largest pair count among the warp's primaries (what a perfectly packed schedule would execute).  Both read 0 unless
 * the library was built with -DENCORE_HARM_STATS (the counters cost a few percent of k_harm). */
int encore_get_harm_steps(const encore_plan_t *plan, uint64_t *executed /* HOST */, uint64_t *ideal /* HOST */);

/* Dependent-DFMA-chain micro-benchmark on the current device: achieved fp64 FLOP/s (FMA = 2) with every SM busy.
 * The ALU roofline denominator reported by bench.py beside the derived 148 SM x 64 lanes x 2 x f_clk. */
int encore_measure_fp64_peak(double *flops_per_s /* HOST */, void *cuda_stream);
/* The same for the fp64 tensor-core path, mma.sync.m8n8k4.f64 in independent accumulator chains on every SM (FLOP/s, FMA = 2):
 * the number that decides whether recasting a contraction as fp64 MMAs could pay. */
int encore_measure_dmma_peak(double *flops_per_s /* HOST */, void *cuda_stream);

const char *encore_strerror(int status);
int encore_last_cuda_error(void); /* cudaError_t of the most recent ENCORE_ECUDA on this thread */

#ifdef __cplusplus
}
#endif
#endif /* ENCORE_H */
