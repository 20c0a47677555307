/*
 * oracle/encore_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement of what the ENCORE hot path computes
 * (arxiv 2105.08722; citations are PAPER.md line + equation).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or constant with the
 * CUDA library under paper_2105_08722_b200/ and neither includes the other.
 *
 * What it computes (fp64 arithmetic, long-double accumulation of every sum over particles):
 *
 *   a^b_lm(s_i) = (1/v_b) sum_{j != i} w_j Y_lm( (r_j - s_i)^ ) Theta^b(|r_j - s_i|)      eq. 35
 *   zeta^B_Lam  = (1/V) sum_i w_i sum_M E(Lam) C^Lam_M prod_k a^{b_k}_{l_k m_k}(s_i)        eq. 34
 *
 * with the FULL sum over M = (m_1..m_{N-1}) (no half-sum trick of eq. 44; that identity is
 * a test), C^Lam_M from eq. 5 specialised as eqs. 16/18/20,
 * Y_lm in the Condon-Shortley convention, bins b_1<b_2<..<b_{N-1} unless an
 * explicit tuple list is passed.
 *
 * Readings of silent / garbled points (DESIGN.md §3 lists them all):
 *   R1  Y_lm = (-1)^m sqrt((2l+1)/(4pi) (l-m)!/(l+m)!) P_l^m(cos th) e^{i m phi}, m>=0, P_l^m without
 *       the CS phase; Y_{l,-m} = (-1)^m conj(Y_lm).
 *   R2  eq. 20 as printed lacks the sqrt(2 l12 + 1) that eq. 5 carries; eq. 5 is followed.
 *   R3  eq. 21's second 3-j bottom row is a misprint; (m12 m3 m4) as in eq. 20.
 *   R5  intermediate l12 is NOT capped at lmax (|l1-l2| <= l12 <= l1+l2).
 *   R7  separation vector is r_j - s_i (eq. 35).
 *   R8  half-open bins e_b <= r < e_{b+1}, decided on squares; additionally r^2 > 0 and j != i.
 *   R10 per axis d = x_j - x_i; if (d > L/2) d -= L; else if (d < -L/2) d += L;
 *       r^2 = fma(dz,dz, fma(dy,dy, dx*dx)).
 *   R11 cell id: see oracle_cell_ids.
 *   R12 V = L^3 (periodic) or 1 (open); 1/v_b inside every a_lm, v_b = 4pi/3 (e_{b+1}^3 - e_b^3).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): exact 3-j values and sum rules; scipy Y_lm;
 * orthonormality sum_M |C|^2 = 1 (decides R2); printed enumeration counts 69/204/381/1126/...
 * (PAPER.md:537,586,594,606); brute-force N-tuple sums with Cartesian closed forms
 * (eq. 17 Legendre, P_110 PAPER.md:558, P_11(0)11) and with eq. 4 via scipy/sympy; the l=0
 * identity; rotation invariance; (l,b) permutation symmetry.  Nothing here is "parity unpinned".
 *
 * Build: gcc -O2 -std=c11 -fopenmp -ffp-contract=off -fcx-limited-range -shared -fPIC
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_MAX_ORDER 6
#define ORACLE_MAX_L 16
#define PI_L 3.14159265358979323846264338327950288L

/* ------------------------------------------------------------------------------------------
 * Wigner 3-j symbol (NIST DLMF 34.2.4, Racah's sum), used by eq. 5.
 * With A=j1+j2-j3, B=j1-j2+j3, C=-j1+j2+j3 every term of Racah's sum is a product of three
 * binomials over A!B!C!:
 *   1/[k!(A-k)! (j1-m1-k)!(B-(j1-m1-k))! (j2+m2-k)!(C-(j2+m2-k))!]
 * so the alternating sum is an exact integer; only the square-root prefactor is floating.
 * ------------------------------------------------------------------------------------------ */
static long double factl(int n)
{
    long double f = 1.0L;
    for (int i = 2; i <= n; ++i) f *= (long double)i;
    return f;
}

static __int128 binom(int n, int k)
{
    if (k < 0 || k > n) return 0;
    __int128 r = 1;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i; /* exact: r holds C(n-k+i, i) */
    return r;
}

double oracle_wigner3j(int j1, int j2, int j3, int m1, int m2, int m3)
{
    if (m1 + m2 + m3 != 0) return 0.0;
    if (abs(m1) > j1 || abs(m2) > j2 || abs(m3) > j3) return 0.0;
    if (j3 < abs(j1 - j2) || j3 > j1 + j2) return 0.0;
    const int A = j1 + j2 - j3, B = j1 - j2 + j3, C = -j1 + j2 + j3;
    __int128 sum = 0;
    for (int k = 0; k <= A; ++k) {
        __int128 t = binom(A, k) * binom(B, j1 - m1 - k) * binom(C, j2 + m2 - k);
        sum += (k & 1) ? -t : t;
    }
    long double pref = factl(j1 + m1) * factl(j1 - m1) * factl(j2 + m2) * factl(j2 - m2) *
                       factl(j3 + m3) * factl(j3 - m3) /
                       (factl(A) * factl(B) * factl(C) * factl(j1 + j2 + j3 + 1));
    long double v = sqrtl(pref) * (long double)sum;
    int ph = j1 - j2 - m3;
    if (ph & 1) v = -v;
    return (double)v;
}

/* ------------------------------------------------------------------------------------------
 * Spherical harmonics, reading R1.  out index: l*l + l + m, -l<=m<=l, 0<=l<=lmax.
 * (x,y,z) must be a unit vector.  cos th = z, sin th = hypot(x,y), e^{i phi} = (x+iy)/sin th.
 * ------------------------------------------------------------------------------------------ */
static double g_norm[ORACLE_MAX_L + 1][ORACLE_MAX_L + 1]; /* sqrt((2l+1)/(4pi) (l-m)!/(l+m)!) */
static int g_norm_ready = 0;
static void norm_init(void) /* called before any parallel region */
{
    if (g_norm_ready) return;
    for (int l = 0; l <= ORACLE_MAX_L; ++l)
        for (int m = 0; m <= l; ++m)
            g_norm[l][m] = (double)sqrtl((2 * l + 1) / (4.0L * PI_L) * factl(l - m) / factl(l + m));
    g_norm_ready = 1;
}

static void ylm_all(int lmax, double x, double y, double z, double complex *out)
{
    double P[ORACLE_MAX_L + 1][ORACLE_MAX_L + 1]; /* P_l^m(z), no Condon-Shortley phase */
    const double s = sqrt(x * x + y * y);
    for (int m = 0; m <= lmax; ++m) {
        double pmm = 1.0; /* (2m-1)!! s^m */
        for (int k = 1; k <= m; ++k) pmm *= (2 * k - 1) * s;
        P[m][m] = pmm;
        if (m + 1 <= lmax) P[m + 1][m] = z * (2 * m + 1) * pmm;
        for (int l = m + 2; l <= lmax; ++l)
            P[l][m] = ((2 * l - 1) * z * P[l - 1][m] - (l + m - 1) * P[l - 2][m]) / (double)(l - m);
    }
    const double complex eiphi = (s > 0.0) ? (x + I * y) / s : 1.0;
    double complex em = 1.0; /* e^{i m phi} */
    for (int m = 0; m <= lmax; ++m) {
        for (int l = m; l <= lmax; ++l) {
            const double norm = g_norm[l][m];
            double complex Y = ((m & 1) ? -1.0 : 1.0) * norm * P[l][m] * em;
            out[l * l + l + m] = Y;
            if (m > 0) out[l * l + l - m] = ((m & 1) ? -1.0 : 1.0) * conj(Y);
        }
        em *= eiphi;
    }
}

void oracle_ylm(int lmax, double x, double y, double z, double *out_re, double *out_im)
{
    double complex Y[(ORACLE_MAX_L + 1) * (ORACLE_MAX_L + 1)];
    norm_init();
    ylm_all(lmax, x, y, z, Y);
    for (int k = 0; k < (lmax + 1) * (lmax + 1); ++k) {
        out_re[k] = creal(Y[k]);
        out_im[k] = cimag(Y[k]);
    }
}

/* ------------------------------------------------------------------------------------------
 * Multiplets Lambda in the order of Alg. 3 / Fig. 4:
 * nested ascending loops, last index fastest.  Width of a row: 2N-5 (N=3: {l}; N=4: {l1,l2,l3};
 * N=5: {l1,l2,l12,l3,l4}; N=6: {l1,l2,l12,l3,l123,l4,l5}).  Intermediates run over their whole
 * triangle range (R5); principal l's up to lmax.  allparity=0 keeps E(Lam)=+1 only (even sum of PRINCIPAL l's).
 * Returns the number of multiplets; writes them if out != NULL.
 * ------------------------------------------------------------------------------------------ */
int oracle_multiplets(int order, int lmax, int allparity, int *out)
{
    int n = 0;
    if (order == 3) {
        for (int l = 0; l <= lmax; ++l) {
            if (out) out[n] = l;
            ++n;
        }
    } else if (order == 4) {
        for (int l1 = 0; l1 <= lmax; ++l1)
            for (int l2 = 0; l2 <= lmax; ++l2)
                for (int l3 = abs(l1 - l2); l3 <= l1 + l2 && l3 <= lmax; ++l3) {
                    if (!allparity && ((l1 + l2 + l3) & 1)) continue;
                    if (out) { out[3 * n] = l1; out[3 * n + 1] = l2; out[3 * n + 2] = l3; }
                    ++n;
                }
    } else if (order == 5) {
        for (int l1 = 0; l1 <= lmax; ++l1)
            for (int l2 = 0; l2 <= lmax; ++l2)
                for (int l12 = abs(l1 - l2); l12 <= l1 + l2; ++l12) /* R5: not capped */
                    for (int l3 = 0; l3 <= lmax; ++l3)
                        for (int l4 = abs(l12 - l3); l4 <= l12 + l3 && l4 <= lmax; ++l4) {
                            if (!allparity && ((l1 + l2 + l3 + l4) & 1)) continue;
                            if (out) {
                                int *o = out + 5 * n;
                                o[0] = l1; o[1] = l2; o[2] = l12; o[3] = l3; o[4] = l4;
                            }
                            ++n;
                        }
    } else if (order == 6) {
        for (int l1 = 0; l1 <= lmax; ++l1)
            for (int l2 = 0; l2 <= lmax; ++l2)
                for (int l12 = abs(l1 - l2); l12 <= l1 + l2; ++l12)          /* R5: not capped */
                    for (int l3 = 0; l3 <= lmax; ++l3)
                        for (int l123 = abs(l12 - l3); l123 <= l12 + l3; ++l123) /* R5: not capped */
                            for (int l4 = 0; l4 <= lmax; ++l4)
                                for (int l5 = abs(l123 - l4); l5 <= l123 + l4 && l5 <= lmax; ++l5) {
                                    if (!allparity && ((l1 + l2 + l3 + l4 + l5) & 1)) continue;
                                    if (out) {
                                        int *o = out + 7 * n;
                                        o[0] = l1; o[1] = l2; o[2] = l12; o[3] = l3; o[4] = l123; o[5] = l4; o[6] = l5;
                                    }
                                    ++n;
                                }
    } else {
        return -1;
    }
    return n;
}

/* principal l's of a multiplet row */
static void principal_ls(int order, const int *Lam, int *l)
{
    if (order == 3) { l[0] = Lam[0]; l[1] = Lam[0]; }
    else if (order == 4) { l[0] = Lam[0]; l[1] = Lam[1]; l[2] = Lam[2]; }
    else if (order == 5) { l[0] = Lam[0]; l[1] = Lam[1]; l[2] = Lam[3]; l[3] = Lam[4]; }
    else { l[0] = Lam[0]; l[1] = Lam[1]; l[2] = Lam[3]; l[3] = Lam[5]; l[4] = Lam[6]; }
}

/* ------------------------------------------------------------------------------------------
 * Coupling coefficient C^Lam_M, eq. 5 with E(Lam) = (-1)^{sum of principal l}:
 *   N=3: eq. 16   (-1)^{l-m1}/sqrt(2l+1) delta_{m1,-m2}
 *   N=4: eq. 18   (-1)^{l1+l2+l3} (l1 l2 l3; m1 m2 m3)
 *   N=5: eq. 5    E sqrt(2 l12+1) sum_{m12} (-1)^{l12-m12} (l1 l2 l12; m1 m2 -m12)(l12 l3 l4; m12 m3 m4)
 *   N=6: eq. 5    E sqrt(2 l12+1) sqrt(2 l123+1) sum_{m12,m123} (-1)^{l12-m12+l123-m123}
 *                 (l1 l2 l12; m1 m2 -m12)(l12 l3 l123; m12 m3 -m123)(l123 l4 l5; m123 m4 m5)
 * (R2: the sqrt(2 l12+1) of eq. 5 is kept although eq. 20 as printed drops it.)
 * ------------------------------------------------------------------------------------------ */
double oracle_coupling(int order, const int *Lam, const int *m)
{
    if (order == 3) {
        int l = Lam[0];
        if (m[0] + m[1] != 0 || abs(m[0]) > l) return 0.0;
        return (((l - m[0]) & 1) ? -1.0 : 1.0) / sqrt(2.0 * l + 1.0);
    }
    if (order == 4) {
        int s = Lam[0] + Lam[1] + Lam[2];
        return ((s & 1) ? -1.0 : 1.0) * oracle_wigner3j(Lam[0], Lam[1], Lam[2], m[0], m[1], m[2]);
    }
    if (order == 5) {
        int l1 = Lam[0], l2 = Lam[1], l12 = Lam[2], l3 = Lam[3], l4 = Lam[4];
        int s = l1 + l2 + l3 + l4;
        double sum = 0.0;
        for (int m12 = -l12; m12 <= l12; ++m12) {
            double t = oracle_wigner3j(l1, l2, l12, m[0], m[1], -m12) *
                       oracle_wigner3j(l12, l3, l4, m12, m[2], m[3]);
            sum += (((l12 - m12) & 1) ? -1.0 : 1.0) * t;
        }
        return ((s & 1) ? -1.0 : 1.0) * sqrt(2.0 * l12 + 1.0) * sum;
    }
    if (order == 6) {
        int l1 = Lam[0], l2 = Lam[1], l12 = Lam[2], l3 = Lam[3], l123 = Lam[4], l4 = Lam[5], l5 = Lam[6];
        int s = l1 + l2 + l3 + l4 + l5;
        double sum = 0.0;
        for (int m12 = -l12; m12 <= l12; ++m12)
            for (int m123 = -l123; m123 <= l123; ++m123) {
                double t = oracle_wigner3j(l1, l2, l12, m[0], m[1], -m12) *
                           oracle_wigner3j(l12, l3, l123, m12, m[2], -m123) *
                           oracle_wigner3j(l123, l4, l5, m123, m[3], m[4]);
                sum += (((l12 - m12 + l123 - m123) & 1) ? -1.0 : 1.0) * t;
            }
        return ((s & 1) ? -1.0 : 1.0) * sqrt(2.0 * l12 + 1.0) * sqrt(2.0 * l123 + 1.0) * sum;
    }
    return 0.0;
}

/* Number of non-zero (Lam, M) terms; half!=0 keeps m_{N-1} >= 0 only (eq. 44).  For the
 * printed task counts of PAPER.md:586, :594. */
int64_t oracle_count_terms(int order, int lmax, int allparity, int half)
{
    int nL = oracle_multiplets(order, lmax, allparity, NULL);
    int width = 2 * order - 5;
    int *Lam = (int *)malloc(sizeof(int) * (size_t)nL * width);
    oracle_multiplets(order, lmax, allparity, Lam);
    int64_t cnt = 0;
    for (int iL = 0; iL < nL; ++iL) {
        int l[5], m[5];
        principal_ls(order, Lam + iL * width, l);
        int nm = order - 1;
        /* odometer over m_1..m_{N-2}; m_{N-1} = -(sum) */
        for (int k = 0; k < nm - 1; ++k) m[k] = -l[k];
        for (;;) {
            int s = 0;
            for (int k = 0; k < nm - 1; ++k) s += m[k];
            m[nm - 1] = -s;
            if (abs(m[nm - 1]) <= l[nm - 1] && (!half || m[nm - 1] >= 0)) {
                double c = oracle_coupling(order, Lam + iL * width, m);
                if (fabs(c) > 1e-14) ++cnt;
            }
            int k = nm - 2;
            while (k >= 0 && ++m[k] > l[k]) { m[k] = -l[k]; --k; }
            if (k < 0) break;
        }
    }
    free(Lam);
    return cnt;
}

/* ------------------------------------------------------------------------------------------
 * Radial bins (R8): e_b = r_min + b*width, width = (r_max-r_min)/nbins, e_nbins = r_max.
 * ------------------------------------------------------------------------------------------ */
void oracle_bin_edges(double rmin, double rmax, int nbins, double *e)
{
    const double width = (rmax - rmin) / (double)nbins;
    for (int b = 0; b < nbins; ++b) e[b] = rmin + (double)b * width;
    e[nbins] = rmax;
}

/* ------------------------------------------------------------------------------------------
 * Cell ids (R11) — an integer side output of the hot path (step a1); the oracle's own
 * neighbour search below does not use it.  `sub[a]` = subdivision S_a of axis a chosen by the plan (a free
 * design parameter, R11/R23; the cell size of axis a is rmax/S_a).
 *   periodic: nc_a = max(1, floor(L / (rmax/S_a))), origin 0, extent L
 *   open    : per axis origin = min coordinate, extent = max - min, nc_a = max(1, floor(extent/(rmax/S_a)))
 *   inv = nc / extent (1 if extent == 0);  i = min(nc-1, (int)((x - origin) * inv));
 *   cid = (iz*nc_y + iy)*nc_x + ix
 * ------------------------------------------------------------------------------------------ */
int oracle_cell_ids(const double *pos, int64_t n, double box, double rmax, const int *sub, int32_t *cid,
                    int *nc_out)
{
    const double *p[3] = {pos, pos + n, pos + 2 * n};
    double org[3], inv[3];
    int nc[3];
    for (int a = 0; a < 3; ++a) {
        const double h = rmax / (double)sub[a];
        double ext;
        if (box > 0.0) { org[a] = 0.0; ext = box; }
        else {
            double lo = p[a][0], hi = p[a][0];
            for (int64_t i = 1; i < n; ++i) { if (p[a][i] < lo) lo = p[a][i]; if (p[a][i] > hi) hi = p[a][i]; }
            org[a] = lo; ext = hi - lo;
        }
        double q = floor(ext / h);
        nc[a] = (q < 1.0) ? 1 : (int)q;
        inv[a] = (ext > 0.0) ? (double)nc[a] / ext : 1.0;
        nc_out[a] = nc[a];
    }
    for (int64_t i = 0; i < n; ++i) {
        int c[3];
        for (int a = 0; a < 3; ++a) {
            int v = (int)((p[a][i] - org[a]) * inv[a]);
            c[a] = v > nc[a] - 1 ? nc[a] - 1 : v;
        }
        cid[i] = (c[2] * nc[1] + c[1]) * nc[0] + c[0];
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * The oracle's own neighbour search: all pairs for small n, else a plain cell list with cells
 * >= rmax wide (27-cell stencil).  Only a way of skipping pairs that are certainly rejected.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    int use;           /* 0: all pairs */
    int nc[3];
    double org[3], inv[3];
    int64_t *start;    /* [ncell+1] */
    int64_t *idx;      /* [n] particle indices grouped by cell */
} cell_list;

static void cl_build(cell_list *cl, const double *pos, int64_t n, double box, double rmax, int force_allpairs)
{
    memset(cl, 0, sizeof(*cl));
    if (force_allpairs || n <= 4096) return;
    const double *p[3] = {pos, pos + n, pos + 2 * n};
    for (int a = 0; a < 3; ++a) {
        double ext;
        if (box > 0.0) { cl->org[a] = 0.0; ext = box; }
        else {
            double lo = p[a][0], hi = p[a][0];
            for (int64_t i = 1; i < n; ++i) { if (p[a][i] < lo) lo = p[a][i]; if (p[a][i] > hi) hi = p[a][i]; }
            cl->org[a] = lo; ext = hi - lo;
        }
        double q = floor(ext / (rmax * 1.000001));
        cl->nc[a] = q < 1.0 ? 1 : (q > 512.0 ? 512 : (int)q);
        cl->inv[a] = ext > 0.0 ? cl->nc[a] / ext : 1.0;
        if (box > 0.0 && cl->nc[a] < 3) return; /* periodic stencil would alias: all pairs */
    }
    cl->use = 1;
    int64_t ncell = (int64_t)cl->nc[0] * cl->nc[1] * cl->nc[2];
    cl->start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
    cl->idx = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    int64_t *cell = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        int c[3];
        for (int a = 0; a < 3; ++a) {
            int v = (int)((p[a][i] - cl->org[a]) * cl->inv[a]);
            if (v < 0) v = 0;
            c[a] = v > cl->nc[a] - 1 ? cl->nc[a] - 1 : v;
        }
        cell[i] = ((int64_t)c[2] * cl->nc[1] + c[1]) * cl->nc[0] + c[0];
        cl->start[cell[i] + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) cl->start[c + 1] += cl->start[c];
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)ncell);
    memcpy(fill, cl->start, sizeof(int64_t) * (size_t)ncell);
    for (int64_t i = 0; i < n; ++i) cl->idx[fill[cell[i]]++] = i;
    free(fill);
    free(cell);
}

static void cl_free(cell_list *cl)
{
    free(cl->start);
    free(cl->idx);
}

/* ------------------------------------------------------------------------------------------
 * a^b_lm(s_i) for one primary (eq. 35; Alg. 1 l.3-13).
 * alm: [nbins][(lmax+1)^2] complex, index l*l+l+m (all m); counts: [nbins] accepted pairs.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    const double *x, *y, *z, *w;
    int64_t n;
    double box, half;
    int nbins, lmax, nlm;
    const double *e2;   /* squared edges [nbins+1] */
    const double *vinv; /* 1/v_b */
} pair_ctx;

static inline void pair_one(const pair_ctx *c, int64_t i, int64_t j, long double *acc_re,
                            long double *acc_im, uint32_t *counts)
{
    if (j == i) return;
    double dx = c->x[j] - c->x[i], dy = c->y[j] - c->y[i], dz = c->z[j] - c->z[i]; /* R7 */
    if (c->box > 0.0) { /* R10 minimal image */
        if (dx > c->half) dx -= c->box; else if (dx < -c->half) dx += c->box;
        if (dy > c->half) dy -= c->box; else if (dy < -c->half) dy += c->box;
        if (dz > c->half) dz -= c->box; else if (dz < -c->half) dz += c->box;
    }
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    if (!(r2 > 0.0) || r2 < c->e2[0] || !(r2 < c->e2[c->nbins])) return; /* R8 */
    int b = 0;
    while (!(r2 < c->e2[b + 1])) ++b; /* R9: e_b^2 <= r2 < e_{b+1}^2 */
    counts[b]++;
    const double r = sqrt(r2);
    double complex Y[(ORACLE_MAX_L + 1) * (ORACLE_MAX_L + 1)];
    ylm_all(c->lmax, dx / r, dy / r, dz / r, Y);
    const double wj = c->w ? c->w[j] : 1.0;
    long double *ar = acc_re + (size_t)b * c->nlm, *ai = acc_im + (size_t)b * c->nlm;
    for (int k = 0; k < c->nlm; ++k) {
        ar[k] += (long double)(wj * creal(Y[k]));
        ai[k] += (long double)(wj * cimag(Y[k]));
    }
}

static void alm_primary(const pair_ctx *c, const cell_list *cl, int64_t i, double complex *alm,
                        uint32_t *counts, long double *acc_re, long double *acc_im)
{
    const size_t tot = (size_t)c->nbins * c->nlm;
    for (size_t k = 0; k < tot; ++k) { acc_re[k] = 0.0L; acc_im[k] = 0.0L; }
    for (int b = 0; b < c->nbins; ++b) counts[b] = 0;
    if (!cl->use) {
        for (int64_t j = 0; j < c->n; ++j) pair_one(c, i, j, acc_re, acc_im, counts);
    } else {
        const double pi[3] = {c->x[i], c->y[i], c->z[i]};
        int ci[3];
        for (int a = 0; a < 3; ++a) {
            int v = (int)((pi[a] - cl->org[a]) * cl->inv[a]);
            if (v < 0) v = 0;
            ci[a] = v > cl->nc[a] - 1 ? cl->nc[a] - 1 : v;
        }
        for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int cc[3] = {ci[0] + dx, ci[1] + dy, ci[2] + dz};
                    int ok = 1;
                    for (int a = 0; a < 3; ++a) {
                        if (c->box > 0.0) cc[a] = (cc[a] + cl->nc[a]) % cl->nc[a];
                        else if (cc[a] < 0 || cc[a] >= cl->nc[a]) ok = 0;
                    }
                    if (!ok) continue;
                    int64_t cell = ((int64_t)cc[2] * cl->nc[1] + cc[1]) * cl->nc[0] + cc[0];
                    for (int64_t t = cl->start[cell]; t < cl->start[cell + 1]; ++t)
                        pair_one(c, i, cl->idx[t], acc_re, acc_im, counts);
                }
    }
    for (int b = 0; b < c->nbins; ++b)
        for (int k = 0; k < c->nlm; ++k) {
            size_t o = (size_t)b * c->nlm + k;
            alm[o] = (double)(acc_re[o] * (long double)c->vinv[b]) +
                     I * (double)(acc_im[o] * (long double)c->vinv[b]);
        }
}

static void ctx_init(pair_ctx *c, const double *pos, const double *w, int64_t n, double box,
                     double rmin, double rmax, int nbins, int lmax, double *e2, double *vinv)
{
    double e[256];
    norm_init();
    oracle_bin_edges(rmin, rmax, nbins, e);
    for (int b = 0; b <= nbins; ++b) e2[b] = e[b] * e[b];
    for (int b = 0; b < nbins; ++b) /* v_b = 4 pi/3 (e_{b+1}^3 - e_b^3) */
        vinv[b] = (double)(1.0L / (4.0L * PI_L / 3.0L *
                  ((long double)e[b + 1] * e[b + 1] * e[b + 1] - (long double)e[b] * e[b] * e[b])));
    c->x = pos; c->y = pos + n; c->z = pos + 2 * n; c->w = w; c->n = n;
    c->box = box; c->half = 0.5 * box; c->nbins = nbins; c->lmax = lmax;
    c->nlm = (lmax + 1) * (lmax + 1); c->e2 = e2; c->vinv = vinv;
}

/* a_lm tile + per-bin counts of one primary (diagnostic / sampled parity). */
int oracle_alm(const double *pos, const double *w, int64_t n, double box, double rmin, double rmax,
               int nbins, int lmax, int64_t i, int force_allpairs, double *alm_re, double *alm_im,
               uint32_t *counts)
{
    if (lmax > ORACLE_MAX_L || nbins > 255 || i < 0 || i >= n) return -1;
    double e2[256], vinv[256];
    pair_ctx c;
    ctx_init(&c, pos, w, n, box, rmin, rmax, nbins, lmax, e2, vinv);
    cell_list cl;
    cl_build(&cl, pos, n, box, rmax, force_allpairs);
    size_t tot = (size_t)nbins * c.nlm;
    double complex *alm = (double complex *)malloc(sizeof(double complex) * tot);
    long double *ar = (long double *)malloc(sizeof(long double) * tot * 2);
    alm_primary(&c, &cl, i, alm, counts, ar, ar + tot);
    for (size_t k = 0; k < tot; ++k) { alm_re[k] = creal(alm[k]); alm_im[k] = cimag(alm[k]); }
    free(alm); free(ar); cl_free(&cl);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * zeta^B_Lam (eq. 34) over the primaries i = prim_offset, prim_offset+prim_stride, ... < n
 * (all of them for offset 0, stride 1; a strided subset is one shard of the sum over i).
 *   bins     : [nB][N-1] explicit bin tuples, or NULL for all b_1<..<b_{N-1} in lexicographic
 *              order (Alg. 3 l.9-13); nB is then ignored and recomputed.
 *   zeta     : [nLam][nB] real part; max_imag: largest |Im| met (must be ~0 for even parity)
 *   zeta_im  : optional [nLam][nB] imaginary part (odd parity) or NULL
 *   bin_counts: [nbins] accepted ordered pairs over the processed primaries
 *   prim_counts: optional [n][nbins] (rows of unprocessed primaries untouched)
 *   stage_seconds: optional [2]: wall-clock seconds spent in step (i) (a_lm of every primary) and in steps
 *              (ii)+(iii) (contraction and sum), each averaged over the OpenMP threads (timing only)
 * ------------------------------------------------------------------------------------------ */
static int64_t n_choose(int n, int k)
{
    if (k < 0 || k > n) return 0;
    int64_t r = 1;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
    return r;
}

int64_t oracle_bin_tuples(int order, int nbins, int *out)
{
    int k = order - 1, b[5];
    int64_t cnt = 0;
    if (k > nbins) return 0;
    for (int i = 0; i < k; ++i) b[i] = i;
    for (;;) {
        if (out) for (int i = 0; i < k; ++i) out[cnt * k + i] = b[i];
        ++cnt;
        int i = k - 1;
        while (i >= 0 && b[i] == nbins - k + i) --i;
        if (i < 0) break;
        ++b[i];
        for (int t = i + 1; t < k; ++t) b[t] = b[t - 1] + 1;
    }
    return cnt;
}

static double wall_seconds(void)
{
#ifdef _OPENMP
    return omp_get_wtime();
#else
    return 0.0;
#endif
}

typedef struct { int idx[5]; double c; } term_t; /* idx[k] = l_k*l_k + l_k + m_k; c = E(Lam) C^Lam_M */

int oracle_zeta(int order, const double *pos, const double *w, int64_t n, double box, double rmin,
                double rmax, int nbins, int lmax, int allparity, const int *bins, int64_t nB,
                int64_t prim_offset, int64_t prim_stride, int force_allpairs, double *zeta,
                double *zeta_im, uint64_t *bin_counts, uint32_t *prim_counts, double *max_imag,
                double *stage_seconds)
{
    if (order < 3 || order > ORACLE_MAX_ORDER || lmax > ORACLE_MAX_L || nbins > 255 || n < 1) return -1;
    if (box > 0.0 && rmax > 0.5 * box) return -2;
    if (prim_stride < 1 || prim_offset < 0) return -3;
    const int nm = order - 1, width = 2 * order - 5;
    double e2[256], vinv[256];
    pair_ctx c;
    ctx_init(&c, pos, w, n, box, rmin, rmax, nbins, lmax, e2, vinv);

    /* bin tuples */
    int *own_bins = NULL;
    if (!bins) {
        nB = n_choose(nbins, nm);
        own_bins = (int *)malloc(sizeof(int) * (size_t)(nB > 0 ? nB : 1) * nm);
        oracle_bin_tuples(order, nbins, own_bins);
        bins = own_bins;
    }
    /* multiplets and their non-zero (M, E*C) lists: the full M sum of eq. 34 */
    const int nL = oracle_multiplets(order, lmax, allparity, NULL);
    int *Lam = (int *)malloc(sizeof(int) * (size_t)nL * width);
    oracle_multiplets(order, lmax, allparity, Lam);
    int64_t *tstart = (int64_t *)calloc((size_t)nL + 1, sizeof(int64_t));
    size_t tcap = 1024, tn = 0;
    term_t *terms = (term_t *)malloc(sizeof(term_t) * tcap);
    for (int iL = 0; iL < nL; ++iL) {
        int l[5], m[5], sl = 0;
        principal_ls(order, Lam + iL * width, l);
        for (int k = 0; k < nm; ++k) sl += l[k];
        const double E = (sl & 1) ? -1.0 : 1.0;
        for (int k = 0; k < nm - 1; ++k) m[k] = -l[k];
        for (;;) {
            int s = 0;
            for (int k = 0; k < nm - 1; ++k) s += m[k];
            m[nm - 1] = -s;
            if (abs(m[nm - 1]) <= l[nm - 1]) {
                double cf = oracle_coupling(order, Lam + iL * width, m);
                if (cf != 0.0) {
                    if (tn == tcap) { tcap *= 2; terms = (term_t *)realloc(terms, sizeof(term_t) * tcap); }
                    for (int k = 0; k < nm; ++k) terms[tn].idx[k] = l[k] * l[k] + l[k] + m[k];
                    terms[tn].c = E * cf;
                    ++tn;
                }
            }
            int k = nm - 2;
            while (k >= 0 && ++m[k] > l[k]) { m[k] = -l[k]; --k; }
            if (k < 0) break;
        }
        tstart[iL + 1] = (int64_t)tn;
    }

    cell_list cl;
    cl_build(&cl, pos, n, box, rmax, force_allpairs);
    const double Vinv = box > 0.0 ? 1.0 / (box * box * box) : 1.0; /* R12 */
    const size_t nout = (size_t)nL * (size_t)nB, tile = (size_t)nbins * c.nlm;

    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
    long double *part = (long double *)calloc(nout * 2 * (size_t)nthreads, sizeof(long double));
    uint64_t *cpart = (uint64_t *)calloc((size_t)nbins * nthreads, sizeof(uint64_t));
    double *imax = (double *)calloc((size_t)nthreads, sizeof(double));
    double *tsec = (double *)calloc((size_t)nthreads * 2, sizeof(double));
    const int64_t nprim = prim_offset < n ? (n - prim_offset + prim_stride - 1) / prim_stride : 0;

#pragma omp parallel
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        long double *zr = part + (size_t)tid * nout * 2, *zi = zr + nout;
        uint64_t *cc = cpart + (size_t)tid * nbins;
        double complex *alm = (double complex *)malloc(sizeof(double complex) * tile);
        long double *acc = (long double *)malloc(sizeof(long double) * tile * 2);
        uint32_t cnt[256];
#pragma omp for schedule(dynamic, 8)
        for (int64_t ip = 0; ip < nprim; ++ip) {
            const int64_t i = prim_offset + ip * prim_stride;
            const double t0 = wall_seconds();
            alm_primary(&c, &cl, i, alm, cnt, acc, acc + tile);      /* step (i) */
            const double t1 = wall_seconds();
            for (int b = 0; b < nbins; ++b) {
                cc[b] += cnt[b];
                if (prim_counts) prim_counts[(size_t)i * nbins + b] = cnt[b];
            }
            const double wi = w ? w[i] : 1.0;
            for (int iL = 0; iL < nL; ++iL)                           /* step (ii) */
                for (int64_t iB = 0; iB < nB; ++iB) {
                    const int *b = bins + iB * nm;
                    double complex H = 0.0;
                    for (int64_t t = tstart[iL]; t < tstart[iL + 1]; ++t) {
                        double complex pr = terms[t].c;
                        for (int k = 0; k < nm; ++k) pr *= alm[(size_t)b[k] * c.nlm + terms[t].idx[k]];
                        H += pr;
                    }
                    zr[(size_t)iL * nB + iB] += (long double)(wi * creal(H)); /* step (iii) */
                    zi[(size_t)iL * nB + iB] += (long double)(wi * cimag(H));
                }
            tsec[2 * tid] += t1 - t0;
            tsec[2 * tid + 1] += wall_seconds() - t1;
        }
        free(alm); free(acc);
    }
    /* combine the per-thread sums in thread order */
    double mi = 0.0;
    for (size_t o = 0; o < nout; ++o) {
        long double sr = 0.0L, si = 0.0L;
        for (int t = 0; t < nthreads; ++t) { sr += part[(size_t)t * nout * 2 + o]; si += part[(size_t)t * nout * 2 + nout + o]; }
        zeta[o] = (double)(sr * (long double)Vinv);
        double im = (double)(si * (long double)Vinv);
        if (zeta_im) zeta_im[o] = im;
        if (fabs(im) > mi) mi = fabs(im);
    }
    if (max_imag) *max_imag = mi;
    if (stage_seconds) {
        stage_seconds[0] = stage_seconds[1] = 0.0;
        for (int t = 0; t < nthreads; ++t) { stage_seconds[0] += tsec[2 * t] / nthreads; stage_seconds[1] += tsec[2 * t + 1] / nthreads; }
    }
    if (bin_counts)
        for (int b = 0; b < nbins; ++b) {
            uint64_t s = 0;
            for (int t = 0; t < nthreads; ++t) s += cpart[(size_t)t * nbins + b];
            bin_counts[b] = s;
        }
    free(part); free(cpart); free(imax); free(tsec); free(terms); free(tstart); free(Lam); free(own_bins);
    cl_free(&cl);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Edge correction (eqs. 37-42).
 * Gaunt integral, eq. 13:
 *   G^{l1 l2 l3}_{m1 m2 m3} = sqrt((2l1+1)(2l2+1)(2l3+1)/(4 pi)) (l1 l2 l3; m1 m2 m3)(l1 l2 l3; 0 0 0)
 *                           = int d r^ Y_{l1 m1} Y_{l2 m2} Y_{l3 m3}.
 * Generalised Gaunt integral, eq. 15, written out from its definition with eq. 4:
 *   G^{Lam Lam' Lam''} = int dR^ P_Lam P_Lam' P_Lam''
 *                      = sum_{M, M'} C^Lam_M C^Lam'_M' C^Lam''_M'' prod_k G^{l_k l'_k l''_k}_{m_k m'_k m''_k},  m''_k = -m_k - m'_k
 * (the Gaunt integral vanishes unless its m's sum to zero).  No 9-j symbols: App. A's closed forms (A1-A3, whose 9-j
 * rows are misprinted, reading R18) are what the TESTS compare this against.
 * ------------------------------------------------------------------------------------------ */
double oracle_gaunt(int l1, int l2, int l3, int m1, int m2, int m3)
{
    return (double)sqrtl((2 * l1 + 1) * (2 * l2 + 1) * (2 * l3 + 1) / (4.0L * PI_L)) *
           oracle_wigner3j(l1, l2, l3, m1, m2, m3) * oracle_wigner3j(l1, l2, l3, 0, 0, 0);
}

double oracle_generalized_gaunt(int order, const int *LamA, const int *LamB, const int *LamC)
{
    if (order < 3 || order > ORACLE_MAX_ORDER) return 0.0;
    const int nm = order - 1;
    int la[5], lb[5], lc[5], ma[5], mb[5], mc[5];
    principal_ls(order, LamA, la);
    principal_ls(order, LamB, lb);
    principal_ls(order, LamC, lc);
    for (int k = 0; k < nm; ++k) /* (l l' l''; 0 0 0) = 0 unless triangle and even sum */
        if (lc[k] < abs(la[k] - lb[k]) || lc[k] > la[k] + lb[k] || ((la[k] + lb[k] + lc[k]) & 1)) return 0.0;
    long double tot = 0.0L;
    for (int k = 0; k < nm - 1; ++k) ma[k] = -la[k];
    for (;;) { /* odometer over M (last m fixed by the sum rule) */
        int sa = 0;
        for (int k = 0; k < nm - 1; ++k) sa += ma[k];
        ma[nm - 1] = -sa;
        if (abs(ma[nm - 1]) <= la[nm - 1]) {
            const double ca = oracle_coupling(order, LamA, ma);
            if (ca != 0.0) {
                for (int k = 0; k < nm - 1; ++k) mb[k] = -lb[k];
                for (;;) { /* odometer over M' */
                    int sb = 0;
                    for (int k = 0; k < nm - 1; ++k) sb += mb[k];
                    mb[nm - 1] = -sb;
                    if (abs(mb[nm - 1]) <= lb[nm - 1]) {
                        int ok = 1;
                        for (int k = 0; k < nm; ++k) { mc[k] = -ma[k] - mb[k]; if (abs(mc[k]) > lc[k]) ok = 0; }
                        if (ok) {
                            const double cb = oracle_coupling(order, LamB, mb);
                            const double cc = cb != 0.0 ? oracle_coupling(order, LamC, mc) : 0.0;
                            if (cc != 0.0) {
                                long double pr = (long double)ca * cb * cc;
                                for (int k = 0; k < nm && pr != 0.0L; ++k) pr *= oracle_gaunt(la[k], lb[k], lc[k], ma[k], mb[k], mc[k]);
                                tot += pr;
                            }
                        }
                    }
                    int k = nm - 2;
                    while (k >= 0 && ++mb[k] > lb[k]) { mb[k] = -lb[k]; --k; }
                    if (k < 0) break;
                }
            }
        }
        int k = nm - 2;
        while (k >= 0 && ++ma[k] > la[k]) { ma[k] = -la[k]; --k; }
        if (k < 0) break;
    }
    return (double)tot;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
