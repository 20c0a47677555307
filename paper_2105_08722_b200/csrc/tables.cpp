// tables.cpp — host-side plan tables of the ENCORE hot path (step a0 of SURVEY.md §8(a)).
// Multiplets Lambda, ordered bin tuples, the non-zero coupling terms of the
// half-sum eq. 44 with C^Lam_M from eq. 5 (N=3: eq. 16, N=4: eq. 18),
// bin edges / volumes and the Y_lm normalisations.  Plain C++, no CUDA, no Python;
// the paper precomputes these with sympy — here they are built at plan time.
#include "common.h"

#include <algorithm>
#include <cmath>
#include <cstdlib>

namespace {

const long double kPi = 3.14159265358979323846264338327950288L;

struct FactTable {
    long double v[256];
    FactTable()
    {
        v[0] = 1.0L;
        for (int i = 1; i < 256; ++i) v[i] = v[i - 1] * (long double)i;
    }
};

long double fact(int n)
{
    static const FactTable tab; // function-local static: initialised once, thread-safe (C++11)
    return tab.v[n];
}

} // namespace

// Wigner 3-j by Racah's single sum (textbook form with factorials, long double throughout).
double encore_host_wigner3j(int j1, int j2, int j3, int m1, int m2, int m3)
{
    if (m1 + m2 + m3 != 0) return 0.0;
    if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(m3) > j3) return 0.0;
    if (j3 > j1 + j2 || j3 < std::abs(j1 - j2)) return 0.0;
    const int kmin = std::max(0, std::max(j2 - j3 - m1, j1 - j3 + m2));
    const int kmax = std::min(j1 + j2 - j3, std::min(j1 - m1, j2 + m2));
    long double s = 0.0L;
    for (int k = kmin; k <= kmax; ++k) {
        long double den = fact(k) * fact(j1 + j2 - j3 - k) * fact(j1 - m1 - k) * fact(j2 + m2 - k) *
                          fact(j3 - j2 + m1 + k) * fact(j3 - j1 - m2 + k);
        s += ((k & 1) ? -1.0L : 1.0L) / den;
    }
    long double tri = fact(j1 + j2 - j3) * fact(j1 - j2 + j3) * fact(-j1 + j2 + j3) / fact(j1 + j2 + j3 + 1);
    long double pre = tri * fact(j1 + m1) * fact(j1 - m1) * fact(j2 + m2) * fact(j2 - m2) * fact(j3 + m3) *
                      fact(j3 - m3);
    long double v = std::sqrt(pre) * s;
    if ((j1 - j2 - m3) & 1) v = -v;
    return (double)v;
}

namespace {

// E(Lam) C^Lam_M for principal m's `m` (sum = 0).  Intermediates of N=5 are NOT capped at lmax (R5).
double coupling(int order, const int *lam, const int *m)
{
    if (order == 3) {
        const int l = lam[0];
        return (((l - m[0]) & 1) ? -1.0 : 1.0) / std::sqrt(2.0 * l + 1.0); // eq. 16; E = (-1)^{2l} = 1
    }
    if (order == 4) { // eq. 18: C = (-1)^{l1+l2+l3} (3j); times E = same sign -> plain 3j
        return encore_host_wigner3j(lam[0], lam[1], lam[2], m[0], m[1], m[2]);
    }
    if (order == 6) {
        // eq. 5 for N=6: two intermediates, kappa = l12 - m12 + l123 - m123; only m12 = m1+m2 and
        // m123 = m12+m3 survive; E*E = 1.
        const int l1 = lam[0], l2 = lam[1], l12 = lam[2], l3 = lam[3], l123 = lam[4], l4 = lam[5], l5 = lam[6];
        const int m12 = m[0] + m[1], m123 = m12 + m[2];
        if (std::abs(m12) > l12 || std::abs(m123) > l123) return 0.0;
        double v = encore_host_wigner3j(l1, l2, l12, m[0], m[1], -m12) * encore_host_wigner3j(l12, l3, l123, m12, m[2], -m123) *
                   encore_host_wigner3j(l123, l4, l5, m123, m[3], m[4]);
        if ((l12 - m12 + l123 - m123) & 1) v = -v;
        return std::sqrt((2.0 * l12 + 1.0) * (2.0 * l123 + 1.0)) * v;
    }
    // eq. 5 for N=5: C = E sqrt(2 l12+1) sum_{m12} (-1)^{l12-m12} (l1 l2 l12; m1 m2 -m12)(l12 l3 l4; m12 m3 m4);
    // only m12 = m1+m2 survives; E*E = 1.
    const int l1 = lam[0], l2 = lam[1], l12 = lam[2], l3 = lam[3], l4 = lam[4];
    const int m12 = m[0] + m[1];
    if (std::abs(m12) > l12) return 0.0;
    double v = encore_host_wigner3j(l1, l2, l12, m[0], m[1], -m12) * encore_host_wigner3j(l12, l3, l4, m12, m[2], m[3]);
    if ((l12 - m12) & 1) v = -v;
    return std::sqrt(2.0 * l12 + 1.0) * v;
}

void enumerate_multiplets(HostTables &t)
{
    const int L = t.lmax;
    if (t.order == 3) {
        for (int l = 0; l <= L; ++l) t.multiplets.push_back(l);
    } else if (t.order == 4) {
        for (int l1 = 0; l1 <= L; ++l1)
            for (int l2 = 0; l2 <= L; ++l2)
                for (int l3 = std::abs(l1 - l2); l3 <= std::min(l1 + l2, L); ++l3)
                    if (t.allparity || ((l1 + l2 + l3) & 1) == 0) { // even parity unless ALLPARITY
                        t.multiplets.push_back(l1); t.multiplets.push_back(l2); t.multiplets.push_back(l3);
                    }
    } else if (t.order == 5) {
        for (int l1 = 0; l1 <= L; ++l1)
            for (int l2 = 0; l2 <= L; ++l2)
                for (int l12 = std::abs(l1 - l2); l12 <= l1 + l2; ++l12)
                    for (int l3 = 0; l3 <= L; ++l3)
                        for (int l4 = std::abs(l12 - l3); l4 <= std::min(l12 + l3, L); ++l4)
                            if (t.allparity || ((l1 + l2 + l3 + l4) & 1) == 0) {
                                const int row[5] = {l1, l2, l12, l3, l4};
                                t.multiplets.insert(t.multiplets.end(), row, row + 5);
                            }
    } else { // N = 6: {l1, l2, (l12), l3, (l123), l4, l5}, intermediates over their whole triangle range (R5)
        for (int l1 = 0; l1 <= L; ++l1)
            for (int l2 = 0; l2 <= L; ++l2)
                for (int l12 = std::abs(l1 - l2); l12 <= l1 + l2; ++l12)
                    for (int l3 = 0; l3 <= L; ++l3)
                        for (int l123 = std::abs(l12 - l3); l123 <= l12 + l3; ++l123)
                            for (int l4 = 0; l4 <= L; ++l4)
                                for (int l5 = std::abs(l123 - l4); l5 <= std::min(l123 + l4, L); ++l5)
                                    if (t.allparity || ((l1 + l2 + l3 + l4 + l5) & 1) == 0) {
                                        const int row[7] = {l1, l2, l12, l3, l123, l4, l5};
                                        t.multiplets.insert(t.multiplets.end(), row, row + 7);
                                    }
    }
}

// E(Lam) = (-1)^{sum of principal l}: 0 = parity-even (zeta real), 1 = parity-odd (zeta imaginary)
void fill_parity(HostTables &t)
{
    const int nL = t.nLam();
    t.parity.assign(nL, 0);
    for (int iL = 0; iL < nL; ++iL) {
        const int *lam = &t.multiplets[(size_t)iL * t.width];
        int s = 0;
        if (t.order == 4) s = lam[0] + lam[1] + lam[2];
        else if (t.order == 5) s = lam[0] + lam[1] + lam[3] + lam[4];
        else if (t.order == 6) s = lam[0] + lam[1] + lam[3] + lam[5] + lam[6];
        t.parity[iL] = s & 1;
    }
}

void enumerate_bins(HostTables &t)
{
    const int k = t.order - 1;
    int b[5];
    for (int i = 0; i < k; ++i) b[i] = i;
    for (;;) {
        t.bin_tuples.insert(t.bin_tuples.end(), b, b + k);
        int i = k - 1;
        while (i >= 0 && b[i] == t.nbins - k + i) --i;
        if (i < 0) break;
        ++b[i];
        for (int j = i + 1; j < k; ++j) b[j] = b[j - 1] + 1;
    }
}

void enumerate_terms(HostTables &t)
{
    const int nm = t.order - 1;
    const int nL = t.nLam();
    t.term_start.assign(1, 0);
    for (int iL = 0; iL < nL; ++iL) {
        const int *lam = &t.multiplets[(size_t)iL * t.width];
        int l[5];
        if (t.order == 3) { l[0] = l[1] = lam[0]; }
        else if (t.order == 4) { l[0] = lam[0]; l[1] = lam[1]; l[2] = lam[2]; }
        else if (t.order == 5) { l[0] = lam[0]; l[1] = lam[1]; l[2] = lam[3]; l[3] = lam[4]; }
        else { l[0] = lam[0]; l[1] = lam[1]; l[2] = lam[3]; l[3] = lam[5]; l[4] = lam[6]; }
        int m[5];
        for (int k = 0; k < nm - 1; ++k) m[k] = -l[k];
        for (;;) {
            int s = 0;
            for (int k = 0; k < nm - 1; ++k) s += m[k];
            m[nm - 1] = -s;
            if (m[nm - 1] >= 0 && m[nm - 1] <= l[nm - 1]) { // half-sum: m_{N-1} >= 0, weight 2 S(m)
                const double c = coupling(t.order, lam, m);
                if (std::fabs(c) > 1e-15) {
                    HostTerm ht{};
                    double W = (m[nm - 1] == 0 ? 1.0 : 2.0) * c;
                    for (int k = 0; k < nm; ++k) {
                        const int am = std::abs(m[k]);
                        ht.re[k] = (int16_t)comp_re(l[k], am);
                        ht.im[k] = (int16_t)comp_im(l[k], am);
                        ht.tau[k] = 1;
                        if (m[k] < 0) { // a_{l,-m} = (-1)^m conj(a_lm)
                            ht.tau[k] = -1;
                            if (am & 1) W = -W;
                        }
                    }
                    for (int k = nm; k < 5; ++k) { ht.re[k] = 0; ht.im[k] = -1; ht.tau[k] = 1; }
                    ht.W = W;
                    t.terms.push_back(ht);
                }
            }
            int k = nm - 2;
            while (k >= 0 && ++m[k] > l[k]) { m[k] = -l[k]; --k; }
            if (k < 0) break;
        }
        t.term_start.push_back((int)t.terms.size());
    }
}

// Terms of sum_{ma+mb=msum} (la lb L; ma mb -msum) a~_{la ma} a~_{lb mb} times `factor`.
void coupled_pair_terms(int la, int lb, int L, int msum, double factor, std::vector<PairTerm> &out)
{
    for (int ma = -la; ma <= la; ++ma) {
        const int mb = msum - ma;
        if (std::abs(mb) > lb) continue;
        double w = factor * encore_host_wigner3j(la, lb, L, ma, mb, -msum);
        if (std::fabs(w) < 1e-15) continue;
        // a~ = sigma (re + i tau im): m >= 0: sigma = tau = 1; m < 0: sigma = (-1)^m, tau = -1
        const int aa = std::abs(ma), ab = std::abs(mb);
        const double ta = ma < 0 ? -1.0 : 1.0, tb = mb < 0 ? -1.0 : 1.0;
        if (ma < 0 && (aa & 1)) w = -w;
        if (mb < 0 && (ab & 1)) w = -w;
        PairTerm t{};
        t.ia_re = aa == 0 ? 0 : 2 * aa - 1;
        t.ib_re = ab == 0 ? 0 : 2 * ab - 1;
        t.ia_im = aa == 0 ? t.ia_re : 2 * aa;   // m = 0: no imaginary part; point at a valid row, zero the weights
        t.ib_im = ab == 0 ? t.ib_re : 2 * ab;
        t.wrr = w;
        t.wii = (aa && ab) ? -w * ta * tb : 0.0;
        t.wri = ab ? w * tb : 0.0;
        t.wir = aa ? w * ta : 0.0;
        out.push_back(t);
    }
}

// Terms of f sum_{m12+m3=M} (-1)^{l12-m12} (l12 l3 l123; m12 m3 -M) U~_{m12} a~_{l3 m3}: the first factor is a coupled pair
// U of (l1,l2,l12) stored for m12 >= 0 as components 2 m12 (real part), 2 m12 + 1 (imaginary part);
// U~_{-m} = sigma (-1)^m conj(U_m), sigma = (-1)^{l1+l2+l12}.
void coupled_triple_terms(int l12, int l3, int l123, int M, double f, int sigma_odd, std::vector<PairTerm> &out)
{
    for (int m12 = -l12; m12 <= l12; ++m12) {
        const int m3 = M - m12;
        if (std::abs(m3) > l3) continue;
        double w = f * (((l12 - m12) & 1) ? -1.0 : 1.0) * encore_host_wigner3j(l12, l3, l123, m12, m3, -M);
        if (std::fabs(w) < 1e-15) continue;
        const int aa = std::abs(m12), ab = std::abs(m3);
        const double ta = m12 < 0 ? -1.0 : 1.0, tb = m3 < 0 ? -1.0 : 1.0;
        if (m12 < 0) { if (sigma_odd) w = -w; if (aa & 1) w = -w; }
        if (m3 < 0 && (ab & 1)) w = -w;
        PairTerm t{};
        t.ia_re = 2 * aa; t.ia_im = 2 * aa + 1;
        t.ib_re = ab == 0 ? 0 : 2 * ab - 1;
        t.ib_im = ab == 0 ? t.ib_re : 2 * ab;
        t.wrr = w;
        t.wii = ab ? -w * ta * tb : 0.0;
        t.wri = ab ? w * tb : 0.0;
        t.wir = w * ta;
        out.push_back(t);
    }
}

void build_factorised(HostTables &t)
{
    const int nL = t.nLam();
    std::vector<double> cost(nL, 0.0);
    if (t.order == 4) {
        for (int iL = 0; iL < nL; ++iL) {
            const int *lam = &t.multiplets[(size_t)iL * 3];
            Lam4 q{};
            q.l1 = lam[0]; q.l2 = lam[1]; q.l3 = lam[2]; q.odd = t.parity[iL];
            // m3 = 0 half terms, m1 = 0 .. min(l1,l2):  with c = (l1 l2 l3; m1 -m1 0), s = (-1)^{m1},
            //   T = c s a1_{m1} conj(a2_{m1}),  G_0 = T(m1=0) + sum_{m1>0} [T + sigma conj T],  sigma = (-1)^{l1+l2+l3}
            //   even: G_0 = c0 r1 r2 + sum 2 c s (r1 r2 + i1 i2)          (real)
            //   odd : G_0 = i sum 2 c s (i1 r2 - r1 i2)                   (imaginary; (l1 l2 l3; 0 0 0) = 0)
            q.tbeg[0] = (int)t.pair_terms.size();
            for (int m1 = 0; m1 <= std::min(q.l1, q.l2); ++m1) {
                const double c = encore_host_wigner3j(q.l1, q.l2, q.l3, m1, -m1, 0);
                if (std::fabs(c) < 1e-15) continue;
                const double w = (m1 == 0 ? 1.0 : 2.0) * ((m1 & 1) ? -c : c);
                const int re = m1 == 0 ? 0 : 2 * m1 - 1, im = m1 == 0 ? 0 : 2 * m1;
                PairTerm pt{};
                if (!q.odd) { pt.ia_re = re; pt.ib_re = re; pt.ia_im = im; pt.ib_im = im; pt.wrr = w; pt.wii = m1 ? w : 0.0; }
                else if (m1 > 0) { pt.ia_re = im; pt.ib_re = re; pt.ia_im = re; pt.ib_im = im; pt.wrr = w; pt.wii = -w; }
                else continue;
                t.pair_terms.push_back(pt);
            }
            for (int m3 = 1; m3 <= q.l3; ++m3) {
                q.tbeg[m3] = (int)t.pair_terms.size();
                // G_{m3} = 2 S(m3) sum_{m1+m2=-m3} (l1 l2 l3; m1 m2 m3) a~1 a~2   (eq. 44 with E C = plain 3-j, eq. 18)
                coupled_pair_terms(q.l1, q.l2, q.l3, -m3, 2.0, t.pair_terms);
            }
            for (int m3 = q.l3 + 1; m3 < ENCORE_MAX_LMAX + 2; ++m3) q.tbeg[m3] = (int)t.pair_terms.size();
            q.nterms = q.tbeg[q.l3 + 1] - q.tbeg[0];
            cost[iL] = (q.tbeg[q.l3 + 1] - q.tbeg[1]) + 0.5 * (q.tbeg[1] - q.tbeg[0]) + 0.3 * (q.l3 + 1);
            t.lam4.push_back(q);
        }
    } else if (t.order == 5) {
        for (int iL = 0; iL < nL; ++iL) {
            const int *lam = &t.multiplets[(size_t)iL * 5];
            Lam5 q{};
            q.l1 = lam[0]; q.l2 = lam[1]; q.l12 = lam[2]; q.l3 = lam[3]; q.l4 = lam[4]; q.odd = t.parity[iL];
            // M = 0: the terms (m, -m) and (-m, m) of a coupled pair are complex conjugates up to sigma = (-1)^{la+lb+l12}
            // (3-j column symmetry, a_{l,-m} = (-1)^m a*_lm), so Y12_0 and R34_0 are real (sigma = +1) or imaginary
            // (sigma = -1): one real number per bin pair from "half terms" m >= 0 (as for N = 4, m3 = 0),
            //   T(m) = c_m (-1)^m a_m conj(b_m),  c_m = (la lb l12; m -m 0)
            //   sigma = +1: Re Y_0 = c_0 r r' + sum_{m>0} 2 c_m (-1)^m (r r' + i i');   sigma = -1: Im Y_0 = sum_{m>0} 2 c_m (-1)^m (i r' - r i')
            // and H_0 = s Ys Rs with s = -1 iff both are imaginary (even multiplet, (i Yi)(i Ri)); s is folded into the left weights.
            auto half_terms = [&](int la, int lb, int L, double factor) {
                const int sig_odd = (la + lb + L) & 1;
                for (int m = 0; m <= std::min(la, lb); ++m) {
                    const double c = encore_host_wigner3j(la, lb, L, m, -m, 0);
                    if (std::fabs(c) < 1e-15) continue;
                    const double w = factor * (m == 0 ? 1.0 : 2.0) * ((m & 1) ? -c : c);
                    const int re = m == 0 ? 0 : 2 * m - 1, im = m == 0 ? 0 : 2 * m;
                    PairTerm pt{};
                    if (!sig_odd) { pt.ia_re = re; pt.ib_re = re; pt.ia_im = im; pt.ib_im = im; pt.wrr = w; pt.wii = m ? w : 0.0; }
                    else if (m > 0) { pt.ia_re = im; pt.ib_re = re; pt.ia_im = re; pt.ib_im = im; pt.wrr = w; pt.wii = -w; }
                    else continue;
                    t.pair_terms.push_back(pt);
                }
            };
            const bool both_imag = ((q.l1 + q.l2 + q.l12) & 1) && ((q.l3 + q.l4 + q.l12) & 1);
            for (int M = 0; M <= q.l12; ++M) {
                const double f = std::sqrt(2.0 * q.l12 + 1.0) * (((q.l12 - M) & 1) ? -1.0 : 1.0) * (M == 0 ? 1.0 : 2.0);
                q.lbeg[M] = (int)t.pair_terms.size();
                if (M == 0) half_terms(q.l1, q.l2, q.l12, both_imag ? -f : f);
                else coupled_pair_terms(q.l1, q.l2, q.l12, M, f, t.pair_terms);   // (l1 l2 l12; m1 m2 -M)
                q.lbeg[M + 1] = (int)t.pair_terms.size();
            }
            for (int M = q.l12 + 1; M < 13; ++M) q.lbeg[M + 1] = q.lbeg[q.l12 + 1];
            for (int M = 0; M <= q.l12; ++M) {
                q.rbeg[M] = (int)t.pair_terms.size();
                if (M == 0) half_terms(q.l3, q.l4, q.l12, 1.0);
                else coupled_pair_terms(q.l3, q.l4, q.l12, -M, 1.0, t.pair_terms); // (l3 l4 l12; m3 m4 M) = (l12 l3 l4; M m3 m4)
                q.rbeg[M + 1] = (int)t.pair_terms.size();
            }
            for (int M = q.l12 + 1; M < 13; ++M) q.rbeg[M + 1] = q.rbeg[q.l12 + 1];
            q.nterms = (q.lbeg[q.l12 + 1] - q.lbeg[0]) + (q.rbeg[q.l12 + 1] - q.rbeg[0]);
            cost[iL] = (q.lbeg[q.l12 + 1] - q.lbeg[1]) + 0.5 * (q.lbeg[1] - q.lbeg[0]) + 3.0 * (q.rbeg[q.l12 + 1] - q.rbeg[1]) +
                       1.5 * (q.rbeg[1] - q.rbeg[0]) + (q.l12 + 1);
            t.lam5.push_back(q);
        }
    }
    else if (t.order == 6) {
        bool ok = true;
        for (int iL = 0; iL < nL && ok; ++iL) ok = t.multiplets[(size_t)iL * 7 + 2] <= 12 && t.multiplets[(size_t)iL * 7 + 4] <= 12;
        for (int iL = 0; iL < nL && ok; ++iL) {
            const int *lam = &t.multiplets[(size_t)iL * 7];
            Lam6 q{};
            q.l1 = lam[0]; q.l2 = lam[1]; q.l12 = lam[2]; q.l3 = lam[3]; q.l123 = lam[4]; q.l4 = lam[5]; q.l5 = lam[6]; q.odd = t.parity[iL];
            for (int m = 0; m <= q.l12; ++m) {
                q.ubeg[m] = (int)t.pair_terms.size();
                coupled_pair_terms(q.l1, q.l2, q.l12, m, 1.0, t.pair_terms);        // (l1 l2 l12; m1 m2 -m)
                q.ubeg[m + 1] = (int)t.pair_terms.size();
            }
            for (int m = q.l12 + 1; m < 13; ++m) q.ubeg[m + 1] = q.ubeg[q.l12 + 1];
            for (int M = 0; M <= q.l123; ++M) {
                const double f = std::sqrt((2.0 * q.l12 + 1.0) * (2.0 * q.l123 + 1.0)) * (((q.l123 - M) & 1) ? -1.0 : 1.0) * (M == 0 ? 1.0 : 2.0);
                q.tbeg[M] = (int)t.pair_terms.size();
                coupled_triple_terms(q.l12, q.l3, q.l123, M, f, (q.l1 + q.l2 + q.l12) & 1, t.pair_terms);
                q.tbeg[M + 1] = (int)t.pair_terms.size();
            }
            for (int M = q.l123 + 1; M < 13; ++M) q.tbeg[M + 1] = q.tbeg[q.l123 + 1];
            for (int M = 0; M <= q.l123; ++M) {
                q.rbeg[M] = (int)t.pair_terms.size();
                coupled_pair_terms(q.l4, q.l5, q.l123, -M, 1.0, t.pair_terms);      // (l4 l5 l123; m4 m5 M) = (l123 l4 l5; M m4 m5)
                q.rbeg[M + 1] = (int)t.pair_terms.size();
            }
            for (int M = q.l123 + 1; M < 13; ++M) q.rbeg[M + 1] = q.rbeg[q.l123 + 1];
            q.nterms = q.rbeg[q.l123 + 1] - q.ubeg[0];
            cost[iL] = (q.ubeg[q.l12 + 1] - q.ubeg[0]) + 2.0 * (q.tbeg[q.l123 + 1] - q.tbeg[0]) + (q.rbeg[q.l123 + 1] - q.rbeg[0]) + 2.0 * (q.l123 + 1);
            t.lam6.push_back(q);
        }
    }
    t.lam_order.resize(nL);
    for (int i = 0; i < nL; ++i) t.lam_order[i] = i;
    std::stable_sort(t.lam_order.begin(), t.lam_order.end(), [&](int x, int y) { return cost[x] > cost[y]; });
}

} // namespace

int encore_build_tables(HostTables &t, int order, double rmin, double rmax, int nbins, int lmax, double box, int allparity)
{
    t = HostTables();
    t.allparity = allparity;
    t.order = order; t.nbins = nbins; t.lmax = lmax; t.rmin = rmin; t.rmax = rmax; t.box = box;
    t.width = 2 * order - 5;
    t.ncomp = (lmax + 1) * (lmax + 1);
    enumerate_multiplets(t);
    fill_parity(t);
    enumerate_bins(t);
    enumerate_terms(t);
    // bins: e_b = r_min + b * width, e_nbins = r_max (R8)
    const double wdt = (rmax - rmin) / (double)nbins;
    t.edges.resize(nbins + 1);
    for (int b = 0; b < nbins; ++b) t.edges[b] = rmin + (double)b * wdt;
    t.edges[nbins] = rmax;
    t.edges2.resize(nbins + 1);
    for (int b = 0; b <= nbins; ++b) t.edges2[b] = t.edges[b] * t.edges[b];
    t.vinv.resize(nbins);
    for (int b = 0; b < nbins; ++b) { // v_b = 4 pi/3 (e_{b+1}^3 - e_b^3)
        long double hi = t.edges[b + 1], lo = t.edges[b];
        t.vinv[b] = (double)(1.0L / (4.0L * kPi / 3.0L * (hi * hi * hi - lo * lo * lo)));
    }
    // Y_lm = (-1)^m N_lm P_l^m(z) e^{i m phi},  P_l^m = k_lm (1-z^2)^{m/2} p_lm(z) with p_lm monic in z, so
    // Y_lm = ynorm * p_lm(z) (x+iy)^m,  k_mm = (2m-1)!!,  k_lm = k_{l-1,m} (2l-1)/(l-m).
    t.ynorm.assign(t.ncomp, 0.0);
    for (int m = 0; m <= lmax; ++m) {
        long double k = 1.0L;
        for (int i = 1; i <= m; ++i) k *= (long double)(2 * i - 1);
        for (int l = m; l <= lmax; ++l) {
            if (l > m) k *= (long double)(2 * l - 1) / (long double)(l - m);
            long double N = std::sqrt((2 * l + 1) / (4.0L * kPi) * fact(l - m) / fact(l + m));
            double v = (double)(((m & 1) ? -1.0L : 1.0L) * N * k);
            t.ynorm[comp_re(l, m)] = v;
            if (m > 0) t.ynorm[comp_im(l, m)] = v;
        }
    }
    // k_harm accumulates S_{m,k} = sum w z^k (x+iy)^m (one FMA per component, no Legendre recurrence per pair) and
    // maps to a_lm once per (primary, bin): Y_lm = sum_k ycoef[c][k] z^k (x+iy)^m with ycoef = ynorm * (coefficient of
    // z^k in the monic p_lm), p_mm = 1, p_{m+1,m} = z, p_lm = z p_{l-1,m} - gamma_lm p_{l-2,m},
    // gamma_lm = ((l-1)^2 - m^2) / (4 (l-1)^2 - 1).
    t.ycoef.assign((size_t)t.ncomp * (lmax + 1), 0.0);
    for (int m = 0; m <= lmax; ++m) {
        std::vector<long double> pm2(lmax + 1, 0.0L), pm1(lmax + 1, 0.0L), p(lmax + 1, 0.0L);
        for (int l = m; l <= lmax; ++l) {
            std::fill(p.begin(), p.end(), 0.0L);
            if (l == m) p[0] = 1.0L;
            else if (l == m + 1) p[1] = 1.0L;
            else {
                const long double gam = (long double)((l - 1) * (l - 1) - m * m) / (long double)(4 * (l - 1) * (l - 1) - 1);
                for (int k = 0; k <= l - m; ++k) p[k] = (k > 0 ? pm1[k - 1] : 0.0L) - gam * pm2[k];
            }
            for (int k = 0; k <= lmax; ++k) {
                t.ycoef[(size_t)comp_re(l, m) * (lmax + 1) + k] = (double)((long double)t.ynorm[comp_re(l, m)] * p[k]);
                if (m > 0) t.ycoef[(size_t)comp_im(l, m) * (lmax + 1) + k] = t.ycoef[(size_t)comp_re(l, m) * (lmax + 1) + k];
            }
            pm2 = pm1; pm1 = p;
        }
    }
    build_factorised(t);
    return 0;
}


// ---- edge correction (App. A :676-691) -------------------------------------
// Wigner 6-j by Racah's formula and 9-j as a sum over products of three 6-j symbols (NIST DLMF 34.4.2, 34.6.1);
// integer arguments only.  The generalised Gaunt integrals then follow from App. A's closed forms (A1-A3) with the 9-j
// rows read as (l_k l'_k l''_k) (R18; the oracle evaluates the defining sum over M instead).
namespace {

bool tri(int a, int b, int c) { return c >= std::abs(a - b) && c <= a + b; }

long double delta_tri(int a, int b, int c)
{
    return std::sqrt(fact(a + b - c) * fact(a - b + c) * fact(-a + b + c) / fact(a + b + c + 1));
}

long double wigner6j(int a, int b, int c, int d, int e, int f)
{
    if (!tri(a, b, c) || !tri(a, e, f) || !tri(d, b, f) || !tri(d, e, c)) return 0.0L;
    const int t0 = std::max(std::max(a + b + c, a + e + f), std::max(d + b + f, d + e + c));
    const int t1 = std::min(std::min(a + b + d + e, b + c + e + f), c + a + f + d);
    long double s = 0.0L;
    for (int t = t0; t <= t1; ++t) {
        const long double den = fact(t - a - b - c) * fact(t - a - e - f) * fact(t - d - b - f) * fact(t - d - e - c) *
                                fact(a + b + d + e - t) * fact(b + c + e + f - t) * fact(c + a + f + d - t);
        s += ((t & 1) ? -1.0L : 1.0L) * fact(t + 1) / den;
    }
    return delta_tri(a, b, c) * delta_tri(a, e, f) * delta_tri(d, b, f) * delta_tri(d, e, c) * s;
}

long double wigner9j(int j1, int j2, int j3, int j4, int j5, int j6, int j7, int j8, int j9)
{
    if (!tri(j1, j2, j3) || !tri(j4, j5, j6) || !tri(j7, j8, j9) || !tri(j1, j4, j7) || !tri(j2, j5, j8) || !tri(j3, j6, j9)) return 0.0L;
    const int x0 = std::max(std::max(std::abs(j1 - j9), std::abs(j4 - j8)), std::abs(j2 - j6));
    const int x1 = std::min(std::min(j1 + j9, j4 + j8), j2 + j6);
    long double s = 0.0L;
    for (int x = x0; x <= x1; ++x)
        s += (long double)(2 * x + 1) * wigner6j(j1, j4, j7, j8, j9, x) * wigner6j(j2, j5, j8, j4, x, j6) * wigner6j(j3, j6, j9, x, j1, j2);
    return s;
}

// sqrt((2a+1)(2b+1)(2c+1)) (a b c; 0 0 0), zero unless triangle and even sum
long double w000(int a, int b, int c)
{
    if (!tri(a, b, c) || ((a + b + c) & 1)) return 0.0L;
    return std::sqrt((long double)((2 * a + 1) * (2 * b + 1) * (2 * c + 1))) * (long double)encore_host_wigner3j(a, b, c, 0, 0, 0);
}

} // namespace

double encore_host_wigner9j(int j1, int j2, int j3, int j4, int j5, int j6, int j7, int j8, int j9)
{
    return (double)wigner9j(j1, j2, j3, j4, j5, j6, j7, j8, j9);
}

// T[(i*n + j)*n + k] = E(Lam_k) G^{Lam_i Lam_j Lam_k} over the plan's multiplet list (N = 3, 4, 5)
int encore_build_gaunt_tensor(const HostTables &t, std::vector<double> &T)
{
    const int n = t.nLam(), N = t.order;
    if (N < 3 || N > 5) return -1;
    T.assign((size_t)n * n * n, 0.0);
    const long double fourpi = 4.0L * kPi;
    for (int i = 0; i < n; ++i)
        for (int j = i; j < n; ++j)       // G is symmetric under Lam <-> Lam'
            for (int k = 0; k < n; ++k) {
                const int *a = &t.multiplets[(size_t)i * t.width], *b = &t.multiplets[(size_t)j * t.width], *c = &t.multiplets[(size_t)k * t.width];
                long double g = 0.0L;
                if (N == 3) {             // A1
                    const long double w = w000(a[0], b[0], c[0]);
                    g = w == 0.0L ? 0.0L : w * w / std::sqrt((long double)((2 * a[0] + 1) * (2 * b[0] + 1) * (2 * c[0] + 1))) / fourpi;
                } else if (N == 4) {      // A2
                    g = w000(a[0], b[0], c[0]);
                    if (g != 0.0L) g *= w000(a[1], b[1], c[1]);
                    if (g != 0.0L) g *= w000(a[2], b[2], c[2]);
                    if (g != 0.0L) g *= wigner9j(a[0], b[0], c[0], a[1], b[1], c[1], a[2], b[2], c[2]) / std::pow(fourpi, 1.5L);
                } else {                  // A3
                    g = w000(a[0], b[0], c[0]);
                    if (g != 0.0L) g *= w000(a[1], b[1], c[1]);
                    if (g != 0.0L) g *= w000(a[3], b[3], c[3]);
                    if (g != 0.0L) g *= w000(a[4], b[4], c[4]);
                    if (g != 0.0L) g *= std::sqrt((long double)((2 * a[2] + 1) * (2 * b[2] + 1) * (2 * c[2] + 1)));
                    if (g != 0.0L) g *= wigner9j(a[0], a[1], a[2], b[0], b[1], b[2], c[0], c[1], c[2]);
                    if (g != 0.0L) g *= wigner9j(a[2], a[3], a[4], b[2], b[3], b[4], c[2], c[3], c[4]) / (fourpi * fourpi);
                }
                // E(Lam'') = (-1)^{parity of Lam''}.  ALLPARITY lists: zeta, N, R rows of odd multiplets hold the imaginary parts
                // (coefficient = i * stored value), so an (odd Lam, odd Lam') pair feeding an even Lam'' carries i * i = -1 in
                // eq. 40; (odd, even) -> odd and (even, odd) -> odd keep their sign (i on both sides).
                long double sgn = t.parity[k] ? -1.0L : 1.0L;
                if (t.parity[i] && t.parity[j]) sgn = -sgn;
                const double v = (double)(sgn * g);
                T[((size_t)i * n + j) * n + k] = v;
                T[((size_t)j * n + i) * n + k] = v;
            }
    return 0;
}
