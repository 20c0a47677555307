// common.h — internal structures shared by the host table builder and the CUDA stages.
// Product code of the ENCORE B200 hot path; never includes or links anything under oracle/.
#pragma once
#include <cstdint>
#include <vector>

#define ENCORE_MAX_ORDER 6
#define ENCORE_MAX_BINS 32
#define ENCORE_MAX_LMAX 10
#define ENCORE_GROUP 32              // primaries per group = lanes of a warp

// Real-component layout of one a_lm tile row (per radial bin): (lmax+1)^2 doubles,
//   (l,0) at l*l;  Re(l,m) at l*l+2m-1;  Im(l,m) at l*l+2m   (m = 1..l).
static inline int comp_re(int l, int m) { return m == 0 ? l * l : l * l + 2 * m - 1; }
static inline int comp_im(int l, int m) { return m == 0 ? -1 : l * l + 2 * m; }

// One non-zero (Lambda, M) term of eq. 44: weight W = 2 S(m_{N-1}) E(Lam) C^Lam_M prod_k sigma_k,
// factor k = a_{l_k |m_k|} for m_k >= 0, (-1)^{m_k} conj(a_{l_k |m_k|}) for m_k < 0:
// re[k]/im[k] are component indices (im = -1: imaginary part is zero), tau[k] = -1 conjugates.
struct HostTerm {
    int16_t re[5];
    int16_t im[5];
    int8_t tau[5];
    double W;
};

// One term of a coupled pair  Y = sum_{m_a, m_b} (3j) a~_{l_a m_a}(b_a) a~_{l_b m_b}(b_b)  with every sign, conjugation
// and overall factor folded into four real weights:
//   Re Y += wrr r_a r_b + wii i_a i_b,   Im Y += wri r_a i_b + wir i_a r_b.
// ia_*, ib_* are component indices INSIDE the l-block of the factor: Re(l,m) at 2m-1 (m>0) or 0, Im(l,m) at 2m.
struct PairTerm {
    int ia_re, ia_im, ib_re, ib_im;
    double wrr, wii, wri, wir;
};

// N=4 multiplet for the factorised contraction:
//   H_i = sum_{m3>=0} Re[ G_{m3}(b1,b2) a_{l3 m3}(b3) ],  G_{m3} = 2 S(m3) sum_{m1+m2=-m3} (l1 l2 l3; m1 m2 m3) a~1 a~2
// m3 = 0: the terms (m1, -m1) and (-m1, m1) are complex conjugates of each other up to the sign (-1)^{l1+l2+l3}
// (3-j column symmetry and a_{l,-m} = (-1)^m a*_lm), so G_0 is real for even and imaginary for odd multiplets and only
// m1 >= 0 is kept: the m3 = 0 terms are "half terms" G_0 += wrr A[ia_re] B[ib_re] + wii A[ia_im] B[ib_im] (two FMAs).
struct Lam4 {
    int l1, l2, l3;
    int odd;            // parity-odd multiplet: the stored result is Im instead of Re (App. B)
    int tbeg[ENCORE_MAX_LMAX + 2]; // terms of m3 are [tbeg[m3], tbeg[m3+1]) in pair_terms; m3 = 0: half terms
    int nterms;
};

// N=5 multiplet:  H_i = sum_{M>=0} Re[ Y12_M(b1,b2) R34_M(b3,b4) ]  with
//   Y12_M = f_M sum_{m1+m2=M} (l1 l2 l12; m1 m2 -M) a~1 a~2,  f_M = sqrt(2 l12+1) (-1)^{l12-M} (2 - delta_M0),
//   R34_M = sum_{m3+m4=-M} (l3 l4 l12; m3 m4 M) a~3 a~4.
struct Lam5 {
    int l1, l2, l12, l3, l4;
    int odd;
    int lbeg[14];       // left terms of M: [lbeg[M], lbeg[M+1])   (M <= l12 <= 12)
    int rbeg[14];       // right terms
    int nterms;
};

// N=6 multiplet for the factorised contraction (contract6.cu):  H_i = sum_{m123>=0} Re[ T_{m123}(b1,b2,b3) R45_{m123}(b4,b5) ],
//   U_m(b1,b2)   = sum_{m1+m2=m} (l1 l2 l12; m1 m2 -m) a~1 a~2,  m = 0..l12   (U_{-m} = (-1)^{l1+l2+l12+m} conj U_m)
//   T_M(b1,b2,b3) = f_M sum_{m12+m3=M} (-1)^{l12-m12} (l12 l3 l123; m12 m3 -M) U~_{m12} a~3,
//                   f_M = sqrt((2 l12+1)(2 l123+1)) (-1)^{l123-M} (2 - delta_M0)                      (eq. 5 with two intermediates)
//   R45_M(b4,b5) = sum_{m4+m5=-M} (l123 l4 l5; M m4 m5) a~4 a~5
// All three are PairTerm lists; the first factor of a T term is a component of U (2|m12| real part, 2|m12|+1 imaginary part).
struct Lam6 {
    int l1, l2, l12, l3, l123, l4, l5;
    int odd;
    int ubeg[14];       // U terms of m12: [ubeg[m], ubeg[m+1])     (l12 <= 12)
    int tbeg[14];       // T terms of M                              (l123 <= 12)
    int rbeg[14];       // R terms of M
    int nterms;         // all of them, contiguous from ubeg[0]
};

// One CTA of the factorised N = 4, 5 kernels: its multiplets and the l-blocks of the a_lm tile they need (only those
// are brought into shared memory; a block l is the (2l+1) x nbins x 32 doubles starting at component l^2).
struct CtaPlan {
    int lam[12];                    // multiplet per slot (at most 12: one warp per multiplet), -1: empty; N = 5 at 9-10 bins and N = 6:
                                    // lam[w] = 8 * multiplet + warp role for w < 8 (N = 5: lam[8 + s] = multiplet staged in term slot s)
    int nblk;
    int bl[ENCORE_MAX_LMAX + 1];    // l of block j
    int off[ENCORE_MAX_LMAX + 1];   // offset (doubles) of block l inside a tile buffer, -1: not staged
    int tile;                       // doubles per tile buffer
    int nbuf;                       // tile buffers of the ring: 1 (single) .. 4
    int scr[8];                     // N = 6: offset (doubles) of warp w's U scratch;  N = 5 at 9-10 bins: term slot of warp w's multiplet
};

struct HostTables {
    int order = 0, nbins = 0, lmax = 0, ncomp = 0, width = 0; // width = 2N-5 columns of a multiplet row
    int allparity = 0;               // 1: odd-parity multiplets too (ALLPARITY mode)
    std::vector<int> parity;         // [nLam] 0 even (zeta real), 1 odd (zeta = i * stored value)
    double rmin = 0, rmax = 0, box = 0;
    std::vector<int> multiplets;     // [nLam][width]
    std::vector<int> bin_tuples;     // [nB][N-1]
    std::vector<HostTerm> terms;     // grouped by multiplet
    std::vector<int> term_start;     // [nLam+1]
    std::vector<double> edges;       // [nbins+1]
    std::vector<double> edges2;      // squared
    std::vector<double> vinv;        // 1/v_b
    std::vector<double> ynorm;       // [ncomp]: (-1)^m N_lm k_lm, turns sum w p_lm(z) (x+iy)^m into sum w Y_lm
    std::vector<double> ycoef;       // [ncomp][lmax+1]: ynorm * coefficient of z^k in the monic p_lm(z)
    std::vector<PairTerm> pair_terms; // factorised contraction (N=4,5)
    std::vector<Lam4> lam4;
    std::vector<Lam5> lam5;
    std::vector<Lam6> lam6;          // N = 6, only when every intermediate is <= 12 (empty otherwise: literal kernel)
    std::vector<int> lam_order;      // multiplets by decreasing work (launch order)
    int nLam() const { return width ? (int)multiplets.size() / width : 0; }
    int nB() const { return order > 1 ? (int)bin_tuples.size() / (order - 1) : 0; }
};

// Host side (tables.cpp)
double encore_host_wigner3j(int j1, int j2, int j3, int m1, int m2, int m3);
double encore_host_wigner9j(int j1, int j2, int j3, int j4, int j5, int j6, int j7, int j8, int j9);
int encore_build_gaunt_tensor(const HostTables &t, std::vector<double> &T); // edge correction: E(Lam'') G^{Lam Lam' Lam''}
int encore_build_tables(HostTables &t, int order, double rmin, double rmax, int nbins, int lmax, double box, int allparity = 0);
