// common.h — internal structures shared by the host table builder and the CUDA stages.
// Product code of the ENCORE B200 hot path; never includes or links anything under oracle/.
#pragma once
#include <cstdint>
#include <vector>

#define ENCORE_MAX_ORDER 5
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
    int16_t re[4];
    int16_t im[4];
    int8_t tau[4];
    double W;
};

struct HostTables {
    int order = 0, nbins = 0, lmax = 0, ncomp = 0, width = 0; // width = 2N-5 columns of a multiplet row
    double rmin = 0, rmax = 0, box = 0;
    std::vector<int> multiplets;     // [nLam][width]
    std::vector<int> bin_tuples;     // [nB][N-1]
    std::vector<HostTerm> terms;     // grouped by multiplet
    std::vector<int> term_start;     // [nLam+1]
    std::vector<double> edges;       // [nbins+1]
    std::vector<double> edges2;      // squared
    std::vector<double> vinv;        // 1/v_b
    std::vector<double> ynorm;       // [ncomp]: (-1)^m N_lm k_lm, turns sum w p_lm(z) (x+iy)^m into sum w Y_lm
    int nLam() const { return width ? (int)multiplets.size() / width : 0; }
    int nB() const { return order > 1 ? (int)bin_tuples.size() / (order - 1) : 0; }
};

// Host side (tables.cpp)
double encore_host_wigner3j(int j1, int j2, int j3, int m1, int m2, int m3);
int encore_build_tables(HostTables &t, int order, double rmin, double rmax, int nbins, int lmax, double box);
