"""Pins of the oracle's tables: 3-j symbols, Y_lm, coupling coefficients, enumeration counts.

Every expected value here is the paper's (cited) or a mathematical identity / an independent
library (scipy Y_lm, sympy 3-j) — never the oracle itself, never the CUDA path.
"""
import itertools
import math

import numpy as np
import pytest
from scipy.special import sph_harm_y
from sympy.physics.wigner import wigner_3j


# ---- 3-j: exact values (closed forms from sympy / DLMF 34.3) -------------
EXACT_3J = [
    ((1, 1, 0, 0, 0, 0), -1 / math.sqrt(3)),
    ((1, 1, 2, 0, 0, 0), math.sqrt(2 / 15)),
    ((2, 2, 2, 0, 0, 0), -math.sqrt(2 / 35)),
    ((1, 1, 1, 1, -1, 0), 1 / math.sqrt(6)),
    ((1, 1, 2, 1, 1, -2), 1 / math.sqrt(5)),
    ((2, 2, 0, 1, -1, 0), -1 / math.sqrt(5)),
    ((3, 2, 1, 0, 0, 0), -math.sqrt(3 / 35)),
    ((5, 5, 4, 2, -3, 1), math.sqrt(2145) / 429),
    ((10, 10, 10, 0, 0, 0), -126 * math.sqrt(233753485) / 33393355),
]


@pytest.mark.parametrize("args,val", EXACT_3J)
def test_3j_exact_values(oracle, args, val):
    assert oracle.wigner3j(*args) == pytest.approx(val, rel=0, abs=2e-15)


def test_3j_against_sympy_random(oracle):
    rng = np.random.default_rng(7)
    for _ in range(300):
        j1, j2 = rng.integers(0, 11, 2)
        j3 = rng.integers(abs(j1 - j2), j1 + j2 + 1)
        m1 = rng.integers(-j1, j1 + 1)
        m2 = rng.integers(-j2, j2 + 1)
        m3 = -m1 - m2
        ref = float(wigner_3j(int(j1), int(j2), int(j3), int(m1), int(m2), int(m3))) if abs(m3) <= j3 else 0.0
        assert oracle.wigner3j(j1, j2, j3, m1, m2, m3) == pytest.approx(ref, abs=3e-15)


def test_3j_selection_rules_and_sum_rule(oracle):
    assert oracle.wigner3j(2, 2, 5, 0, 0, 0) == 0.0          # triangle
    assert oracle.wigner3j(2, 2, 2, 1, 1, -1) == 0.0         # sum m != 0
    assert oracle.wigner3j(1, 1, 1, 0, 0, 0) == 0.0          # odd sum, all m = 0
    for (j1, j2, j3) in [(1, 1, 2), (3, 4, 5), (10, 9, 4), (5, 5, 0)]:
        s = sum(oracle.wigner3j(j1, j2, j3, m1, m2, -m1 - m2) ** 2
                for m1 in range(-j1, j1 + 1) for m2 in range(-j2, j2 + 1))
        assert s == pytest.approx(1.0, abs=1e-14)            # orthogonality, DLMF 34.3.16
    # (l l 0; m -m 0) = (-1)^{l-m}/sqrt(2l+1): turns eq. 5 into eq. 16
    for l in range(0, 11):
        for m in range(-l, l + 1):
            assert oracle.wigner3j(l, l, 0, m, -m, 0) == pytest.approx((-1) ** (l - m) / math.sqrt(2 * l + 1), abs=1e-15)
    # column swap sign (-1)^{l1+l2+l3}
    assert oracle.wigner3j(3, 2, 2, 1, -2, 1) == pytest.approx(-oracle.wigner3j(2, 3, 2, -2, 1, 1), abs=1e-15)


# ---- Y_lm (reading R1) ----------------------------------------------------------------------
def test_ylm_against_scipy(oracle):
    rng = np.random.default_rng(11)
    lmax = 10
    vs = rng.standard_normal((40, 3))
    vs = np.vstack([vs, [[0, 0, 1], [0, 0, -1], [1, 0, 0], [0, -1, 0], [1e-9, 0, 1]]])
    for v in vs:
        v = v / np.linalg.norm(v)
        Y = oracle.ylm(lmax, v)
        th, ph = math.atan2(math.hypot(v[0], v[1]), v[2]), math.atan2(v[1], v[0])   # acos loses the pole
        for l in range(lmax + 1):
            for m in range(-l, l + 1):
                assert abs(Y[l * l + l + m] - sph_harm_y(l, m, th, ph)) < 5e-14, (l, m, v)


def test_ylm_paper_closed_forms(oracle):
    v = np.array([0.3, -0.5, 0.4])
    v /= np.linalg.norm(v)
    Y = oracle.ylm(2, v)
    assert Y[0] == pytest.approx((4 * math.pi) ** -0.5, abs=1e-16)
    # Y_{2,-1} ∝ (dx - i dy) dz; constant sqrt(15/(8 pi))
    assert abs(Y[4 + 2 - 1] - math.sqrt(15 / (8 * math.pi)) * (v[0] - 1j * v[1]) * v[2]) < 1e-15
    # Y_{l,-m} = (-1)^m conj(Y_lm)
    assert abs(Y[4 + 2 - 2] - np.conj(Y[4 + 2 + 2])) < 1e-16
    assert abs(Y[1 + 1 - 1] + np.conj(Y[1 + 1 + 1])) < 1e-16
    # addition theorem -> eq. 17 at r1 = r2: sum_m |Y_lm|^2 = (2l+1)/(4 pi)
    Y = oracle.ylm(8, v)
    for l in range(9):
        assert sum(abs(Y[l * l + l + m]) ** 2 for m in range(-l, l + 1)) == pytest.approx((2 * l + 1) / (4 * math.pi), rel=1e-13)


# ---- multiplets and term counts printed in the paper --------------------
def test_multiplet_counts_and_order(oracle):
    assert len(oracle.multiplets(3, 10)) == 11
    assert len(oracle.multiplets(4, 5)) == 69                  # PAPER.md:606  8 280 = 69 x 120
    assert len(oracle.multiplets(4, 10)) == 381                # PAPER.md:537, :586  45 720 = 381 x 120
    assert len(oracle.multiplets(5, 3)) == 204                 # PAPER.md:606, :644  42 840 = 204 x 210
    assert len(oracle.multiplets(5, 5)) == 1406                # PAPER.md:594  295 260 = 1 406 x 210 (R5: l12 uncapped)
    assert len(oracle.multiplets(4, 5, allparity=True)) == 111  # PAPER.md:602  13 320 = 111 x 120
    assert len(oracle.multiplets(4, 10, allparity=True)) == 671  # PAPER.md:602  80 520 = 671 x 120
    lam = oracle.multiplets(4, 5)
    # order printed for Fig. 4: {0,0,0},{0,1,1},{0,2,2},...,{1,0,1},{1,1,0}
    assert lam[:3].tolist() == [[0, 0, 0], [0, 1, 1], [0, 2, 2]]
    assert lam[6:8].tolist() == [[1, 0, 1], [1, 1, 0]]
    for row in oracle.multiplets(5, 3):
        l1, l2, l12, l3, l4 = row
        assert abs(l1 - l2) <= l12 <= l1 + l2 and abs(l12 - l3) <= l4 <= l12 + l3
        assert max(l1, l2, l3, l4) <= 3 and (l1 + l2 + l3 + l4) % 2 == 0


def _enumerate6(lmax, cap):
    """6PCF multiplets {l1,l2,(l12),l3,(l123),l4,l5} written out here from the triangle rules of eq. 5,
    even parity; cap: intermediates limited to lmax as well (the counting behind PAPER.md:537)"""
    rows = []
    top = lmax if cap else 10 ** 9
    for l1 in range(lmax + 1):
        for l2 in range(lmax + 1):
            for l12 in range(abs(l1 - l2), min(l1 + l2, top) + 1):
                for l3 in range(lmax + 1):
                    for l123 in range(abs(l12 - l3), min(l12 + l3, top) + 1):
                        for l4 in range(lmax + 1):
                            for l5 in range(abs(l123 - l4), min(l123 + l4, lmax) + 1):
                                if (l1 + l2 + l3 + l4 + l5) % 2 == 0:
                                    rows.append([l1, l2, l12, l3, l123, l4, l5])
    return rows


def test_6pcf_multiplet_counts(oracle):
    """PAPER.md:537 prints 1 558 six-point multiplets at lmax = 3: that is the count with the intermediates capped at
    lmax; reading R5 leaves them uncapped as for the 5PCF (204 / 1 406 of PAPER.md:606, :594), which gives
    2 212.  Both enumerations are written out above; the oracle's is the uncapped one, in nested-loop order."""
    assert len(_enumerate6(3, cap=True)) == 1558
    assert len(_enumerate6(3, cap=False)) == 2212
    assert oracle.multiplets(6, 3).tolist() == _enumerate6(3, cap=False)
    assert oracle.multiplets(6, 2).tolist() == _enumerate6(2, cap=False)
    assert len(oracle.multiplets(6, 1, allparity=True)) > len(oracle.multiplets(6, 1))
    assert len(oracle.bin_tuples(6, 10)) == 252                  # C(10,5), PAPER.md:537 (R6)
    assert oracle.bin_tuples(6, 6).tolist() == [list(c) for c in itertools.combinations(range(6), 5)]


def test_6pcf_coupling(oracle):
    """eq. 5 for N = 6: orthonormality (eq. 9), orthogonality across intermediates, eq. 6, against sympy, and the
    closed form P_{11(0)0(0)11} = (4 pi)^{-1/2} 3 (4 pi)^{-2} (r1.r2)(r4.r5) (two eq.-17 functions times Y_00)."""
    lams = oracle.multiplets(6, 1, allparity=True)
    for lam in lams:
        ls = (lam[0], lam[1], lam[3], lam[5], lam[6])
        assert sum(oracle.coupling(6, lam, M) ** 2 for M in _all_M(ls)) == pytest.approx(1.0, abs=1e-13), lam
    for lam in ([2, 1, 3, 2, 1, 1, 2], [1, 2, 2, 2, 4, 2, 2], [2, 2, 4, 2, 6, 2, 2 + 2]):   # intermediates above the principal l's
        ls = (lam[0], lam[1], lam[3], lam[5], lam[6])
        assert sum(oracle.coupling(6, lam, M) ** 2 for M in _all_M(ls)) == pytest.approx(1.0, abs=1e-12), lam
    ls = (1, 1, 1, 1, 1, )
    fam = [r for r in lams.tolist() if (r[0], r[1], r[3], r[5], r[6]) == (1, 1, 1, 1, 1) or False]
    same = [r for r in oracle.multiplets(6, 1, allparity=True).tolist() if [r[0], r[1], r[3], r[5], r[6]] == [1, 1, 1, 1, 0]]
    assert len(same) >= 2
    for a in same:
        for b in same:
            s = sum(oracle.coupling(6, a, M) * oracle.coupling(6, b, M) for M in _all_M((1, 1, 1, 1, 0)))
            assert s == pytest.approx(1.0 if a == b else 0.0, abs=1e-13)
    rng = np.random.default_rng(66)
    for lam in ([1, 1, 2, 1, 1, 1, 0], [1, 2, 1, 1, 2, 2, 1], [2, 1, 3, 1, 2, 1, 1]):
        E = (-1) ** (lam[0] + lam[1] + lam[3] + lam[5] + lam[6])
        l1, l2, l12, l3, l123, l4, l5 = lam
        for M in _all_M((l1, l2, l3, l4, l5)):
            c = oracle.coupling(6, lam, M)
            assert oracle.coupling(6, lam, [-m for m in M]) == pytest.approx(E * c, abs=1e-15)      # eq. 6
            m12, m123 = M[0] + M[1], M[0] + M[1] + M[2]
            ref = 0.0
            if abs(m12) <= l12 and abs(m123) <= l123:
                ref = (E * math.sqrt((2 * l12 + 1) * (2 * l123 + 1)) * (-1) ** (l12 - m12 + l123 - m123)
                       * float(wigner_3j(l1, l2, l12, M[0], M[1], -m12)) * float(wigner_3j(l12, l3, l123, m12, M[2], -m123))
                       * float(wigner_3j(l123, l4, l5, m123, M[3], M[4])))
            assert c == pytest.approx(ref, abs=1e-14)
    u = rng.standard_normal((5, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    Y = [oracle.ylm(2, v) for v in u]
    lam, ls = [1, 1, 0, 0, 0, 1, 1], (1, 1, 0, 1, 1)
    tot = 0.0
    for M in _all_M(ls):
        pr = oracle.coupling(6, lam, M)
        for k, (l, m) in enumerate(zip(ls, M)):
            pr = pr * Y[k][l * l + l + m]
        tot += pr
    fourpi = 4 * math.pi
    assert abs(tot - fourpi ** -0.5 * 3 / fourpi ** 2 * (u[0] @ u[1]) * (u[3] @ u[4])) < 1e-15


def test_bin_tuple_counts_and_order(oracle):
    assert len(oracle.bin_tuples(3, 10)) == 45
    assert len(oracle.bin_tuples(4, 10)) == 120
    assert len(oracle.bin_tuples(5, 10)) == 210
    assert len(oracle.bin_tuples(5, 8)) == 70
    bt = oracle.bin_tuples(4, 5)
    assert bt.tolist() == [list(c) for c in itertools.combinations(range(5), 3)]


def test_term_counts_printed_in_paper(oracle):
    # GPU-b task counts (one per Lambda, B, M with m_{N-1} >= 0): PAPER.md:586, :594
    assert oracle.count_terms(4, 5, half=True) * 120 == 135120
    assert oracle.count_terms(4, 10, half=True) * 120 == 2499480
    assert oracle.count_terms(5, 5, half=True) * 210 == 29606430
    assert oracle.count_terms(3, 10, half=True) == 66          # 660 = 66 x 10
    assert oracle.count_terms(3, 10, half=False) == 121


# ---- coupling coefficients ------------------------------------------------------------------
def _all_M(ls):
    for ms in itertools.product(*[range(-l, l + 1) for l in ls[:-1]]):
        mlast = -sum(ms)
        if abs(mlast) <= ls[-1]:
            yield (*ms, mlast)


@pytest.mark.parametrize("order,lmax", [(3, 6), (4, 4), (5, 2)])
def test_coupling_orthonormality(oracle, order, lmax):
    """eq. 9 ⇒ sum_M C^Lam_M C^Lam'_M = delta_{Lam Lam'} for multiplets sharing their
    principal l's; decides reading R2 (the sqrt(2 l12+1) of eq. 5 is required)."""
    lams = oracle.multiplets(order, lmax, allparity=True)

    def principal(lam):
        return {3: lambda x: (x[0], x[0]), 4: tuple, 5: lambda x: (x[0], x[1], x[3], x[4])}[order](lam)
    for lam in lams:
        ls = principal(lam)
        s = sum(oracle.coupling(order, lam, M) ** 2 for M in _all_M(ls))
        assert s == pytest.approx(1.0, abs=1e-13), lam
    if order == 5:   # different l12, same principal l's: orthogonal
        a, b = [1, 1, 0, 1, 1], [1, 1, 2, 1, 1]
        s = sum(oracle.coupling(5, a, M) * oracle.coupling(5, b, M) for M in _all_M((1, 1, 1, 1)))
        assert abs(s) < 1e-14


def test_coupling_special_cases(oracle):
    assert oracle.coupling(3, [0], [0, 0]) == 1.0              # C^0_0 = 1
    assert oracle.coupling(4, [0, 0, 0], [0, 0, 0]) == 1.0
    assert oracle.coupling(5, [0, 0, 0, 0, 0], [0, 0, 0, 0]) == pytest.approx(1.0, abs=1e-15)
    # eq. 16
    for l in range(5):
        for m in range(-l, l + 1):
            assert oracle.coupling(3, [l], [m, -m]) == pytest.approx((-1) ** (l - m) / math.sqrt(2 * l + 1), abs=1e-15)
    # eq. 18 against sympy
    for lam, M in [([1, 1, 2], (1, -1, 0)), ([2, 3, 3], (-2, 1, 1)), ([5, 4, 3], (2, -3, 1))]:
        ref = (-1) ** sum(lam) * float(wigner_3j(*lam, *M))
        assert oracle.coupling(4, lam, M) == pytest.approx(ref, abs=1e-15)
    # eq. 6: C_{-M} = E(Lam) C_M, incl. odd parity
    for lam in ([1, 1, 1], [2, 1, 2], [2, 2, 2]):
        E = (-1) ** sum(lam)
        for M in _all_M(lam):
            assert oracle.coupling(4, lam, [-m for m in M]) == pytest.approx(E * oracle.coupling(4, lam, M), abs=1e-15)
    for lam in ([1, 1, 2, 1, 1], [1, 2, 2, 1, 1], [1, 1, 1, 2, 1]):
        E = (-1) ** (lam[0] + lam[1] + lam[3] + lam[4])
        for M in _all_M((lam[0], lam[1], lam[3], lam[4])):
            assert oracle.coupling(5, lam, [-m for m in M]) == pytest.approx(E * oracle.coupling(5, lam, M), abs=1e-15)


def test_basis_closed_forms_through_oracle_tables(oracle):
    """P_Lam(R) = sum_M C^Lam_M prod Y (eq. 4) assembled from the oracle's own C and Y
    must equal the closed forms the paper prints."""
    rng = np.random.default_rng(3)
    u = rng.standard_normal((4, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    Y = [oracle.ylm(4, v) for v in u]

    def P(order, lam, ls):
        tot = 0.0
        for M in _all_M(ls):
            c = oracle.coupling(order, lam, M)
            pr = c
            for k, (l, m) in enumerate(zip(ls, M)):
                pr = pr * Y[k][l * l + l + m]
            tot += pr
        return tot
    fourpi = 4 * math.pi
    assert P(3, [0], (0, 0)) == pytest.approx(1 / fourpi, abs=1e-15)                   # eq. 11
    assert P(4, [0, 0, 0], (0, 0, 0)) == pytest.approx(fourpi ** -1.5, abs=1e-15)
    from numpy.polynomial.legendre import legval
    for l in range(5):                                                                  # eq. 17
        mu = float(u[0] @ u[1])
        ref = math.sqrt(2 * l + 1) / fourpi * (-1) ** l * legval(mu, [0] * l + [1])
        assert abs(P(3, [l], (l, l)) - ref) < 1e-14
    assert abs(P(4, [1, 1, 0], (1, 1, 0)) + math.sqrt(3) * fourpi ** -1.5 * (u[0] @ u[1])) < 1e-15
    ref111 = -(3j / math.sqrt(2)) * fourpi ** -1.5 * (u[0] @ np.cross(u[1], u[2]))     # odd parity: imaginary (eq. 8)
    assert abs(P(4, [1, 1, 1], (1, 1, 1)) - ref111) < 1e-15
    ref = 3 / fourpi ** 2 * (u[0] @ u[1]) * (u[2] @ u[3])                               # product of two eq.-17 functions
    assert abs(P(5, [1, 1, 0, 1, 1], (1, 1, 1, 1)) - ref) < 1e-15
