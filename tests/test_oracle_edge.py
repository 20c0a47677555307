"""Pins of the oracle's edge-correction pieces (SURVEY.md §8(f2); PAPER.md:113-127 eqs. 12-15, :297-331 eqs. 37-43,
:676-691 App. A).  The oracle evaluates the generalised Gaunt integral from its definition (sum over M, M' of three
coupling coefficients and N-1 Gaunt integrals); here it is checked against the paper's closed forms A1-A3 with sympy's
3-j / 9-j symbols (which decides reading R18: the 9-j rows are (l_k l'_k l''_k)), against the product-to-sum relations
eq. 12 and eq. 14 evaluated at random directions, and against the uniform-geometry limit of eq. 43."""
import itertools
import math

import numpy as np
import pytest
from sympy.physics.wigner import wigner_3j, wigner_9j

FOURPI = 4 * math.pi


def _w3(a, b, c):
    return float(wigner_3j(a, b, c, 0, 0, 0))


def test_gaunt_integral_eq12_eq13(oracle):
    assert oracle.gaunt(0, 0, 0, 0, 0, 0) == pytest.approx(FOURPI ** -0.5, abs=1e-15)
    rng = np.random.default_rng(12)
    u = rng.standard_normal(3)
    u /= np.linalg.norm(u)
    Y = oracle.ylm(8, u)
    for (l1, m1, l2, m2) in [(1, 0, 1, 1), (2, -1, 3, 2), (4, 3, 2, -2), (3, 0, 3, 0)]:
        lhs = Y[l1 * l1 + l1 + m1] * Y[l2 * l2 + l2 + m2]
        rhs = 0.0
        for l3 in range(abs(l1 - l2), l1 + l2 + 1):
            m3 = m1 + m2
            if abs(m3) <= l3:   # eq. 12: sum_{l3 m3} G^{l1 l2 l3}_{m1 m2 -m3} (-1)^{m3} Y_{l3 m3}
                rhs += oracle.gaunt(l1, l2, l3, m1, m2, -m3) * (-1) ** m3 * Y[l3 * l3 + l3 + m3]
        assert abs(lhs - rhs) < 1e-14


def test_generalized_gaunt_closed_forms(oracle):
    # A1
    for l, lp, lpp in [(1, 1, 2), (2, 2, 2), (0, 3, 3), (2, 1, 3), (1, 1, 1), (4, 2, 2)]:
        ref = math.sqrt((2 * l + 1) * (2 * lp + 1) * (2 * lpp + 1)) / FOURPI * _w3(l, lp, lpp) ** 2
        assert oracle.generalized_gaunt(3, [l], [lp], [lpp]) == pytest.approx(ref, abs=1e-15)

    # A2 with the 9-j rows (l_k l'_k l''_k): reading R18
    def a2(a, b, c):
        pre = FOURPI ** -1.5
        for k in range(3):
            pre *= math.sqrt((2 * a[k] + 1) * (2 * b[k] + 1) * (2 * c[k] + 1)) * _w3(a[k], b[k], c[k])
        return pre * float(wigner_9j(a[0], b[0], c[0], a[1], b[1], c[1], a[2], b[2], c[2]))
    for a, b, c in [([1, 1, 0], [1, 1, 2], [2, 2, 2]), ([1, 1, 2], [1, 1, 0], [0, 2, 2]), ([1, 2, 3], [1, 2, 1], [2, 2, 2]),
                    ([1, 1, 1], [1, 1, 1], [2, 2, 2]), ([1, 1, 1], [1, 2, 2], [2, 1, 1]), ([2, 2, 0], [2, 0, 2], [2, 2, 2])]:
        assert oracle.generalized_gaunt(4, a, b, c) == pytest.approx(a2(a, b, c), abs=1e-15)

    # A3 with rows (l1 l2 l12; ' ; '') and (l12 l3 l4; ' ; '')
    def a3(a, b, c):
        pr = lambda x: (x[0], x[1], x[3], x[4])
        pre = FOURPI ** -2 * math.sqrt((2 * a[2] + 1) * (2 * b[2] + 1) * (2 * c[2] + 1))
        for x, y, z in zip(pr(a), pr(b), pr(c)):
            pre *= math.sqrt((2 * x + 1) * (2 * y + 1) * (2 * z + 1)) * _w3(x, y, z)
        return pre * float(wigner_9j(a[0], a[1], a[2], b[0], b[1], b[2], c[0], c[1], c[2])) * \
            float(wigner_9j(a[2], a[3], a[4], b[2], b[3], b[4], c[2], c[3], c[4]))
    for a, b, c in [([1, 1, 0, 1, 1], [1, 1, 2, 1, 1], [2, 2, 2, 2, 2]), ([1, 0, 1, 1, 0], [1, 1, 1, 0, 1], [2, 1, 2, 1, 1]),
                    ([1, 1, 1, 1, 1], [1, 1, 1, 1, 1], [2, 2, 2, 2, 2]), ([1, 1, 2, 1, 1], [0, 1, 1, 1, 0], [1, 2, 1, 2, 1])]:
        assert oracle.generalized_gaunt(5, a, b, c) == pytest.approx(a3(a, b, c), abs=1e-15)


def _all_M(ls):
    for ms in itertools.product(*[range(-l, l + 1) for l in ls[:-1]]):
        mlast = -sum(ms)
        if abs(mlast) <= ls[-1]:
            yield (*ms, mlast)


def _principal(order, lam):
    lam = [int(v) for v in lam]
    return {3: lambda x: (x[0], x[0]), 4: tuple, 5: lambda x: (x[0], x[1], x[3], x[4])}[order](lam)


def _P(oracle, order, lam, Y):
    ls = _principal(order, lam)
    tot = 0.0
    for M in _all_M(ls):
        pr = oracle.coupling(order, lam, M)
        for k, (l, m) in enumerate(zip(ls, M)):
            pr = pr * Y[k][l * l + l + m]
        tot += pr
    return tot


@pytest.mark.parametrize("order,a,b", [(3, [2], [1]), (4, [1, 1, 0], [1, 1, 2]), (4, [1, 1, 1], [1, 0, 1]), (5, [1, 1, 0, 1, 1], [1, 0, 1, 1, 0])])
def test_product_to_sum_identity_eq14(oracle, order, a, b):
    """P_Lam(R) P_Lam'(R) = sum_Lam'' E(Lam'') G^{Lam Lam' Lam''} P_Lam''(R)  (eq. 14) at a random R,
    the sum running over ALL multiplets (both parities, intermediates uncapped) with l'' <= l + l'."""
    rng = np.random.default_rng(140 + order)
    u = rng.standard_normal((order - 1, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    Y = [oracle.ylm(4, v) for v in u]
    lhs = _P(oracle, order, a, Y) * _P(oracle, order, b, Y)
    lmax2 = max(x + y for x, y in zip(_principal(order, a), _principal(order, b)))
    rhs = 0.0
    for c in oracle.multiplets(order, lmax2, allparity=True):
        g = oracle.generalized_gaunt(order, a, b, c)
        if g != 0.0:
            e = -1.0 if oracle.principal_sum(order, c) % 2 else 1.0
            rhs += e * g * _P(oracle, order, c, Y)
    assert abs(lhs - rhs) < 1e-13 * max(1.0, abs(lhs))
    assert abs(lhs) > 1e-6


def test_uniform_geometry_limit_and_round_trip(oracle):
    """eq. 43: with R_Lam' = delta_{Lam' 0} R_0 the coupling matrix is (4 pi)^{-(N-1)/2} times the
    identity, so zeta = (4 pi)^{(N-1)/2} N / R_0; and a generic f: eq. 41 followed by eq. 42 returns the input zeta."""
    for order, lmax in [(3, 4), (4, 2), (5, 1)]:
        lams = oracle.multiplets(order, lmax)
        T = oracle.gaunt_tensor(order, lams)
        n = len(lams)
        assert np.abs(T[:, 0, :] - FOURPI ** (-(order - 1) / 2) * np.eye(n)).max() < 1e-14       # G^{Lam 0 Lam''}
        assert np.abs(T - T.transpose(1, 0, 2)).max() < 1e-14                                     # symmetric in (Lam, Lam')
        rng = np.random.default_rng(order)
        nB = 3
        zeta = rng.standard_normal((n, nB))
        R = np.zeros((n, nB))
        R[0] = rng.uniform(1.0, 2.0, nB)
        N = zeta * R[0] * FOURPI ** (-(order - 1) / 2)
        assert np.abs(oracle.edge_correct(order, lams, N, R, T) - zeta).max() < 1e-12
        R[1:] = 0.2 * rng.standard_normal((n - 1, nB)) * R[0]                                     # a survey-like f_Lam
        N = np.stack([np.einsum("i,j,ijk->k", zeta[:, b], R[:, b] / R[0, b], T) * R[0, b] for b in range(nB)], axis=1)   # eq. 41
        assert np.abs(oracle.edge_correct(order, lams, N, R, T) - zeta).max() < 1e-10


@pytest.mark.parametrize("order,lmax", [(4, 1), (5, 1)])
def test_parity_odd_multiplets_in_the_edge_correction(oracle, order, lmax):
    """ALLPARITY lists: odd multiplets have imaginary coefficients and odd basis functions are imaginary.
    (i) eqs. 39-40 in complex arithmetic at a random set of directions: with zeta_Lam = i z_Lam and
    R_Lam' = i phi_Lam' for odd multiplets, zeta(R^) and R(R^) are real, and the coefficients N_Lam'' = sum zeta_Lam R_Lam'
    E(Lam'') G^{Lam Lam' Lam''}, summed over ALL Lam'' the product reaches, rebuild the function zeta(R^) R(R^); they are
    real for even and imaginary for odd Lam''.  (ii) the stored (Re / Im) rows of that N and R, on a list closed under the
    product, go through oracle.edge_correct and return the stored zeta - which fails if the factor i * i = -1 of an
    (odd, odd) -> even coupling, e.g. G^{111,111,000} = -(4 pi)^{-3/2}, is dropped."""
    rng = np.random.default_rng(4100 + order)
    lams = oracle.multiplets(order, lmax, allparity=True)
    odd = np.array([oracle.principal_sum(order, lam) % 2 == 1 for lam in lams])
    assert odd.any() and not odd[0]
    n = len(lams)
    z = rng.standard_normal(n)                       # stored values
    phi = 0.3 * rng.standard_normal(n)
    phi[0] = 1.5
    unit = np.where(odd, 1j, 1.0)
    zc, rc = unit * z, unit * phi
    # every multiplet the products P_Lam P_Lam' reach: principal l'' <= 2 lmax, intermediates free
    big = oracle.multiplets(order, 2 * lmax, allparity=True)
    if order == 5:   # the intermediate l12'' of a product is not capped by 2 lmax in `multiplets`; list them all
        big = np.array([[a, b, c, d, e] for a in range(2 * lmax + 1) for b in range(2 * lmax + 1) for c in range(abs(a - b), a + b + 1)
                        for d in range(2 * lmax + 1) for e in range(abs(c - d), c + d + 1) if e <= 2 * lmax], dtype=np.int32)
    big_odd = np.array([oracle.principal_sum(order, lam) % 2 == 1 for lam in big])
    Nc = np.zeros(len(big), dtype=complex)
    for k, c in enumerate(big):
        e = -1.0 if big_odd[k] else 1.0
        for i in range(n):
            for j in range(n):
                g = oracle.generalized_gaunt(order, lams[i], lams[j], c)
                if g != 0.0:
                    Nc[k] += zc[i] * rc[j] * e * g
    assert np.abs(np.where(big_odd, Nc.real, Nc.imag)).max() < 1e-14
    assert np.abs(Nc[big_odd]).max() > 1e-3 and np.abs(Nc[~big_odd]).max() > 1e-3
    u = rng.standard_normal((order - 1, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    Y = [oracle.ylm(2 * lmax, v) for v in u]
    zeta_fn = sum(zc[i] * _P(oracle, order, lams[i], Y) for i in range(n))
    rand_fn = sum(rc[i] * _P(oracle, order, lams[i], Y) for i in range(n))
    n_fn = sum(Nc[k] * _P(oracle, order, big[k], Y) for k in range(len(big)) if Nc[k] != 0)
    assert abs(zeta_fn.imag) < 1e-13 and abs(rand_fn.imag) < 1e-13          # real functions (eq. 8)
    assert abs(n_fn - zeta_fn * rand_fn) < 1e-12 * max(1.0, abs(zeta_fn * rand_fn))
    # (ii) truncated to `lams`, as the estimator does: eq. 41 forward in complex arithmetic, eq. 42 back through the oracle
    T = oracle.gaunt_tensor(order, lams)
    Nl = np.einsum("i,j,ijk->k", zc, rc, T.astype(complex))
    N_stored = np.where(odd, Nl.imag, Nl.real)
    back = oracle.edge_correct(order, lams, N_stored[:, None], phi[:, None], T)[:, 0]
    assert np.abs(back - z).max() < 1e-11
    # the (odd, odd) -> even couplings are there and carry weight: dropping their sign changes N
    oo = np.einsum("i,j,ijk->k", np.where(odd, z, 0.0), np.where(odd, phi, 0.0), T)
    assert np.abs(oo[~odd]).max() > 1e-3
