"""Tier-0 brute force: the NPCF multiplets as explicit N-tuple sums (eq. 46, PAPER.md:556,
with weights and the 1/(V prod v_b) normalisation of eq. 34 restored).

Pure numpy + scipy (+ sympy for 3-j); knows nothing of the oracle's C code.  The angular basis
function of a tuple is evaluated either from a Cartesian closed form or from eq. 4 with
scipy's Y_lm and sympy's 3-j, tuple by tuple — the sum is never factorised into a_lm's.
"""
import itertools

import numpy as np
from scipy.special import sph_harm_y
from sympy.physics.wigner import wigner_3j


def bin_volumes(rmin, rmax, nbins):
    e = rmin + (rmax - rmin) / nbins * np.arange(nbins + 1)
    e[-1] = rmax
    return e, 4.0 * np.pi / 3.0 * (e[1:] ** 3 - e[:-1] ** 3)


def neighbours(pos, box, rmin, rmax, nbins):
    """per primary: list over bins of (secondary indices, unit vectors r_j - s_i)."""
    e, _ = bin_volumes(rmin, rmax, nbins)
    n = pos.shape[1]
    out = []
    for i in range(n):
        d = pos - pos[:, i:i + 1]
        if box > 0:
            d = d - box * np.round(d / box)
        r = np.sqrt((d ** 2).sum(axis=0))
        per_bin = []
        for b in range(nbins):
            sel = np.where((r >= e[b]) & (r < e[b + 1]) & (r > 0) & (np.arange(n) != i))[0]
            per_bin.append((sel, d[:, sel] / r[sel]))
        out.append(per_bin)
    return out


def tuple_sum(pos, w, box, rmin, rmax, nbins, bins, basis):
    """sum_i w_i sum_{j_k in b_k(i)} prod w_jk conj(basis(rhat_1..rhat_{N-1})) / (V prod v_b).

    basis(list of unit-vector arrays broadcast over the tuple grid) -> complex array.
    Returns complex array [len(bins)].
    """
    _, vb = bin_volumes(rmin, rmax, nbins)
    nb = neighbours(pos, box, rmin, rmax, nbins)
    V = box ** 3 if box > 0 else 1.0
    res = np.zeros(len(bins), dtype=complex)
    for iB, B in enumerate(bins):
        k = len(B)
        tot = 0.0 + 0.0j
        for i in range(pos.shape[1]):
            sels = [nb[i][b] for b in B]
            if any(len(s[0]) == 0 for s in sels):
                continue
            # explicit tuple grid: axis t of the grid runs over the secondaries of bin b_t
            vecs, wts = [], 1.0
            for t, (idx, u) in enumerate(sels):
                shape = [1] * k
                shape[t] = len(idx)
                vecs.append(u.reshape(3, *shape))
                wts = wts * w[idx].reshape(shape)
            val = np.conj(basis(vecs)) * wts
            tot += w[i] * val.sum()
        res[iB] = tot / (V * np.prod(vb[list(B)]))
    return res


def _Y(l, m, u):
    theta = np.arccos(np.clip(u[2], -1.0, 1.0))
    phi = np.arctan2(u[1], u[0])
    return sph_harm_y(l, m, theta, phi)


def basis_eq4(order, lam):
    """P_Lambda by eq. 4/5 with scipy Y_lm and sympy 3-j (independent of the oracle)."""
    lam = [int(v) for v in lam]
    if order == 3:
        l = lam[0]
        terms = [((m, -m), (-1) ** (l - m) / np.sqrt(2 * l + 1)) for m in range(-l, l + 1)]
        ls = (l, l)
    elif order == 4:
        l1, l2, l3 = lam
        ls = (l1, l2, l3)
        terms = []
        for m1 in range(-l1, l1 + 1):
            for m2 in range(-l2, l2 + 1):
                m3 = -m1 - m2
                if abs(m3) > l3:
                    continue
                c = (-1) ** (l1 + l2 + l3) * float(wigner_3j(l1, l2, l3, m1, m2, m3))
                if c != 0.0:
                    terms.append(((m1, m2, m3), c))
    elif order == 5:
        l1, l2, l12, l3, l4 = lam
        ls = (l1, l2, l3, l4)
        terms = []
        for m1, m2, m3 in itertools.product(range(-l1, l1 + 1), range(-l2, l2 + 1), range(-l3, l3 + 1)):
            m4 = -m1 - m2 - m3
            m12 = m1 + m2
            if abs(m4) > l4 or abs(m12) > l12:
                continue
            c = ((-1) ** (l1 + l2 + l3 + l4) * np.sqrt(2 * l12 + 1) * (-1) ** (l12 - m12)
                 * float(wigner_3j(l1, l2, l12, m1, m2, -m12)) * float(wigner_3j(l12, l3, l4, m12, m3, m4)))
            if c != 0.0:
                terms.append(((m1, m2, m3, m4), c))
    elif order == 6:
        # eq. 5 with two intermediates: kappa = l12 - m12 + l123 - m123
        l1, l2, l12, l3, l123, l4, l5 = lam
        ls = (l1, l2, l3, l4, l5)
        terms = []
        for m1, m2, m3, m4 in itertools.product(range(-l1, l1 + 1), range(-l2, l2 + 1), range(-l3, l3 + 1), range(-l4, l4 + 1)):
            m5 = -m1 - m2 - m3 - m4
            m12, m123 = m1 + m2, m1 + m2 + m3
            if abs(m5) > l5 or abs(m12) > l12 or abs(m123) > l123:
                continue
            c = ((-1) ** (l1 + l2 + l3 + l4 + l5) * np.sqrt((2 * l12 + 1) * (2 * l123 + 1)) * (-1) ** (l12 - m12 + l123 - m123)
                 * float(wigner_3j(l1, l2, l12, m1, m2, -m12)) * float(wigner_3j(l12, l3, l123, m12, m3, -m123))
                 * float(wigner_3j(l123, l4, l5, m123, m4, m5)))
            if c != 0.0:
                terms.append(((m1, m2, m3, m4, m5), c))
    else:
        raise ValueError(order)

    def f(vecs):
        tot = 0.0
        for ms, c in terms:
            pr = c
            for l, m, u in zip(ls, ms, vecs):
                pr = pr * _Y(l, m, u)
            tot = tot + pr
        return tot
    return f


def dot(a, b):
    return (a * b).sum(axis=0)
