"""Pins of the oracle's estimator (eq. 34/35) — the four self-checks north_star asks for plus
neighbour-search and integer-output checks.  Expected values come from tests/tier0.py (explicit
N-tuple sums, eq. 46, with scipy/sympy or Cartesian closed forms), from closed-form identities,
or from invariances — never from the oracle's own code path and never from the CUDA path.
"""
import math

import numpy as np
import pytest
from numpy.polynomial.legendre import legval

import workloads as W
from tests import tier0

FOURPI = 4 * math.pi


def cloud(n, seed, scale=60.0, weights=True):
    rng = np.random.default_rng(seed)
    pos = np.ascontiguousarray(rng.uniform(0, scale, (3, n)))
    w = rng.uniform(0.5, 1.5, n) * rng.choice([-1.0, 1.0], n, p=[0.25, 0.75]) if weights else np.ones(n)
    return pos, w


# ---- (i) Tier 1 == Tier 0 -------------------------------------------------------------------
def test_3pcf_bruteforce_c1_subset_legendre(oracle):
    """40-point subset of c1 (BASELINE.json configs[0]); triplet sums of eq. 17."""
    cfg = W.CONFIGS["c1"]
    pos, w = W.make(cfg)
    sel = W.nearest_subset(pos, (500.0, 500.0, 500.0), 40)
    p, ww = np.ascontiguousarray(pos[:, sel]), w[sel]
    res = oracle.zeta(3, p, ww, 0.0, cfg.rmin, cfg.rmax, cfg.nbins, cfg.lmax)
    bins = [tuple(b) for b in res["bins"]]
    for il, lam in enumerate(res["multiplets"]):
        l = int(lam[0])
        basis = lambda v, l=l: math.sqrt(2 * l + 1) / FOURPI * (-1) ** l * legval(tier0.dot(v[0], v[1]), [0] * l + [1])
        ref = tier0.tuple_sum(p, ww, 0.0, cfg.rmin, cfg.rmax, cfg.nbins, bins, basis)
        scale = np.abs(ref).max()
        assert np.abs(res["zeta"][il] - ref.real).max() <= 1e-12 * scale
    assert res["max_imag"] <= 1e-12 * np.abs(res["zeta"]).max()


def test_3pcf_bruteforce_periodic_eq4(oracle):
    """periodic wrap exercised; basis from eq. 4 with scipy Y_lm (independent of the oracle's Y_lm)."""
    pos, w = cloud(18, 5, scale=50.0)
    box, rmin, rmax, nb, lmax = 50.0, 2.0, 25.0, 3, 3
    res = oracle.zeta(3, pos, w, box, rmin, rmax, nb, lmax)
    bins = [tuple(b) for b in res["bins"]]
    for il, lam in enumerate(res["multiplets"]):
        ref = tier0.tuple_sum(pos, w, box, rmin, rmax, nb, bins, tier0.basis_eq4(3, lam))
        assert np.abs(res["zeta"][il] - ref.real).max() <= 1e-12 * np.abs(ref).max() + 1e-30
        assert np.abs(ref.imag).max() <= 1e-12 * np.abs(ref).max() + 1e-30


def test_4pcf_bruteforce(oracle):
    pos, w = cloud(14, 21)
    rmin, rmax, nb, lmax = 5.0, 65.0, 4, 2
    res = oracle.zeta(4, pos, w, 0.0, rmin, rmax, nb, lmax, allparity=True)
    bins = [tuple(b) for b in res["bins"]]
    zc = res["zeta"] + 1j * res["zeta_im"]
    scale = np.abs(zc).max()
    for il, lam in enumerate(res["multiplets"]):
        ref = tier0.tuple_sum(pos, w, 0.0, rmin, rmax, nb, bins, tier0.basis_eq4(4, lam))
        assert np.abs(zc[il] - ref).max() <= 1e-12 * scale, lam
        if sum(lam) % 2 == 0:
            assert np.abs(zc[il].imag).max() <= 1e-13 * scale          # eq. 8: even parity real
        else:
            assert np.abs(zc[il].real).max() <= 1e-13 * scale          # odd parity imaginary
    # closed forms: P_000 and P_110
    lams = [tuple(r) for r in res["multiplets"]]
    ref = tier0.tuple_sum(pos, w, 0.0, rmin, rmax, nb, bins, lambda v: FOURPI ** -1.5 + 0 * v[0][0])
    assert np.abs(zc[lams.index((0, 0, 0))] - ref).max() <= 1e-12 * scale
    ref = tier0.tuple_sum(pos, w, 0.0, rmin, rmax, nb, bins, lambda v: -math.sqrt(3) * FOURPI ** -1.5 * tier0.dot(v[0], v[1]) + 0 * v[2][0])
    assert np.abs(zc[lams.index((1, 1, 0))] - ref).max() <= 1e-12 * scale


def test_5pcf_bruteforce(oracle):
    pos, w = cloud(11, 33)
    rmin, rmax, nb, lmax = 5.0, 70.0, 5, 1
    res = oracle.zeta(5, pos, w, 0.0, rmin, rmax, nb, lmax)
    bins = [tuple(b) for b in res["bins"]]
    scale = np.abs(res["zeta"]).max()
    lams = [tuple(r) for r in res["multiplets"]]
    assert (1, 1, 2, 1, 1) in lams and (1, 1, 1, 1, 1) in lams            # R5: intermediates above lmax
    for il, lam in enumerate(lams):
        ref = tier0.tuple_sum(pos, w, 0.0, rmin, rmax, nb, bins, tier0.basis_eq4(5, lam))
        assert np.abs(res["zeta"][il] - ref.real).max() <= 1e-12 * scale, lam
    ref = tier0.tuple_sum(pos, w, 0.0, rmin, rmax, nb, bins,
                          lambda v: 3 / FOURPI ** 2 * tier0.dot(v[0], v[1]) * tier0.dot(v[2], v[3]))
    assert np.abs(res["zeta"][lams.index((1, 1, 0, 1, 1))] - ref.real).max() <= 1e-12 * scale
    assert res["max_imag"] <= 1e-12 * scale


def test_6pcf_bruteforce(oracle):
    """N = 6 (two intermediates): eq. 34/35 through the oracle against explicit 6-tuple sums of
    the basis functions of eq. 4/5 (scipy Y_lm, sympy 3-j), every multiplet of lmax = 1 incl. intermediates above lmax"""
    pos, w = cloud(14, 66)
    rmin, rmax, nb, lmax = 2.0, 62.0, 5, 1
    res = oracle.zeta(6, pos, w, 0.0, rmin, rmax, nb, lmax)
    bins = [tuple(b) for b in res["bins"]]
    assert bins == [(0, 1, 2, 3, 4)]
    scale = np.abs(res["zeta"]).max()
    assert scale > 0
    lams = [tuple(r) for r in res["multiplets"]]
    assert (1, 1, 2, 1, 1, 1, 0) in lams and (1, 1, 2, 1, 3, 1, 0) not in lams and (1, 1, 2, 0, 2, 1, 1) in lams   # R5
    for il, lam in enumerate(lams):
        ref = tier0.tuple_sum(pos, w, 0.0, rmin, rmax, nb, bins, tier0.basis_eq4(6, lam))
        assert np.abs(res["zeta"][il] - ref.real).max() <= 1e-12 * scale, lam
    ref = tier0.tuple_sum(pos, w, 0.0, rmin, rmax, nb, bins,
                          lambda v: FOURPI ** -0.5 * 3 / FOURPI ** 2 * tier0.dot(v[0], v[1]) * tier0.dot(v[3], v[4]) + 0 * v[2][0])
    assert np.abs(res["zeta"][lams.index((1, 1, 0, 0, 0, 1, 1))] - ref.real).max() <= 1e-12 * scale
    assert res["max_imag"] <= 1e-12 * scale
    # odd-parity multiplets are imaginary, and equal the tuple sums too (ALLPARITY)
    res = oracle.zeta(6, pos, w, 0.0, rmin, rmax, nb, lmax, allparity=True)
    lams = [tuple(r) for r in res["multiplets"]]
    odd = [il for il, lam in enumerate(lams) if (lam[0] + lam[1] + lam[3] + lam[5] + lam[6]) % 2]
    assert odd
    for il in odd[:6]:
        ref = tier0.tuple_sum(pos, w, 0.0, rmin, rmax, nb, bins, tier0.basis_eq4(6, lams[il]))
        assert abs(res["zeta_im"][il, 0] - ref.imag[0]) <= 1e-12 * scale and abs(res["zeta"][il, 0]) <= 1e-12 * scale


# ---- (ii) l = 0 identity --------------------------------------------------------------------
@pytest.mark.parametrize("order", [3, 4, 5])
def test_l0_identity_c1(oracle, order):
    """zeta_{0..0}^B = (4 pi)^{-(N-1)/2}/V sum_i w_i prod_k n^w_i(b_k)/v_{b_k}  (Y_00 = (4pi)^-1/2, C = 1;
    PAPER.md:107-109) with n^w_i(b) counted here by numpy all-pairs."""
    cfg = W.CONFIGS["c1"]
    pos, _ = W.make(cfg)
    rng = np.random.default_rng(9)
    w = rng.uniform(0.8, 1.2, cfg.n)
    n = 600 if order == 5 else cfg.n
    pos, w = np.ascontiguousarray(pos[:, :n]), w[:n]
    nb = cfg.nbins
    res = oracle.zeta(order, pos, w, cfg.box, cfg.rmin, cfg.rmax, nb, 0 if order > 3 else 2, want_prim_counts=True)
    e, vb = tier0.bin_volumes(cfg.rmin, cfg.rmax, nb)
    nw = np.zeros((n, nb))
    cnt = np.zeros((n, nb), dtype=np.int64)
    for i in range(n):
        d = pos - pos[:, i:i + 1]
        d -= cfg.box * np.round(d / cfg.box)
        r = np.sqrt((d ** 2).sum(0))
        r[i] = -1.0
        b = np.searchsorted(e, r, side="right") - 1
        ok = (r > 0) & (b >= 0) & (b < nb)
        nw[i] = np.bincount(b[ok], weights=w[ok], minlength=nb)
        cnt[i] = np.bincount(b[ok], minlength=nb)
    assert (res["prim_counts"] == cnt).all()
    assert (res["bin_counts"] == cnt.sum(0)).all()
    a = nw / vb
    for iB, B in enumerate(res["bins"]):
        ref = FOURPI ** (-(order - 1) / 2) / cfg.box ** 3 * (w * np.prod(a[:, list(B)], axis=1)).sum()
        assert res["zeta"][0, iB] == pytest.approx(ref, rel=1e-12)


# ---- (iii) rotation invariance --------------------------------------------------------------
def _random_rotation(seed):
    rng = np.random.default_rng(seed)
    q, r = np.linalg.qr(rng.standard_normal((3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


@pytest.mark.parametrize("order,lmax,n", [(3, 6, 300), (4, 3, 200), (5, 2, 60), (6, 2, 24)])
def test_rotation_invariance(oracle, order, lmax, n):
    pos, w = cloud(n, 100 + order, scale=100.0)
    args = (0.0, 10.0, 70.0, 5, lmax)
    z0 = oracle.zeta(order, pos, w, *args, allparity=(order == 4))
    R = _random_rotation(order)
    c = pos.mean(axis=1, keepdims=True)
    z1 = oracle.zeta(order, np.ascontiguousarray(R @ (pos - c)), w, *args, allparity=(order == 4))
    scale = np.abs(z0["zeta"]).max()
    assert np.abs(z0["zeta"] - z1["zeta"]).max() <= 1e-11 * scale
    assert np.abs(z0["zeta_im"] - z1["zeta_im"]).max() <= 1e-11 * scale
    # binning is decided on r^2 which a rotation perturbs by rounding only: same counts unless a
    # pair sits on an edge to 1 ulp, which these seeds do not
    assert (z0["bin_counts"] == z1["bin_counts"]).all()


# ---- (iv) permutation symmetry of (l, b) pairs ----------------------------------------------
def test_permutation_symmetry_3pcf_4pcf(oracle):
    pos, w = cloud(120, 77, scale=90.0)
    rmin, rmax, nb, lmax = 5.0, 75.0, 4, 3
    z3 = oracle.zeta(3, pos, w, 0.0, rmin, rmax, nb, lmax, bins=[(0, 2), (2, 0), (1, 3), (3, 1)])["zeta"]
    assert np.allclose(z3[:, 0], z3[:, 1], rtol=1e-12, atol=0) and np.allclose(z3[:, 2], z3[:, 3], rtol=1e-12, atol=0)
    perms = [(0, 1, 2), (1, 0, 2), (0, 2, 1), (2, 1, 0), (1, 2, 0), (2, 0, 1)]
    B = (0, 2, 3)
    res = oracle.zeta(4, pos, w, 0.0, rmin, rmax, nb, lmax, allparity=True, bins=[tuple(B[p] for p in pm) for pm in perms])
    zc = res["zeta"] + 1j * res["zeta_im"]
    lams = [tuple(r) for r in res["multiplets"]]
    scale = np.abs(zc).max()
    for lam in lams:
        for ip, pm in enumerate(perms):
            lam_p = tuple(lam[p] for p in pm)
            if lam_p not in lams:
                continue
            odd_perm = pm in [(1, 0, 2), (0, 2, 1), (2, 1, 0)]
            sign = (-1) ** sum(lam) if odd_perm else 1           # 3-j column permutation symmetry
            assert abs(zc[lams.index(lam_p), ip] - sign * zc[lams.index(lam), 0]) <= 1e-12 * scale, (lam, pm)


def test_permutation_symmetry_5pcf(oracle):
    pos, w = cloud(40, 78, scale=90.0)
    rmin, rmax, nb, lmax = 5.0, 80.0, 5, 2
    B = (0, 1, 3, 4)
    swaps = {"id": (0, 1, 2, 3), "12": (1, 0, 2, 3), "34": (0, 1, 3, 2), "pairs": (2, 3, 0, 1)}
    res = oracle.zeta(5, pos, w, 0.0, rmin, rmax, nb, lmax, bins=[tuple(B[p] for p in pm) for pm in swaps.values()])
    z = res["zeta"]
    lams = [tuple(r) for r in res["multiplets"]]
    scale = np.abs(z).max()
    checked = 0
    for (l1, l2, l12, l3, l4) in lams:
        i0 = lams.index((l1, l2, l12, l3, l4))
        assert abs(z[lams.index((l2, l1, l12, l3, l4)), 1] - (-1) ** (l1 + l2 + l12) * z[i0, 0]) <= 1e-12 * scale
        assert abs(z[lams.index((l1, l2, l12, l4, l3)), 2] - (-1) ** (l12 + l3 + l4) * z[i0, 0]) <= 1e-12 * scale
        assert abs(z[lams.index((l3, l4, l12, l1, l2)), 3] - z[i0, 0]) <= 1e-12 * scale
        checked += 1
    assert checked == len(lams) > 30


# ---- neighbour search, a_lm symmetry, cell ids ---------------------------------------------
def test_cell_list_equals_all_pairs(oracle):
    cfg = W.scaled(W.CONFIGS["c3"], box=640.0, n=5000, grid=64)       # > 4096 points: cell list path
    pos, w = W.make(cfg)
    a = oracle.zeta(3, pos, w, cfg.box, cfg.rmin, cfg.rmax, 4, 2, prim_stride=50, want_prim_counts=True)
    b = oracle.zeta(3, pos, w, cfg.box, cfg.rmin, cfg.rmax, 4, 2, prim_stride=50, want_prim_counts=True, force_allpairs=True)
    assert (a["bin_counts"] == b["bin_counts"]).all() and (a["prim_counts"] == b["prim_counts"]).all()
    assert a["bin_counts"].sum() > 10000
    assert np.abs(a["zeta"] - b["zeta"]).max() <= 1e-13 * np.abs(b["zeta"]).max()
    pos, w = W.make(W.scaled(W.CONFIGS["c4"], n=6000))                 # open geometry
    a = oracle.zeta(3, pos, w, 0.0, 20.0, 160.0, 4, 2, prim_stride=60)
    b = oracle.zeta(3, pos, w, 0.0, 20.0, 160.0, 4, 2, prim_stride=60, force_allpairs=True)
    assert (a["bin_counts"] == b["bin_counts"]).all() and a["bin_counts"].sum() > 10000
    assert np.abs(a["zeta"] - b["zeta"]).max() <= 1e-12 * np.abs(b["zeta"]).max()


def test_alm_conjugation_and_counts(oracle):
    pos, w = cloud(200, 5, scale=100.0)
    a, cnt = oracle.alm(pos, w, 0.0, 10.0, 60.0, 5, 4, 17)
    for l in range(5):
        for m in range(1, l + 1):                                      # a_{l,-m} = (-1)^m a*_{lm}
            assert np.abs(a[:, l * l + l - m] - (-1) ** m * np.conj(a[:, l * l + l + m])).max() < 1e-18
    d = pos - pos[:, 17:18]
    r = np.sqrt((d ** 2).sum(0))
    e, vb = tier0.bin_volumes(10.0, 60.0, 5)
    ref = np.array([((r >= e[b]) & (r < e[b + 1])).sum() for b in range(5)])
    assert (cnt == ref).all()
    nw = np.array([w[(r >= e[b]) & (r < e[b + 1])].sum() for b in range(5)])
    assert np.allclose(a[:, 0].real, nw / vb / math.sqrt(FOURPI), rtol=1e-13)


def test_cell_ids_are_valid_cells(oracle):
    """Reading R11: the id is the linear index of the cell that geometrically contains the point."""
    for cfg, sub in [(W.CONFIGS["c1"], (2, 2, 2)), (W.CONFIGS["c1"], (8, 2, 3)), (W.scaled(W.CONFIGS["c4"], n=4000), (12, 3, 3))]:
        pos, _ = W.make(cfg)
        cid, nc = oracle.cell_ids(pos, cfg.box, cfg.rmax, sub)
        sub = np.asarray(sub)
        if cfg.box > 0:
            org, ext = np.zeros(3), np.full(3, cfg.box)
            assert (nc == np.floor(cfg.box / (cfg.rmax / sub))).all()
        else:
            org, ext = pos.min(1), pos.max(1) - pos.min(1)
            assert (nc == np.maximum(1, np.floor(ext / (cfg.rmax / sub)))).all()
        ix, iy, iz = cid % nc[0], (cid // nc[0]) % nc[1], cid // (nc[0] * nc[1])
        assert iz.max() < nc[2] and cid.min() >= 0
        for a, idx in enumerate((ix, iy, iz)):
            h = ext[a] / nc[a]
            lo, hi = org[a] + idx * h, org[a] + (idx + 1) * h
            tol = 1e-9 * h
            assert ((pos[a] >= lo - tol) & (pos[a] <= hi + tol)).all()


def test_strided_primary_subsets_add_up_to_the_full_sum(oracle):
    """prim_offset / prim_stride (what bench.py's cpu_baseline and --impl reference time): the s shards offset = 0..s-1
    with stride s partition the primaries, so their zeta and counts add up to the stride-1 result, and each shard
    holds exactly the primaries offset, offset+s, ... (checked through the per-primary counts it fills)"""
    rng = np.random.default_rng(31)
    n = 157                                              # not a multiple of the strides
    pos = np.ascontiguousarray(rng.uniform(0, 60.0, (3, n)))
    w = rng.uniform(0.5, 1.5, n)
    full = oracle.zeta(4, pos, w, 0.0, 3.0, 30.0, 4, 2, want_prim_counts=True)
    for stride in (2, 3, 7):
        z = np.zeros_like(full["zeta"])
        bc = np.zeros_like(full["bin_counts"])
        for off in range(stride):
            part = oracle.zeta(4, pos, w, 0.0, 3.0, 30.0, 4, 2, prim_offset=off, prim_stride=stride, want_prim_counts=True)
            z += part["zeta"]
            bc += part["bin_counts"]
            mine = np.zeros(n, dtype=bool)
            mine[off::stride] = True
            assert (part["prim_counts"][mine] == full["prim_counts"][mine]).all()
            assert not part["prim_counts"][~mine].any()          # rows of other primaries stay untouched (zero-initialised)
            assert part["bin_counts"].sum() == full["prim_counts"][mine].sum()
        assert (bc == full["bin_counts"]).all()
        assert np.abs(z - full["zeta"]).max() <= 1e-13 * np.abs(full["zeta"]).max()
    # an offset beyond n processes nothing
    none = oracle.zeta(4, pos, w, 0.0, 3.0, 30.0, 4, 2, prim_offset=n, prim_stride=5)
    assert not none["zeta"].any() and not none["bin_counts"].any()
    assert full["stage_seconds"][0] >= 0.0 and full["stage_seconds"][1] >= 0.0


def test_gridded_definition_against_fft_convolution(oracle):
    """eq. 36: a^b_lm(s) = F^-1[ F[delta] F[Y_lm Theta^b] ] / int Theta^b.  The oracle's gridded estimator is
    the direct lattice sum; here the same a_lm field comes from numpy FFTs of the mesh (cyclic cross-correlation with the
    kernel sampled at the minimal-image lattice offsets) and must agree with `oracle.alm` at the cell centres, and the
    3PCF assembled from the FFT fields by eq. 16 must agree with `oracle.zeta_grid`."""
    from scipy.special import sph_harm_y
    G, box, rmin, rmax, nb, lmax = 12, 60.0, 0.0, 24.0, 3, 2
    rng = np.random.default_rng(36)
    delta = rng.standard_normal((G, G, G))
    delta[rng.random((G, G, G)) < 0.5] = 0.0
    h = box / G
    res = oracle.zeta_grid(3, delta, box, rmin, rmax, nb, lmax)
    # lattice offsets (minimal image), radius, bin
    o = (np.arange(G) + G // 2) % G - G // 2
    ox, oy, oz = np.meshgrid(o, o, o, indexing="ij")
    r = h * np.sqrt(ox ** 2 + oy ** 2 + oz ** 2)
    e = np.linspace(rmin, rmax, nb + 1)
    vb = 4 * np.pi / 3 * (e[1:] ** 3 - e[:-1] ** 3)
    with np.errstate(invalid="ignore", divide="ignore"):
        theta = np.arccos(np.where(r > 0, h * oz / r, 1.0))
    phi = np.arctan2(oy, ox)
    Fd = np.fft.fftn(delta * h ** 3)
    a = np.zeros((nb, lmax + 1, 2 * lmax + 1, G, G, G), dtype=complex)
    for b in range(nb):
        sel = (r >= e[b]) & (r < e[b + 1]) & (r > 0)
        for l in range(lmax + 1):
            for m in range(-l, l + 1):
                K = np.where(sel, sph_harm_y(l, m, theta, phi), 0.0)
                # a(s) = sum_x delta(x) K(x - s): cross-correlation = F^-1[ F[delta] conj(F[conj K]) ]
                a[b, l, m + l] = np.fft.ifftn(Fd * np.conj(np.fft.fftn(np.conj(K)))) / vb[b]
    # one cell against the oracle's a_lm of the lattice particles
    idx = np.argwhere(delta != 0.0)
    pos = np.ascontiguousarray(((idx + 0.5) * h).T)
    w = delta[idx[:, 0], idx[:, 1], idx[:, 2]] * h ** 3
    for p in (0, 17, len(idx) - 1):
        a_o, _ = oracle.alm(pos, w, box, rmin, rmax, nb, lmax, p)
        ix, iy, iz = idx[p]
        for b in range(nb):
            for l in range(lmax + 1):
                for m in range(-l, l + 1):
                    assert abs(a[b, l, m + l, ix, iy, iz] - a_o[b, l * l + l + m]) <= 1e-12 * np.abs(a_o).max()
    # eq. 16 from the FFT fields
    V = box ** 3
    for il in range(lmax + 1):
        for iB, (b1, b2) in enumerate(res["bins"]):
            tot = 0.0
            for m in range(-il, il + 1):
                tot += (-1) ** (il - m) / np.sqrt(2 * il + 1) * (delta * h ** 3 * a[b1, il, m + il] * a[b2, il, -m + il]).sum()
            assert abs(tot.real / V - res["zeta"][il, iB]) <= 1e-12 * np.abs(res["zeta"]).max()
