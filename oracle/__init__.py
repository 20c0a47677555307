"""ctypes front-end of the CPU oracle (oracle/encore_oracle.c) — TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It never imports paper_2105_08722_b200 and shares nothing with it.
The C file is compiled on first use with gcc (OpenMP) into oracle/libencore_oracle.so.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "encore_oracle.c")
_LIB = os.path.join(_HERE, "libencore_oracle.so")
_lib = None

CFLAGS = ["-O2", "-std=gnu11", "-fopenmp", "-ffp-contract=off", "-fcx-limited-range",
          "-shared", "-fPIC", "-Wall"]


def build(force: bool = False) -> str:
    """Compile the oracle (gcc).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.run(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    dp = C.POINTER(C.c_double)
    ip = C.POINTER(C.c_int)
    lib.oracle_wigner3j.restype = C.c_double
    lib.oracle_wigner3j.argtypes = [C.c_int] * 6
    lib.oracle_ylm.restype = None
    lib.oracle_ylm.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, dp, dp]
    lib.oracle_multiplets.restype = C.c_int
    lib.oracle_multiplets.argtypes = [C.c_int, C.c_int, C.c_int, ip]
    lib.oracle_coupling.restype = C.c_double
    lib.oracle_coupling.argtypes = [C.c_int, ip, ip]
    lib.oracle_count_terms.restype = C.c_int64
    lib.oracle_count_terms.argtypes = [C.c_int] * 4
    lib.oracle_bin_edges.restype = None
    lib.oracle_bin_edges.argtypes = [C.c_double, C.c_double, C.c_int, dp]
    lib.oracle_cell_ids.restype = C.c_int
    lib.oracle_cell_ids.argtypes = [dp, C.c_int64, C.c_double, C.c_double, ip,
                                    C.POINTER(C.c_int32), ip]
    lib.oracle_bin_tuples.restype = C.c_int64
    lib.oracle_bin_tuples.argtypes = [C.c_int, C.c_int, ip]
    lib.oracle_alm.restype = C.c_int
    lib.oracle_alm.argtypes = [dp, dp, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_int,
                               C.c_int, C.c_int64, C.c_int, dp, dp, C.POINTER(C.c_uint32)]
    lib.oracle_zeta.restype = C.c_int
    lib.oracle_zeta.argtypes = [C.c_int, dp, dp, C.c_int64, C.c_double, C.c_double, C.c_double,
                                C.c_int, C.c_int, C.c_int, ip, C.c_int64, C.c_int64, C.c_int64,
                                C.c_int, dp, dp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint32), dp, dp]
    lib.oracle_num_threads.restype = C.c_int
    lib.oracle_gaunt.restype = C.c_double
    lib.oracle_gaunt.argtypes = [C.c_int] * 6
    lib.oracle_generalized_gaunt.restype = C.c_double
    lib.oracle_generalized_gaunt.argtypes = [C.c_int, ip, ip, ip]
    _lib = lib
    return lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _pos(pos):
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    assert pos.ndim == 2 and pos.shape[0] == 3, "positions are SoA (3, n)"
    return pos


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def wigner3j(j1, j2, j3, m1, m2, m3) -> float:
    return float(_load().oracle_wigner3j(j1, j2, j3, m1, m2, m3))


def ylm(lmax: int, v) -> np.ndarray:
    """Y_lm of a unit vector, complex array indexed l*l+l+m."""
    n = (lmax + 1) ** 2
    re, im = np.empty(n), np.empty(n)
    _load().oracle_ylm(lmax, float(v[0]), float(v[1]), float(v[2]), _dp(re), _dp(im))
    return re + 1j * im


def multiplets(order: int, lmax: int, allparity: bool = False) -> np.ndarray:
    lib = _load()
    n = lib.oracle_multiplets(order, lmax, int(allparity), None)
    out = np.empty((n, 2 * order - 5), dtype=np.int32)
    lib.oracle_multiplets(order, lmax, int(allparity), _ip(out))
    return out


def coupling(order: int, lam, m) -> float:
    lam = np.ascontiguousarray(lam, dtype=np.int32)
    m = np.ascontiguousarray(m, dtype=np.int32)
    return float(_load().oracle_coupling(order, _ip(lam), _ip(m)))


def count_terms(order: int, lmax: int, allparity: bool = False, half: bool = False) -> int:
    return int(_load().oracle_count_terms(order, lmax, int(allparity), int(half)))


def bin_edges(rmin: float, rmax: float, nbins: int) -> np.ndarray:
    e = np.empty(nbins + 1)
    _load().oracle_bin_edges(rmin, rmax, nbins, _dp(e))
    return e


def bin_tuples(order: int, nbins: int) -> np.ndarray:
    lib = _load()
    n = lib.oracle_bin_tuples(order, nbins, None)
    out = np.empty((n, order - 1), dtype=np.int32)
    lib.oracle_bin_tuples(order, nbins, _ip(out))
    return out


def cell_ids(pos, box: float, rmax: float, sub):
    """(cid int32[n], nc[3]) by the formula of reading R11; sub = S or (S_x, S_y, S_z)."""
    pos = _pos(pos)
    n = pos.shape[1]
    cid = np.empty(n, dtype=np.int32)
    nc = np.zeros(3, dtype=np.int32)
    sub = np.ascontiguousarray(np.broadcast_to(np.asarray(sub, dtype=np.int32), (3,)))
    rc = _load().oracle_cell_ids(_dp(pos), n, box, rmax, _ip(sub),
                                 cid.ctypes.data_as(C.POINTER(C.c_int32)), _ip(nc))
    assert rc == 0
    return cid, nc


def alm(pos, w, box, rmin, rmax, nbins, lmax, i, force_allpairs=False):
    """(a[nbins, (lmax+1)^2] complex, counts[nbins] uint32) of primary i (eq. 35)."""
    pos = _pos(pos)
    n = pos.shape[1]
    nlm = (lmax + 1) ** 2
    re, im = np.empty((nbins, nlm)), np.empty((nbins, nlm))
    cnt = np.zeros(nbins, dtype=np.uint32)
    wp = None if w is None else _dp(np.ascontiguousarray(w, dtype=np.float64))
    rc = _load().oracle_alm(_dp(pos), wp, n, box, rmin, rmax, nbins, lmax, int(i),
                            int(force_allpairs), _dp(re), _dp(im),
                            cnt.ctypes.data_as(C.POINTER(C.c_uint32)))
    assert rc == 0, rc
    return re + 1j * im, cnt


def zeta(order, pos, w, box, rmin, rmax, nbins, lmax, *, allparity=False, bins=None,
         prim_offset=0, prim_stride=1, force_allpairs=False, want_prim_counts=False):
    """zeta^B_Lambda by eq. 34/35 over primaries offset, offset+stride, ...

    Returns dict(zeta[nLam,nB], zeta_im, bin_counts[nbins] uint64, prim_counts or None,
    max_imag, multiplets, bins, stage_seconds=(a_lm stage, contraction) wall seconds).
    """
    lib = _load()
    pos = _pos(pos)
    n = pos.shape[1]
    lam = multiplets(order, lmax, allparity)
    if bins is None:
        bt = bin_tuples(order, nbins)
        bptr, nB = None, bt.shape[0]
    else:
        bt = np.ascontiguousarray(bins, dtype=np.int32).reshape(-1, order - 1)
        bptr, nB = _ip(bt), bt.shape[0]
    z = np.zeros((lam.shape[0], nB))
    zi = np.zeros((lam.shape[0], nB))
    bc = np.zeros(nbins, dtype=np.uint64)
    pc = np.zeros((n, nbins), dtype=np.uint32) if want_prim_counts else None
    mi = C.c_double(0.0)
    secs = np.zeros(2)
    wa = None if w is None else np.ascontiguousarray(w, dtype=np.float64)
    rc = lib.oracle_zeta(order, _dp(pos), None if wa is None else _dp(wa), n, float(box),
                         float(rmin), float(rmax), nbins, lmax, int(allparity), bptr, nB,
                         int(prim_offset), int(prim_stride), int(force_allpairs), _dp(z), _dp(zi),
                         bc.ctypes.data_as(C.POINTER(C.c_uint64)),
                         None if pc is None else pc.ctypes.data_as(C.POINTER(C.c_uint32)),
                         C.byref(mi), _dp(secs))
    if rc != 0:
        raise ValueError(f"oracle_zeta failed with status {rc}")
    return dict(zeta=z, zeta_im=zi, bin_counts=bc, prim_counts=pc, max_imag=mi.value,
                multiplets=lam, bins=bt, stage_seconds=(float(secs[0]), float(secs[1])))


# ---- edge correction (eqs. 39-42) ------------------------------------------
def gaunt(l1, l2, l3, m1, m2, m3) -> float:
    """Gaunt integral, eq. 13."""
    return float(_load().oracle_gaunt(l1, l2, l3, m1, m2, m3))


def generalized_gaunt(order: int, lam_a, lam_b, lam_c) -> float:
    """G^{Lam Lam' Lam''} = int dR P_Lam P_Lam' P_Lam'' (eq. 15) from its definition (sum over M, M' of C C C prod Gaunt)."""
    a, b, c = (np.ascontiguousarray(v, dtype=np.int32) for v in (lam_a, lam_b, lam_c))
    return float(_load().oracle_generalized_gaunt(order, _ip(a), _ip(b), _ip(c)))


def principal_sum(order: int, lam) -> int:
    lam = [int(v) for v in lam]
    return {3: lambda x: 2 * x[0], 4: sum, 5: lambda x: x[0] + x[1] + x[3] + x[4], 6: lambda x: x[0] + x[1] + x[3] + x[5] + x[6]}[order](lam)


def gaunt_tensor(order: int, lams) -> np.ndarray:
    """T[Lam, Lam', Lam''] = E(Lam'') G^{Lam Lam' Lam''} over the given multiplet list (the bracket of eq. 41 before
    the f_Lam' weights)."""
    lams = np.ascontiguousarray(lams, dtype=np.int32)
    n = len(lams)
    T = np.zeros((n, n, n))
    for i in range(n):
        for j in range(n):
            for k in range(n):
                e = -1.0 if principal_sum(order, lams[k]) % 2 else 1.0
                T[i, j, k] = e * generalized_gaunt(order, lams[i], lams[j], lams[k])
    return T


def edge_correct(order: int, lams, N, R, T=None) -> np.ndarray:
    """Edge-corrected multiplets, eq. 42, one linear system per bin tuple B:
        f_Lam'(B) = R_Lam'^B / R_0^B;   M_{Lam Lam''}(B) = sum_Lam' f_Lam'(B) E(Lam'') G^{Lam Lam' Lam''}   (eq. 41)
        sum_Lam zeta_Lam(B) M_{Lam Lam''}(B) = N_Lam''^B / R_0^B                                       (eq. 41) -> solve
    N, R: [nLam, nB] raw multiplets of the data-minus-random and the random field on the multiplet list `lams`, whose
    first row is the all-zero multiplet.  The basis is truncated to `lams` (as the paper truncates at lmax).

    Parity-odd multiplets (ALLPARITY lists): their coefficients are purely imaginary (eq. 8) and the rows of
    N, R and of the result hold the IMAGINARY part for them (the real part for even multiplets), as `zeta` stores them.
    Eqs. 40-42 are relations between the complex coefficients, so they are evaluated here in complex arithmetic:
    coefficient = stored value for even, i * stored value for odd multiplets; the solution is real for even and
    imaginary for odd multiplets (checked) and is returned in the stored form."""
    lams = np.ascontiguousarray(lams, dtype=np.int32)
    assert not lams[0].any(), "the first multiplet must be Lambda = 0"
    N, R = np.asarray(N, dtype=np.float64), np.asarray(R, dtype=np.float64)
    if T is None:
        T = gaunt_tensor(order, lams)
    odd = np.array([principal_sum(order, lam) % 2 == 1 for lam in lams])
    unit = np.where(odd, 1j, 1.0)                       # stored value -> complex coefficient
    out = np.empty_like(N)
    for iB in range(N.shape[1]):
        f = unit * R[:, iB] / R[0, iB]
        M = np.einsum("j,ijk->ik", f, T.astype(np.complex128))   # M[Lam, Lam'']
        z = np.linalg.solve(M.T, unit * N[:, iB] / R[0, iB])
        stored = np.where(odd, z.imag, z.real)
        other = np.where(odd, z.real, z.imag)
        assert np.abs(other).max() <= 1e-9 * max(np.abs(stored).max(), 1e-300), "solution has the wrong reality"
        out[:, iB] = stored
    return out


# ---- gridded estimator (eq. 36) ---------------------------------------------
def zeta_grid(order, delta, box, rmin, rmax, nbins, lmax, *, allparity=False):
    """NPCF multiplets of a density field given on a periodic G^3 mesh (cell size h = box / G, value delta[ix, iy, iz] at
    the cell centre (ix + 1/2, iy + 1/2, iz + 1/2) h).

    Discretising eq. 35/36 on the mesh, int dr -> h^3 sum over cells, gives
        a^b_lm(s) = (1/v_b) sum_{cells x != s} delta(x) h^3 Y_lm((x - s)^) Theta^b(|x - s|),   v_b = int dr Theta^b(r)
        zeta^B_Lam = (1/V) sum_cells s  delta(s) h^3  sum_M E(Lam) C^Lam_M prod_k a^{b_k}_{l_k m_k}(s)            (steps i-iii)
    which is eq. 34/35 for particles at the cell centres with weights delta h^3 (minimal-image separations of the
    periodic mesh): the definition is evaluated by the direct sums of `zeta`, no FFT.  Cells with delta = 0 contribute
    nothing and are left out."""
    delta = np.asarray(delta, dtype=np.float64)
    G = delta.shape[0]
    assert delta.shape == (G, G, G)
    h = box / G
    idx = np.argwhere(delta != 0.0)
    pos = np.ascontiguousarray(((idx + 0.5) * h).T)
    w = delta[idx[:, 0], idx[:, 1], idx[:, 2]] * h ** 3
    return zeta(order, pos, w, box, rmin, rmax, nbins, lmax, allparity=allparity)
