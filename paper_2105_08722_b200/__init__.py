"""Thin Python binding of the C ABI in include/encore.h (argument marshalling only).

Every step of the hot path runs in the CUDA library `libencore_b200.so`; this module loads it with
ctypes, checks status codes and passes raw pointers (`tensor.data_ptr()`) and sizes.  PyTorch is used
by callers for device memory and streams only.  There is no CPU fallback: if the library is missing it
is built with nvcc (paper_2105_08722_b200/build.py); if that fails, importing raises.

Functions carry the names of the C entry points: encore_plan, encore_compute, encore_compute_host,
encore_destroy, encore_zeta_len, encore_get_* ...; `Plan` is a small RAII convenience around them.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

OK, EINVAL, EDOMAIN, EALLOC, ECUDA, ESTATE, EUNSUPPORTED, EINTERNAL, ECAPACITY, ETOOBIG = 0, -1, -2, -3, -4, -5, -6, -7, -8, -9

# every symbol include/encore.h declares (tests check the .so exports all of them)
SYMBOLS = [
    "encore_plan", "encore_plan_flags", "encore_get_multiplet_parity", "encore_compute", "encore_compute_enqueue", "encore_query_grid", "encore_compute_host", "encore_compute_shard", "encore_get_shard_groups", "encore_get_pair_steps", "encore_set_option", "encore_get_status", "encore_edge_correct", "encore_edge_correct_noalloc", "encore_get_gaunt_tensor", "encore_compute_grid",
    "encore_destroy", "encore_zeta_len",
    "encore_num_multiplets", "encore_num_bin_tuples", "encore_num_terms", "encore_get_multiplets",
    "encore_get_bin_tuples", "encore_get_bin_edges", "encore_contraction_flops", "encore_get_contraction_layout", "encore_get_grid",
    "encore_get_cell_ids", "encore_get_bin_counts", "encore_get_primary_counts", "encore_get_alm",
    "encore_get_stage_ms", "encore_get_kernel_ms", "encore_set_timing", "encore_get_launch_count", "encore_get_candidate_pairs", "encore_get_harm_steps",
    "encore_measure_fp64_peak", "encore_measure_dmma_peak", "encore_strerror", "encore_last_cuda_error",
]


class EncoreError(RuntimeError):
    def __init__(self, status: int):
        self.status = status
        msg = lib().encore_strerror(status)
        super().__init__(f"encore status {status}: {msg.decode() if msg else '?'}")


def lib():
    """Load (building first if needed) the CUDA library.  Fails loudly; never falls back."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    L.encore_plan.argtypes = [C.POINTER(vp), C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double]
    L.encore_plan_flags.argtypes = [C.POINTER(vp), C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double, C.c_uint]
    L.encore_get_multiplet_parity.argtypes = [vp, ip]
    L.encore_compute.argtypes = [vp, vp, vp, C.c_int64, vp, vp]
    L.encore_compute_host.argtypes = [vp, vp, vp, C.c_int64, vp]
    L.encore_compute_enqueue.argtypes = [vp, vp, vp, C.c_int64, dp, dp, vp, vp]
    L.encore_query_grid.argtypes = [vp, C.c_int64, dp, dp, ip, ip]
    L.encore_compute_shard.argtypes = [vp, vp, vp, C.c_int64, C.c_int, C.c_int, vp, vp]
    L.encore_get_shard_groups.argtypes = [vp, ip]
    L.encore_get_pair_steps.argtypes = [vp]
    L.encore_set_option.argtypes = [vp, C.c_char_p, C.c_longlong]
    L.encore_get_status.argtypes = [vp]
    L.encore_edge_correct.argtypes = [vp, vp, vp, vp, vp]
    L.encore_edge_correct_noalloc.argtypes = [vp, vp, vp, C.c_int, C.c_int, vp, vp]
    L.encore_get_gaunt_tensor.argtypes = [vp, dp]
    L.encore_get_contraction_layout.argtypes = [vp, ip]
    L.encore_compute_grid.argtypes = [vp, vp, C.c_int, vp, vp]
    L.encore_destroy.argtypes = [vp]
    L.encore_zeta_len.argtypes = [vp]
    L.encore_zeta_len.restype = C.c_int64
    L.encore_num_multiplets.argtypes = [vp]
    L.encore_num_bin_tuples.argtypes = [vp]
    L.encore_num_terms.argtypes = [vp]
    L.encore_num_terms.restype = C.c_int64
    L.encore_get_multiplets.argtypes = [vp, ip]
    L.encore_get_bin_tuples.argtypes = [vp, ip]
    L.encore_get_bin_edges.argtypes = [vp, dp]
    L.encore_contraction_flops.argtypes = [vp, dp, dp]
    L.encore_get_grid.argtypes = [vp, ip, ip]
    L.encore_get_cell_ids.argtypes = [vp, vp]
    L.encore_get_bin_counts.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.encore_get_primary_counts.argtypes = [vp, vp]
    L.encore_get_alm.argtypes = [vp, C.c_int64, dp]
    L.encore_get_stage_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.encore_set_timing.argtypes = [vp, C.c_int]
    L.encore_get_kernel_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.encore_get_launch_count.argtypes = [vp]
    L.encore_get_candidate_pairs.argtypes = [vp, C.POINTER(C.c_uint64)]
    L.encore_measure_fp64_peak.argtypes = [dp, vp]
    L.encore_measure_dmma_peak.argtypes = [dp, vp]
    L.encore_get_harm_steps.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.encore_strerror.argtypes = [C.c_int]
    L.encore_strerror.restype = C.c_char_p
    L.encore_last_cuda_error.argtypes = []
    _lib = L
    return L


def _check(status: int):
    if status != OK:
        raise EncoreError(status)


def _ptr(t):
    """device/host pointer of a torch tensor, numpy array or int; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, int):
        return C.c_void_p(t)
    if isinstance(t, np.ndarray):
        return C.c_void_p(t.ctypes.data)
    return C.c_void_p(t.data_ptr())


# ---- the C entry points, same names ------------------------------------------------------------------
def encore_plan(npcf_order: int, r_min: float, r_max: float, nbins: int, lmax: int, box_size: float):
    h = C.c_void_p()
    _check(lib().encore_plan(C.byref(h), npcf_order, r_min, r_max, nbins, lmax, box_size))
    return h


ALLPARITY = 1
FP32_HARMONICS = 2


def encore_plan_flags(npcf_order: int, r_min: float, r_max: float, nbins: int, lmax: int, box_size: float, flags: int):
    h = C.c_void_p()
    _check(lib().encore_plan_flags(C.byref(h), npcf_order, r_min, r_max, nbins, lmax, box_size, flags))
    return h


def encore_get_multiplet_parity(plan) -> np.ndarray:
    out = np.zeros(encore_num_multiplets(plan), dtype=np.int32)
    _check(lib().encore_get_multiplet_parity(plan, out.ctypes.data_as(C.POINTER(C.c_int))))
    return out


def encore_compute(plan, positions, weights, n: int, zeta_out, cuda_stream: int = 0):
    """positions/weights/zeta_out: CUDA tensors (fp64, contiguous) or raw device pointers."""
    _check(lib().encore_compute(plan, _ptr(positions), _ptr(weights), n, _ptr(zeta_out), C.c_void_p(cuda_stream)))


def encore_compute_shard(plan, positions, weights, n: int, shard: int, nshards: int, zeta_partial_out, cuda_stream: int = 0):
    _check(lib().encore_compute_shard(plan, _ptr(positions), _ptr(weights), n, shard, nshards, _ptr(zeta_partial_out),
                                      C.c_void_p(cuda_stream)))


def encore_get_shard_groups(plan):
    out = (C.c_int * 3)()
    _check(lib().encore_get_shard_groups(plan, out))
    return int(out[0]), int(out[1]), int(out[2])


def encore_get_pair_steps(plan) -> int:
    v = lib().encore_get_pair_steps(plan)
    if v < 0:
        _check(v)
    return int(v)


def _d3(v):
    return None if v is None else (C.c_double * 3)(*[float(x) for x in v])


def encore_compute_enqueue(plan, positions, weights, n: int, bbox_lo, bbox_hi, zeta_out, cuda_stream: int = 0):
    """positions / weights / zeta_out: CUDA tensors (or raw device pointers); bbox_lo / bbox_hi: 3 floats each or None."""
    _check(lib().encore_compute_enqueue(plan, _ptr(positions), _ptr(weights), n, _d3(bbox_lo), _d3(bbox_hi), _ptr(zeta_out),
                                        C.c_void_p(cuda_stream)))


def encore_query_grid(plan, n: int, bbox_lo=None, bbox_hi=None):
    nc, sub = (C.c_int * 3)(), (C.c_int * 3)()
    _check(lib().encore_query_grid(plan, n, _d3(bbox_lo), _d3(bbox_hi), nc, sub))
    return list(nc), list(sub)


def encore_set_option(plan, key: str, value: int):
    _check(lib().encore_set_option(plan, key.encode(), int(value)))


def encore_edge_correct(plan, n_raw, r_raw, zeta_out, cuda_stream: int = 0):
    """n_raw, r_raw, zeta_out: CUDA fp64 tensors [n_lambda, n_b] (or raw device pointers)."""
    _check(lib().encore_edge_correct(plan, _ptr(n_raw), _ptr(r_raw), _ptr(zeta_out), C.c_void_p(cuda_stream)))


def encore_edge_correct_noalloc(gaunt, n_raw, r_raw, n_lambda: int, n_b: int, zeta_out, cuda_stream: int = 0):
    """Edge correction for callers that must not allocate device memory (a process whose HBM belongs to its own pool
    allocator, a fixed memory quota, a loop that cannot take the device-wide stalls of cudaMalloc / cudaFree).
    gaunt: CUDA fp64 tensor [n_lambda]^3, the caller's device copy of encore_get_gaunt_tensor; n_raw, r_raw, zeta_out:
    CUDA fp64 [n_lambda, n_b].  The library allocates nothing: its scratch is a fixed 8 MiB device array, which limits
    n_b * n_lambda * (n_lambda + 1) to ENCORE_EDGE_NOALLOC_MAX_DOUBLES = 2^20 (ETOOBIG beyond).  Calls on one device
    share that array: keep them on one stream.  The first call on a device should come before any stream capture."""
    _check(lib().encore_edge_correct_noalloc(_ptr(gaunt), _ptr(n_raw), _ptr(r_raw), int(n_lambda), int(n_b), _ptr(zeta_out),
                                             C.c_void_p(cuda_stream)))


def encore_compute_grid(plan, delta, G: int, zeta_out, cuda_stream: int = 0):
    _check(lib().encore_compute_grid(plan, _ptr(delta), G, _ptr(zeta_out), C.c_void_p(cuda_stream)))


def encore_get_gaunt_tensor(plan) -> np.ndarray:
    n = encore_num_multiplets(plan)
    out = np.empty((n, n, n))
    _check(lib().encore_get_gaunt_tensor(plan, out.ctypes.data_as(C.POINTER(C.c_double))))
    return out


def encore_get_contraction_layout(plan) -> dict:
    """{'kernel': 3..6 (factorised) or 0 (literal eq. 44), 'ctas': CTA work plans, 'nbuf_min', 'nbuf_max': a_lm tile buffers per CTA}"""
    out = (C.c_int * 4)()
    _check(lib().encore_get_contraction_layout(plan, out))
    return {"kernel": out[0], "ctas": out[1], "nbuf_min": out[2], "nbuf_max": out[3]}


def encore_get_status(plan) -> int:
    return int(lib().encore_get_status(plan))


def encore_compute_host(plan, positions, weights, n: int, zeta_out):
    """positions/weights/zeta_out: host buffers (numpy arrays or CPU tensors, fp64, contiguous)."""
    _check(lib().encore_compute_host(plan, _ptr(positions), _ptr(weights), n, _ptr(zeta_out)))


def encore_destroy(plan):
    _check(lib().encore_destroy(plan))


def encore_zeta_len(plan) -> int:
    return int(lib().encore_zeta_len(plan))


def encore_num_multiplets(plan) -> int:
    return int(lib().encore_num_multiplets(plan))


def encore_num_bin_tuples(plan) -> int:
    return int(lib().encore_num_bin_tuples(plan))


def encore_num_terms(plan) -> int:
    return int(lib().encore_num_terms(plan))


def encore_get_multiplets(plan, order: int) -> np.ndarray:
    out = np.empty((encore_num_multiplets(plan), 2 * order - 5), dtype=np.int32)
    _check(lib().encore_get_multiplets(plan, out.ctypes.data_as(C.POINTER(C.c_int))))
    return out


def encore_get_bin_tuples(plan, order: int) -> np.ndarray:
    out = np.empty((encore_num_bin_tuples(plan), order - 1), dtype=np.int32)
    _check(lib().encore_get_bin_tuples(plan, out.ctypes.data_as(C.POINTER(C.c_int))))
    return out


def encore_get_bin_edges(plan, nbins: int) -> np.ndarray:
    out = np.empty(nbins + 1)
    _check(lib().encore_get_bin_edges(plan, out.ctypes.data_as(C.POINTER(C.c_double))))
    return out


def encore_contraction_flops(plan):
    ex, ca = C.c_double(), C.c_double()
    _check(lib().encore_contraction_flops(plan, C.byref(ex), C.byref(ca)))
    return ex.value, ca.value


def encore_get_grid(plan):
    nc, sub = (C.c_int * 3)(), (C.c_int * 3)()
    _check(lib().encore_get_grid(plan, nc, sub))
    return list(nc), list(sub)


def encore_get_cell_ids(plan, out):
    _check(lib().encore_get_cell_ids(plan, _ptr(out)))


def encore_get_bin_counts(plan, nbins: int):
    counts = (C.c_uint64 * nbins)()
    tot = C.c_uint64()
    _check(lib().encore_get_bin_counts(plan, counts, C.byref(tot)))
    return np.array(list(counts), dtype=np.uint64), int(tot.value)


def encore_get_primary_counts(plan, out):
    _check(lib().encore_get_primary_counts(plan, _ptr(out)))


def encore_get_alm(plan, i: int, nbins: int, lmax: int) -> np.ndarray:
    """complex array [nbins, (lmax+1)(lmax+2)/2], (l, m>=0) at l(l+1)/2+m."""
    nlm = (lmax + 1) * (lmax + 2) // 2
    out = np.empty((nbins, nlm, 2))
    _check(lib().encore_get_alm(plan, i, out.ctypes.data_as(C.POINTER(C.c_double))))
    return out[..., 0] + 1j * out[..., 1]


def encore_get_stage_ms(plan):
    ms = (C.c_float * 5)()
    _check(lib().encore_get_stage_ms(plan, ms))
    return dict(zip(("grid", "sort", "pair", "contraction", "reduce"), [float(v) for v in ms]))


def encore_get_kernel_ms(plan):
    ms = (C.c_float * 7)()
    _check(lib().encore_get_kernel_ms(plan, ms))
    return dict(zip(("grid", "sort", "bounds", "k_fill", "k_harm", "k_contract", "reduce"), [float(v) for v in ms]))


def encore_set_timing(plan, enabled: bool):
    _check(lib().encore_set_timing(plan, int(enabled)))


def encore_get_launch_count(plan) -> int:
    v = lib().encore_get_launch_count(plan)
    if v < 0:
        raise EncoreError(v)
    return v


def encore_get_candidate_pairs(plan) -> int:
    v = C.c_uint64()
    _check(lib().encore_get_candidate_pairs(plan, C.byref(v)))
    return int(v.value)


def encore_get_harm_steps(plan):
    ex, ideal = C.c_uint64(), C.c_uint64()
    _check(lib().encore_get_harm_steps(plan, C.byref(ex), C.byref(ideal)))
    return int(ex.value), int(ideal.value)


def encore_measure_fp64_peak(cuda_stream: int = 0) -> float:
    v = C.c_double()
    _check(lib().encore_measure_fp64_peak(C.byref(v), C.c_void_p(cuda_stream)))
    return v.value


def encore_measure_dmma_peak(cuda_stream: int = 0) -> float:
    v = C.c_double()
    _check(lib().encore_measure_dmma_peak(C.byref(v), C.c_void_p(cuda_stream)))
    return v.value


class Plan:
    """RAII wrapper: Plan(order, r_min, r_max, nbins, lmax, box) -> .compute(pos, w) on CUDA tensors."""

    def __init__(self, order, r_min, r_max, nbins, lmax, box=0.0, allparity=False, fp32_harmonics=False):
        self.order, self.r_min, self.r_max, self.nbins, self.lmax, self.box = order, r_min, r_max, nbins, lmax, box
        flags = (ALLPARITY if allparity else 0) | (FP32_HARMONICS if fp32_harmonics else 0)
        self.h = encore_plan_flags(order, r_min, r_max, nbins, lmax, box, flags) if flags else encore_plan(order, r_min, r_max, nbins, lmax, box)
        self.n_lambda = encore_num_multiplets(self.h)
        self.n_b = encore_num_bin_tuples(self.h)

    def close(self):
        if getattr(self, "h", None) is not None:
            encore_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:      # interpreter shutdown: module globals may already be gone
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    @property
    def multiplets(self):
        return encore_get_multiplets(self.h, self.order)

    @property
    def bin_tuples(self):
        return encore_get_bin_tuples(self.h, self.order)

    def compute(self, positions, weights=None, out=None, stream=None):
        """positions: CUDA fp64 tensor (3, n) SoA; weights: CUDA fp64 (n,) or None; returns zeta (n_lambda, n_b)."""
        import torch
        assert positions.is_cuda and positions.dtype == torch.float64 and positions.is_contiguous()
        assert positions.dim() == 2 and positions.shape[0] == 3
        n = positions.shape[1]
        if weights is not None:
            assert weights.is_cuda and weights.dtype == torch.float64 and weights.is_contiguous() and weights.numel() == n
        if out is None:
            out = torch.empty((self.n_lambda, self.n_b), dtype=torch.float64, device=positions.device)
        st = torch.cuda.current_stream(positions.device).cuda_stream if stream is None else stream
        encore_compute(self.h, positions, weights, n, out, st)
        return out

    def compute_enqueue(self, positions, weights, out, bbox_lo=None, bbox_hi=None, stream=None):
        """encore_compute_enqueue: enqueue only (no read-back, no allocation; CUDA-graph capturable).  `out` must exist."""
        import torch
        assert positions.is_cuda and positions.dtype == torch.float64 and positions.is_contiguous()
        assert positions.dim() == 2 and positions.shape[0] == 3
        n = positions.shape[1]
        if weights is not None:
            assert weights.is_cuda and weights.dtype == torch.float64 and weights.is_contiguous() and weights.numel() == n
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.n_lambda * self.n_b
        st = torch.cuda.current_stream(positions.device).cuda_stream if stream is None else stream
        encore_compute_enqueue(self.h, positions, weights, n, bbox_lo, bbox_hi, out, st)
        return out

    def compute_shard(self, positions, weights, shard: int, nshards: int, out=None, stream=None):
        """Partial zeta over the primaries of shard `shard` of `nshards` (encore_compute_shard); same arguments as compute."""
        import torch
        assert positions.is_cuda and positions.dtype == torch.float64 and positions.is_contiguous()
        assert positions.dim() == 2 and positions.shape[0] == 3
        n = positions.shape[1]
        if weights is not None:
            assert weights.is_cuda and weights.dtype == torch.float64 and weights.is_contiguous() and weights.numel() == n
        if out is None:
            out = torch.empty((self.n_lambda, self.n_b), dtype=torch.float64, device=positions.device)
        st = torch.cuda.current_stream(positions.device).cuda_stream if stream is None else stream
        encore_compute_shard(self.h, positions, weights, n, shard, nshards, out, st)
        return out

    def compute_grid(self, delta, out=None, stream=None):
        """zeta of a density field on a periodic mesh: delta CUDA fp64 tensor (G, G, G) (encore_compute_grid, eq. 36)."""
        import torch
        assert delta.is_cuda and delta.dtype == torch.float64 and delta.is_contiguous() and delta.dim() == 3
        G = delta.shape[0]
        assert tuple(delta.shape) == (G, G, G)
        if out is None:
            out = torch.empty((self.n_lambda, self.n_b), dtype=torch.float64, device=delta.device)
        st = torch.cuda.current_stream(delta.device).cuda_stream if stream is None else stream
        encore_compute_grid(self.h, delta, G, out, st)
        return out

    def edge_correct(self, n_raw, r_raw, out=None, stream=None):
        """Edge-corrected zeta [n_lambda, n_b] from the raw multiplets of the D-R field and of the random field (eq. 42)."""
        import torch
        for t in (n_raw, r_raw):
            assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == (self.n_lambda, self.n_b)
        if out is None:
            out = torch.empty_like(n_raw)
        st = torch.cuda.current_stream(n_raw.device).cuda_stream if stream is None else stream
        encore_edge_correct(self.h, n_raw, r_raw, out, st)
        return out

    def compute_host(self, positions: np.ndarray, weights=None) -> np.ndarray:
        positions = np.ascontiguousarray(positions, dtype=np.float64)
        assert positions.ndim == 2 and positions.shape[0] == 3
        n = positions.shape[1]
        if weights is not None:
            weights = np.ascontiguousarray(weights, dtype=np.float64)
        out = np.empty((self.n_lambda, self.n_b))
        encore_compute_host(self.h, positions, weights, n, out)
        return out
