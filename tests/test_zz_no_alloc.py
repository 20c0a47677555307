"""encore_edge_correct_noalloc: the edge correction (eqs. 41-42) for callers that must not allocate.

Why the entry point exists: encore_edge_correct cudaMallocs plan-owned scratch (the per-bin-tuple matrices).  A process
that has given all of HBM to its own pool allocator, one that runs under a fixed device-memory quota, or a latency-bound
loop that cannot take the device-wide stalls of cudaMalloc / cudaFree cannot use it.  The no-alloc variant runs the same
two kernels with the scratch in a fixed 8 MiB device array compiled into the library, so the sizes it accepts are
limited (n_b * n_lambda * (n_lambda + 1) <= ENCORE_EDGE_NOALLOC_MAX_DOUBLES = 2^20) and calls on one device share it.

What is checked: on two calls in a row - the second with a different, smaller shape, so that it runs on top of what the
first left in the shared array - the output equals that of the existing allocating path within the tolerance of the
other parity tests (1e-9 of max|zeta|), and oversized or malformed requests are refused with a status, not a crash.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (first use of the array on the device) and after the other tests.
"""
import ctypes as C

import numpy as np
import pytest

import paper_2105_08722_b200 as E

TOL = 1e-9   # the parity tolerance of tests/test_gpu_parity.py
MAX_DOUBLES = 1 << 20   # ENCORE_EDGE_NOALLOC_MAX_DOUBLES in include/encore.h


def test_noalloc_refuses_what_does_not_fit_before_touching_the_gpu():
    """Size and argument checks come before any CUDA call, so they can be exercised without a GPU.  The pointers are
    never dereferenced on these paths."""
    lib = E.lib()
    hdr = open(E._build.INCLUDE + "/encore.h").read()
    assert f"#define ENCORE_EDGE_NOALLOC_MAX_DOUBLES {MAX_DOUBLES}" in hdr
    p = C.c_void_p(256)   # non-NULL stand-in
    call = lib.encore_edge_correct_noalloc
    # 69 multiplets: 120 bin tuples fit (579 600 doubles), 218 do not (1 052 940 > 2^20); 1023 x 1 is the widest system
    assert 120 * 69 * 70 <= MAX_DOUBLES < 218 * 69 * 70
    assert call(p, p, p, 69, 218, p, None) == E.ETOOBIG
    assert call(p, p, p, 1024, 1, p, None) == E.ETOOBIG
    assert call(p, p, p, 2 ** 31 - 1, 2 ** 31 - 1, p, None) == E.ETOOBIG      # no overflow in the size product
    assert call(p, p, p, 0, 5, p, None) == E.EINVAL
    assert call(p, p, p, 5, 0, p, None) == E.EINVAL
    assert call(p, p, p, -3, 4, p, None) == E.EINVAL
    for k in range(4):
        args = [p, p, p, 5, 5, p, None]
        args[k if k < 3 else 5] = None
        assert call(*args) == E.EINVAL
    assert b"ENCORE_EDGE_NOALLOC_MAX_DOUBLES" in lib.encore_strerror(E.ETOOBIG)
    with pytest.raises(E.EncoreError) as ei:
        E.encore_edge_correct_noalloc(256, 256, 256, 69, 218, 256)
    assert ei.value.status == E.ETOOBIG


@pytest.mark.gpu
def test_noalloc_matches_the_allocating_path_on_two_calls_in_a_row():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(20211)

    def inputs(plan):
        # synthetic raw multiplets with strong geometry terms (as in test_edge_correction_matches_the_oracle): R_0 > 0
        R = rng.standard_normal((plan.n_lambda, plan.n_b)) * 0.3
        R[0] = rng.uniform(1.0, 2.0, plan.n_b)
        R[1:] *= R[0]
        N = rng.standard_normal((plan.n_lambda, plan.n_b))
        return torch.from_numpy(N).to(dev), torch.from_numpy(R).to(dev)

    # first call: 4PCF, lmax 5, 10 bins - the c3/c4 shape, 69 x 120 (579 600 doubles of the array);
    # second call: 3PCF, lmax 6, 6 bins - 7 x 15, a different shape on top of the first call's leftovers;
    # third: the first shape again with new numbers
    shapes = [(4, 10, 5), (3, 6, 6), (4, 10, 5)]
    for order, nbins, lmax in shapes:
        with E.Plan(order, 20.0, 160.0, nbins, lmax, 0.0) as plan:
            n, nb = plan.n_lambda, plan.n_b
            assert nb * n * (n + 1) <= MAX_DOUBLES
            N, R = inputs(plan)
            want = plan.edge_correct(N, R)                                   # existing path: plan-owned cudaMalloc'd scratch
            gaunt = torch.from_numpy(E.encore_get_gaunt_tensor(plan.h)).to(dev)   # the caller's own device copy of E G
            got = torch.full_like(want, float("nan"))
            st = torch.cuda.current_stream(dev).cuda_stream
            E.encore_edge_correct_noalloc(gaunt, N, R, n, nb, got, st)
            torch.cuda.synchronize()
            want, got = want.cpu().numpy(), got.cpu().numpy()
            assert np.isfinite(got).all()
            assert np.abs(got - want).max() <= TOL * np.abs(want).max()
            # same inputs again, straight after: the array now holds this very call's LU factors
            got2 = torch.full((n, nb), float("nan"), dtype=torch.float64, device=dev)
            E.encore_edge_correct_noalloc(gaunt, N, R, n, nb, got2, st)
            torch.cuda.synchronize()
            assert np.abs(got2.cpu().numpy() - want).max() <= TOL * np.abs(want).max()
    # a request beyond the array is refused and leaves the output alone
    with E.Plan(4, 20.0, 160.0, 10, 5, 0.0) as plan:
        big_nb = MAX_DOUBLES // (plan.n_lambda * (plan.n_lambda + 1)) + 1
        out = torch.zeros((plan.n_lambda, big_nb), dtype=torch.float64, device=dev)
        with pytest.raises(E.EncoreError) as ei:
            E.encore_edge_correct_noalloc(gaunt, out, out, plan.n_lambda, big_nb, out)
        assert ei.value.status == E.ETOOBIG
        torch.cuda.synchronize()
        assert float(out.abs().max()) == 0.0
