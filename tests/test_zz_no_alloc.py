"""cbgmres_k_multidot_noalloc (include/cbgmres.h): the multi-dot S2 (Fig. 1 l.5) for callers that
cannot call cudaMalloc -- no handle, the reduction scratch in a file-scope device array of the library.

Checked against the existing path (cbgmres_k_multidot through a handle) and the oracle's extended-precision
reference, on two calls in a row (the static scratch keeps the first call's contents), and that the call itself
allocates no device memory and rejects k beyond the static scratch.  Named test_zz_* so that pytest collects it last.
"""
import numpy as np
import pytest

import oracle
from workloads import ortho_basis

pytestmark = pytest.mark.gpu

TOL = 1e-12  # the bar of tests/test_gpu_kernels.py: |h_c - h_c^ref| <= 1e-12 ||v^_c|| ||w||


def _basis(fmt, n, k, seed):
    import torch

    from paper_2009_12101_b200 import payload_dtype

    V, w = ortho_basis(n, k, seed=seed)
    P, sig = oracle.enc_basis(fmt, V)
    ld = (n + 63) // 64 * 64
    Ppad = np.zeros((k, ld), dtype=P.dtype)
    Ppad[:, :n] = P
    dP = torch.as_tensor(Ppad, device="cuda").view(payload_dtype(fmt))
    return Ppad, sig, w, dP, torch.as_tensor(sig, device="cuda"), torch.as_tensor(w, device="cuda")


@pytest.mark.parametrize("fmt,n,k", [("fp64", 50021, 33), ("fp16", 200003, 100), ("int16", 50021, 9), ("fp32", 4096, 8),
                                     ("int32", 70001, 128)])
def test_noalloc_multidot_matches_existing_path_twice(fmt, n, k):
    import torch

    from paper_2009_12101_b200 import Solver
    from paper_2009_12101_b200.binding import k_multidot_noalloc

    P, sig, w, dP, dsig, dw = _basis(fmt, n, k, seed=900 + n + k)
    w2 = np.random.default_rng(901).standard_normal(n)
    dw2 = torch.as_tensor(w2, device="cuda")
    s = Solver(0)
    try:
        ref = [s.k_multidot(fmt, dP, dsig, x, n=n, k=k).cpu().numpy() for x in (dw, dw2)]
    finally:
        s.destroy()
    h = torch.full((2, k), float("nan"), dtype=torch.float64, device="cuda")  # caller-owned outputs
    # two calls in a row, different w: the second starts from the scratch the first left behind
    k_multidot_noalloc(fmt, dP, dsig, dw, h[0], n=n, k=k)
    k_multidot_noalloc(fmt, dP, dsig, dw2, h[1], n=n, k=k)
    torch.cuda.synchronize()
    got = h.cpu().numpy()
    # ... and two more with the device's free memory read on both sides: the calls take none
    before = torch.cuda.memory_allocated()
    free0, _ = torch.cuda.mem_get_info()
    k_multidot_noalloc(fmt, dP, dsig, dw2, h[0], n=n, k=k)
    k_multidot_noalloc(fmt, dP, dsig, dw, h[1], n=n, k=k)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_allocated() == before
    assert free1 >= free0, "the no-allocation entry point took device memory"
    assert np.array_equal(h.cpu().numpy(), got[::-1])
    Vn = np.array([np.linalg.norm(oracle.dec(fmt, P[c, :n], sig[c])) for c in range(k)])
    for i, x in enumerate((w, w2)):
        assert np.all(np.isfinite(got[i]))
        assert np.all(np.abs(got[i] - ref[i]) <= TOL * Vn * np.linalg.norm(x))  # the existing path
        assert np.array_equal(got[i], ref[i])  # same kernels, same launch configuration: the same bits
        h_or = oracle.ref_multidot(fmt, P, sig, x, k=k)
        assert np.all(np.abs(got[i] - h_or) <= TOL * Vn * np.linalg.norm(x))  # the oracle


def test_noalloc_multidot_rejects_sizes_beyond_the_static_scratch():
    import torch

    from paper_2009_12101_b200 import CbgmresError
    from paper_2009_12101_b200.binding import NOALLOC_MAX_K, k_multidot_noalloc

    n, k = 4096, NOALLOC_MAX_K + 1
    V = torch.zeros((k, n), dtype=torch.float64, device="cuda")
    w = torch.ones(n, dtype=torch.float64, device="cuda")
    h = torch.full((k,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(CbgmresError) as ei:
        k_multidot_noalloc("fp64", V, None, w, h)
    assert ei.value.code == 1 and "at most 128" in str(ei.value)
    torch.cuda.synchronize()
    assert torch.all(h == 7.0)  # nothing was enqueued
    # k = 0 is a no-op; fixed point without scales is an argument error
    k_multidot_noalloc("fp64", V, None, w, h, k=0)
    with pytest.raises(CbgmresError):
        k_multidot_noalloc("int16", V.to(torch.int16), None, w, h, k=4)
    torch.cuda.synchronize()
    assert torch.all(h == 7.0)
