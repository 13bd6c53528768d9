"""Pins for the oracle's SpMV and the extended-precision per-kernel references
(SURVEY.md §8(c) C-D).  Library routines (scipy, numpy, math.fsum) and closed forms only."""
import math

import numpy as np
import pytest

import oracle
from workloads import laplace2d_5pt, make_config, ortho_basis


def test_spmv_equals_scipy():
    for name, kw in (("C1", {}), ("C2", {"grid": 20}), ("C4", {"n": 20000}), ("C5", {"grid": 12})):
        p = make_config(name, **kw)
        x = np.random.default_rng(20).standard_normal(p.A.n)
        ref = p.A.to_scipy() @ x
        scale = abs(p.A.to_scipy()) @ np.abs(x)
        assert np.all(np.abs(oracle.spmv(p.A, x) - ref) <= 1e-13 * scale)
        y, rowabs = oracle.ref_spmv(p.A, x)
        assert np.all(np.abs(y - ref) <= 1e-13 * scale)
        assert np.allclose(rowabs, scale, rtol=1e-13)


def test_spmv_row_sums_closed_form():
    # A * 1 = row sums: 0 on interior rows of the 5-point Laplacian, 1 on edges, 2 in corners
    g = 16
    A = laplace2d_5pt(g, g)
    y = oracle.spmv(A, np.ones(A.n)).reshape(g, g)
    assert np.all(y[1:-1, 1:-1] == 0.0)
    assert y[0, 0] == 2.0 and y[0, 5] == 1.0 and y[7, 0] == 1.0 and y[-1, -1] == 2.0
    # e_k picks column k
    e = np.zeros(A.n)
    e[g + 1] = 1.0
    col = oracle.spmv(A, e)
    assert col[g + 1] == 4.0 and col[g] == -1.0 and col[g + 2] == -1.0 and col[1] == -1.0 and col[2 * g + 1] == -1.0
    assert np.count_nonzero(col) == 5


def test_spmv_is_not_transposed():
    # C2 is nonsymmetric: -1.3 below the diagonal, -0.7 above (reading Q16)
    p = make_config("C2", grid=6)
    e = np.zeros(p.A.n)
    e[50] = 1.0
    col = oracle.spmv(p.A, e)  # column 50 of A: A[51,50] is the (i - stride) coefficient of row 51
    assert col[51] == -1.3 and col[49] == -0.7 and col[50] == 6.0


@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_ref_multidot_and_update_closed_form(fmt):
    """w = V^T c for orthonormal V (C3's Q factor): the dots return c and the update annihilates w
    (exactly so for fp64 storage; to the storage precision otherwise)."""
    n, k = 3000, 12
    V, _ = ortho_basis(n, k, seed=2)
    rng = np.random.default_rng(21)
    c = rng.standard_normal(k)
    P, sig = oracle.enc_basis(fmt, V)
    Vhat = np.stack([oracle.dec(fmt, P[i], sig[i]) for i in range(k)])
    w = c @ Vhat
    h = oracle.ref_multidot(fmt, P, sig, w)
    # independent reference: exactly rounded sums (math.fsum) of the decoded products
    h_fsum = np.array([math.fsum(Vhat[i] * w) for i in range(k)])
    assert np.all(np.abs(h - h_fsum) <= 1e-15 * np.linalg.norm(Vhat, axis=1) * np.linalg.norm(w))
    if fmt == "fp64":
        assert np.allclose(h, c, rtol=0, atol=1e-13)
    w2, ss, am = oracle.ref_update(fmt, P, sig, h, w)
    w2_np = w - h @ Vhat
    assert np.linalg.norm(w2 - w2_np) <= 1e-14 * np.linalg.norm(w)
    assert abs(ss - math.fsum(w2 * w2)) <= 1e-15 * max(ss, 1e-300)
    assert am == np.abs(w2).max()
    tol = {"fp64": 1e-13, "fp32": 1e-6, "int32": 1e-7, "fp16": 5e-3, "int16": 5e-3}[fmt]
    assert np.linalg.norm(w2) <= tol * np.linalg.norm(w)


def test_ref_multidot_uses_leading_dimension_and_k():
    n, k = 257, 5
    rng = np.random.default_rng(22)
    P = rng.standard_normal((k, n + 7))  # ld = n + 7, only the first n entries belong to the vectors
    w = rng.standard_normal(n)
    h = oracle.ref_multidot("fp64", P, np.ones(k), w, k=3)
    assert h.shape == (3,)
    assert np.allclose(h, P[:3, :n] @ w, rtol=1e-13)


def test_norm_helpers():
    a = np.random.default_rng(23).standard_normal(10001)
    assert abs(oracle.nrm2(a) - np.linalg.norm(a)) <= 1e-13 * np.linalg.norm(a)
    assert oracle.amax(a) == np.abs(a).max()
