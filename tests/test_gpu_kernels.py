"""GPU parity, per kernel, through the C ABI (BASELINE.json north_star): compression of a given fp64
vector is bit-exact; dot / update / SpMV agree with the oracle's extended-precision references to
1e-12 in the norm-wise metrics of DESIGN.md."""
import numpy as np
import pytest

import oracle
from workloads import make_config, ortho_basis

pytestmark = pytest.mark.gpu

FORMATS = oracle.FORMATS
TOL = 1e-12


@pytest.fixture(scope="module")
def solver():
    from paper_2009_12101_b200 import Solver

    s = Solver(0)
    yield s
    s.destroy()


def _dev(a, dtype=None):
    import torch

    t = torch.as_tensor(np.ascontiguousarray(a), device="cuda")
    return t if dtype is None else t.to(dtype)


def _basis(fmt, n, k, seed, ld_extra=0):
    """k unit vectors (orthonormalised Gaussian), oracle-encoded, laid out [k, ld] on host and device."""
    import torch

    V, w = ortho_basis(n, k, seed=seed)
    P, sig = oracle.enc_basis(fmt, V)
    ld = (n + 63) // 64 * 64 + ld_extra
    Ppad = np.zeros((k, ld), dtype=P.dtype)
    Ppad[:, :n] = P
    # poison the padding: the kernels must never let entries at or beyond n reach a result
    if P.dtype.kind == "f":
        Ppad[:, n:] = np.nan
    else:
        Ppad[:, n:] = np.iinfo(P.dtype).max
    from paper_2009_12101_b200 import payload_dtype

    dP = torch.as_tensor(Ppad, device="cuda").view(payload_dtype(fmt))
    return Ppad, sig, w, dP, _dev(sig)


# ------------------------------------------------------------------------------------------ codecs
@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("n", [1, 7, 64, 1000, 100003])
def test_compress_bit_exact(solver, fmt, n):
    rng = np.random.default_rng(100 + n)
    w = rng.standard_normal(n)
    v = w / np.linalg.norm(w)
    if n > 20:  # ties, zeros, tiny values, the extremes
        v[3] = 0.0
        v[5] = -0.0
        v[7] = 1e-30
        v[11] = 2.0 ** -25
        v[13] = -(2.0 ** -24 + 2.0 ** -25)
    exp_p, exp_s = oracle.enc(fmt, v)
    p, s = solver.k_compress(fmt, _dev(v))
    got = p.cpu().numpy()
    assert got.dtype == exp_p.dtype
    assert np.array_equal(got.view(np.uint8), exp_p.view(np.uint8))
    assert s.item() == exp_s
    d = solver.k_decode(fmt, p, s).cpu().numpy()
    assert np.array_equal(d, oracle.dec(fmt, exp_p, exp_s))


@pytest.mark.parametrize("fmt", ["fp16", "fp32"])
def test_compress_midpoints_and_subnormals(solver, fmt):
    if fmt == "fp16":
        bits = np.arange(0, 0x7BFF, dtype=np.uint16)
        a = bits.view(np.float16).astype(np.float64)
        up = (bits + 1).astype(np.uint16).view(np.float16).astype(np.float64)
    else:
        a32 = np.abs(np.random.default_rng(5).uniform(-1, 1, 50000).astype(np.float32))
        a32 = np.concatenate([a32, np.float32([0.0, 1e-45, 1.1754942e-38, 1.17549435e-38])])
        a = a32.astype(np.float64)
        up = np.nextafter(a32, np.float32(np.inf)).astype(np.float64)
    mid = (a + up) / 2
    v = np.concatenate([mid, -mid, np.nextafter(mid, 0.0), np.nextafter(mid, np.inf)])
    exp_p, _ = oracle.enc(fmt, v)
    p, _ = solver.k_compress(fmt, _dev(v))
    assert np.array_equal(p.cpu().numpy().view(np.uint8), exp_p.view(np.uint8))


@pytest.mark.parametrize("fmt", ["int16", "int32"])
def test_compress_fixed_point_ties_and_zero_vector(solver, fmt):
    M = 32767 if fmt == "int16" else 2147483647
    a = M * 2.0 ** -40
    ties = np.array([0.5, 1.5, 2.5, -0.5, -1.5, -2.5, M - 0.5, -(M - 0.5), 3.25, -3.75]) * 2.0 ** -40
    v = np.concatenate([[a, -a], ties])
    exp_p, exp_s = oracle.enc(fmt, v)
    p, s = solver.k_compress(fmt, _dev(v))
    assert np.array_equal(p.cpu().numpy(), exp_p) and s.item() == exp_s == 2.0 ** -40
    z, sz = solver.k_compress(fmt, _dev(np.zeros(100)))
    assert not z.cpu().numpy().any() and sz.item() == 0.0


# ------------------------------------------------------------------------------------------ store
@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("n", [5, 4099, 70001])
def test_store_normalises_and_compresses(solver, fmt, n):
    rng = np.random.default_rng(200 + n)
    w = rng.standard_normal(n) * 37.5
    hn = float(np.linalg.norm(w))
    amax = float(np.abs(w).max())
    v = w / hn  # IEEE division per element (reading Q8)
    exp_p, exp_s = oracle.enc(fmt, v)
    p, s, vout = solver.k_store(fmt, _dev(w), hn, amax)
    assert np.array_equal(vout.cpu().numpy(), v)
    assert np.array_equal(p.cpu().numpy().view(np.uint8), exp_p.view(np.uint8))
    assert s.item() == exp_s


# ------------------------------------------------------------------------------------------ block-Jacobi(4)
@pytest.mark.parametrize("cfg,kw", [("C5", {"grid": 12}), ("C4", {"n": 5003}), ("C2", {"grid": 11}), ("C1", {"grid": 5})])
def test_bj4_setup_matches_oracle_blocks(cfg, kw):
    """The inverted 4 x 4 diagonal blocks of stencil and power-law matrices, ragged last blocks
    included (n = 5003, 1331, 25), against the oracle's Gauss-Jordan inverses."""
    from paper_2009_12101_b200 import Solver

    p = make_config(cfg, **kw)
    s = Solver(0)
    try:
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        got = s.k_bj4_setup().cpu().numpy()
    finally:
        s.destroy()
    exp = oracle.block_jacobi4(p.A)
    assert got.shape == exp.shape
    scale = np.abs(exp).max(axis=(1, 2), keepdims=True)
    assert np.all(np.abs(got - exp) <= 1e-12 * scale)
    r = p.A.n % 4
    if r:  # identity completion of the last block, bit for bit
        assert np.array_equal(got[-1, r:, :], exp[-1, r:, :]) and np.array_equal(got[-1, :, r:], exp[-1, :, r:])


@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("n", [1, 3, 4, 7, 4099, 70002])
def test_store_bj4_compresses_v_and_hands_minv_v_to_the_spmv(solver, fmt, n):
    """S4 under block-Jacobi: the payload is still enc(v), bit-exact; the fp64 output is z = M^-1 v (Fig. 1 l.3)."""
    rng = np.random.default_rng(300 + n)
    w = rng.standard_normal(n) * 3.5
    hn, amax = float(np.linalg.norm(w)), float(np.abs(w).max())
    v = w / hn
    nb = (n + 3) // 4
    inv = rng.standard_normal((nb, 4, 4)) * 10.0 ** rng.uniform(-2, 2, (nb, 1, 1))
    if n % 4:
        r = n % 4
        inv[-1, r:, :] = 0.0
        inv[-1, :, r:] = 0.0
        inv[-1, np.arange(r, 4), np.arange(r, 4)] = 1.0
    exp_p, exp_s = oracle.enc(fmt, v)
    z_ref = oracle.apply_minv("block_jacobi4", inv, v)
    vpad = np.zeros(4 * nb)
    vpad[:n] = v
    zabs = np.einsum("brc,bc->br", np.abs(inv), np.abs(vpad.reshape(nb, 4))).ravel()[:n]
    pl, sc, z = solver.k_store_bj4(fmt, _dev(w), hn, amax, _dev(inv))
    assert np.array_equal(pl.cpu().numpy().view(np.uint8), exp_p.view(np.uint8))
    assert sc.item() == exp_s
    assert np.all(np.abs(z.cpu().numpy() - z_ref) <= TOL * np.maximum(zabs, 1e-300))


# ------------------------------------------------------------------------------------------ multi-dot / update
@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("n,k", [(1, 1), (63, 3), (4096, 8), (50021, 1), (50021, 9), (50021, 33), (200003, 100)])
def test_multidot_matches_oracle(solver, fmt, n, k):
    k = min(k, n)
    P, sig, w, dP, dsig = _basis(fmt, n, k, seed=300 + n + k, ld_extra=64)
    h_ref = oracle.ref_multidot(fmt, P, sig, w, k=k)
    h = solver.k_multidot(fmt, dP, dsig, _dev(w), n=n, k=k).cpu().numpy()
    Vhat_norm = np.array([np.linalg.norm(oracle.dec(fmt, P[c, :n], sig[c])) for c in range(k)])
    assert np.all(np.isfinite(h))
    assert np.all(np.abs(h - h_ref) <= TOL * Vhat_norm * np.linalg.norm(w))


@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("n,k", [(1, 1), (63, 3), (4096, 8), (50021, 1), (50021, 9), (50021, 33), (200003, 100)])
def test_update_matches_oracle(solver, fmt, n, k):
    import torch

    k = min(k, n)
    P, sig, w, dP, dsig = _basis(fmt, n, k, seed=400 + n + k)
    h = np.random.default_rng(401).standard_normal(k)
    w_ref, ss_ref, am_ref = oracle.ref_update(fmt, P[:k], sig[:k], h, w)
    dw = _dev(w).clone()
    out = solver.k_update(fmt, dP[:k], dsig[:k], _dev(h), dw, n=n)
    torch.cuda.synchronize()
    w_gpu = dw.cpu().numpy()
    nrm2, amax = out.cpu().numpy()
    scale = np.linalg.norm(w) + np.linalg.norm(h)  # ||w|| + ||V^|| ||h||, ||V^|| ~ 1
    assert np.linalg.norm(w_gpu - w_ref) <= TOL * scale
    assert abs(nrm2 - np.sqrt(ss_ref)) <= TOL * scale
    assert amax == np.abs(w_gpu).max()


@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("n,k", [(1, 1), (63, 3), (4096, 8), (50021, 9), (50021, 33), (200003, 100), (9473, 128)])
def test_update_multidot_fused_matches_oracle(solver, fmt, n, k):
    """S3 + S2' from one read of V: w_new = w - V^ h and u = V^^T w_new, against the oracle's
    extended-precision update followed by its extended-precision multi-dot of the updated w."""
    import torch

    k = min(k, n)
    P, sig, w, dP, dsig = _basis(fmt, n, k, seed=450 + n + k, ld_extra=64)
    h = np.random.default_rng(451).standard_normal(k)
    w_ref, ss_ref, am_ref = oracle.ref_update(fmt, P[:k], sig[:k], h, w)
    u_ref = oracle.ref_multidot(fmt, P, sig, w_ref, k=k)
    dw = _dev(w).clone()
    u, out = solver.k_update_multidot(fmt, dP[:k], dsig[:k], _dev(h), dw, n=n)
    torch.cuda.synchronize()
    w_gpu, u_gpu = dw.cpu().numpy(), u.cpu().numpy()
    nrm2, amax = out.cpu().numpy()
    scale = np.linalg.norm(w) + np.linalg.norm(h)
    Vhat_norm = np.array([np.linalg.norm(oracle.dec(fmt, P[c, :n], sig[c])) for c in range(k)])
    assert np.linalg.norm(w_gpu - w_ref) <= TOL * scale
    assert abs(nrm2 - np.sqrt(ss_ref)) <= TOL * scale
    assert amax == np.abs(w_gpu).max()
    assert np.all(np.isfinite(u_gpu))
    # u inherits the update's error through V^^T: |du_c| <= ||v^_c|| ||dw|| + the dot's own rounding
    assert np.all(np.abs(u_gpu - u_ref) <= 2 * TOL * Vhat_norm * scale)


@pytest.mark.parametrize("fmt", ["fp32", "fp16", "int32", "int16"])
@pytest.mark.parametrize("rows_mapped,seg_kb", [(1, 0), (1, 1), (1, 2), (0, 0)])
@pytest.mark.parametrize("n,k,ld_extra", [(9, 9, 64), (1000, 9, 64), (40000, 17, 64), (70001, 128, 64), (200003, 33, 64),
                                          (300000, 100, 0), (148 * 1024 * 3 + 5, 12, 64), (70001, 50, 8)])
def test_fused_pass_both_mappings(fmt, rows_mapped, seg_kb, n, k, ld_extra):
    """The fused update + multi-dot of the reduced formats in both mappings: warps own rows with a shuffle reduction
    (orth_fused_kernel, 1 or 2 KB column segments: option orth_fused_rows = 1) and the column-mapped kind of
    orth_kernel (= 0, also the fall-back when a column's stride is not a multiple of 128 bytes: ld_extra = 8).
    Ragged last tiles, odd n, NaN-poisoned padding, k up to the 128 columns of one launch."""
    import torch

    from paper_2009_12101_b200 import Solver

    s = Solver(0)
    try:
        s.set_option("orth_fused_rows", rows_mapped)
        s.set_option("orth_seg_kb", seg_kb)
        P, sig, w, dP, dsig = _basis(fmt, n, k, seed=480 + n + k, ld_extra=ld_extra)
        h = np.random.default_rng(481).standard_normal(k)
        w_ref, ss_ref, am_ref = oracle.ref_update(fmt, P[:k], sig[:k], h, w)
        u_ref = oracle.ref_multidot(fmt, P, sig, w_ref, k=k)
        dw = _dev(w).clone()
        u, out = s.k_update_multidot(fmt, dP[:k], dsig[:k], _dev(h), dw, n=n)
        torch.cuda.synchronize()
        w_gpu, u_gpu = dw.cpu().numpy(), u.cpu().numpy()
        nrm2, amax = out.cpu().numpy()
        scale = np.linalg.norm(w) + np.linalg.norm(h)
        Vhat_norm = np.array([np.linalg.norm(oracle.dec(fmt, P[c, :n], sig[c])) for c in range(k)])
        assert np.linalg.norm(w_gpu - w_ref) <= TOL * scale
        assert abs(nrm2 - np.sqrt(ss_ref)) <= TOL * scale
        assert amax == np.abs(w_gpu).max()
        assert np.all(np.isfinite(u_gpu))
        assert np.all(np.abs(u_gpu - u_ref) <= 2 * TOL * Vhat_norm * scale)
        # bitwise repeatable (fixed summation order)
        dw2 = _dev(w).clone()
        u2, out2 = s.k_update_multidot(fmt, dP[:k], dsig[:k], _dev(h), dw2, n=n)
        torch.cuda.synchronize()
        assert torch.equal(dw, dw2) and torch.equal(u, u2) and torch.equal(out, out2)
    finally:
        s.destroy()


@pytest.mark.parametrize("fmt", FORMATS)
@pytest.mark.parametrize("seg_kb", [1, 2, 4])
@pytest.mark.parametrize("n,k", [(148 * 64 + 1, 5), (31111, 40), (70001, 129), (131072, 16)])
def test_orth_passes_every_tile_height(fmt, seg_kb, n, k):
    """Every column-segment size of the row tiles (1, 2, 4 KB), ragged tails, an odd n, more than
    128 columns (two launches per pass)."""
    import torch

    from paper_2009_12101_b200 import Solver

    s = Solver(0)
    try:
        s.set_option("orth_seg_kb", seg_kb)
        P, sig, w, dP, dsig = _basis(fmt, n, k, seed=470 + n + k, ld_extra=64)
        Vhat_norm = np.array([np.linalg.norm(oracle.dec(fmt, P[c, :n], sig[c])) for c in range(k)])
        h_ref = oracle.ref_multidot(fmt, P, sig, w, k=k)
        h = s.k_multidot(fmt, dP, dsig, _dev(w), n=n, k=k).cpu().numpy()
        assert np.all(np.abs(h - h_ref) <= TOL * Vhat_norm * np.linalg.norm(w))
        hh = np.random.default_rng(471).standard_normal(k)
        w_ref, ss_ref, _ = oracle.ref_update(fmt, P[:k], sig[:k], hh, w)
        dw = _dev(w).clone()
        out = s.k_update(fmt, dP[:k], dsig[:k], _dev(hh), dw, n=n)
        torch.cuda.synchronize()
        scale = np.linalg.norm(w) + np.linalg.norm(hh)
        assert np.linalg.norm(dw.cpu().numpy() - w_ref) <= TOL * scale
        assert abs(out.cpu().numpy()[0] - np.sqrt(ss_ref)) <= TOL * scale
        if k <= 128:
            dw = _dev(w).clone()
            u, out = s.k_update_multidot(fmt, dP[:k], dsig[:k], _dev(hh), dw, n=n)
            u_ref = oracle.ref_multidot(fmt, P, sig, w_ref, k=k)
            assert np.linalg.norm(dw.cpu().numpy() - w_ref) <= TOL * scale
            assert np.all(np.abs(u.cpu().numpy() - u_ref) <= 2 * TOL * Vhat_norm * scale)
    finally:
        s.destroy()


@pytest.mark.parametrize("fmt", ["fp32", "fp16", "int16"])
def test_multidot_many_tiles_per_cta_repeats_bitwise(solver, fmt):
    """A million rows and few vectors: every CTA walks many row tiles while its shared-memory ring
    holds several of them at once -- the regime in which a slot handed back before its loads had
    completed once gave wrong inner products.  Checked against the oracle and for bitwise repeatability."""
    import torch

    n, kmax = 1_000_003, 33
    rng = np.random.default_rng(480)
    V = rng.standard_normal((kmax, n)) / np.sqrt(n)
    w = rng.standard_normal(n)
    P, sig = oracle.enc_basis(fmt, V)
    ld = (n + 63) // 64 * 64
    Ppad = np.zeros((kmax, ld), dtype=P.dtype)
    Ppad[:, :n] = P
    from paper_2009_12101_b200 import payload_dtype

    dP = torch.as_tensor(Ppad, device="cuda").view(payload_dtype(fmt))
    dsig, dw = _dev(sig), _dev(w)
    for k in (1, 9, 33):
        h_ref = oracle.ref_multidot(fmt, Ppad, sig, w, k=k)
        hs = [solver.k_multidot(fmt, dP, dsig, dw, n=n, k=k).clone() for _ in range(12)]
        torch.cuda.synchronize()
        assert all(torch.equal(hs[0], h) for h in hs[1:])
        assert np.all(np.abs(hs[0].cpu().numpy() - h_ref) <= 2 * TOL * np.linalg.norm(w))


@pytest.mark.parametrize("fmt", FORMATS)
def test_cgs_closed_form(solver, fmt):
    """w in span(V^): the dots return the coefficients and the update annihilates w."""
    n, k = 30011, 16
    P, sig, _, dP, dsig = _basis(fmt, n, k, seed=500)
    Vhat = np.stack([oracle.dec(fmt, P[c, :n], sig[c]) for c in range(k)])
    c = np.random.default_rng(501).standard_normal(k)
    w = c @ Vhat
    dw = _dev(w).clone()
    h = solver.k_multidot(fmt, dP, dsig, dw, n=n, k=k)
    G = Vhat @ Vhat.T
    assert np.allclose(h.cpu().numpy(), G @ c, rtol=0, atol=1e-12 * np.linalg.norm(w))
    if fmt == "fp64":
        out = solver.k_update(fmt, dP, dsig, h, dw, n=n)
        assert out.cpu().numpy()[0] <= 1e-12 * np.linalg.norm(w)


# ------------------------------------------------------------------------------------------ SpMV
@pytest.mark.parametrize("name,kw", [("C1", {}), ("C2", {"grid": 30}), ("C4", {"n": 60000}), ("C5", {"grid": 20})])
@pytest.mark.parametrize("kernel", [0, 2, 4, 8, 16, 32, 64, 65, 129, 130, 132, 146, 148, 152])
def test_spmv_matches_oracle(name, kw, kernel):
    from paper_2009_12101_b200 import Solver

    p = make_config(name, **kw)
    s = Solver(0)
    try:
        s.set_option("spmv_kernel", kernel)
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        x = np.random.default_rng(600).standard_normal(p.A.n)
        y_ref, rowabs = oracle.ref_spmv(p.A, x)
        w, nrm = s.k_spmv(_dev(x))
        y = w.cpu().numpy()
        assert np.all(np.abs(y - y_ref) <= TOL * np.maximum(rowabs, 1e-300))
        assert abs(nrm.item() - np.linalg.norm(y_ref)) <= TOL * np.linalg.norm(y_ref)
    finally:
        s.destroy()


def test_spmv_empty_rows_and_long_rows():
    """Degenerate CSR shapes: empty rows, one dense row longer than the streaming buffer."""
    import scipy.sparse as sp

    from paper_2009_12101_b200 import Solver
    from workloads import CSR

    rng = np.random.default_rng(601)
    n = 9000
    M = sp.random(n, n, density=0.0005, random_state=7, format="lil")
    M[17, :] = rng.standard_normal(n)      # a full row (9000 > 6000-entry product buffer)
    M[4000, :3000] = 1.0                   # a long row inside an otherwise sparse block
    M[100:140, :] = 0.0                    # empty rows
    M = sp.csr_matrix(M)
    M.sort_indices()
    A = CSR(n, M.indptr.astype(np.int32), M.indices.astype(np.int32), M.data.astype(np.float64))
    x = rng.standard_normal(n)
    y_ref, rowabs = oracle.ref_spmv(A, x)
    for kernel in (0, 8, 32, 64, 65):
        s = Solver(0)
        try:
            s.set_option("spmv_kernel", kernel)
            s.set_matrix(A.row_ptr, A.col_idx, A.vals)
            y = s.k_spmv(_dev(x))[0].cpu().numpy()
            assert np.all(np.abs(y - y_ref) <= TOL * np.maximum(rowabs, 1e-300) + 0.0)
            assert np.all(y[100:140] == 0.0)
        finally:
            s.destroy()


# ------------------------------------------------------------------------------------------ errors
def test_invalid_arguments_return_status_codes(solver):
    import torch

    from paper_2009_12101_b200 import CbgmresError, Solver

    s = Solver(0)
    try:
        with pytest.raises(CbgmresError) as e:
            s.k_spmv(torch.zeros(4, dtype=torch.float64, device="cuda"), torch.zeros(4, dtype=torch.float64, device="cuda"))
        assert e.value.code == 2  # E_NOMATRIX
        V = torch.zeros((2, 72), dtype=torch.float16, device="cuda")  # ld*2 bytes not a multiple of 16
        with pytest.raises(CbgmresError) as e:
            s.k_multidot("fp16", V[:, :70].contiguous(), None, torch.zeros(60, dtype=torch.float64, device="cuda"))
        assert e.value.code == 1
        with pytest.raises(CbgmresError) as e:
            s.k_multidot("int16", torch.zeros((2, 64), dtype=torch.int16, device="cuda"), None,
                         torch.zeros(60, dtype=torch.float64, device="cuda"))
        assert e.value.code == 1  # fixed point without scales
        with pytest.raises(CbgmresError):
            s.set_option("no_such_option", 1)
    finally:
        s.destroy()
