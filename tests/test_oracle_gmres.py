"""Pins for the oracle's restarted CB-GMRES (Fig. 1) against what the mathematics
fixes (BASELINE.json north_star): direct dense solves, <= n-step convergence,
the Arnoldi relation, basis orthogonality, the least-squares problem via numpy.linalg.lstsq, the
recurrence-vs-explicit residual, a library GMRES (scipy), and for compressed storage the mixed
Arnoldi relation of reading Q1, |V^| <= 1 and the paper's qualitative claims
(Table 2)."""
import numpy as np
import pytest

import oracle
from workloads import make_config, random_dense_system

RSQ2 = 1.0 / np.sqrt(2.0)


@pytest.mark.parametrize("n,seed", [(8, 30), (33, 31), (64, 32)])
@pytest.mark.parametrize("reorth", ["never", "cond", "always"])
def test_fp64_tiny_dense_matches_direct_solve_and_converges_in_n_steps(n, seed, reorth):
    A, Ad, b = random_dense_system(n, seed)
    r = oracle.gmres(A, b, np.zeros(n), restart=n, rel_tol=1e-13, max_iters=4 * n, fmt="fp64", reorth=reorth)
    xs = np.linalg.solve(Ad, b)
    assert r.converged
    assert r.iters <= n  # Krylov space of dimension n is the whole space
    assert np.linalg.norm(r.x - xs) <= 1e-10 * np.linalg.norm(xs)
    assert r.rel_res_true <= 1e-13


def test_fp64_restarted_matches_direct_solve_nonzero_x0():
    n = 40
    A, Ad, b = random_dense_system(n, 33, density=0.3)
    x0 = np.random.default_rng(34).standard_normal(n)
    r = oracle.gmres(A, b, x0, restart=7, rel_tol=1e-12, max_iters=2000, fmt="fp64")
    assert r.converged and r.restarts > 1
    xs = np.linalg.solve(Ad, b)
    assert np.linalg.norm(r.x - xs) <= 1e-9 * np.linalg.norm(xs)
    # threshold is relative to ||b||, not ||r0|| (reading Q9)
    assert np.linalg.norm(b - Ad @ r.x) <= 1e-12 * np.linalg.norm(b) * (1 + 1e-6)
    assert r.b_norm == pytest.approx(np.linalg.norm(b), rel=1e-14)


def _first_cycle(fmt, reorth="cond", grid=12, m=30):
    p = make_config("C2", grid=grid)
    r = oracle.gmres(p.A, p.b, p.x0, restart=m, rel_tol=1e-30, max_iters=m, fmt=fmt, reorth=reorth,
                     capture_cycle=0)
    return p, r


@pytest.mark.parametrize("reorth", ["cond", "always"])
def test_fp64_arnoldi_relation_and_orthogonality(reorth):
    p, r = _first_cycle("fp64", reorth)
    cap = r.capture
    k = cap["k"]
    assert k == 30
    S = p.A.to_scipy()
    V = cap["Vhat"]  # (k+1) x n, fp64 storage: identical to the fp64 vectors
    assert np.array_equal(V, cap["Vfp64"])
    AV = (S @ V[:k].T)  # n x k
    lhs = AV - V.T @ cap["Hbar"]
    normA = np.sqrt((p.A.vals ** 2).sum())
    assert np.linalg.norm(lhs) <= 1e-12 * normA
    G = V @ V.T
    assert np.linalg.norm(np.eye(k + 1) - G, 2) < 1e-12
    # v_1 = r_0 / beta
    assert cap["beta"] == pytest.approx(np.linalg.norm(p.b), rel=1e-14)
    assert np.allclose(V[0], p.b / cap["beta"], rtol=1e-15, atol=0)
    # Hessenberg structure
    H = cap["Hbar"]
    assert np.all(np.tril(H, -2) == 0)
    assert np.all(np.diag(H, -1) > 0)


def test_cgs_without_reorth_loses_orthogonality_but_keeps_arnoldi_relation():
    # the reason for l.7-11: classical Gram-Schmidt alone is not orthogonal to working precision
    p, r = _first_cycle("fp64", "never", grid=16, m=60)
    cap = r.capture
    k = cap["k"]
    V = cap["Vhat"]
    S = p.A.to_scipy()
    assert np.linalg.norm(S @ V[:k].T - V.T @ cap["Hbar"]) <= 1e-12 * np.sqrt((p.A.vals ** 2).sum())
    loss_never = np.linalg.norm(np.eye(k + 1) - V @ V.T, 2)
    _, r2 = _first_cycle("fp64", "cond", grid=16, m=60)
    V2 = r2.capture["Vhat"]
    loss_cond = np.linalg.norm(np.eye(k + 1) - V2 @ V2.T, 2)
    assert loss_cond < 1e-13 < loss_never


def test_least_squares_update_matches_numpy_lstsq():
    p, r = _first_cycle("fp64")
    cap = r.capture
    k, H, beta = cap["k"], cap["Hbar"], cap["beta"]
    rhs = np.zeros(k + 1)
    rhs[0] = beta
    y_ref, res, *_ = np.linalg.lstsq(H, rhs, rcond=None)
    assert np.allclose(cap["y"], y_ref, rtol=1e-10, atol=1e-14)
    resid = np.linalg.norm(rhs - H @ y_ref)
    assert abs(abs(cap["g"][k]) - resid) <= 1e-10 * beta
    # x_m = x_0 + V_m y_m
    assert np.allclose(r.x, cap["y"] @ cap["Vhat"][:k], rtol=1e-12, atol=1e-15)
    # recurrence residual equals the explicit residual after the first cycle
    S = p.A.to_scipy()
    expl = np.linalg.norm(p.b - S @ r.x) / np.linalg.norm(p.b)
    assert r.rel_res_recurrence == pytest.approx(expl, rel=1e-8)
    assert r.expl_history[1] == pytest.approx(expl, rel=1e-10)


def test_residual_estimate_non_increasing_within_a_cycle_and_matches_scipy():
    import scipy.sparse.linalg as spla

    p = make_config("C2", grid=10)
    m = 25
    r = oracle.gmres(p.A, p.b, p.x0, restart=m, rel_tol=1e-10, max_iters=400, fmt="fp64")
    assert r.converged
    h = r.rec_history
    for c in range(0, r.iters, m):  # inside each cycle (cycles are m long until the last)
        seg = h[c:c + m]
        assert np.all(np.diff(seg) <= 1e-14)
    # library special case: same minimisation problem per inner step
    hist = []
    spla.gmres(p.A.to_scipy(), p.b, x0=p.x0, restart=m, rtol=1e-10, atol=0.0, maxiter=400,
               callback=lambda rk: hist.append(rk), callback_type="pr_norm")
    hist = np.array(hist)
    kmax = min(len(hist), len(h))
    sel = h[:kmax] > 1e-9
    assert sel.sum() > 20
    assert np.allclose(h[:kmax][sel], hist[:kmax][sel], rtol=1e-6)
    assert abs(len(hist) - r.iters) <= 1


@pytest.mark.parametrize("fmt", ["fp32", "fp16", "int32", "int16"])
def test_compressed_mixed_arnoldi_relation_and_bounds(fmt):
    """Reading Q1: the SpMV multiplies the fp64 v_j while the orthogonalisation reads the decoded
    basis, so  A v_j = V^_j h_{1:j,j} + h_{j+1,j} v_{j+1}  holds to fp64 round-off."""
    p, r = _first_cycle(fmt)
    cap = r.capture
    k, H = cap["k"], cap["Hbar"]
    Vh, Vf = cap["Vhat"], cap["Vfp64"]
    S = p.A.to_scipy()
    normA = np.sqrt((p.A.vals ** 2).sum())
    err = 0.0
    for j in range(k):
        lhs = S @ Vf[j]
        rhs = H[: j + 1, j] @ Vh[: j + 1] + H[j + 1, j] * Vf[j + 1]
        err = max(err, np.linalg.norm(lhs - rhs))
    assert err <= 1e-12 * normA
    # the plain relation does NOT hold for compressed storage (it would if SpMV read V^)
    plain = np.linalg.norm(S @ Vh[:k].T - Vh.T @ H)
    assert plain > 100 * err
    # stored entries bounded by 1; decoded vectors close to the fp64 ones to the format's precision
    assert np.abs(Vh).max() <= 1.0
    u = {"fp32": 2.0 ** -24, "int32": 2.0 ** -31, "fp16": 2.0 ** -11, "int16": 2.0 ** -15}[fmt]
    assert np.abs(Vh - Vf).max() <= u * 1.0001
    assert np.abs(Vf).max() <= 1.0 and np.allclose(np.linalg.norm(Vf, axis=1), 1.0, rtol=1e-14)
    # orthogonality of the decoded basis degrades only to the storage precision
    G = Vh @ Vh.T
    assert np.abs(np.eye(k + 1) - G).max() <= 8 * u * np.sqrt(p.A.n)


@pytest.mark.parametrize("fmt", ["fp64", "fp32", "fp16", "int32", "int16"])
def test_converged_means_explicit_residual_below_threshold(fmt):
    p = make_config("C2", grid=14)
    r = oracle.gmres(p.A, p.b, p.x0, restart=20, rel_tol=1e-8, max_iters=3000, fmt=fmt)
    S = p.A.to_scipy()
    true = np.linalg.norm(p.b - S @ r.x) / np.linalg.norm(p.b)
    assert r.converged and true <= 1e-8 * (1 + 1e-6)
    assert r.rel_res_true == pytest.approx(true, rel=1e-6)
    assert r.expl_history[0] == pytest.approx(1.0, rel=1e-14)  # x0 = 0
    assert len(r.expl_history) == r.restarts + 1


def test_paper_qualitative_iteration_counts():
    # Table 2: 32-bit formats match fp64's iteration count, 16-bit formats need
    # at least as many.  Exact counts on synthetic inputs are unpinned.
    p = make_config("C2", grid=24)
    it = {f: oracle.gmres(p.A, p.b, p.x0, restart=p.restart, rel_tol=p.rel_tol, max_iters=5000, fmt=f).iters
          for f in oracle.FORMATS}
    # ("match ... in almost all cases, and only need a few additional iterations")
    assert abs(it["fp32"] - it["fp64"]) <= 0.05 * it["fp64"]
    assert abs(it["int32"] - it["fp64"]) <= 0.05 * it["fp64"]
    assert it["fp16"] >= it["fp64"] and it["int16"] >= it["fp64"]


def test_max_iters_and_zero_rhs_and_immediate_convergence():
    p = make_config("C1", grid=16)
    r = oracle.gmres(p.A, p.b, p.x0, restart=10, rel_tol=1e-14, max_iters=25, fmt="fp64")
    assert not r.converged and r.iters == 25 and r.restarts == 3
    z = oracle.gmres(p.A, np.zeros(p.A.n), np.ones(p.A.n), restart=10, rel_tol=1e-10, max_iters=50)
    assert z.converged and z.iters == 0 and not z.x.any()
    xs = p.meta["xstar"]
    e = oracle.gmres(p.A, p.b, xs, restart=10, rel_tol=1e-10, max_iters=50)
    assert e.converged and e.iters == 0 and e.restarts == 0 and np.array_equal(e.x, xs)


def test_breakdown_on_invariant_subspace():
    # b is an eigenvector of the identity-like matrix: the Krylov space is 1-dimensional, h_{2,1} = 0
    n = 10
    A, Ad, b = random_dense_system(n, 35)
    import scipy.sparse as sp
    from workloads import CSR

    D = sp.csr_matrix(np.diag(np.full(n, 3.0)))
    A = CSR(n, D.indptr.astype(np.int32), D.indices.astype(np.int32), D.data.astype(np.float64))
    r = oracle.gmres(A, b, np.zeros(n), restart=5, rel_tol=1e-12, max_iters=20)
    assert r.converged and r.iters == 1 and r.breakdown == 1
    assert np.allclose(r.x, b / 3.0, rtol=1e-15)


# ---- scalar Jacobi right preconditioner (Fig. 1 l.3 "w := A(M^-1 v_j)", l.17 "x_0 + M^-1(V_m y_m)") ----

def _badly_scaled_system(n, seed):
    """Dense nonsymmetric system whose diagonal spans four orders of magnitude (column scaling of a
    well-conditioned matrix): input construction only."""
    from workloads import CSR
    import scipy.sparse as sp

    _, Ad, b = random_dense_system(n, seed)
    col = 10.0 ** np.random.default_rng(seed + 1).uniform(-2.0, 2.0, n)
    col[::3] *= -1.0  # negative diagonal entries too: M^-1 is a division by d_i, not by |d_i|
    Ad = Ad * col[None, :]
    S = sp.csr_matrix(Ad)
    S.sort_indices()
    return CSR(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(np.float64)), Ad, b


def test_jacobi_diag_is_the_matrix_diagonal():
    A, Ad, _ = _badly_scaled_system(17, 70)
    assert np.array_equal(oracle.jacobi_diag(A), np.diag(Ad))
    p = make_config("C1", grid=6)
    assert np.array_equal(oracle.jacobi_diag(p.A), np.full(p.A.n, 4.0))
    # a row without a stored diagonal entry is left unscaled
    from workloads import CSR
    B = CSR(2, np.array([0, 1, 2], np.int32), np.array([1, 1], np.int32), np.array([5.0, 7.0]))
    assert np.array_equal(oracle.jacobi_diag(B), np.array([1.0, 7.0]))


@pytest.mark.parametrize("n,seed", [(12, 71), (40, 72)])
def test_jacobi_tiny_dense_matches_direct_solve(n, seed):
    A, Ad, b = _badly_scaled_system(n, seed)
    x0 = np.random.default_rng(seed + 2).standard_normal(n)
    r = oracle.gmres(A, b, x0, restart=n, rel_tol=1e-13, max_iters=4 * n, fmt="fp64", precond="jacobi")
    xs = np.linalg.solve(Ad, b)
    assert r.converged and r.iters <= n + 1
    assert np.linalg.norm(r.x - xs) <= 1e-9 * np.linalg.norm(xs)
    # the stopping test is on the residual of the ORIGINAL system
    assert np.linalg.norm(b - Ad @ r.x) <= 1e-13 * np.linalg.norm(b) * (1 + 1e-6)


def test_jacobi_equals_plain_gmres_on_the_column_scaled_matrix():
    """Right preconditioning is GMRES on A M^-1 in the variable u = M x with the SAME residuals:
    the recurrence history of the preconditioned run on A equals that of the plain run on the
    explicitly formed A D^-1 (scipy, input construction), and x = D^-1 u.  A left-preconditioned or
    un-preconditioned implementation, or one that drops M^-1 in l.17, fails here."""
    from workloads import CSR
    import scipy.sparse as sp

    n = 60
    A, Ad, b = _badly_scaled_system(n, 73)
    d = np.diag(Ad).copy()
    S = sp.csr_matrix(Ad / d[None, :])
    S.sort_indices()
    Ahat = CSR(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(np.float64))
    kw = dict(restart=3, rel_tol=1e-11, max_iters=400, fmt="fp64")
    rp = oracle.gmres(A, b, np.zeros(n), precond="jacobi", **kw)
    ru = oracle.gmres(Ahat, b, np.zeros(n), precond="none", **kw)
    assert rp.converged and ru.converged and rp.restarts > 2
    assert rp.iters == ru.iters
    live = ru.rec_history > 1e-9
    assert np.allclose(rp.rec_history[live], ru.rec_history[live], rtol=1e-6)
    assert np.linalg.norm(rp.x - ru.x / d) <= 1e-9 * np.linalg.norm(rp.x)
    # and it is not the un-preconditioned iteration (which needs many more steps on this matrix)
    r0 = oracle.gmres(A, b, np.zeros(n), precond="none", **kw)
    assert (not r0.converged) or r0.iters > rp.iters


@pytest.mark.parametrize("fmt", ["fp64", "fp32", "int16"])
def test_jacobi_is_a_no_op_up_to_rounding_on_a_constant_diagonal(fmt):
    """C2 has the constant diagonal 6: A D^-1 = A / 6 spans the same Krylov spaces, so the residual
    history is that of the plain solver (the paper's stencil-like problems)."""
    p = make_config("C2", grid=10)
    kw = dict(restart=20, rel_tol=1e-8, max_iters=400, fmt=fmt)
    a = oracle.gmres(p.A, p.b, p.x0, precond="none", **kw)
    j = oracle.gmres(p.A, p.b, p.x0, precond="jacobi", **kw)
    assert a.converged and j.converged
    assert abs(a.iters - j.iters) <= (0 if fmt == "fp64" else 2)
    if fmt == "fp64":
        live = a.rec_history > 1e-7
        assert np.allclose(a.rec_history[live], j.rec_history[live], rtol=1e-6)
    S = p.A.to_scipy()
    assert np.linalg.norm(p.b - S @ j.x) <= 1e-8 * np.linalg.norm(p.b)


def test_jacobi_makes_the_power_law_config_converge():
    """C4's diagonal (1.1 x row abs-sum of power-law rows) spans orders of magnitude; with the paper's
    default preconditioner the restarted solver converges where M = I stalls."""
    p = make_config("C4", n=3000)
    kw = dict(restart=p.restart, rel_tol=p.rel_tol, max_iters=600, fmt="fp64")
    j = oracle.gmres(p.A, p.b, p.x0, precond="jacobi", **kw)
    assert j.converged
    S = p.A.to_scipy()
    assert np.linalg.norm(p.b - S @ j.x) <= p.rel_tol * np.linalg.norm(p.b) * (1 + 1e-6)
    a = oracle.gmres(p.A, p.b, p.x0, precond="none", **kw)
    assert (not a.converged) or a.iters > 2 * j.iters


# ---- block-Jacobi right preconditioner, block size 4 (section 6.5) ---------------------------

def _csr_from_dense(Ad):
    from workloads import CSR
    import scipy.sparse as sp

    S = sp.csr_matrix(Ad)
    S.sort_indices()
    return CSR(Ad.shape[0], S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(np.float64))


def _block_system(n, seed, coupling=0.05):
    """Dense nonsymmetric system A = (I + coupling G) M with M block diagonal: strong, badly scaled 4 x 4
    diagonal blocks (scales spanning two decades, a large ANTI-diagonal inside each block, so that
    pivoting is needed and the scalar diagonal is a poor preconditioner) and weak coupling between the
    blocks.  Input construction only."""
    rng = np.random.default_rng(seed)
    M = np.zeros((n, n))
    for b0 in range(0, n, 4):
        b1 = min(n, b0 + 4)
        blk = 0.3 * rng.standard_normal((b1 - b0, b1 - b0)) + 2.0 * np.eye(b1 - b0)[::-1] + 0.5 * np.eye(b1 - b0)
        M[b0:b1, b0:b1] = 10.0 ** rng.uniform(-1.0, 1.0) * blk
    Ad = (np.eye(n) + coupling * rng.standard_normal((n, n))) @ M
    b = rng.standard_normal(n)
    return _csr_from_dense(Ad), Ad, b


@pytest.mark.parametrize("n", [16, 18, 19, 3])
def test_block_jacobi4_blocks_match_numpy_inv(n):
    A, Ad, _ = _block_system(n, 80 + n)
    inv = oracle.block_jacobi4(A)
    assert inv.shape == ((n + 3) // 4, 4, 4)
    for b in range(inv.shape[0]):
        b0, b1 = 4 * b, min(n, 4 * b + 4)
        s = b1 - b0
        ref = np.linalg.inv(Ad[b0:b1, b0:b1])
        assert np.allclose(inv[b, :s, :s], ref, rtol=1e-11, atol=1e-13 * np.abs(ref).max())
        # ragged last block: completed by the identity, nothing couples into the real rows
        assert np.array_equal(inv[b, s:, s:], np.eye(4 - s)) and not inv[b, :s, s:].any() and not inv[b, s:, :s].any()
    # apply: z = M^-1 v block by block
    v = np.random.default_rng(5).standard_normal(n)
    z = oracle.apply_minv("block_jacobi4", inv, v)
    M = np.zeros((n, n))
    for b0 in range(0, n, 4):
        b1 = min(n, b0 + 4)
        M[b0:b1, b0:b1] = Ad[b0:b1, b0:b1]
    assert np.allclose(z, np.linalg.solve(M, v), rtol=1e-10, atol=1e-13 * np.abs(z).max())


def test_block_jacobi4_sparse_pattern_absent_entries_are_zero_and_singular_block_is_identity():
    from workloads import CSR

    # rows 0..3: only part of the block is stored; rows 4..7: a singular block (two equal rows)
    Ad = np.zeros((8, 8))
    Ad[0, 0], Ad[0, 2], Ad[1, 1], Ad[2, 0], Ad[2, 2], Ad[3, 3], Ad[1, 6] = 2.0, 1.0, 4.0, 1.0, 3.0, 5.0, 9.0
    Ad[4, 4:8] = [1.0, 2.0, 3.0, 4.0]
    Ad[5, 4:8] = [1.0, 2.0, 3.0, 4.0]
    Ad[6, 6], Ad[7, 7] = 1.0, 1.0
    inv = oracle.block_jacobi4(_csr_from_dense(Ad))
    assert np.allclose(inv[0], np.linalg.inv(Ad[:4, :4]), rtol=1e-14)
    assert np.array_equal(inv[1], np.eye(4))


@pytest.mark.parametrize("n,seed", [(24, 90), (41, 91)])
def test_block_jacobi4_tiny_dense_matches_direct_solve(n, seed):
    A, Ad, b = _block_system(n, seed)
    x0 = np.random.default_rng(seed + 2).standard_normal(n)
    r = oracle.gmres(A, b, x0, restart=n, rel_tol=1e-11, max_iters=4 * n, fmt="fp64", precond="block_jacobi4")
    xs = np.linalg.solve(Ad, b)
    assert r.converged and r.iters <= n and r.restarts == 1  # the Krylov space of dimension n is the whole space
    assert np.linalg.norm(r.x - xs) <= 1e-8 * np.linalg.norm(xs)
    assert np.linalg.norm(b - Ad @ r.x) <= 1e-11 * np.linalg.norm(b) * (1 + 1e-6)  # residual of the ORIGINAL system


def test_block_jacobi4_equals_plain_gmres_on_the_explicit_product():
    """Right preconditioning is GMRES on A M^-1 in u = M x with the same residuals: the history of the
    preconditioned run on A equals the plain run on the explicitly formed A M^-1 (numpy, input
    construction), and x = M^-1 u.  Left / missing / transposed-block / l.17-without-M^-1 variants fail."""
    n = 42  # ragged last block (2 rows)
    A, Ad, b = _block_system(n, 92, coupling=0.08)
    M = np.zeros((n, n))
    for b0 in range(0, n, 4):
        b1 = min(n, b0 + 4)
        M[b0:b1, b0:b1] = Ad[b0:b1, b0:b1]
    Minv = np.linalg.inv(M)
    Ahat = _csr_from_dense(Ad @ Minv)
    kw = dict(restart=5, rel_tol=1e-11, max_iters=600, fmt="fp64")
    rp = oracle.gmres(A, b, np.zeros(n), precond="block_jacobi4", **kw)
    ru = oracle.gmres(Ahat, b, np.zeros(n), precond="none", **kw)
    assert rp.converged and ru.converged and rp.restarts > 2
    assert rp.iters == ru.iters
    live = ru.rec_history > 1e-9
    assert np.allclose(rp.rec_history[live], ru.rec_history[live], rtol=1e-6)
    assert np.linalg.norm(rp.x - Minv @ ru.x) <= 1e-9 * np.linalg.norm(rp.x)
    # the transposed blocks are a different (here: much worse) preconditioner -- and so is none at all
    AhatT = _csr_from_dense(Ad @ Minv.T)
    rt = oracle.gmres(AhatT, b, np.zeros(n), precond="none", **kw)
    assert (not rt.converged) or rt.iters != rp.iters
    r0 = oracle.gmres(A, b, np.zeros(n), precond="none", **kw)
    assert (not r0.converged) or r0.iters > rp.iters


@pytest.mark.parametrize("fmt", ["fp64", "int16"])
def test_block_jacobi4_reduces_to_scalar_jacobi_without_in_block_coupling(fmt):
    """If no off-diagonal entry falls inside a 4 x 4 diagonal block, M is diag(A): same iteration as
    the scalar preconditioner up to rounding (1/d * v against v / d)."""
    n = 64
    rng = np.random.default_rng(93)
    G = 0.05 * rng.standard_normal((n, n))
    for b0 in range(0, n, 4):
        G[b0:b0 + 4, b0:b0 + 4] = 0.0
    Ad = (np.eye(n) + G) * (10.0 ** rng.uniform(-1.0, 2.0, n) * rng.choice([-1.0, 1.0], n))[None, :]  # column scaling
    A, b = _csr_from_dense(Ad), rng.standard_normal(n)
    kw = dict(restart=8, rel_tol=1e-9, max_iters=4000, fmt=fmt)
    s = oracle.gmres(A, b, np.zeros(n), precond="jacobi", **kw)
    q = oracle.gmres(A, b, np.zeros(n), precond="block_jacobi4", **kw)
    assert s.converged and q.converged
    if fmt == "fp64":
        assert s.iters == q.iters
        live = s.rec_history > 1e-7
        assert np.allclose(s.rec_history[live], q.rec_history[live], rtol=1e-6)
    else:
        assert abs(s.iters - q.iters) <= max(2, 0.05 * s.iters)
    inv = oracle.block_jacobi4(A)
    assert np.allclose(inv.reshape(-1, 4, 4)[:, np.arange(4), np.arange(4)].ravel(), 1.0 / np.diag(Ad), rtol=1e-15)


def test_block_jacobi4_beats_scalar_jacobi_on_block_structured_matrix():
    """What section 6.5 uses it for: on a matrix with strong 4 x 4 blocks the block preconditioner needs
    fewer iterations than the scalar one."""
    A, Ad, b = _block_system(200, 94, coupling=0.03)
    kw = dict(restart=30, rel_tol=1e-9, max_iters=3000, fmt="fp64")
    q = oracle.gmres(A, b, np.zeros(200), precond="block_jacobi4", **kw)
    s = oracle.gmres(A, b, np.zeros(200), precond="jacobi", **kw)
    assert q.converged and ((not s.converged) or s.iters > 2 * q.iters)


# ---- Fig. 1 l.12: the second Gram-Schmidt pass again lost more than eta (reading Q4) -------------------------

def invariant_subspace_problem(n=40, d=6, seed=95):
    """A = blockdiag(A1, I): b lives in the first d coordinates, so the Krylov space closes at dimension
    d: A v_d lies in span(V_d).  With a QUANTISED basis V^ the first pass leaves w1 = -V^ E c (E = V^T V^ - I,
    about the format's unit roundoff), which triggers l.7, and the second pass leaves about E^2 c: it again
    loses far more than eta while h_{d+1,d} stays nonzero -- only the clause `hn < eta * omega1` of l.12
    ends the cycle there.  Hand computation: x* = [A1^-1 b1; 0]."""
    rng = np.random.default_rng(seed)
    A1 = rng.standard_normal((d, d)) + d * np.eye(d)
    Ad = np.eye(n)
    Ad[:d, :d] = A1
    b = np.zeros(n)
    b[:d] = rng.standard_normal(d)
    xs = np.zeros(n)
    xs[:d] = np.linalg.solve(A1, b[:d])
    return _csr_from_dense(Ad), Ad, b, xs


@pytest.mark.parametrize("fmt,u", [("fp64", 2.0 ** -53), ("fp32", 2.0 ** -24), ("fp16", 2.0 ** -11), ("int32", 2.0 ** -31),
                                   ("int16", 2.0 ** -15)])
def test_second_pass_breakdown_clause_ends_the_cycle(fmt, u):
    n, d, m = 40, 6, 20
    A, Ad, b, xs = invariant_subspace_problem(n, d)
    # tau = 0 is out of reach, so the recurrence-residual test cannot end the cycle: only l.12 can.
    # One cycle only (the iteration bound is met at the next restart).
    r = oracle.gmres(A, b, np.zeros(n), restart=m, rel_tol=0.0, max_iters=d, fmt=fmt, capture_cycle=0)
    cap = r.capture
    H = cap["Hbar"]
    assert cap["k"] == d and r.iters == d and r.restarts == 1
    assert r.breakdown == 1 and not r.converged
    # it is the eta clause, not hn == 0: h_{d+1,d} is nonzero (about omega * u^2) and far below eta * omega1
    hn = H[d, d - 1]
    assert 0.0 < hn < 1e-3 * cap["omega"][d - 1]
    assert cap["reorth_log"][d - 1] == 1
    assert r.rel_res_recurrence > 0.0
    # no earlier step broke down although every one re-orthogonalised: there the second pass kept the norm
    assert np.all(cap["reorth_log"] == 1) and np.all(np.diag(H, -1)[: d - 1] > 1e-2)
    # x of that cycle against the hand computation: the minimiser over span(V^_d) = the first d coordinates,
    # accurate to the storage format's roundoff
    assert np.linalg.norm(r.x - xs) <= 50 * u * np.linalg.norm(xs)
    assert not r.x[d:].any()
    # with a reachable tau the solver restarts from the explicit residual and converges; every
    # cycle is cut at (or before) step d -- without the clause the first one would run on to m = 20
    full = oracle.gmres(A, b, np.zeros(n), restart=m, rel_tol=1e-12, max_iters=200, fmt=fmt)
    assert full.converged and np.linalg.norm(full.x - xs) <= 1e-10 * np.linalg.norm(xs)
    assert full.iters <= d * full.restarts and full.iters <= 6 * d


def test_second_pass_breakdown_needs_the_clause():
    """The same problem with REORTH_NEVER has no l.12 clause (breakdown is hn == 0 only): the cycle then runs past
    step d with a basis vector made of rounding noise -- the behaviour the clause exists to prevent."""
    n, d, m = 40, 6, 20
    A, Ad, b, xs = invariant_subspace_problem(n, d)
    r = oracle.gmres(A, b, np.zeros(n), restart=m, rel_tol=0.0, max_iters=m, fmt="fp16", reorth="never",
                     capture_cycle=0)
    assert r.capture["k"] == m and r.breakdown == 0
