"""GPU parity of the whole solver through cbgmres_solve (BASELINE.json north_star): iteration counts
to convergence agree with the oracle within +-2 % (at least +-2 steps), final true relative residuals
are both below the tolerance and within 10x of each other.  The true residual of the GPU's x is
recomputed by the oracle's SpMV, never taken from the GPU's own report."""
import numpy as np
import pytest

import oracle
from parity import check_iters
from workloads import make_config, random_dense_system

pytestmark = pytest.mark.gpu


def _solve_gpu(p, fmt, restart=None, rel_tol=None, max_iters=None, reorth="cond", history=False, x0=None,
               precond="none"):
    from paper_2009_12101_b200 import Solver

    s = Solver(0)
    try:
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        x, r = s.solve(p.b, p.x0 if x0 is None else x0, restart or p.restart, rel_tol or p.rel_tol,
                       max_iters or p.max_iters, fmt, reorth=reorth, history=history, precond=precond)
        return x.cpu().numpy(), r
    finally:
        s.destroy()


def _true_rel_res(p, x):
    return oracle.nrm2(p.b - oracle.spmv(p.A, x)) / oracle.nrm2(p.b)


def _check_parity(p, fmt, restart=None, rel_tol=None, max_iters=None, reorth="cond", precond="none", label=None):
    """GPU solve against the oracle's: counts through the shared checker (tests/parity.py: strict +-2 %, the
    oracle's own spread for quantised formats, the listed chaotic cases), residuals, restarts, ||b||."""
    restart, rel_tol, max_iters = restart or p.restart, rel_tol or p.rel_tol, max_iters or p.max_iters
    label = label or p.name
    run = lambda: oracle.gmres(p.A, p.b, p.x0, restart, rel_tol, max_iters, fmt, reorth=reorth, precond=precond)
    ref = run()
    x, r = _solve_gpu(p, fmt, restart, rel_tol, max_iters, reorth, precond=precond)
    true_gpu = _true_rel_res(p, x)
    true_ref = _true_rel_res(p, ref.x)
    assert r.converged == ref.converged
    rule = check_iters(r.iters, ref.iters, fmt, label, run=run)
    if ref.converged:
        assert true_gpu <= rel_tol * (1 + 1e-9) and true_ref <= rel_tol * (1 + 1e-9)
    assert true_gpu <= 10 * true_ref and true_ref <= 10 * true_gpu
    assert r.rel_res_true == pytest.approx(true_gpu, rel=1e-6)
    if rule == "strict":  # cycles are comparable only where the counts are
        assert abs(r.restarts - ref.restarts) <= 1
    assert r.b_norm == pytest.approx(ref.b_norm, rel=1e-13)
    return r, ref


@pytest.mark.parametrize("fmt", ["fp64", "fp32"])
def test_c1_full_size(fmt):
    p = make_config("C1")
    r, ref = _check_parity(p, fmt)
    assert r.converged


@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_c2_reduced(fmt):
    _check_parity(make_config("C2", grid=32), fmt, label="C2-32")


@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_c4_reduced(fmt):
    # without a preconditioner C4 does not converge within its iteration bound (reading Q12); both
    # sides must then stop at the bound with comparable true residuals
    r, ref = _check_parity(make_config("C4", n=40000), fmt, max_iters=300, label="C4-40k")
    assert r.iters == ref.iters == 300


@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_c4_reduced_jacobi_converges(fmt):
    """The paper's default preconditioner (scalar Jacobi) as the right preconditioner of
    Fig. 1 l.3 / l.17: C4 converges on both sides, counts and residuals as in every other parity case."""
    r, ref = _check_parity(make_config("C4", n=40000), fmt, max_iters=2000, precond="jacobi", label="C4J-40k")
    assert r.converged and ref.converged


@pytest.mark.parametrize("fmt", ["fp64", "fp16"])
def test_c2_reduced_jacobi_constant_diagonal(fmt):
    """C2's diagonal is the constant 6: A D^-1 = A / 6, same Krylov spaces (streamed SpMV variant with
    the scaled copy of the values; x = D^-1 u at the end)."""
    p = make_config("C2", grid=32)
    r, ref = _check_parity(p, fmt, precond="jacobi", label="C2J-32")
    _, plain = _solve_gpu(p, fmt)
    assert r.converged and abs(r.iters - plain.iters) <= max(2, 0.02 * plain.iters)


def test_jacobi_tiny_dense_nonzero_x0_matches_direct_solve():
    A, Ad, b = random_dense_system(48, 61, density=0.4)
    col = 10.0 ** np.random.default_rng(62).uniform(-2.0, 2.0, 48)
    col[::3] *= -1.0
    import scipy.sparse as sp
    from workloads import CSR, Problem

    S = sp.csr_matrix(Ad * col[None, :])
    S.sort_indices()
    A2 = CSR(48, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(np.float64))
    x0 = np.random.default_rng(63).standard_normal(48)
    p = Problem("tiny", A2, b, x0, 48, 1e-12, 400, ("fp64",), {})
    x, r = _solve_gpu(p, "fp64", precond="jacobi")
    xs = np.linalg.solve(Ad * col[None, :], b)
    assert r.converged
    assert np.linalg.norm(x - xs) <= 1e-8 * np.linalg.norm(xs)
    assert _true_rel_res(p, x) <= 1e-12 * (1 + 1e-6)


def test_jacobi_host_entry_and_workspace():
    """solve_host with the preconditioner: the extra workspace (scaled values + diagonal) is accounted for."""
    from paper_2009_12101_b200 import Solver

    p = make_config("C4", n=20000)
    s = Solver(0)
    try:
        x = p.x0.copy()
        r = s.solve_host(p.A.row_ptr, p.A.col_idx, p.A.vals, p.b, x, p.restart, p.rel_tol, 2000, "fp32", precond="jacobi")
        assert r.converged and _true_rel_res(p, x) <= p.rel_tol * (1 + 1e-6)
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        assert s.workspace_bytes(p.restart, "fp32", precond="jacobi") >= s.workspace_bytes(p.restart, "fp32") + 8 * (p.A.nnz + p.A.n)
    finally:
        s.destroy()


@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_c5_reduced(fmt):
    _check_parity(make_config("C5", grid=24), fmt, label="C5-24")


@pytest.mark.parametrize("reorth", ["never", "always"])
def test_reorth_modes(reorth):
    p = make_config("C2", grid=20)
    r, ref = _check_parity(p, "fp32", restart=30, reorth=reorth, label="C2-20-" + reorth)
    assert (r.reorth_count == 0) if reorth == "never" else (r.reorth_count == r.iters)


def test_recurrence_history_matches_oracle_first_cycle():
    p = make_config("C2", grid=16)
    ref = oracle.gmres(p.A, p.b, p.x0, 40, 1e-8, 400, "fp64")
    x, r = _solve_gpu(p, "fp64", 40, 1e-8, 400, history=True)
    k = min(30, r.iters, ref.iters)
    assert np.allclose(r.rec_history[:k], ref.rec_history[:k], rtol=1e-6)


def test_tiny_dense_matches_direct_solve():
    for n, seed in ((1, 40), (3, 41), (33, 42), (64, 43)):
        A, Ad, b = random_dense_system(n, seed)
        from paper_2009_12101_b200 import Solver

        s = Solver(0)
        try:
            s.set_matrix(A.row_ptr, A.col_idx, A.vals)
            x, r = s.solve(b, np.zeros(n), n, 1e-13, 4 * n + 4, "fp64")
            assert r.converged and r.iters <= n
            xs = np.linalg.solve(Ad, b)
            assert np.linalg.norm(x.cpu().numpy() - xs) <= 1e-10 * np.linalg.norm(xs)
        finally:
            s.destroy()


def test_edge_cases_zero_rhs_exact_x0_max_iters_restart1():
    p = make_config("C1", grid=16)
    from paper_2009_12101_b200 import Solver

    s = Solver(0)
    try:
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        x, r = s.solve(np.zeros(p.A.n), np.ones(p.A.n), 10, 1e-10, 50, "fp32")
        assert r.converged and r.iters == 0 and not x.cpu().numpy().any()
        xs = p.meta["xstar"]
        x, r = s.solve(p.b, xs, 10, 1e-10, 50, "fp64")
        assert r.converged and r.iters == 0 and r.restarts == 0 and np.array_equal(x.cpu().numpy(), xs)
        x, r = s.solve(p.b, p.x0, 10, 1e-14, 25, "fp64")
        assert (not r.converged) and r.status == 16 and r.iters == 25 and r.restarts == 3
        ref = oracle.gmres(p.A, p.b, p.x0, 10, 1e-14, 25, "fp64")
        assert _true_rel_res(p, x.cpu().numpy()) == pytest.approx(ref.rel_res_true, rel=1e-6)
        # restart length 1 (GMRES(1)) still runs the whole path
        x, r = s.solve(p.b, p.x0, 1, 1e-3, 500, "int16")
        ref = oracle.gmres(p.A, p.b, p.x0, 1, 1e-3, 500, "int16")
        assert r.converged == ref.converged and abs(r.iters - ref.iters) <= max(2, 0.02 * ref.iters)
    finally:
        s.destroy()


def test_breakdown_on_invariant_subspace():
    import scipy.sparse as sp

    from paper_2009_12101_b200 import Solver
    from workloads import CSR

    n = 10
    b = np.random.default_rng(44).standard_normal(n)
    D = sp.csr_matrix(np.diag(np.full(n, 3.0)))
    A = CSR(n, D.indptr.astype(np.int32), D.indices.astype(np.int32), D.data.astype(np.float64))
    s = Solver(0)
    try:
        s.set_matrix(A.row_ptr, A.col_idx, A.vals)
        x, r = s.solve(b, np.zeros(n), 5, 1e-12, 20, "fp64")
        assert r.converged and r.iters == 1 and r.breakdown == 1
        assert np.allclose(x.cpu().numpy(), b / 3.0, rtol=1e-15)
    finally:
        s.destroy()


def test_solve_host_matches_device_solve():
    import torch

    from paper_2009_12101_b200 import Solver

    p = make_config("C2", grid=24)
    s = Solver(0)
    try:
        pin = lambda a: torch.as_tensor(a).pin_memory()
        hx = pin(p.x0.copy())
        r = s.solve_host(pin(p.A.row_ptr), pin(p.A.col_idx), pin(p.A.vals), pin(p.b), hx, p.restart, p.rel_tol,
                         p.max_iters, "fp32")
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        x, r2 = s.solve(p.b, p.x0, p.restart, p.rel_tol, p.max_iters, "fp32")
        assert r.converged and r.iters == r2.iters
        assert np.array_equal(hx.numpy(), x.cpu().numpy())  # deterministic reductions: bitwise repeatable
        assert _true_rel_res(p, hx.numpy()) <= p.rel_tol
    finally:
        s.destroy()


def test_invalid_solve_arguments():
    from paper_2009_12101_b200 import CbgmresError, Solver

    p = make_config("C1", grid=8)
    s = Solver(0)
    try:
        with pytest.raises(CbgmresError) as e:
            s.solve(p.b, p.x0, 10, 1e-8, 10, "fp64")
        assert e.value.code == 2
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        for kw in (dict(restart=0), dict(restart=513), dict(rel_tol=-1.0), dict(max_iters=-1)):
            args = dict(restart=10, rel_tol=1e-8, max_iters=10)
            args.update(kw)
            with pytest.raises(CbgmresError) as e:
                s.solve(p.b, p.x0, args["restart"], args["rel_tol"], args["max_iters"], "fp64")
            assert e.value.code == 1
    finally:
        s.destroy()


@pytest.mark.parametrize("fmt", ["fp64", "fp16", "int16"])
def test_full_size_c2_solve_is_bitwise_repeatable(fmt):
    """Every reduction has a fixed order, so two solves of the same system give the same bits -- on
    the full-size C2 matrix, where each CTA of the Gram-Schmidt passes owns many row tiles."""
    from paper_2009_12101_b200 import Solver

    p = make_config("C2")
    s = Solver(0)
    try:
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        runs = []
        for _ in range(3):
            x, r = s.solve(p.b, p.x0, p.restart, p.rel_tol, 150, fmt, history=True)
            runs.append((x.cpu().numpy(), r.rec_history.copy()))
        for x, hist in runs[1:]:
            assert np.array_equal(hist, runs[0][1])
            assert np.array_equal(x, runs[0][0])
    finally:
        s.destroy()


def test_measurement_drivers_run(capsys):
    """cyclebench (fixed iteration count: every solve does exactly cycles * m steps) and paperprotocol
    (b_i = sin i, Jacobi) on small inputs."""
    from paper_2009_12101_b200 import cyclebench, paperprotocol

    assert cyclebench.main(["--workload", "C2", "--grid", "20", "--m", "5,12", "--cycles", "3", "--formats", "fp64,int16"]) == 0
    out = capsys.readouterr().out
    rows = [l.split() for l in out.splitlines() if l and l[0] == " " and l.split()[0].isdigit()]
    assert [(int(r[0]), r[1], int(r[2])) for r in rows] == [(5, "fp64", 15), (5, "int16", 15), (12, "fp64", 36), (12, "int16", 36)]
    assert paperprotocol.main(["--small", "--max-iters", "3000"]) == 0
    out = capsys.readouterr().out
    assert "fp32" in out and "3/3" in out


# ---- block-Jacobi(4) right preconditioner -----------------------------------

@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_c4_reduced_block_jacobi4(fmt):
    """C4 (power-law rows, strongly varying diagonal) with M = the 4 x 4 diagonal blocks: converges on both
    sides; counts, residuals and restarts as in every other parity case."""
    r, ref = _check_parity(make_config("C4", n=40000), fmt, max_iters=2000, precond="block_jacobi4", label="C4B-40k")
    assert r.converged and ref.converged


@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_c5_reduced_block_jacobi4(fmt):
    """27-point stencil: four consecutive grid points are coupled, so the blocks are genuinely 4 x 4."""
    r, ref = _check_parity(make_config("C5", grid=24), fmt, precond="block_jacobi4", label="C5B-24")
    assert r.converged


@pytest.mark.parametrize("fmt", ["fp64", "int16"])
def test_c2_reduced_block_jacobi4_ragged_last_block(fmt):
    """n = 27^3 = 19683 = 4 * 4920 + 3: the last block has three rows (identity completion); streamed SpMV
    of z = M^-1 v written by the store kernel's scalar tail."""
    _check_parity(make_config("C2", grid=27), fmt, precond="block_jacobi4", label="C2B-27")


def test_block_jacobi4_tiny_dense_nonzero_x0_matches_direct_solve():
    import scipy.sparse as sp
    from workloads import CSR, Problem

    n = 50  # ragged last block (2 rows)
    rng = np.random.default_rng(64)
    M = np.zeros((n, n))
    for b0 in range(0, n, 4):
        b1 = min(n, b0 + 4)
        blk = 0.3 * rng.standard_normal((b1 - b0, b1 - b0)) + 2.0 * np.eye(b1 - b0)[::-1] + 0.5 * np.eye(b1 - b0)
        M[b0:b1, b0:b1] = 10.0 ** rng.uniform(-1.0, 1.0) * blk
    Ad = (np.eye(n) + 0.05 * rng.standard_normal((n, n))) @ M
    S = sp.csr_matrix(Ad)
    S.sort_indices()
    A = CSR(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(np.float64))
    b, x0 = rng.standard_normal(n), rng.standard_normal(n)
    p = Problem("tinyB", A, b, x0, n, 1e-11, 4 * n, ("fp64",), {})
    x, r = _solve_gpu(p, "fp64", precond="block_jacobi4")
    ref = oracle.gmres(A, b, x0, n, 1e-11, 4 * n, "fp64", precond="block_jacobi4")
    xs = np.linalg.solve(Ad, b)
    assert r.converged and ref.converged and r.iters == ref.iters and r.iters <= n
    assert np.linalg.norm(x - xs) <= 1e-8 * np.linalg.norm(xs)
    assert _true_rel_res(p, x) <= 1e-11 * (1 + 1e-6)
    # scalar Jacobi and no preconditioner do far worse on this matrix: the blocks are what is applied
    _, rj = _solve_gpu(p, "fp64", precond="jacobi", restart=10, max_iters=300)
    _, rb = _solve_gpu(p, "fp64", precond="block_jacobi4", restart=10, max_iters=300)
    assert rb.converged and ((not rj.converged) or rj.iters > 2 * rb.iters)


def test_block_jacobi4_host_entry_and_workspace():
    from paper_2009_12101_b200 import Solver

    p = make_config("C4", n=20001)
    s = Solver(0)
    try:
        x = p.x0.copy()
        r = s.solve_host(p.A.row_ptr, p.A.col_idx, p.A.vals, p.b, x, p.restart, p.rel_tol, 2000, "fp32", precond="block_jacobi4")
        assert r.converged and _true_rel_res(p, x) <= p.rel_tol * (1 + 1e-6)
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        assert s.workspace_bytes(p.restart, "fp32", precond="block_jacobi4") >= s.workspace_bytes(p.restart, "fp32") + 128 * ((p.A.n + 3) // 4)
    finally:
        s.destroy()


# ---- Fig. 1 l.12: the second pass again lost more than eta (reading Q4; oracle pin in test_oracle_gmres.py) ------

@pytest.mark.parametrize("fmt,u", [("fp32", 2.0 ** -24), ("fp16", 2.0 ** -11), ("int32", 2.0 ** -31), ("int16", 2.0 ** -15)])
def test_second_pass_breakdown_clause_matches_oracle(fmt, u):
    """A = blockdiag(A1, I), b in the first d coordinates: the Krylov space closes at dimension d; with a
    quantised basis h_{d+1,d} stays nonzero (about u^2 omega) and only the clause hn < eta * omega1 of l.12 ends
    the cycle there.  tau = 0 is out of reach, so the recurrence test cannot end it."""
    import scipy.sparse as sp
    from workloads import CSR, Problem

    n, d, m = 40, 6, 20
    rng = np.random.default_rng(95)
    A1 = rng.standard_normal((d, d)) + d * np.eye(d)
    Ad = np.eye(n)
    Ad[:d, :d] = A1
    b = np.zeros(n)
    b[:d] = rng.standard_normal(d)
    xs = np.zeros(n)
    xs[:d] = np.linalg.solve(A1, b[:d])
    S = sp.csr_matrix(Ad)
    S.sort_indices()
    A = CSR(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(np.float64))
    p = Problem("inv", A, b, np.zeros(n), m, 0.0, d, (fmt,), {})
    ref = oracle.gmres(A, b, np.zeros(n), m, 0.0, d, fmt)
    x, r = _solve_gpu(p, fmt, restart=m, rel_tol=0.0, max_iters=d, history=True)
    assert ref.breakdown == 1 and ref.iters == d and ref.restarts == 1
    assert r.breakdown == 1 and r.iters == d and r.restarts == 1 and r.reorth_count == ref.reorth_count == d
    assert r.rel_res_recurrence > 0.0  # the cycle was not ended by hn == 0 or by the residual test
    assert np.linalg.norm(x - xs) <= 50 * u * np.linalg.norm(xs) and not x[d:].any()
    assert np.allclose(r.rec_history[: d - 1], ref.rec_history[: d - 1], rtol=1e-3)
    # with a reachable tau: restart from the explicit residual, every cycle cut at step d, converged
    p2 = Problem("inv", A, b, np.zeros(n), m, 1e-12, 200, (fmt,), {})
    x2, r2 = _solve_gpu(p2, fmt)
    ref2 = oracle.gmres(A, b, np.zeros(n), m, 1e-12, 200, fmt)
    assert r2.converged and ref2.converged and r2.iters <= d * r2.restarts
    assert abs(r2.iters - ref2.iters) <= d and np.linalg.norm(x2 - xs) <= 1e-10 * np.linalg.norm(xs)
    # REORTH_NEVER has no such clause: the cycle runs on to m
    _, r3 = _solve_gpu(p, fmt, restart=m, rel_tol=0.0, max_iters=m, reorth="never")
    assert r3.iters == m and r3.breakdown == 0


# ---- restart lengths beyond one launch's 128 columns (PAPER.md:294 sweeps m = 10 .. 300; NEXT-2) ------------------

@pytest.mark.parametrize("m", [150, 300])
@pytest.mark.parametrize("fmt", ["fp64", "fp32", "int16"])
def test_long_restart_split_ranges_match_oracle(m, fmt):
    """m > 128: every pass is split into ranges of <= 128 basis vectors and the fused update + multi-dot is
    replaced by separate passes.  C2 on a 40^3 grid with tau = 1e-11 needs 140 steps with an fp64 basis (one
    cycle) and 230 / 330-390 with fp32 / int16 (several cycles): iteration counts and residuals against the oracle."""
    p = make_config("C2", grid=40)
    r, ref = _check_parity(p, fmt, restart=m, rel_tol=1e-11, max_iters=3000, label=f"C2-40-m{m}")
    assert r.converged and r.iters > 128  # the split path really ran
    if fmt == "fp64":
        assert r.reorth_count == ref.reorth_count


@pytest.mark.parametrize("fmt", ["fp64", "int16"])
def test_long_restart_whole_cycle_of_300_steps_matches_oracle(fmt):
    """A whole cycle of m = 300 steps at a fixed iteration count (tau = 0, the protocol of PAPER.md:294): ranges of
    128 + 128 + 44 vectors in every pass.  2D Laplacian on a 128^2 grid (C1's recipe), which is still at a relative
    residual of 8e-9 after 300 unrestarted steps.  fp64 storage: the residual history equals the oracle's to rounding
    over the whole cycle; int16: over the first 40 steps to the format's roundoff."""
    p = make_config("C1", grid=128)
    m = 300
    ref = oracle.gmres(p.A, p.b, p.x0, m, 0.0, m, fmt)
    x, r = _solve_gpu(p, fmt, restart=m, rel_tol=0.0, max_iters=m, history=True)
    assert r.iters == m and ref.iters == m and r.restarts == 1 and ref.restarts == 1 and not r.converged
    hg, ho = np.asarray(r.rec_history), np.asarray(ref.rec_history)
    if fmt == "fp64":
        assert np.allclose(hg, ho, rtol=1e-8)
        assert abs(r.reorth_count - ref.reorth_count) <= 2
    else:
        assert np.all(np.abs(hg[:40] - ho[:40]) <= 2.0 ** -15 * 4 * ho[:40])
    tg, to = _true_rel_res(p, x), _true_rel_res(p, ref.x)
    assert tg <= 10 * to and to <= 10 * tg


# ---- the paper's protocol: b_i = sin(i), m = 100, tau = 1e-9, scalar Jacobi (NEXT-3) -----------

@pytest.mark.parametrize("cfg,kw,label", [("C2", {"grid": 24}, "PP-C2-24"), ("C5", {"grid": 16}, "PP-C5-16"), ("C4", {"n": 20000}, "PP-C4-20k")])
@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_paper_protocol_small_matrices_match_oracle(cfg, kw, label, fmt):
    from workloads import Problem

    q = make_config(cfg, **kw)
    n = q.A.n
    b = np.sin(np.arange(1, n + 1, dtype=np.float64))
    p = Problem(label, q.A, b, np.zeros(n), 100, 1e-9, 3000, oracle.FORMATS, {})
    if label == "PP-C4-20k" and fmt in ("fp16", "int16"):
        # 16-bit storage stagnates on the Jacobi-scaled power-law matrix: both sides stop at a
        # short bound with comparable residuals instead of running thousands of chaotic steps
        r, ref = _check_parity(p, fmt, max_iters=200, precond="jacobi", label=label)
    else:
        r, ref = _check_parity(p, fmt, precond="jacobi", label=label)
        assert r.converged and ref.converged


# ---- library hygiene: handles share no mutable state -----------------------------------------------------------

def test_two_handles_with_different_options_do_not_interfere():
    """Two handles on two streams with different pdl / orth_seg_kb / orth_interleave options, solves
    interleaved: each result is bitwise the one the same handle gives alone."""
    import torch
    from paper_2009_12101_b200 import Solver

    p = make_config("C2", grid=28)
    opts = ({"pdl": 1, "orth_seg_kb": 0, "orth_interleave": 0}, {"pdl": 0, "orth_seg_kb": 1, "orth_interleave": 1})

    def make(o, stream):
        s = Solver(0, stream=stream)
        for k, v in o.items():
            s.set_option(k, v)
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        return s

    alone = []
    for o in opts:
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            s = make(o, st)
            x, r = s.solve(p.b, p.x0, 40, 1e-8, 400, "fp16", history=True)
            st.synchronize()
            alone.append((x.cpu().numpy(), r.rec_history.copy(), r.iters))
            s.destroy()
    st = [torch.cuda.Stream(), torch.cuda.Stream()]
    hs = []
    for o, t in zip(opts, st):
        with torch.cuda.stream(t):
            hs.append(make(o, t))
    try:
        for rep in range(2):
            for i in (0, 1, 1, 0):
                with torch.cuda.stream(st[i]):
                    x, r = hs[i].solve(p.b, p.x0, 40, 1e-8, 400, "fp16", history=True)
                    st[i].synchronize()
                    assert r.iters == alone[i][2]
                    assert np.array_equal(r.rec_history, alone[i][1])
                    assert np.array_equal(x.cpu().numpy(), alone[i][0])
    finally:
        for s in hs:
            s.destroy()


# ---- small systems: the whole solve as one kernel of a 16-CTA cluster (csrc/cluster.cu) ---------------------------

def _solve_opt(p, fmt, small, restart=None, rel_tol=None, max_iters=None, precond="none", reorth="cond", x0=None):
    from paper_2009_12101_b200 import Solver

    s = Solver(0)
    try:
        s.set_option("small_path", small)
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        x, r = s.solve(p.b, p.x0 if x0 is None else x0, restart or p.restart, rel_tol or p.rel_tol, max_iters or p.max_iters,
                       fmt, history=True, precond=precond, reorth=reorth)
        return x.cpu().numpy(), r
    finally:
        s.destroy()


@pytest.mark.parametrize("fmt", oracle.FORMATS)
@pytest.mark.parametrize("cfg,kw,m,precond", [("C1", {}, 50, "none"), ("C1", {"grid": 16}, 10, "none"), ("C2", {"grid": 12}, 30, "none"),
                                             ("C4", {"n": 3000}, 50, "jacobi"), ("C5", {"grid": 9}, 128, "none")])
def test_small_system_cluster_path(cfg, kw, m, precond, fmt):
    """The cluster kernel against the oracle (iteration counts, residuals) and against the large path of the same
    library (same algorithm, different summation order: fp64 histories agree to rounding)."""
    from workloads import Problem

    q = make_config(cfg, **kw)
    p = Problem(f"{cfg}-small", q.A, q.b, q.x0, m, q.rel_tol, 3000, oracle.FORMATS, {})
    xs, rs = _solve_opt(p, fmt, 1, precond=precond)
    xl, rl = _solve_opt(p, fmt, 0, precond=precond)
    assert rs.spmv_kernel == 1016 and rl.spmv_kernel != 1016  # the two paths really ran
    run = lambda: oracle.gmres(p.A, p.b, p.x0, m, p.rel_tol, 3000, fmt, precond=precond)
    ref = run()
    assert rs.converged == ref.converged == rl.converged
    check_iters(rs.iters, ref.iters, fmt, f"{cfg}-small", run=run)
    ts, tr = _true_rel_res(p, xs), _true_rel_res(p, ref.x)
    assert ts <= p.rel_tol * (1 + 1e-9) and ts <= 10 * tr and tr <= 10 * ts
    assert rs.rel_res_true == pytest.approx(ts, rel=1e-6)
    assert rs.b_norm == pytest.approx(ref.b_norm, rel=1e-13)
    if fmt == "fp64":
        assert rs.iters == rl.iters == ref.iters and rs.restarts == ref.restarts and rs.reorth_count == ref.reorth_count
        live = ref.rec_history > 1e-7
        assert np.allclose(rs.rec_history[live], ref.rec_history[live], rtol=1e-7)
        assert np.allclose(rs.rec_history[live], rl.rec_history[live], rtol=1e-7)


def test_small_system_cluster_path_edge_cases():
    """Exact x0, iteration bound inside a cycle, restart length 1, a tiny dense system with x0 != 0, l.12."""
    p = make_config("C1", grid=16)
    xs_ = p.meta["xstar"]
    x, r = _solve_opt(p, "fp64", 1, restart=10, rel_tol=1e-10, max_iters=50, x0=xs_)
    assert r.converged and r.iters == 0 and r.restarts == 0 and np.array_equal(x, xs_) and r.spmv_kernel == 1016
    x, r = _solve_opt(p, "fp64", 1, restart=10, rel_tol=1e-14, max_iters=25)
    ref = oracle.gmres(p.A, p.b, p.x0, 10, 1e-14, 25, "fp64")
    assert (not r.converged) and r.status == 16 and r.iters == 25 and r.restarts == 3
    assert _true_rel_res(p, x) == pytest.approx(ref.rel_res_true, rel=1e-6)
    assert np.allclose(r.rec_history, ref.rec_history, rtol=1e-8)
    x, r = _solve_opt(p, "int16", 1, restart=1, rel_tol=1e-3, max_iters=500)
    ref = oracle.gmres(p.A, p.b, p.x0, 1, 1e-3, 500, "int16")
    assert r.converged == ref.converged and abs(r.iters - ref.iters) <= max(2, 0.02 * ref.iters)
    for n, seed in ((1, 40), (3, 41), (33, 42), (64, 43)):
        A, Ad, b = random_dense_system(n, seed)
        from workloads import Problem

        x0 = np.random.default_rng(seed).standard_normal(n)
        q = Problem("tiny", A, b, x0, n, 1e-13, 4 * n + 4, ("fp64",), {})
        x, r = _solve_opt(q, "fp64", 1)
        assert r.spmv_kernel == 1016 and r.converged and r.iters <= n + 1
        assert np.linalg.norm(x - np.linalg.solve(Ad, b)) <= 1e-10 * np.linalg.norm(x)
