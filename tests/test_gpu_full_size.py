"""GPU parity at BASELINE.json's FULL sizes, in the launch configurations bench.py and the C3
microbench time: outputs the oracle can compute one by one are compared on samples (columns of
the multi-dot, rows of the update, every row of the SpMV -- the oracle's SpMV is fast enough), the
rest through properties that hold at any size (norms of the GPU's own output, true residuals,
residual histories over a bounded prefix of the solve)."""
import numpy as np
import pytest

import json
import os

import oracle
from parity import check_iters
from workloads import make_config

pytestmark = pytest.mark.gpu

TOL = 1e-12
N_C3 = 4_194_304  # BASELINE.json configs[2]


def _dev(a):
    import torch

    return torch.as_tensor(np.ascontiguousarray(a), device="cuda")


@pytest.fixture(scope="module")
def solver():
    from paper_2009_12101_b200 import Solver

    s = Solver(0)
    yield s
    s.destroy()


@pytest.fixture(scope="module")
def c3_vectors():
    """k = 100 vectors of n = 4,194,304 entries of typical size n^-1/2 (the value distribution of the
    decode path), scaled to unit 2-norm; w standard normal.  No QR at this
    size (minutes on the host): orthogonality plays no role in per-kernel parity."""
    rng = np.random.default_rng(2)
    k = 100
    V = rng.standard_normal((k, N_C3))
    V /= np.linalg.norm(V, axis=1, keepdims=True)
    w = rng.standard_normal(N_C3)
    h = rng.standard_normal(k)
    return V, w, h


@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_c3_size_passes_sampled(solver, c3_vectors, fmt):
    import torch
    from paper_2009_12101_b200 import payload_dtype

    V, w, h = c3_vectors
    k, n = V.shape
    P, sig = oracle.enc_basis(fmt, V)
    dP = torch.as_tensor(P, device="cuda").view(payload_dtype(fmt))
    dsig, dw = _dev(sig), _dev(w)
    wn = np.linalg.norm(w)

    # S2: sampled columns against the oracle's extended-precision dot
    cols = [0, 1, 37, 63, 64, 99]
    hg = solver.k_multidot(fmt, dP, dsig, dw, n=n, k=k).cpu().numpy()
    assert np.all(np.isfinite(hg))
    for c in cols:
        ref = oracle.ref_multidot(fmt, P[c:c + 1], sig[c:c + 1], w, k=1)[0]
        vn = np.linalg.norm(oracle.dec(fmt, P[c], sig[c]))
        assert abs(hg[c] - ref) <= TOL * vn * wn

    # S3 (+ S2' fused): sampled rows -- first and last tiles, tile borders, random interior rows
    rng = np.random.default_rng(7)
    rows = np.unique(np.concatenate([np.arange(0, 2048), np.arange(n - 2048, n),
                                     rng.integers(0, n, 4096), np.arange(1 << 20, (1 << 20) + 64)]))
    w_ref_rows, _, _ = oracle.ref_update(fmt, np.ascontiguousarray(P[:, rows]), sig, h, w[rows])
    row_tol = TOL * (np.abs(w[rows]) + np.linalg.norm(h))  # |dw_i| <= tol (|w_i| + ||V^_{i,:}|| ||h||), ||V^_{i,:}|| << 1

    d1 = dw.clone()
    out = solver.k_update(fmt, dP, dsig, _dev(h), d1, n=n)
    torch.cuda.synchronize()
    w1 = d1.cpu().numpy()
    nrm2, amax = out.cpu().numpy()
    assert np.all(np.abs(w1[rows] - w_ref_rows) <= row_tol)
    assert abs(nrm2 - np.linalg.norm(w1)) <= 1e-13 * np.linalg.norm(w1)  # the norm of the kernel's own output
    assert amax == np.abs(w1).max()

    d2 = dw.clone()
    u, out2 = solver.k_update_multidot(fmt, dP, dsig, _dev(h), d2, n=n)
    torch.cuda.synchronize()
    w2 = d2.cpu().numpy()
    assert np.all(np.abs(w2[rows] - w_ref_rows) <= row_tol)
    nrm2f, amaxf = out2.cpu().numpy()
    assert abs(nrm2f - np.linalg.norm(w2)) <= 1e-13 * np.linalg.norm(w2)
    assert amaxf == np.abs(w2).max()
    ug = u.cpu().numpy()
    for c in cols:  # u = dec(V)^T w_new, on the GPU's own w_new (exactly representable input for the oracle)
        ref = oracle.ref_multidot(fmt, P[c:c + 1], sig[c:c + 1], w2, k=1)[0]
        vn = np.linalg.norm(oracle.dec(fmt, P[c], sig[c]))
        assert abs(ug[c] - ref) <= TOL * vn * np.linalg.norm(w2)


@pytest.mark.parametrize("name", ["C2", "C4", "C5"])
def test_full_size_spmv_every_row(name):
    """S1 on the full-size matrices with the kernel set_matrix selects (the one bench.py times)."""
    from paper_2009_12101_b200 import Solver

    p = make_config(name)
    s = Solver(0)
    try:
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        x = np.random.default_rng(600).standard_normal(p.A.n)
        y_ref, rowabs = oracle.ref_spmv(p.A, x)
        w, nrm = s.k_spmv(_dev(x))
        y = w.cpu().numpy()
        assert np.all(np.abs(y - y_ref) <= TOL * np.maximum(rowabs, 1e-300))
        assert abs(nrm.item() - np.linalg.norm(y_ref)) <= TOL * np.linalg.norm(y_ref)
    finally:
        s.destroy()


@pytest.fixture(scope="module")
def c2_full():
    from paper_2009_12101_b200 import Solver

    p = make_config("C2")
    s = Solver(0)
    s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
    yield p, s
    s.destroy()


@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_full_size_c2_solve_properties(c2_full, fmt):
    """The solve bench.py times.  Properties: converged, the explicit residual of the returned x
    (recomputed with the oracle's SpMV) is below tolerance and equals the reported one."""
    p, s = c2_full
    x, r = s.solve(p.b, p.x0, p.restart, p.rel_tol, p.max_iters, fmt)
    xh = x.cpu().numpy()
    true = np.linalg.norm(p.b - oracle.spmv(p.A, xh)) / np.linalg.norm(p.b)
    assert r.converged
    assert true <= p.rel_tol * (1 + 1e-9)
    assert r.rel_res_true == pytest.approx(true, rel=1e-6)
    assert r.iters <= p.max_iters and r.restarts >= r.iters // p.restart


# relative agreement of the residual histories: fp64 storage reproduces the oracle to rounding; with
# reduced storage a rounding-level difference in w can move an entry of v across a rounding boundary
# of the format at the store, a perturbation of one unit of the format's precision
HIST_TOL = {"fp64": 1e-12, "fp32": 2.0 ** -24, "fp16": 2.0 ** -11, "int32": 1.0 / 2147483647, "int16": 1.0 / 32767}


@pytest.mark.parametrize("fmt", oracle.FORMATS)
def test_full_size_c2_residual_history_prefix(c2_full, fmt):
    """Bounded prefix of the full-size solve against the oracle: the recurrence residual of the first
    40 Arnoldi steps (one step = SpMV + both Gram-Schmidt passes + store at n = 1e6) and the
    re-orthogonalisation decisions (reading Q11: the iterates differ by summation order only)."""
    p, s = c2_full
    steps = 40
    ref = oracle.gmres(p.A, p.b, p.x0, p.restart, p.rel_tol, steps, fmt=fmt)
    _, r = s.solve(p.b, p.x0, p.restart, p.rel_tol, steps, fmt, history=True)
    assert r.iters == ref.iters == steps
    hg, ho = np.asarray(r.rec_history[:steps]), np.asarray(ref.rec_history[:steps])
    assert np.all(np.abs(hg - ho) <= HIST_TOL[fmt] * ho)
    assert r.reorth_count == ref.reorth_count


# ---- full-size solves to convergence against the oracle's cached results -----------------------------------------
# tests/golden/fullsize_oracle.json is written by tests/golden/make_fullsize_oracle_cache.py, which calls only
# oracle/ (hours of CPU work: SURVEY.md 8(d) "cache its result keyed by config + format").  north_star: iteration
# counts to convergence within +-2 %, true residuals both below the tolerance and within 10x of each other.
_CACHE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fullsize_oracle.json")
_PRECOND = {"C2": "none", "C5": "none", "C4J": "jacobi", "C4B": "block_jacobi4", "C4": "none"}


def _cached(case, fmt):
    if not os.path.exists(_CACHE):
        pytest.fail("tests/golden/fullsize_oracle.json is missing: run tests/golden/make_fullsize_oracle_cache.py")
    with open(_CACHE) as f:
        data = json.load(f)
    entry = data["cases"].get(case)
    if entry is None or "iters" not in entry["formats"].get(fmt, {}):
        pytest.skip(f"{case} {fmt}: no cached oracle result")
    return entry, entry["formats"][fmt]


@pytest.fixture(scope="module")
def full_solvers():
    """One handle + matrix per full-size config, made on first use and kept for the module."""
    from paper_2009_12101_b200 import Solver

    made = {}

    def get(cfg):
        if cfg not in made:
            p = make_config(cfg)
            s = Solver(0)
            s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
            made[cfg] = (p, s)
        return made[cfg]

    yield get
    for _, s in made.values():
        s.destroy()


@pytest.mark.parametrize("fmt", oracle.FORMATS)
@pytest.mark.parametrize("case", ["C2", "C5", "C4J", "C4B", "C4"])
def test_full_size_solve_matches_cached_oracle(full_solvers, case, fmt):
    entry, o = _cached(case, fmt)
    p, s = full_solvers(entry["config"])
    assert (p.A.n, p.A.nnz, p.restart, p.rel_tol) == (entry["n"], entry["nnz"], entry["restart"], entry["rel_tol"])
    x, r = s.solve(p.b, p.x0, p.restart, p.rel_tol, entry["max_iters"], fmt, precond=_PRECOND[case], history=True)
    xh = x.cpu().numpy()
    true = np.linalg.norm(p.b - oracle.spmv(p.A, xh)) / np.linalg.norm(p.b)  # recomputed with the oracle's SpMV
    assert bool(r.converged) == o["converged"], (case, fmt, r.iters, o["iters"])
    draws = [d["iters"] for d in o.get("spread", {}).values()]
    rule = check_iters(r.iters, o["iters"], fmt, case, draws=draws if draws else None)
    assert r.rel_res_true == pytest.approx(true, rel=1e-6)
    if o["converged"]:
        assert true <= p.rel_tol * (1 + 1e-9) and o["rel_res_true_recomputed"] <= p.rel_tol * (1 + 1e-9)
    # "within 10x of each other" (north_star), against the range of the oracle's own residuals: its base run and the same
    # solve under other summation orders.  The range is a point for every case but the 16-bit solves that do not converge
    # (int16 on the Jacobi- / block-Jacobi-preconditioned power-law matrix: the oracle's own residuals at the iteration
    # bound run from 3 to 2e5, reading Q11 and DESIGN.md section 6.6)
    ores = [o["rel_res_true_recomputed"]] + [d["rel_res_true"] for d in o.get("spread", {}).values()]
    assert true <= 10 * max(ores) and min(ores) <= 10 * true
    if rule == "strict":
        assert abs(r.restarts - o["restarts"]) <= 1
        # l.7 fires on almost every step of these solves, so the two counts can only be compared after allowing for the
        # steps one side did and the other did not (reading Q11: the step counts themselves agree to +-2 %)
        assert abs(r.reorth_count - o["reorth_count"]) <= max(2, 0.02 * o["reorth_count"]) + abs(r.iters - o["iters"])
    # the first steps are before any decorrelation: the recurrence residuals agree to the format's roundoff (40 steps on
    # the stencils; 12 on the power-law matrix, whose quantised histories part within some tens of steps: reading Q11)
    c4 = case.startswith("C4")
    k = min(12 if c4 else 40, r.iters, o["iters"])
    hg, ho = np.asarray(r.rec_history[:k]), np.asarray(o["rec_history"][:k])
    assert np.all(np.abs(hg - ho) <= HIST_TOL[fmt] * ho * (100 if c4 else 1))
    print(f"[full-size] {case} {fmt}: gpu iters {r.iters} restarts {r.restarts} | oracle {o['iters']} {o['restarts']} "
          f"draws {sorted(draws)} | rule {rule} | true residual gpu {true:.3e} oracle {o['rel_res_true_recomputed']:.3e}")
