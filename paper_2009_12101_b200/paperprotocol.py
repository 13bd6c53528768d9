"""The paper's experimental protocol on the synthetic matrix set.

PAPER.md:251: right-hand side b_i = sin(i), x0 = 0, restart m = 100, stop at ||A x - b|| <= 1e-9 ||b||;
PAPER.md:186: scalar Jacobi preconditioner.  For every matrix and storage format the solver runs to
convergence (or to the iteration bound); the table printed at the end has the form of the paper's
Table 2: mean, median and variance over the matrices of the iteration count
relative to the fp64 basis, over the problems every format of the row solved.  The SuiteSparse
matrices of the paper are not available; BASELINE.json's synthetic families at several sizes stand
in for them, so the numbers compare with Table 2 only qualitatively.

    python -m paper_2009_12101_b200.paperprotocol [--max-iters 20000] [--json out.json] [--small]

Runs through cbgmres_solve (C ABI) on cuda:0.
"""
from __future__ import annotations

import argparse
import json
import statistics
import sys

import numpy as np

from .binding import FORMATS, Solver

MATRICES = (  # (label, config, keyword arguments of workloads.make_config)
    ("convdiff7pt-60^3", "C2", {"grid": 60}),
    ("convdiff7pt-80^3", "C2", {"grid": 80}),
    ("convdiff7pt-100^3", "C2", {}),
    ("stencil27pt-64^3", "C5", {"grid": 64}),
    ("stencil27pt-100^3", "C5", {"grid": 100}),
    ("stencil27pt-160^3", "C5", {}),
    ("powerlaw-5e5", "C4", {"n": 500_000}),
    ("powerlaw-2e6", "C4", {}),
    ("laplace5pt-64^2", "C1", {}),
)
SMALL = (("convdiff7pt-24^3", "C2", {"grid": 24}), ("stencil27pt-16^3", "C5", {"grid": 16}), ("powerlaw-2e4", "C4", {"n": 20_000}))


def main(argv=None) -> int:
    from workloads import make_config

    ap = argparse.ArgumentParser()
    ap.add_argument("--max-iters", type=int, default=20000)
    ap.add_argument("--restart", type=int, default=100)
    ap.add_argument("--tol", type=float, default=1e-9)
    ap.add_argument("--precond", default="jacobi", choices=("none", "jacobi"))
    ap.add_argument("--small", action="store_true", help="three small matrices (a quick check of the script)")
    ap.add_argument("--json", default="")
    args = ap.parse_args(argv)
    s = Solver(0)
    rows = []
    print(f"# b_i = sin(i), x0 = 0, m = {args.restart}, tol = {args.tol:g}, precond = {args.precond}, max_iters = {args.max_iters}")
    print(f"{'matrix':20s} {'n':>9s} {'nnz':>10s} " + " ".join(f"{f:>16s}" for f in FORMATS))
    for label, cfg, kw in (SMALL if args.small else MATRICES):
        p = make_config(cfg, **kw)
        n = p.A.n
        b = np.sin(np.arange(1, n + 1, dtype=np.float64))  # PAPER.md:251, 1-based i
        x0 = np.zeros(n)
        s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        rec = {"matrix": label, "n": n, "nnz": p.A.nnz, "formats": {}}
        cells = []
        for fmt in FORMATS:
            s.solve(b, x0, args.restart, args.tol, 3, fmt, precond=args.precond)  # warm-up: one-time kernel set-up
            _, r = s.solve(b, x0, args.restart, args.tol, args.max_iters, fmt, precond=args.precond)
            rec["formats"][fmt] = {"iters": r.iters, "converged": bool(r.converged), "rel_res_true": r.rel_res_true,
                                   "solve_ms": r.solve_ms, "reorth_count": r.reorth_count}
            cells.append(f"{r.iters:6d}{'' if r.converged else '*'} {r.solve_ms:8.1f}ms")
        rows.append(rec)
        print(f"{label:20s} {n:9d} {p.A.nnz:10d} " + " ".join(f"{c:>16s}" for c in cells))
    print("# (* = not converged within the bound)")
    print("\n# iteration count relative to the fp64 basis over the matrices both solved (cf. Table 2, PAPER.md:281-290)")
    print(f"{'format':8s} {'solved':>8s} {'mean':>8s} {'median':>8s} {'variance':>10s} {'time ratio (median)':>20s}")
    table = {}
    for fmt in FORMATS[1:]:
        ratios, tratios = [], []
        for rec in rows:
            a, c = rec["formats"]["fp64"], rec["formats"][fmt]
            if a["converged"] and c["converged"] and a["iters"] > 0:
                ratios.append(c["iters"] / a["iters"])
                tratios.append(a["solve_ms"] / c["solve_ms"])
        if ratios:
            var = statistics.pvariance(ratios) if len(ratios) > 1 else 0.0
            table[fmt] = {"solved": len(ratios), "mean": statistics.fmean(ratios), "median": statistics.median(ratios),
                          "variance": var, "speedup_median": statistics.median(tratios)}
            print(f"{fmt:8s} {len(ratios):5d}/{len(rows):<2d} {table[fmt]['mean']:8.2f} {table[fmt]['median']:8.2f} {var:10.3f} "
                  f"{table[fmt]['speedup_median']:20.2f}")
        else:
            print(f"{fmt:8s} {0:5d}/{len(rows):<2d}")
    if args.json:
        with open(args.json, "w") as f:
            json.dump({"protocol": vars(args), "rows": rows, "table": table}, f, indent=1)
    s.destroy()
    return 0


if __name__ == "__main__":
    sys.exit(main())
