"""Restart-length sweep (Fig. 9; SURVEY.md §8(d) "per-cycle time at fixed iteration count"
and §8(f) NEXT-2): time per restart cycle of every storage format at a FIXED number of Arnoldi steps
(`--cycles` full cycles of m steps, tolerance 0, so the convergence test never ends a cycle) --
"numerical effects are ignored" as in the paper -- and the speedup over the fp64 basis next to the
ratio of the algorithmic bytes (the 2x / 4x asymptotes of PAPER.md:294 are its limit for m -> inf).

    python -m paper_2009_12101_b200.cyclebench [--workload C2] [--m 10,20,50,100,150,200,300]
                                               [--cycles 10] [--reorth cond|never|always] [--json out.json]

Runs through cbgmres_solve (C ABI) on cuda:0; inputs are the seeded synthetic workloads of
workloads/generators.py.  Times are the device time of the whole solve (CUDA events on the solver's
stream, one warm-up solve first) divided by the cycles done.
"""
from __future__ import annotations

import argparse
import json
import sys

from . import model
from .binding import FORMATS, Solver


def cycle_bytes(n: int, nnz: int, m: int, fmt: str, reorth_share: float) -> float:
    """Algorithmic bytes of one restart cycle: m Arnoldi steps at basis sizes 1..m (a share of them
    re-orthogonalised: S2' + S3' read the basis twice more), the cycle-end x update over m vectors
    and the explicit residual."""
    steps = 0.0
    for j in range(1, m + 1):
        once = model.arnoldi_step_bytes(n, nnz, j, fmt, reorth=False)
        # re-orthogonalised: S2, then S3 + S2' from one read of the basis, then S3' (three reads)
        twice = once + model.update_bytes(n, j, fmt)
        steps += (1.0 - reorth_share) * once + reorth_share * twice
    return steps + model.update_bytes(n, m, fmt) + model.spmv_bytes(n, nnz) + 8 * n + model.store_bytes(n, fmt)


def run(s, p, ms, cycles, fmts, reorth="cond", out=None):
    """The sweep on handle `s` (matrix of problem `p` already registered).  Returns the rows."""
    import torch

    n, nnz = p.A.n, p.A.nnz
    b = torch.as_tensor(p.b, device=s.device)
    x0 = torch.as_tensor(p.x0, device=s.device)
    rows = []
    for m in ms:
        base_ms = base_bytes = None
        for fmt in fmts:
            iters = cycles * m
            s.solve(b, x0, m, 0.0, m, fmt, reorth=reorth)  # warm-up: one cycle
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            _, r = s.solve(b, x0, m, 0.0, iters, fmt, reorth=reorth)
            e1.record()
            e1.synchronize()
            cyc = max(1, r.iters // m)
            per_cycle = e0.elapsed_time(e1) / cyc
            share = r.reorth_count / max(1, r.iters)
            by = cycle_bytes(n, nnz, m, fmt, share)
            if fmt == "fp64":
                base_ms, base_bytes = per_cycle, by
            row = {"m": m, "format": fmt, "iters": r.iters, "reorth_count": r.reorth_count, "ms_per_cycle": per_cycle,
                   "us_per_step": per_cycle * 1e3 / m, "speedup_vs_fp64": base_ms / per_cycle,
                   "bytes_ratio_vs_fp64": base_bytes / by, "GBps": by / per_cycle / 1e6}
            rows.append(row)
            if out:
                out(f"{m:4d} {fmt:6s} {r.iters:6d} {r.reorth_count:6d} {per_cycle:9.3f} {row['us_per_step']:8.1f} "
                    f"{row['speedup_vs_fp64']:8.2f} {row['bytes_ratio_vs_fp64']:11.2f} {row['GBps']:7.0f}")
    return rows


def main(argv=None) -> int:
    from workloads import make_config

    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="C2")
    ap.add_argument("--m", default="10,20,50,100,150,200,300")
    ap.add_argument("--cycles", type=int, default=10)
    ap.add_argument("--formats", default=",".join(FORMATS))
    ap.add_argument("--reorth", default="cond")
    ap.add_argument("--json", default="")
    ap.add_argument("--grid", type=int, default=0, help="shrink a stencil workload to grid^d points (same recipe)")
    args = ap.parse_args(argv)
    ms = [int(x) for x in args.m.split(",") if x]
    fmts = [f for f in args.formats.split(",") if f]
    if "fp64" not in fmts:
        fmts.insert(0, "fp64")
    p = make_config(args.workload, **({"grid": args.grid} if args.grid else {}))
    n, nnz = p.A.n, p.A.nnz
    s = Solver(0)
    s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
    print(f"# {args.workload}: n={n} nnz={nnz} cycles={args.cycles} reorth={args.reorth} (tolerance 0: fixed iteration count)")
    print(f"{'m':>4s} {'fmt':6s} {'iters':>6s} {'reorth':>6s} {'ms/cycle':>9s} {'us/step':>8s} {'speedup':>8s} {'bytes ratio':>11s} {'GB/s':>7s}")
    rows = run(s, p, ms, args.cycles, fmts, args.reorth, out=print)
    if args.json:
        with open(args.json, "w") as f:
            json.dump({"workload": args.workload, "n": n, "nnz": nnz, "cycles": args.cycles, "reorth": args.reorth,
                       "rows": rows}, f, indent=1)
    s.destroy()
    return 0


if __name__ == "__main__":
    sys.exit(main())
