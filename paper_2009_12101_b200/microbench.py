"""Per-kernel microbenchmark (BASELINE.json configs[2], "C3"): multi-dot, update + norms and
normalise + compress-store timed separately over a basis of k vectors of n rows in every storage
format, through the per-kernel hooks of the C ABI, with CUDA events on the launching stream.

    python -m paper_2009_12101_b200.microbench [--n 4194304] [--k 1,2,4,8,16,32,64,100] [--formats ...]
                                               [--reps 20] [--flush] [--spmv C2,C5] [--json out.json]

Inputs are synthetic and made on the device: basis vector c = N(0,1)/sqrt(n) entries (the magnitude
distribution of a unit vector, |v_i| <= 1) pushed through cbgmres_k_compress; w ~ N(0,1).  The values
do not need to be orthonormal for timing (parity with the oracle on the orthonormal C3 recipe is
tests/test_gpu_kernels.py).  GB/s = ALGORITHMIC bytes / median time.
--flush writes a 512 MB buffer between launches so nothing is L2-resident; without it a working set
below ~126 MB is served from L2 and the figure is not an HBM bandwidth.
"""
from __future__ import annotations

import argparse
import json
import statistics
import sys

from . import model
from .binding import FORMATS, Solver, payload_dtype


def _time(fn, reps, flush_buf, torch):
    ts = []
    for i in range(reps + 3):
        if flush_buf is not None:
            flush_buf.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        e1.synchronize()
        if i >= 3:
            ts.append(e0.elapsed_time(e1) * 1e-3)
    return statistics.median(ts), min(ts)


def run(s, n, ks, fmts, reps=20, flush=True, log=None):
    """Times S2 (multi-dot), S3 (update + norms), the fused S3 + S2' and S4 (store) separately on handle `s`.
    Returns a list of rows {"kernel", "format", "k", "median_us", "best_us", "bytes", "GBps"}."""
    import torch

    dev = s.device
    kmax = max(ks)
    flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device=dev) if flush else None
    rows = []
    g = torch.Generator(device=dev)
    g.manual_seed(2)
    w0 = torch.randn(n, dtype=torch.float64, device=dev, generator=g)
    for fmt in fmts:
        ld = (n + 63) // 64 * 64
        V = torch.zeros((kmax, ld), dtype=payload_dtype(fmt), device=dev)
        sig = torch.ones(kmax, dtype=torch.float64, device=dev)
        for c in range(kmax):
            v = torch.randn(n, dtype=torch.float64, device=dev, generator=g) / n ** 0.5
            pay, sc = s.k_compress(fmt, v)
            V[c, :n] = pay
            sig[c] = sc[0]
        for k in ks:
            h = s.k_multidot(fmt, V, sig, w0, n=n, k=k).clone()
            w = w0.clone()
            med, best = _time(lambda: s.k_multidot(fmt, V, sig, w0, n=n, k=k), reps, flush_buf, torch)
            rows.append(("multidot", fmt, k, med, best, model.multidot_bytes(n, k, fmt)))
            hz = torch.zeros_like(h)  # w -= V*0 keeps w bounded over the repetitions; same traffic and flops
            med, best = _time(lambda: s.k_update(fmt, V[:k], sig, hz, w, n=n), reps, flush_buf, torch)
            rows.append(("update", fmt, k, med, best, model.update_bytes(n, k, fmt)))
            if k <= 128:
                med, best = _time(lambda: s.k_update_multidot(fmt, V[:k], sig, hz, w, n=n), reps, flush_buf, torch)
                rows.append(("update_multidot", fmt, k, med, best, model.update_bytes(n, k, fmt)))
        col = torch.empty(ld, dtype=payload_dtype(fmt), device=dev)
        vout = torch.empty(n, dtype=torch.float64, device=dev)
        med, best = _time(lambda: s.k_store(fmt, w0, 2.0, 6.0, col, vout), reps, flush_buf, torch)
        rows.append(("store", fmt, 1, med, best, model.store_bytes(n, fmt)))
        del V
        if log:
            log(f"microbench {fmt} done")
    return [{"kernel": name, "format": fmt, "k": k, "median_us": med * 1e6, "best_us": best * 1e6, "bytes": by,
             "GBps": by / med / 1e9} for name, fmt, k, med, best, by in rows]


def main(argv=None) -> int:
    import torch

    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=4_194_304)
    ap.add_argument("--k", default="1,2,4,8,16,32,50,64,100")
    ap.add_argument("--formats", default=",".join(FORMATS))
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--flush", action="store_true")
    ap.add_argument("--spmv", default="")
    ap.add_argument("--json", default="")
    ap.add_argument("--interleave", type=int, default=0, help="orth_interleave option: 0 auto, 1 blocked, 2 interleaved")
    ap.add_argument("--spmv-kernel", default="0", help="comma list of spmv_kernel options to time (0 = auto)")
    ap.add_argument("--seg-kb", type=int, default=0, help="orth_seg_kb option: 0 auto, 1, 2, 4")
    ap.add_argument("--opt", action="append", default=[], help="name=value, passed to cbgmres_set_option (repeatable)")
    args = ap.parse_args(argv)
    ks = [int(x) for x in args.k.split(",") if x]
    fmts = [f for f in args.formats.split(",") if f]
    n = args.n
    s = Solver(0)
    s.set_option("orth_seg_kb", args.seg_kb)
    s.set_option("orth_interleave", args.interleave)
    for o in args.opt:
        name, val = o.split("=")
        s.set_option(name, int(val))
    dev = s.device
    out = run(s, n, ks, fmts, args.reps, args.flush) if ks and fmts else []
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev) if args.flush else None
    g = torch.Generator(device=dev)
    g.manual_seed(3)
    for name in [x for x in args.spmv.split(",") if x]:
        from workloads import make_config

        p = make_config(name)
        x = torch.randn(p.A.n, dtype=torch.float64, device=dev, generator=g)
        y = torch.empty_like(x)
        for kern in [int(v) for v in args.spmv_kernel.split(",")]:
            s.set_option("spmv_kernel", kern)
            s.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
            med, best = _time(lambda: s.k_spmv(x, y, want_norm=False), args.reps, flush, torch)
            by = model.spmv_bytes(p.A.n, p.A.nnz)
            out.append({"kernel": f"spmv[{name},opt={kern}]", "format": "fp64", "k": 0, "median_us": med * 1e6,
                        "best_us": best * 1e6, "bytes": by, "GBps": by / med / 1e9})
    print(f"# n={n} reps={args.reps} flush={args.flush}  GB/s = algorithmic bytes / median time")
    print(f"{'kernel':28s} {'fmt':6s} {'k':>4s} {'median_us':>10s} {'best_us':>10s} {'MB':>9s} {'GB/s':>8s}")
    for r in out:
        print(f"{r['kernel']:28s} {r['format']:6s} {r['k']:4d} {r['median_us']:10.1f} {r['best_us']:10.1f} "
              f"{r['bytes'] / 1e6:9.1f} {r['GBps']:8.0f}")
    if args.json:
        with open(args.json, "w") as f:
            json.dump({"n": n, "flush": args.flush, "rows": out}, f, indent=1)
    s.destroy()
    return 0


if __name__ == "__main__":
    sys.exit(main())
