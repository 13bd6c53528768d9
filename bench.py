"""bench.py -- CB-GMRES (arXiv 2009.12101) on B200: Arnoldi iterations / second and time-to-solution
per basis storage format, with the roofline of the dominant kernel and the oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C2]

Workload (BASELINE.json configs[1], "C2"): 3D 7-point convection-diffusion on a 100^3 grid
(n = 1e6, nnz = 6.94e6), b ~ U[-1,1] seed 1, x0 = 0, restart m = 100, tol 1e-8, all five storage
formats.  One STEP = one pass of the whole hot path over that input: one CB-GMRES solve to
convergence per storage format (fp64, fp32, fp16, int32, int16), i.e. rows S1-S7 of DESIGN.md for
every format.  value = Arnoldi iterations done by all ranks / device time (max over ranks).

N > 1 (torchrun): the path is partitioned by independent problems -- every rank solves its own copy
of the workload on its own GPU, no data-path collective ("scaling": "weak").

--impl reference: the oracle (oracle/, plain C, fp64, as it stands) on the host cores, on a bounded
sample of the same workload (each step = the first REF_ITERS Arnoldi steps of every format's solve).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FORMATS = ("fp64", "fp32", "fp16", "int32", "int16")
FORMAT_BYTES = {"fp64": 8, "fp32": 4, "fp16": 2, "int32": 4, "int16": 2}
METRIC = "arnoldi_iters_per_sec"
UNIT = "iters/s"
PROFILE_EVERY = 8       # CUDA-event brackets around the kernels of every 8th Arnoldi step of the timed region
REF_ITERS = 60          # Arnoldi steps per format in one step of the reference arm / cpu_baseline
PRECOND = "none"        # --precond jacobi: the paper's scalar Jacobi right preconditioner on both arms
WORKLOADS = {"C2": {}, "C1": {}, "C5": {}, "C4": {}, "C2small": {"name": "C2", "grid": 32}}


def _peaks():
    """Measured roofline denominators (MEASURED_PEAKS.json, driver-written); else the guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def _make_problem(workload: str):
    from workloads import make_config

    kw = dict(WORKLOADS[workload])
    name = kw.pop("name", workload)
    return make_config(name, **kw)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
                power.append(float(f[2]))
            except ValueError:
                continue
            for nm, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---- the oracle arm (cpu_baseline leg and --impl reference) ---------------------------------------
def _oracle_step(p, iters_per_format: int):
    """One bounded sample of the workload on the host cores: the first `iters_per_format` Arnoldi
    steps of the solve in every storage format.  Returns (iterations done, seconds)."""
    import oracle

    t0 = time.perf_counter()
    done = 0
    for fmt in p.formats:
        r = oracle.gmres(p.A, p.b, p.x0, p.restart, p.rel_tol, iters_per_format, fmt, precond=PRECOND)
        done += r.iters
    return done, time.perf_counter() - t0


def _sample_text(p, iters_per_format: int) -> str:
    return (f"first {iters_per_format} Arnoldi steps of the {p.name} solve in each of {len(p.formats)} storage formats "
            f"(n={p.A.n}, nnz={p.A.nnz}, m={p.restart})")


def run_reference(args) -> int:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0  # rank 0 alone runs the oracle
    import oracle

    p = _make_problem(args.workload)
    REF = REF_ITERS
    for _ in range(args.warmup):
        _oracle_step(p, REF)
    total_it, total_s = 0, 0.0
    for _ in range(args.steps):
        it, s = _oracle_step(p, REF)
        total_it += it
        total_s += s
    value = total_it / total_s
    cores = oracle.num_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total_s / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "precond": PRECOND, "n": p.A.n, "nnz": p.A.nnz, "restart": p.restart, "rel_tol": p.rel_tol,
                   "formats": list(p.formats), "bounded_sample": _sample_text(p, REF)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": _sample_text(p, REF)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---- our arm ----------------------------------------------------------------------------------------
def _solve_all_formats(solver, p, dev, host=None):
    """One step: one solve per storage format.  Returns {fmt: SolveResult}."""
    out = {}
    for fmt in p.formats:
        if host is None:
            solver.profile_reset()
            _, r = solver.solve(dev["b"], dev["x0"], p.restart, p.rel_tol, p.max_iters, fmt, precond=PRECOND)
            r.prof = solver.profile_get()
        else:
            host["x"].copy_(host["x0"])
            r = solver.solve_host(host["row_ptr"], host["col_idx"], host["vals"], host["b"], host["x"], p.restart,
                                  p.rel_tol, p.max_iters, fmt, precond=PRECOND)
        out[fmt] = r
    return out


def aggregate_over_ranks(world: int, device, ms: float, e_ms: float, iters: int, e_iters: int, launches: int):
    """Whole-job figures of N independent replicas ("replicas only"): the timed
    regions are bracketed by barriers, so the job takes the MAX of the ranks' times; iterations and
    launches are SUMMED.  No data-path collective exists; this is the only cross-rank exchange."""
    if world <= 1:
        return ms, e_ms, iters, e_iters, launches
    import torch
    import torch.distributed as dist

    t = torch.tensor([ms, e_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([iters, e_iters, launches], dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), int(c[0]), int(c[1]), int(c[2])


def run_ours(args) -> int:
    import torch
    import torch.distributed as dist

    from paper_2009_12101_b200 import PROF_FAMILIES, Solver

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (sm_100a); there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    p = _make_problem(args.workload)
    n, nnz = p.A.n, p.A.nnz
    solver = Solver(local)
    solver.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
    dev = {"b": torch.as_tensor(p.b, device=solver.device), "x0": torch.as_tensor(p.x0, device=solver.device)}
    host = {k: torch.as_tensor(v).pin_memory() for k, v in
            (("row_ptr", p.A.row_ptr), ("col_idx", p.A.col_idx), ("vals", p.A.vals), ("b", p.b), ("x0", p.x0))}
    host["x"] = torch.empty(n, dtype=torch.float64).pin_memory()
    solver.set_option("profile", PROFILE_EVERY)

    # -- device-resident arm: W warm-up steps, K timed steps --
    for _ in range(args.warmup):
        _solve_all_formats(solver, p, dev)
    sampler = ClockSampler(local)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = solver.launch_count()
    barrier()
    sampler.start()
    ev0.record()
    steps = [_solve_all_formats(solver, p, dev) for _ in range(args.steps)]
    ev1.record()
    barrier()
    clocks = sampler.stop()
    launches = solver.launch_count() - launches0
    ms = ev0.elapsed_time(ev1)
    iters = sum(r.iters for st in steps for r in st.values())

    # -- end-to-end arm: host buffers through cbgmres_solve_host, copies inside the timed region --
    solver.set_option("profile", 0)
    for _ in range(min(args.warmup, 1)):
        _solve_all_formats(solver, p, dev, host)
    barrier()
    t0 = time.perf_counter()
    e_steps = [_solve_all_formats(solver, p, dev, host) for _ in range(args.steps)]
    barrier()
    e_s = time.perf_counter() - t0
    e_iters = sum(r.iters for st in e_steps for r in st.values())
    nf = len(p.formats)
    h2d = nf * (4 * (n + 1) + 12 * nnz + 16 * n)
    d2h = nf * 8 * n

    ms, e_ms, iters, e_iters, launches = aggregate_over_ranks(world, solver.device, ms, e_s * 1e3, iters, e_iters, launches)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # -- per-format table (time-to-solution, iterations/s) from the timed steps --
    per_format = {}
    for fmt in p.formats:
        rs = [st[fmt] for st in steps]
        t_ms = sum(r.solve_ms for r in rs) / len(rs)
        it = rs[-1].iters
        per_format[fmt] = {"iters": it, "restarts": rs[-1].restarts, "reorth_count": rs[-1].reorth_count,
                           "converged": bool(rs[-1].converged), "rel_res_true": rs[-1].rel_res_true,
                           "time_to_solution_ms": t_ms, "iters_per_sec": it / (t_ms * 1e-3) if t_ms > 0 else None}
    t64 = per_format.get("fp64", {}).get("time_to_solution_ms")
    for fmt, d in per_format.items():
        d["speedup_vs_fp64"] = (t64 / d["time_to_solution_ms"]) if t64 and d["time_to_solution_ms"] else None

    # -- roofline of the dominant kernel family: CUDA events around every launch of the timed region --
    peak, peak_src = _peaks()
    fam = {name: {"ms": 0.0, "bytes": 0.0, "launches": 0} for name in PROF_FAMILIES}
    kernels = []
    for fmt in p.formats:
        acc = {name: {"ms": 0.0, "bytes": 0.0, "launches": 0} for name in PROF_FAMILIES}
        for st in steps:
            for name, d in st[fmt].prof.items():
                for k in ("ms", "bytes", "launches"):
                    acc[name][k] += d[k]
                    fam[name][k] += d[k]
        for name, d in acc.items():
            if d["launches"]:
                gbs = d["bytes"] / (d["ms"] * 1e-3) / 1e9 if d["ms"] > 0 else None
                kernels.append({"kernel": name, "format": fmt, "launches": d["launches"], "ms": round(d["ms"], 3),
                                "GBps": round(gbs, 1) if gbs else None, "frac": round(gbs / peak, 4) if gbs else None})
    total_prof_ms = sum(d["ms"] for d in fam.values()) or 1.0
    dom = max(fam, key=lambda k: fam[k]["ms"])
    d = fam[dom]
    achieved = d["bytes"] / (d["ms"] * 1e-3) / 1e9 if d["ms"] > 0 else 0.0
    # ncu dram__bytes_read + dram__bytes_write of this family, per launch: the ratio traffic / algorithmic
    # bytes of the captured launches (profiles/ncu_traffic.csv, written from the --set full captures)
    # applied to the average launch of this run
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if os.path.exists(tpath):
        import csv

        with open(tpath, newline="") as f:
            ratios = {r["family"]: float(r["traffic_over_algorithmic"]) for r in csv.DictReader(f)}
        if dom in ratios and d["launches"]:
            traffic = round(ratios[dom] * d["bytes"] / d["launches"])
    roofline = {"bound": "hbm", "kernel": dom, "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
                "frac": round(achieved / peak, 4), "traffic": traffic, "peak_source": peak_src,
                "launches": d["launches"], "avg_launch_us": round(1e3 * d["ms"] / max(d["launches"], 1), 2),
                "algorithmic_bytes_per_launch": round(d["bytes"] / max(d["launches"], 1)),
                "share_of_step": round(d["ms"] / total_prof_ms, 4),
                "shares": {k: round(v["ms"] / total_prof_ms, 4) for k, v in fam.items()}}

    # -- the oracle on this box's host cores, bounded sample of the same workload --
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle

        c_it, c_s = _oracle_step(p, REF_ITERS)
        cpu = {"value": c_it / c_s, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": _sample_text(p, REF_ITERS), "seconds": round(c_s, 2)}

    line = {
        "metric": METRIC, "value": iters / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "precond": PRECOND, "n": n, "nnz": nnz, "restart": p.restart, "rel_tol": p.rel_tol,
                   "max_iters": p.max_iters, "formats": list(p.formats), "reorth": "cond (eta = 1/sqrt 2)",
                   "step": "one solve to convergence per storage format",
                   "l2": "no flush: basis (0.2-0.8 GB) + matrix exceed the 126 MB L2; reuse inside a solve is the workload's own",
                   "parallelism": f"{world} independent solves, one per GPU" if world > 1 else "1 GPU"},
        "iters_per_step": iters / args.steps / world,
        "e2e": {"value": e_iters / (e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e_ms / args.steps},
        "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
        "per_format": per_format, "kernels": kernels,
    }
    print(json.dumps(line))
    solver.destroy()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--workload", choices=tuple(WORKLOADS), default="C2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--precond", choices=("none", "jacobi"), default="none")
    args = ap.parse_args()
    global PRECOND
    PRECOND = args.precond
    if args.steps < 1:
        ap.error("--steps must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
