"""bench.py -- CB-GMRES (arXiv 2009.12101) on B200: Arnoldi iterations / second and time-to-solution
per basis storage format, with the roofline of the dominant kernel and the oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C5]
                    [--precond none|jacobi|block_jacobi4] [--no-extras] [--no-cpu-baseline]

Workload (default): BASELINE.json configs[4], "C5", the largest single-GPU configuration: 3D 27-point stencil
on a 160^3 grid (n = 4,096,000, nnz = 109,215,352), b ~ U[-1,1] seed 4, x0 = 0, restart m = 100, tol 1e-8,
all five storage formats.  One STEP = one pass of the whole hot path over that input: one CB-GMRES solve to
convergence per storage format (fp64, fp32, fp16, int32, int16), i.e. rows S1-S7 of DESIGN.md for every format.
value = Arnoldi iterations done by all ranks / device time (max over ranks).

Protocol.  W warm-up steps, then K timed steps between CUDA events on the solver's stream with a barrier and a
device synchronisation on both sides -- with the library's per-kernel event brackets OFF.  Then the same K steps
through cbgmres_solve_host with pinned HOST buffers (e2e: every solve copies the CSR arrays, b and x0 in and x
out).  Only after both timed regions: one more step with event brackets around the launches of every 2nd Arnoldi
step (`roofline`, `kernels`), and -- on rank 0 at N = 1 -- the other configs (`per_config`: C1, C2, C4 with
none / Jacobi / block-Jacobi), the C3 microbenchmark at n = 4,194,304 (`c3`), the restart sweep at a fixed
iteration count on this workload (`msweep`, Fig. 9 of the paper) and the oracle on the host cores
(`cpu_baseline`).  `--no-extras` drops per_config / c3 / msweep.

N > 1 (torchrun): the path is partitioned by independent problems -- every rank solves its own copy of the
workload on its own GPU, no data-path collective ("scaling": "weak").

--impl reference: the oracle (oracle/, plain C, fp64, as it stands) on the host cores, on a bounded sample of
the same workload (each step = the first REF_ITERS[workload] Arnoldi steps of every format's solve).
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
PROFILE_EVERY = 2       # separate pass after the timed regions: CUDA-event brackets around the kernels of every 2nd Arnoldi step
# Arnoldi steps per format in one step of the reference arm / cpu_baseline: sized so that `--steps 20 --warmup 5` of the
# reference arm ends within a few minutes on the GPU box's host cores (an oracle step at basis size j streams about
# 12 nnz + 100 j n bytes: on 16 cores one such step of the reference arm takes ~ 7 s on C5, ~ 2 s on C2)
REF_ITERS = {"C5": 24, "C2": 60, "C2small": 60, "C4": 20, "C1": 3000}
PRECOND = "none"        # --precond: the paper's right preconditioners on both arms
WORKLOADS = {"C5": {}, "C2": {}, "C1": {}, "C4": {}, "C2small": {"name": "C2", "grid": 32}}
NOMINAL_HBM_GBS = 8000.0  # BASELINE.json north_star: "B200 peak (~8 TB/s)"
C3_N = 4_194_304
C3_KS = (1, 2, 4, 8, 16, 32, 50, 64, 100)
MSWEEP = (10, 50, 100, 200)
TRAFFIC_CSV = os.path.join("profiles", "ncu_traffic.csv")


def _peaks():
    """Measured roofline denominator (MEASURED_PEAKS.json, driver-written); else the guide's fallback."""
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


def _log(msg: str):
    print(f"[bench {time.strftime('%H:%M:%S')}] {msg}", file=sys.stderr, flush=True)


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
            f"(n={p.A.n}, nnz={p.A.nnz}, m={p.restart}); basis sizes 1..{iters_per_format} only, so the work per "
            f"iteration is smaller than in the GPU arm's whole solves (mean basis size m/2)")


def run_reference(args) -> int:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0  # rank 0 alone runs the oracle
    import oracle

    p = _make_problem(args.workload)
    REF = REF_ITERS[args.workload]
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
def _solve_all_formats(solver, p, dev, host=None, profile=False, precond=None, max_iters=None, reorth="cond"):
    """One step: one solve per storage format.  Returns {fmt: SolveResult}."""
    out = {}
    pc = PRECOND if precond is None else precond
    for fmt in p.formats:
        if host is None:
            if profile:
                solver.profile_reset()
            _, r = solver.solve(dev["b"], dev["x0"], p.restart, p.rel_tol, max_iters or p.max_iters, fmt, precond=pc, reorth=reorth)
            if profile:
                r.prof = solver.profile_get()
        else:
            host["x"].copy_(host["x0"])
            r = solver.solve_host(host["row_ptr"], host["col_idx"], host["vals"], host["b"], host["x"], p.restart,
                                  p.rel_tol, max_iters or p.max_iters, fmt, precond=pc)
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


def _format_table(p, results_per_step, peak):
    """Per-format time to solution, iterations/s and whole-solve fraction of the HBM roofline (algorithmic bytes of every
    launch that ran / device time of the solve) from a list of {fmt: SolveResult}."""
    table = {}
    for fmt in p.formats:
        rs = [st[fmt] for st in results_per_step]
        t_ms = sum(r.solve_ms for r in rs) / len(rs)
        last = rs[-1]
        gbs = last.algorithmic_bytes / (last.solve_ms * 1e-3) / 1e9 if last.solve_ms > 0 else None
        table[fmt] = {"iters": last.iters, "restarts": last.restarts, "reorth_count": last.reorth_count,
                      "converged": bool(last.converged), "rel_res_true": last.rel_res_true,
                      "time_to_solution_ms": round(t_ms, 3), "us_per_iter": round(1e3 * t_ms / max(last.iters, 1), 2),
                      "iters_per_sec": round(last.iters / (t_ms * 1e-3), 1) if t_ms > 0 else None,
                      "whole_solve_GBps": round(gbs, 1) if gbs else None,
                      "whole_solve_frac_measured": round(gbs / peak, 4) if gbs else None,
                      "whole_solve_frac_nominal_8TBs": round(gbs / NOMINAL_HBM_GBS, 4) if gbs else None}
    t64 = table.get("fp64", {}).get("time_to_solution_ms")
    b64 = results_per_step[-1]["fp64"].algorithmic_bytes if "fp64" in table else None
    for fmt, d in table.items():
        d["speedup_vs_fp64"] = round(t64 / d["time_to_solution_ms"], 3) if t64 and d["time_to_solution_ms"] else None
        by = results_per_step[-1][fmt].algorithmic_bytes
        d["bytes_ratio_vs_fp64"] = round(b64 / by, 3) if b64 and by else None  # "in proportion to the bytes saved" (north_star)
    return table


def _other_config(Solver, local, name, precond, peak, max_iters=None, steps=2):
    """A per_config entry: `steps` solves per format (the first is the warm-up) of another BASELINE config."""
    import torch

    p = _make_problem(name)
    solver = Solver(local)
    try:
        solver.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
        dev = {"b": torch.as_tensor(p.b, device=solver.device), "x0": torch.as_tensor(p.x0, device=solver.device)}
        res = [_solve_all_formats(solver, p, dev, precond=precond, max_iters=max_iters) for _ in range(steps)][1:]
        tab = _format_table(p, res, peak)
        return {"n": p.A.n, "nnz": p.A.nnz, "restart": p.restart, "rel_tol": p.rel_tol, "precond": precond,
                "max_iters": max_iters or p.max_iters, "spmv_kernel": res[-1][p.formats[0]].spmv_kernel, "formats": tab}
    finally:
        solver.destroy()


def _c3_cpu_oracle(n, ks=(1, 10, 100), fmts=("fp32", "int16")):
    """CPU time of the oracle's multi-dot, update + norms and compress-store at the C3 size.
    The oracle's per-kernel references (long double accumulation), as they stand, on the host cores."""
    import numpy as np

    import oracle

    rng = np.random.default_rng(2)
    kmax = max(ks)
    V = rng.standard_normal((kmax, n)) / np.sqrt(n)
    w = rng.standard_normal(n)
    rows = []
    for fmt in fmts:
        t0 = time.perf_counter()
        P, sig = oracle.enc_basis(fmt, V)
        t_enc = (time.perf_counter() - t0) / kmax
        rows.append({"kernel": "compress-store (enc)", "format": fmt, "k": 1, "ms": round(1e3 * t_enc, 2)})
        for k in ks:
            h = np.zeros(k)
            t0 = time.perf_counter()
            oracle.ref_multidot(fmt, P[:k], sig[:k], w, k=k)
            t1 = time.perf_counter()
            oracle.ref_update(fmt, P[:k], sig[:k], h, w)
            t2 = time.perf_counter()
            rows.append({"kernel": "multidot", "format": fmt, "k": k, "ms": round(1e3 * (t1 - t0), 2)})
            rows.append({"kernel": "update+norms", "format": fmt, "k": k, "ms": round(1e3 * (t2 - t1), 2)})
    return {"n": n, "cores": oracle.num_threads(), "rows": rows}


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

    _log(f"building workload {args.workload}")
    p = _make_problem(args.workload)
    n, nnz = p.A.n, p.A.nnz
    solver = Solver(local)
    for o in args.opt:
        name, val = o.split("=")
        solver.set_option(name, int(val))
    solver.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
    dev = {"b": torch.as_tensor(p.b, device=solver.device), "x0": torch.as_tensor(p.x0, device=solver.device)}
    host = {k: torch.as_tensor(v).pin_memory() for k, v in
            (("row_ptr", p.A.row_ptr), ("col_idx", p.A.col_idx), ("vals", p.A.vals), ("b", p.b), ("x0", p.x0))}
    host["x"] = torch.empty(n, dtype=torch.float64).pin_memory()
    solver.set_option("profile", 0)  # no event brackets inside either timed region

    # -- device-resident arm: W warm-up steps, K timed steps --
    _log("warm-up")
    for _ in range(args.warmup):
        _solve_all_formats(solver, p, dev)
    sampler = ClockSampler(local)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = solver.launch_count()
    barrier()
    sampler.start()
    torch.cuda.profiler.start()  # cudaProfilerStart: `ncu --profile-from-start off` sees exactly the timed region (no-op otherwise)
    ev0.record()
    steps = [_solve_all_formats(solver, p, dev) for _ in range(args.steps)]
    ev1.record()
    barrier()
    torch.cuda.profiler.stop()
    clocks = sampler.stop()
    launches = solver.launch_count() - launches0
    ms = ev0.elapsed_time(ev1)
    iters = sum(r.iters for st in steps for r in st.values())
    _log(f"timed region done: {ms / args.steps:.1f} ms per step")

    # -- end-to-end arm: host buffers through cbgmres_solve_host, copies inside the timed region --
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
    _log(f"e2e region done: {1e3 * e_s / args.steps:.1f} ms per step")

    ms, e_ms, iters, e_iters, launches = aggregate_over_ranks(world, solver.device, ms, e_s * 1e3, iters, e_iters, launches)
    if rank != 0:
        solver.destroy()
        if world > 1:
            dist.destroy_process_group()
        return 0

    peak, peak_src = _peaks()
    per_format = _format_table(p, steps, peak)

    # -- separate pass, after both timed regions: per-kernel CUDA-event brackets (solve_host re-registered the matrix) --
    solver.set_matrix(p.A.row_ptr, p.A.col_idx, p.A.vals)
    solver.set_option("profile", PROFILE_EVERY)
    prof_step = _solve_all_formats(solver, p, dev, profile=True)
    solver.set_option("profile", 0)
    fam = {name: {"ms": 0.0, "bytes": 0.0, "launches": 0} for name in PROF_FAMILIES}
    kernels = []
    for fmt in p.formats:
        for name, d in prof_step[fmt].prof.items():
            for k in ("ms", "bytes", "launches"):
                fam[name][k] += d[k]
            if d["launches"]:
                gbs = d["bytes"] / (d["ms"] * 1e-3) / 1e9 if d["ms"] > 0 else None
                kernels.append({"kernel": name, "format": fmt, "launches": d["launches"], "ms": round(d["ms"], 3),
                                "avg_us": round(1e3 * d["ms"] / d["launches"], 2),
                                "GBps": round(gbs, 1) if gbs else None, "frac": round(gbs / peak, 4) if gbs else None,
                                "frac_nominal_8TBs": round(gbs / NOMINAL_HBM_GBS, 4) if gbs else None})
    total_prof_ms = sum(d["ms"] for d in fam.values()) or 1.0
    dom = max(fam, key=lambda k: fam[k]["ms"])
    d = fam[dom]
    achieved = d["bytes"] / (d["ms"] * 1e-3) / 1e9 if d["ms"] > 0 else 0.0
    # ncu dram__bytes_read + dram__bytes_write of this family per launch: the ratio traffic / algorithmic bytes of the
    # captured launches (profiles/ncu_traffic.csv, written by paper_2009_12101_b200/profsummary.py from the --set full
    # captures named in its `capture` column) applied to the average launch of this run
    traffic, traffic_src = None, None
    tpath = os.path.join(ROOT, TRAFFIC_CSV)
    if os.path.exists(tpath):
        import csv

        with open(tpath, newline="") as f:
            rows = {r["family"]: r for r in csv.DictReader(f)}
        if dom in rows and d["launches"]:
            traffic = round(float(rows[dom]["traffic_over_algorithmic"]) * d["bytes"] / d["launches"])
            traffic_src = {"file": TRAFFIC_CSV, "capture": rows[dom].get("capture"), "workload": rows[dom].get("workload"),
                           "ratio": float(rows[dom]["traffic_over_algorithmic"])}
    roofline = {"bound": "hbm", "kernel": dom, "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
                "frac": round(achieved / peak, 4), "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "frac_nominal_8TBs": round(achieved / NOMINAL_HBM_GBS, 4),
                "how": "algorithmic bytes of the family's bracketed launches / their summed CUDA-event durations, in a separate "
                       f"pass after the timed regions (brackets around every {PROFILE_EVERY}nd Arnoldi step)",
                "launches": d["launches"], "avg_launch_us": round(1e3 * d["ms"] / max(d["launches"], 1), 2),
                "algorithmic_bytes_per_launch": round(d["bytes"] / max(d["launches"], 1)),
                "share_of_step": round(d["ms"] / total_prof_ms, 4),
                "shares": {k: round(v["ms"] / total_prof_ms, 4) for k, v in fam.items()}}
    _log("profile pass done")

    extras = {}
    if world == 1 and not args.no_extras:
        from paper_2009_12101_b200 import cyclebench, microbench

        # -- Fig. 9: per-cycle time at a fixed iteration count, tolerance 0, this workload --
        rows = cyclebench.run(solver, p, MSWEEP, 3, list(p.formats))
        extras["msweep"] = {"workload": args.workload, "cycles": 3, "protocol": "full cycles of m steps, tolerance 0 (numerical effects ignored, PAPER.md:294)",
                            "rows": [{k: (round(v, 4) if isinstance(v, float) else v) for k, v in r.items()} for r in rows]}
        _log("msweep done")
        # -- the two-read regime of the paper's memop model (PAPER.md:116 assumes l.7 never fires): same workload, reorth = never --
        never = [_solve_all_formats(solver, p, dev, reorth="never") for _ in range(2)][1:]
        extras_never = {"n": n, "nnz": nnz, "restart": p.restart, "rel_tol": p.rel_tol, "precond": PRECOND, "reorth": "never",
                        "formats": _format_table(p, never, peak)}
        _log("reorth=never done")
        # -- C3 (BASELINE.json configs[2]): S2 / S3 / S3+S2' / S4 timed separately at n = 4,194,304 --
        rows = microbench.run(solver, C3_N, list(C3_KS), list(FORMATS), reps=10, flush=True)
        extras["c3"] = {"n": C3_N, "ks": list(C3_KS), "l2": "512 MB written between launches (nothing L2-resident)",
                        "reps": 10, "stat": "median", "peak_measured_GBps": peak,
                        "rows": [{"kernel": r["kernel"], "format": r["format"], "k": r["k"], "us": round(r["median_us"], 1),
                                  "GBps": round(r["GBps"]), "frac": round(r["GBps"] / peak, 3)} for r in rows]}
        _log("c3 done")
        solver.destroy()
        solver = None
        per_config = {args.workload + ("" if PRECOND == "none" else "+" + PRECOND): {
            "n": n, "nnz": nnz, "restart": p.restart, "rel_tol": p.rel_tol, "precond": PRECOND, "reorth": "cond", "formats": per_format},
            args.workload + " reorth=never": extras_never}
        for name, pc, bound in (("C1", "none", None), ("C2", "none", None), ("C4", "none", 500), ("C4", "jacobi", 1000),
                                ("C4", "block_jacobi4", 1000)):
            if name == args.workload and pc == PRECOND:
                continue
            per_config[name + ("" if pc == "none" else "+" + pc)] = _other_config(Solver, local, name, pc, peak, bound)
            _log(f"per_config {name} {pc} done")
        extras["per_config"] = per_config

    # -- the oracle on this box's host cores, bounded sample of the same workload --
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle

        REF = REF_ITERS[args.workload]
        c_it, c_s = _oracle_step(p, REF)
        cpu = {"value": c_it / c_s, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": _sample_text(p, REF), "seconds": round(c_s, 2)}
        if "c3" in extras:
            extras["c3"]["cpu_oracle"] = _c3_cpu_oracle(C3_N)
        _log("cpu baseline done")

    line = {
        "metric": METRIC, "value": iters / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "precond": PRECOND, "n": n, "nnz": nnz, "restart": p.restart, "rel_tol": p.rel_tol,
                   "max_iters": p.max_iters, "formats": list(p.formats), "reorth": "cond (eta = 1/sqrt 2)", "options": list(args.opt),
                   "step": "one solve to convergence per storage format",
                   "timed_region": "library event brackets off (profile = 0); roofline/kernels from a separate pass afterwards",
                   "l2": "no flush: the basis (0.8-3.3 GB on C5) + matrix (1.3 GB) exceed the 126 MB L2; reuse inside a solve is the workload's own",
                   "parallelism": f"{world} independent solves, one per GPU" if world > 1 else "1 GPU"},
        "iters_per_step": iters / args.steps / world,
        "e2e": {"value": e_iters / (e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e_ms / args.steps},
        "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
        "per_format": per_format, "kernels": kernels,
    }
    line.update(extras)
    print(json.dumps(line))
    if solver is not None:
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
    ap.add_argument("--workload", choices=tuple(WORKLOADS), default="C5")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip per_config, c3 and msweep")
    ap.add_argument("--precond", choices=("none", "jacobi", "block_jacobi4"), default="none")
    ap.add_argument("--opt", action="append", default=[], help="name=value for cbgmres_set_option (tuning experiments; repeatable)")
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
