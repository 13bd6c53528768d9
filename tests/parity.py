"""The ONE checker of iteration-count parity between a CUDA solve and the oracle, shared by the GPU
tests and by __graft_entry__.smoke() (test infrastructure: imports oracle/, never the CUDA package).

BASELINE.json north_star: "iteration counts to convergence agree within +-2 %".  That is the default
and the only bar for fp64 storage.  With a QUANTISED basis the store is a discontinuous map: a last-bit
difference in one inner product flips a rounding decision at the store, and from there the two residual
histories decorrelate at the level of the format's unit roundoff (reading Q11).  The oracle
shows the same sensitivity against ITSELF when only the order of its dot()'s block sums changes (other
thread counts; nothing else about it changes).  So, for quantised formats only:

  * strict:  |gpu - oracle| <= max(2, 2 %)                                   -- always tried first;
  * band:    min(draws) - 2 % <= gpu <= max(draws) + 2 % over the oracle's own counts ("draws": the base run plus
             the runs at other thread counts) -- for any quantised format whose oracle draws differ among themselves;
  * chaotic: the band extended by two sample standard deviations of the draws -- ONLY for the 16-bit formats
             (the paper's own Table 2 puts the variance of their iteration overhead at 62.3 / 46.95 against 0.01
             for the 32-bit formats), only with at least MIN_DRAWS_FOR_SD draws (a further draw
             falls outside the range of five with probability 1/3, so a range of few draws is no band), and never wider
             than +-MAX_REL_HALF_WIDTH around the draws' median unless the case is listed in KNOWN_WIDE.  These cases pin
             nothing about kernel quality; tests/test_gpu_step_parity.py (teacher-forced single Arnoldi steps,
             where nothing is chaotic) is what discriminates there.

Every use of a band is printed with all counts, so the test log (-s) shows which cases needed which rule.
"""
from __future__ import annotations

import numpy as np

import oracle

SIXTEEN_BIT = ("fp16", "int16")
MIN_DRAWS_FOR_SD = 10
MAX_REL_HALF_WIDTH = 0.15
# (case label, format) pairs whose oracle draws scatter by tens of per cent (Q11): 16-bit storage on the
# Jacobi- / block-Jacobi-preconditioned power-law matrix stagnates near tau for hundreds of steps (oracle draws
# 731 .. 1125 for int16).  Only these may exceed MAX_REL_HALF_WIDTH.
KNOWN_WIDE = {("C4J-40k", "int16"), ("C4B-40k", "int16")}
SPREAD_THREADS = (1, 2, 3, 5)
CHAOTIC_THREADS = (4, 6, 7, 9, 10, 11, 12)  # on top of SPREAD_THREADS: 12 draws with the base run


def tol2(c: float) -> float:
    return max(2.0, 0.02 * c)


def strict_ok(gpu_iters: int, ref_iters: int) -> bool:
    return abs(gpu_iters - ref_iters) <= tol2(ref_iters)


def band_of(draws, allow_sd: bool):
    """[lo, hi] admitted for the GPU's count given the oracle's own counts."""
    lo, hi = min(draws), max(draws)
    ext_lo, ext_hi = tol2(lo), tol2(hi)
    if allow_sd and len(draws) >= MIN_DRAWS_FOR_SD:
        sd = float(np.std(draws, ddof=1))
        ext_lo, ext_hi = max(ext_lo, 2 * sd), max(ext_hi, 2 * sd)
    return lo - ext_lo, hi + ext_hi


def oracle_draws(run, threads) -> list:
    """Iteration counts of `run()` (a closure calling oracle.gmres) at the given thread counts."""
    base = oracle.num_threads()
    out = []
    try:
        for t in threads:
            oracle.set_num_threads(t)
            out.append(run().iters)
    finally:
        oracle.set_num_threads(base)
    return out


def check_iters(gpu_iters: int, ref_iters: int, fmt: str, label: str, draws=None, run=None) -> str:
    """Asserts iteration-count parity; returns which rule admitted the count ("strict", "band", "chaotic").
    draws: the oracle's own counts at other summation orders if already known (cached full-size runs);
    run:   else a closure that re-runs the oracle (reduced sizes), called only if the strict rule fails."""
    if strict_ok(gpu_iters, ref_iters):
        return "strict"
    assert fmt != "fp64", f"{label} fp64: gpu {gpu_iters} vs oracle {ref_iters}: fp64 storage has no quantisation, no band"
    if draws is None:
        assert run is not None, f"{label} {fmt}: gpu {gpu_iters} vs oracle {ref_iters} and no oracle spread available"
        draws = oracle_draws(run, SPREAD_THREADS)
    draws = [ref_iters] + list(draws)
    lo, hi = band_of(draws, allow_sd=False)
    if lo <= gpu_iters <= hi:
        print(f"[parity] {label} {fmt}: gpu {gpu_iters}, oracle draws {sorted(draws)} -> band [{lo:.1f}, {hi:.1f}]")
        return "band"
    assert fmt in SIXTEEN_BIT, (label, fmt, gpu_iters, sorted(draws), "32-bit storage: no statistical band")
    if len(draws) < MIN_DRAWS_FOR_SD and run is not None:
        draws += oracle_draws(run, CHAOTIC_THREADS)
    assert len(draws) >= MIN_DRAWS_FOR_SD, (label, fmt, gpu_iters, sorted(draws), "too few oracle draws for a statistical band")
    lo, hi = band_of(draws, allow_sd=True)
    med = float(np.median(draws))
    if (label, fmt) not in KNOWN_WIDE:
        lo, hi = max(lo, med * (1 - MAX_REL_HALF_WIDTH)), min(hi, med * (1 + MAX_REL_HALF_WIDTH))
    print(f"[parity] {label} {fmt}: gpu {gpu_iters}, oracle draws {sorted(draws)} -> chaotic [{lo:.1f}, {hi:.1f}]")
    assert lo <= gpu_iters <= hi, (label, fmt, gpu_iters, sorted(draws), "chaotic")
    return "chaotic"
