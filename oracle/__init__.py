"""ctypes front end of the CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2009_12101_b200/ and imports nothing from it.
Every function is a thin marshalling layer over oracle/cbgmres_oracle.c, where the arithmetic
and the PAPER.md citations live.
"""
from __future__ import annotations

import ctypes as C
import math
from dataclasses import dataclass, field

import numpy as np

from .build import build as _build

FORMATS = ("fp64", "fp32", "fp16", "int32", "int16")
FORMAT_CODE = {f: i for i, f in enumerate(FORMATS)}
PAYLOAD_DTYPE = {"fp64": np.float64, "fp32": np.float32, "fp16": np.float16, "int32": np.int32, "int16": np.int16}
REORTH_CODE = {"never": 0, "cond": 1, "always": 2}

_lib = None


class _Params(C.Structure):
    _fields_ = [("restart", C.c_int32), ("max_iters", C.c_int32), ("format", C.c_int32), ("reorth", C.c_int32),
                ("rel_tol", C.c_double), ("eta", C.c_double)]


class _Result(C.Structure):
    _fields_ = [("iters", C.c_int32), ("restarts", C.c_int32), ("reorth_count", C.c_int32), ("breakdown", C.c_int32),
                ("converged", C.c_int32), ("pad_", C.c_int32), ("rel_res_recurrence", C.c_double),
                ("rel_res_true", C.c_double), ("b_norm", C.c_double)]


class _Capture(C.Structure):
    _fields_ = [("cycle", C.c_int32), ("k", C.c_int32), ("beta", C.c_double), ("Vhat", C.c_void_p),
                ("Vfp64", C.c_void_p), ("Hbar", C.c_void_p), ("y", C.c_void_p), ("g", C.c_void_p),
                ("reorth_log", C.c_void_p), ("omega", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        L.orc_set_num_threads.restype = None
        L.orc_format_bytes.restype = C.c_int64
        L.orc_format_bytes.argtypes = [C.c_int]
        L.orc_enc.argtypes = [C.c_int, C.c_int64, C.c_void_p, C.c_void_p, C.POINTER(C.c_double)]
        L.orc_dec.argtypes = [C.c_int, C.c_int64, C.c_void_p, C.c_double, C.c_void_p]
        L.orc_spmv.argtypes = [C.c_int64] + [C.c_void_p] * 5
        L.orc_spmv.restype = None
        L.orc_nrm2.restype = C.c_double
        L.orc_nrm2.argtypes = [C.c_int64, C.c_void_p]
        L.orc_amax.restype = C.c_double
        L.orc_amax.argtypes = [C.c_int64, C.c_void_p]
        L.orc_ref_multidot.argtypes = [C.c_int, C.c_int64, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_void_p]
        L.orc_ref_multidot.restype = None
        L.orc_ref_update.argtypes = [C.c_int, C.c_int64, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_ref_update.restype = None
        L.orc_ref_spmv.argtypes = [C.c_int64] + [C.c_void_p] * 6
        L.orc_ref_spmv.restype = None
        L.orc_gmres.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                C.POINTER(_Params), C.POINTER(_Result), C.c_void_p, C.c_int32, C.c_void_p, C.c_int32,
                                C.POINTER(_Capture)]
        L.orc_gmres.restype = C.c_int
        L.orc_gmres_m.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                  C.POINTER(_Params), C.POINTER(_Result), C.c_void_p, C.c_int32, C.c_void_p, C.c_int32,
                                  C.POINTER(_Capture)]
        L.orc_gmres_m.restype = C.c_int
        L.orc_jacobi_diag.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_jacobi_diag.restype = None
        L.orc_block_jacobi4.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_block_jacobi4.restype = None
        L.orc_apply_minv.argtypes = [C.c_int, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        L.orc_apply_minv.restype = None
        L.orc_gmres_p.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                                  C.c_void_p, C.POINTER(_Params), C.POINTER(_Result), C.c_void_p, C.c_int32, C.c_void_p,
                                  C.c_int32, C.POINTER(_Capture)]
        L.orc_gmres_p.restype = C.c_int
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(t: int) -> None:
    """Thread count of later calls: changes only the order of dot()'s block sums (reading Q11)."""
    lib().orc_set_num_threads(int(t))


def format_bytes(fmt: str) -> int:
    return int(lib().orc_format_bytes(FORMAT_CODE[fmt]))


def enc(fmt: str, v):
    """enc: fp64[n] -> (payload in the storage dtype, sigma)."""
    v = _f64(v)
    out = np.empty(v.shape[0], dtype=PAYLOAD_DTYPE[fmt])
    s = C.c_double(0.0)
    rc = lib().orc_enc(FORMAT_CODE[fmt], v.shape[0], _p(v), _p(out), C.byref(s))
    assert rc == 0
    return out, s.value


def dec(fmt: str, payload, sigma: float = 1.0) -> np.ndarray:
    payload = np.ascontiguousarray(payload, dtype=PAYLOAD_DTYPE[fmt])
    out = np.empty(payload.shape[0], dtype=np.float64)
    rc = lib().orc_dec(FORMAT_CODE[fmt], payload.shape[0], _p(payload), float(sigma), _p(out))
    assert rc == 0
    return out


def enc_basis(fmt: str, V):
    """Encode k fp64 vectors (rows of V [k, n]) -> payload [k, n] and sigma [k]."""
    V = _f64(V)
    k, n = V.shape
    P = np.empty((k, n), dtype=PAYLOAD_DTYPE[fmt])
    sig = np.empty(k, dtype=np.float64)
    for c in range(k):
        P[c], sig[c] = enc(fmt, V[c])
    return P, sig


def spmv(A, x) -> np.ndarray:
    x = _f64(x)
    y = np.empty(A.n, dtype=np.float64)
    lib().orc_spmv(A.n, _p(A.row_ptr), _p(A.col_idx), _p(A.vals), _p(x), _p(y))
    return y


def nrm2(a) -> float:
    a = _f64(a)
    return float(lib().orc_nrm2(a.shape[0], _p(a)))


def amax(a) -> float:
    a = _f64(a)
    return float(lib().orc_amax(a.shape[0], _p(a)))


def ref_multidot(fmt: str, P, sigma, w, k=None) -> np.ndarray:
    """h_c = sum_i dec(P)[c, i] w_i with long double accumulation.  P: [kmax, ld] payload."""
    P = np.ascontiguousarray(P, dtype=PAYLOAD_DTYPE[fmt])
    sigma = _f64(sigma)
    w = _f64(w)
    k = P.shape[0] if k is None else k
    h = np.empty(k, dtype=np.float64)
    lib().orc_ref_multidot(FORMAT_CODE[fmt], w.shape[0], P.shape[1], k, _p(P), _p(sigma), _p(w), _p(h))
    return h


def ref_update(fmt: str, P, sigma, h, w):
    """Returns (w - dec(P)^T-combination, sum w^2, max |w|), long double accumulation."""
    P = np.ascontiguousarray(P, dtype=PAYLOAD_DTYPE[fmt])
    sigma = _f64(sigma)
    h = _f64(h)
    w = _f64(w).copy()
    s, a = C.c_double(0.0), C.c_double(0.0)
    lib().orc_ref_update(FORMAT_CODE[fmt], w.shape[0], P.shape[1], h.shape[0], _p(P), _p(sigma), _p(h), _p(w),
                         C.byref(s), C.byref(a))
    return w, s.value, a.value


def ref_spmv(A, x):
    x = _f64(x)
    y = np.empty(A.n, dtype=np.float64)
    ra = np.empty(A.n, dtype=np.float64)
    lib().orc_ref_spmv(A.n, _p(A.row_ptr), _p(A.col_idx), _p(A.vals), _p(x), _p(y), _p(ra))
    return y, ra


@dataclass
class OracleResult:
    x: np.ndarray
    iters: int
    restarts: int
    reorth_count: int
    breakdown: int
    converged: bool
    rel_res_recurrence: float
    rel_res_true: float
    b_norm: float
    rec_history: np.ndarray
    expl_history: np.ndarray
    capture: dict = field(default_factory=dict)


def jacobi_diag(A) -> np.ndarray:
    """M = diag(A) of the scalar Jacobi preconditioner; absent / zero entries give 1."""
    d = np.empty(A.n)
    lib().orc_jacobi_diag(A.n, _p(A.row_ptr), _p(A.col_idx), _p(A.vals), _p(d))
    return d


PRECOND_CODE = {"none": 0, "jacobi": 1, "block_jacobi4": 2}


def block_jacobi4(A) -> np.ndarray:
    """The inverted 4 x 4 diagonal blocks of A, [ceil(n/4), 4, 4] (orc_block_jacobi4)."""
    inv = np.empty(((A.n + 3) // 4, 4, 4))
    lib().orc_block_jacobi4(A.n, _p(A.row_ptr), _p(A.col_idx), _p(A.vals), _p(inv))
    return inv


def apply_minv(precond: str, pdata, v) -> np.ndarray:
    """z = M^-1 v as the solver applies it in Fig. 1 l.3 / l.17 (pdata: jacobi_diag / block_jacobi4 output)."""
    v = _f64(v)
    z = np.empty_like(v)
    pd = _f64(pdata) if pdata is not None else None
    lib().orc_apply_minv(PRECOND_CODE[precond], _p(pd) if pd is not None else None, v.shape[0], _p(v), _p(z))
    return z


def gmres(A, b, x0, restart: int, rel_tol: float, max_iters: int, fmt: str = "fp64", reorth: str = "cond",
          eta: float = 1.0 / math.sqrt(2.0), capture_cycle: int | None = None, precond: str = "none") -> OracleResult:
    """Restarted CB-GMRES (Fig. 1).  See orc_gmres_p in cbgmres_oracle.c.
    precond = "jacobi": right preconditioner M = diag(A) (Fig. 1 l.3 and l.17);
    precond = "block_jacobi4": M = the 4 x 4 diagonal blocks of A."""
    if precond not in PRECOND_CODE:
        raise ValueError(precond)
    b = _f64(b)
    x = _f64(x0).copy()
    n, m = A.n, restart
    prm = _Params(restart, max_iters, FORMAT_CODE[fmt], REORTH_CODE[reorth], rel_tol, eta)
    res = _Result()
    rec = np.full(max(max_iters, 1), np.nan)
    expl = np.full(max_iters + 2, np.nan)
    cap = None
    bufs = {}
    if capture_cycle is not None:
        bufs = dict(Vhat=np.zeros((m + 1, n)), Vfp64=np.zeros((m + 1, n)), Hbar=np.zeros((m, m + 1)),
                    y=np.zeros(m), g=np.zeros(m + 1), reorth_log=np.zeros(m, dtype=np.int32), omega=np.zeros(m))
        cap = _Capture(capture_cycle, 0, 0.0, *[bufs[k].ctypes.data for k in ("Vhat", "Vfp64", "Hbar", "y", "g",
                                                                              "reorth_log", "omega")])
    pdata = jacobi_diag(A) if precond == "jacobi" else block_jacobi4(A) if precond == "block_jacobi4" else None
    rc = lib().orc_gmres_p(n, _p(A.row_ptr), _p(A.col_idx), _p(A.vals), PRECOND_CODE[precond],
                           _p(pdata) if pdata is not None else None,
                           _p(b), _p(x), C.byref(prm), C.byref(res), _p(rec), rec.shape[0], _p(expl), expl.shape[0],
                           C.byref(cap) if cap else None)
    if rc != 0:
        raise RuntimeError(f"orc_gmres failed with {rc}")
    capture = {}
    if cap is not None:
        k = cap.k
        capture = dict(k=k, beta=cap.beta, Vhat=bufs["Vhat"][: k + 1], Vfp64=bufs["Vfp64"][: k + 1],
                       Hbar=bufs["Hbar"].T[: k + 1, :k].copy(), y=bufs["y"][:k], g=bufs["g"][: k + 1],
                       reorth_log=bufs["reorth_log"][:k].copy(), omega=bufs["omega"][:k].copy())
    return OracleResult(x, res.iters, res.restarts, res.reorth_count, res.breakdown, bool(res.converged),
                        res.rel_res_recurrence, res.rel_res_true, res.b_norm, rec[: res.iters],
                        expl[~np.isnan(expl)], capture)
