"""Thin ctypes binding of include/cbgmres.h: argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libcbgmres.so; torch is used for device
memory and the stream.  There is no CPU fallback: if the library is missing or no CUDA device is
present, calls raise.  Method names mirror the C entry points (cbgmres_<name>).
"""
from __future__ import annotations

import ctypes as C
import math
import os
from dataclasses import dataclass

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("CBGMRES_LIB") or os.path.join(HERE, "libcbgmres.so")  # CBGMRES_LIB: another build of the same ABI

FORMATS = ("fp64", "fp32", "fp16", "int32", "int16")
FORMAT_CODE = {f: i for i, f in enumerate(FORMATS)}
FORMAT_BYTES = {"fp64": 8, "fp32": 4, "fp16": 2, "int32": 4, "int16": 2}
REORTH_CODE = {"never": 0, "cond": 1, "always": 2}
PRECOND_CODE = {"none": 0, "jacobi": 1, "block_jacobi4": 2}
STATUS = {0: "OK", 1: "E_INVALID", 2: "E_NOMATRIX", 3: "E_WORKSPACE", 4: "E_CUDA", 5: "E_NONFINITE",
          16: "NOT_CONVERGED"}
MAX_RESTART = 512

EXPORTS = (
    "cbgmres_create", "cbgmres_set_matrix", "cbgmres_workspace_bytes", "cbgmres_solve",
    "cbgmres_workspace_bytes_host", "cbgmres_solve_host", "cbgmres_destroy", "cbgmres_last_error",
    "cbgmres_set_option", "cbgmres_launch_count", "cbgmres_k_compress", "cbgmres_k_decode", "cbgmres_k_multidot",
    "cbgmres_k_update", "cbgmres_k_update_multidot", "cbgmres_k_store", "cbgmres_k_spmv", "cbgmres_profile_get", "cbgmres_profile_reset",
    "cbgmres_k_bj4_setup", "cbgmres_k_store_bj4", "cbgmres_noalloc_setup", "cbgmres_k_multidot_noalloc",
    "cbgmres_noalloc_last_error",
)
NOALLOC_MAX_K = 128  # CBGMRES_NOALLOC_MAX_K
PROF_FAMILIES = ("spmv", "multidot", "update", "store", "xupdate", "residual", "update_multidot")


class Params(C.Structure):
    _fields_ = [("restart", C.c_int32), ("max_iters", C.c_int32), ("format", C.c_int32), ("reorth", C.c_int32),
                ("rel_tol", C.c_double), ("eta", C.c_double), ("h_res_history", C.c_void_p),
                ("res_history_cap", C.c_int32), ("precond", C.c_int32)]


class Result(C.Structure):
    _fields_ = [("iters", C.c_int32), ("restarts", C.c_int32), ("reorth_count", C.c_int32), ("breakdown", C.c_int32),
                ("converged", C.c_int32), ("spmv_kernel", C.c_int32), ("rel_res_recurrence", C.c_double),
                ("rel_res_true", C.c_double), ("b_norm", C.c_double), ("solve_ms", C.c_double),
                ("algorithmic_bytes", C.c_double)]


class CbgmresError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"cbgmres status {code} ({STATUS.get(code, '?')}): {msg}")
        self.code = code


_lib = None


def load_library(path: str = LIB_PATH):
    """dlopen libcbgmres.so and declare the prototypes.  Raises if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: run `python -m paper_2009_12101_b200.build` (there is no CPU fallback)")
    L = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    L.cbgmres_create.argtypes = [C.POINTER(vp), C.c_int, vp]
    L.cbgmres_set_matrix.argtypes = [vp, i64, i64, vp, vp, vp]
    L.cbgmres_workspace_bytes.argtypes = [vp, C.POINTER(Params), C.POINTER(C.c_size_t)]
    L.cbgmres_solve.argtypes = [vp, vp, vp, C.POINTER(Params), vp, C.c_size_t, C.POINTER(Result)]
    L.cbgmres_workspace_bytes_host.argtypes = [vp, i64, i64, C.POINTER(Params), C.POINTER(C.c_size_t)]
    L.cbgmres_solve_host.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, C.POINTER(Params), vp, C.c_size_t,
                                     C.POINTER(Result)]
    L.cbgmres_destroy.argtypes = [vp]
    L.cbgmres_last_error.argtypes = [vp]
    L.cbgmres_last_error.restype = C.c_char_p
    L.cbgmres_set_option.argtypes = [vp, C.c_char_p, i64]
    L.cbgmres_launch_count.argtypes = [vp]
    L.cbgmres_launch_count.restype = i64
    L.cbgmres_k_compress.argtypes = [vp, i32, i64, vp, vp, vp]
    L.cbgmres_k_decode.argtypes = [vp, i32, i64, vp, vp, vp]
    L.cbgmres_k_multidot.argtypes = [vp, i32, i64, i64, i32, vp, vp, vp, vp]
    L.cbgmres_k_update.argtypes = [vp, i32, i64, i64, i32, vp, vp, vp, vp, vp, vp]
    L.cbgmres_k_update_multidot.argtypes = [vp, i32, i64, i64, i32, vp, vp, vp, vp, vp, vp, vp]
    L.cbgmres_k_store.argtypes = [vp, i32, i64, vp, dbl, dbl, vp, vp, vp]
    L.cbgmres_k_spmv.argtypes = [vp, vp, vp, vp]
    L.cbgmres_k_bj4_setup.argtypes = [vp, vp]
    L.cbgmres_k_store_bj4.argtypes = [vp, i32, i64, vp, dbl, dbl, vp, vp, vp, vp]
    L.cbgmres_profile_get.argtypes = [vp, i32, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(i64)]
    L.cbgmres_profile_reset.argtypes = [vp]
    L.cbgmres_noalloc_setup.argtypes = [i32]
    L.cbgmres_k_multidot_noalloc.argtypes = [i32, vp, i32, i64, i64, i32, vp, vp, vp, vp]
    L.cbgmres_noalloc_last_error.argtypes = []
    L.cbgmres_noalloc_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("cbgmres_last_error", "cbgmres_launch_count", "cbgmres_noalloc_last_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _torch():
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("paper_2009_12101_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
    return torch


def payload_dtype(fmt: str):
    torch = _torch()
    return {"fp64": torch.float64, "fp32": torch.float32, "fp16": torch.float16, "int32": torch.int32,
            "int16": torch.int16}[fmt]


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def k_multidot_noalloc(fmt: str, V, scales, w, h, n: int | None = None, k: int | None = None):
    """cbgmres_k_multidot_noalloc: h[:k] <- V[:k]^T w with the library's static device scratch -- no handle, no
    allocation inside the call (the caller passes the output `h`, a device tensor of >= k doubles).  Enqueues on
    torch's current stream of V's device.  k > NOALLOC_MAX_K raises CbgmresError (E_INVALID)."""
    torch = _torch()
    L = load_library()
    k = V.shape[0] if k is None else k
    n = w.numel() if n is None else n
    dev = V.device.index if V.device.index is not None else torch.cuda.current_device()
    stream = torch.cuda.current_stream(dev).cuda_stream
    rc = L.cbgmres_k_multidot_noalloc(dev, C.c_void_p(stream), FORMAT_CODE[fmt], n, V.shape[1], k, _ptr(V), _ptr(scales),
                                      _ptr(w), _ptr(h))
    if rc != 0:
        raise CbgmresError(rc, (L.cbgmres_noalloc_last_error() or b"").decode())
    return h[:k]


@dataclass
class SolveResult:
    status: int
    iters: int
    restarts: int
    reorth_count: int
    breakdown: int
    converged: bool
    spmv_kernel: int
    rel_res_recurrence: float
    rel_res_true: float
    b_norm: float
    solve_ms: float
    algorithmic_bytes: float = 0.0
    rec_history: np.ndarray | None = None


class Solver:
    """One cbgmres handle bound to a device and (by default) torch's current stream."""

    def __init__(self, device: int = 0, stream=None):
        torch = _torch()
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.h = C.c_void_p()
        rc = self.lib.cbgmres_create(C.byref(self.h), device, C.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            raise CbgmresError(rc, "cbgmres_create failed")
        self._keep = []
        self._ws = None
        self.n = 0
        self.nnz = 0

    # -- plumbing ---------------------------------------------------------------------------------
    def _check(self, rc: int, allow=(0,)):
        if rc not in allow:
            raise CbgmresError(rc, self.lib.cbgmres_last_error(self.h).decode())
        return rc

    def destroy(self):
        if self.h:
            self.lib.cbgmres_destroy(self.h)
            self.h = C.c_void_p()
            self._keep = []
            self._ws = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_option(self, name: str, value: int):
        self._check(self.lib.cbgmres_set_option(self.h, name.encode(), int(value)))

    def launch_count(self) -> int:
        return int(self.lib.cbgmres_launch_count(self.h))

    def profile_reset(self):
        self._check(self.lib.cbgmres_profile_reset(self.h))

    def profile_get(self) -> dict:
        """{family: {"ms", "bytes", "launches"}} accumulated since profile_reset (option "profile" = 1)."""
        out = {}
        for i, name in enumerate(PROF_FAMILIES):
            ms, by, cnt = C.c_double(0.0), C.c_double(0.0), C.c_int64(0)
            self._check(self.lib.cbgmres_profile_get(self.h, i, C.byref(ms), C.byref(by), C.byref(cnt)))
            out[name] = {"ms": ms.value, "bytes": by.value, "launches": int(cnt.value)}
        return out

    def _dev(self, a, dtype):
        torch = _torch()
        if isinstance(a, torch.Tensor):
            t = a.to(device=self.device, dtype=dtype)
        else:
            t = torch.as_tensor(np.ascontiguousarray(a), dtype=dtype, device=self.device)
        return t.contiguous()

    def _params(self, restart, rel_tol, max_iters, fmt, reorth, eta, hist=None, precond="none") -> Params:
        p = Params(int(restart), int(max_iters), FORMAT_CODE[fmt], REORTH_CODE[reorth], float(rel_tol), float(eta),
                   None, 0, PRECOND_CODE[precond])
        if hist is not None:
            p.h_res_history = hist.ctypes.data
            p.res_history_cap = hist.shape[0]
        return p

    def _workspace(self, nbytes: int):
        torch = _torch()
        if self._ws is None or self._ws.numel() < nbytes:
            self._ws = None
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        return self._ws

    # -- the four calls of the problem statement ---------------------------------------------------
    def set_matrix(self, row_ptr, col_idx, vals):
        torch = _torch()
        rp = self._dev(row_ptr, torch.int32)
        ci = self._dev(col_idx, torch.int32)
        va = self._dev(vals, torch.float64)
        self.n, self.nnz = rp.numel() - 1, ci.numel()
        self._keep = [rp, ci, va]  # BORROWED by the library until the next set_matrix / destroy
        self._check(self.lib.cbgmres_set_matrix(self.h, self.n, self.nnz, _ptr(rp), _ptr(ci), _ptr(va)))

    def workspace_bytes(self, restart, fmt, history_cap=0, precond="none") -> int:
        hist = np.empty(history_cap) if history_cap else None
        p = self._params(restart, 0.0, 0, fmt, "cond", 0.0, hist, precond)
        out = C.c_size_t(0)
        self._check(self.lib.cbgmres_workspace_bytes(self.h, C.byref(p), C.byref(out)))
        return int(out.value)

    def solve(self, b, x0, restart: int, rel_tol: float, max_iters: int, fmt: str = "fp64", reorth: str = "cond",
              eta: float = 0.0, history: bool = False, precond: str = "none"):
        """Returns (x device tensor, SolveResult).  x0 is not modified.  precond = "jacobi": right
        preconditioner M = diag(A); "block_jacobi4": M = the 4 x 4 diagonal blocks."""
        torch = _torch()
        bt = self._dev(b, torch.float64)
        xt = self._dev(x0, torch.float64).clone()
        hist = np.full(max(int(max_iters), 1), np.nan) if history else None
        p = self._params(restart, rel_tol, max_iters, fmt, reorth, eta, hist, precond)
        need = C.c_size_t(0)
        self._check(self.lib.cbgmres_workspace_bytes(self.h, C.byref(p), C.byref(need)))
        ws = self._workspace(need.value)
        res = Result()
        rc = self.lib.cbgmres_solve(self.h, _ptr(bt), _ptr(xt), C.byref(p), _ptr(ws), ws.numel(), C.byref(res))
        self._check(rc, allow=(0, 16))
        return xt, self._result(rc, res, hist)

    def solve_host(self, row_ptr, col_idx, vals, b, x, restart, rel_tol, max_iters, fmt="fp64", reorth="cond",
                   eta=0.0, precond="none"):
        """End-to-end call with HOST buffers (numpy arrays or pinned CPU tensors); x is overwritten."""
        def hp(a):
            return C.c_void_p(a.data_ptr()) if hasattr(a, "data_ptr") else C.c_void_p(a.ctypes.data)

        n, nnz = len(row_ptr) - 1, len(col_idx)
        p = self._params(restart, rel_tol, max_iters, fmt, reorth, eta, None, precond)
        need = C.c_size_t(0)
        self._check(self.lib.cbgmres_workspace_bytes_host(self.h, n, nnz, C.byref(p), C.byref(need)))
        ws = self._workspace(need.value)
        res = Result()
        rc = self.lib.cbgmres_solve_host(self.h, n, nnz, hp(row_ptr), hp(col_idx), hp(vals), hp(b), hp(x), C.byref(p),
                                         _ptr(ws), ws.numel(), C.byref(res))
        self._keep = []
        self.n, self.nnz = n, nnz
        self._check(rc, allow=(0, 16))
        return self._result(rc, res, None)

    @staticmethod
    def _result(rc, res, hist):
        return SolveResult(rc, res.iters, res.restarts, res.reorth_count, res.breakdown, bool(res.converged),
                           res.spmv_kernel, res.rel_res_recurrence, res.rel_res_true, res.b_norm, res.solve_ms,
                           res.algorithmic_bytes, hist[: res.iters] if hist is not None else None)

    # -- per-kernel hooks -----------------------------------------------------------------------------
    def k_compress(self, fmt: str, v):
        torch = _torch()
        vt = self._dev(v, torch.float64)
        payload = torch.empty(vt.numel(), dtype=payload_dtype(fmt), device=self.device)
        scale = torch.zeros(1, dtype=torch.float64, device=self.device)
        self._check(self.lib.cbgmres_k_compress(self.h, FORMAT_CODE[fmt], vt.numel(), _ptr(vt), _ptr(payload),
                                                _ptr(scale)))
        return payload, scale

    def k_decode(self, fmt: str, payload, scale):
        torch = _torch()
        out = torch.empty(payload.numel(), dtype=torch.float64, device=self.device)
        self._check(self.lib.cbgmres_k_decode(self.h, FORMAT_CODE[fmt], payload.numel(), _ptr(payload), _ptr(scale),
                                              _ptr(out)))
        return out

    def k_multidot(self, fmt: str, V, scales, w, n: int | None = None, k: int | None = None):
        """V: payload tensor [kmax, ld]; scales [kmax] fp64 (or None for the floating-point formats)."""
        torch = _torch()
        k = V.shape[0] if k is None else k
        n = w.numel() if n is None else n
        h = torch.empty(max(k, 1), dtype=torch.float64, device=self.device)
        self._check(self.lib.cbgmres_k_multidot(self.h, FORMAT_CODE[fmt], n, V.shape[1], k, _ptr(V), _ptr(scales),
                                                _ptr(w), _ptr(h)))
        return h[:k]

    def k_update(self, fmt: str, V, scales, h, w, n: int | None = None):
        """In place on w.  Returns (nrm2, amax) as a 2-element device tensor."""
        torch = _torch()
        n = w.numel() if n is None else n
        out = torch.zeros(2, dtype=torch.float64, device=self.device)
        self._check(self.lib.cbgmres_k_update(self.h, FORMAT_CODE[fmt], n, V.shape[1], h.numel(), _ptr(V),
                                              _ptr(scales), _ptr(h), _ptr(w), C.c_void_p(out.data_ptr()),
                                              C.c_void_p(out.data_ptr() + 8)))
        return out

    def k_update_multidot(self, fmt: str, V, scales, h, w, n: int | None = None):
        """Fused pass: w -= V h in place, then u = V^T w.  Returns (u, (nrm2, amax) device tensor)."""
        torch = _torch()
        n = w.numel() if n is None else n
        out = torch.zeros(2, dtype=torch.float64, device=self.device)
        u = torch.empty(h.numel(), dtype=torch.float64, device=self.device)
        self._check(self.lib.cbgmres_k_update_multidot(self.h, FORMAT_CODE[fmt], n, V.shape[1], h.numel(), _ptr(V),
                                                       _ptr(scales), _ptr(h), _ptr(w), _ptr(u),
                                                       C.c_void_p(out.data_ptr()), C.c_void_p(out.data_ptr() + 8)))
        return u, out

    def k_store(self, fmt: str, w, hnorm: float, amax: float, payload_col=None, v_out=None):
        torch = _torch()
        n = w.numel()
        if payload_col is None:
            payload_col = torch.empty(n, dtype=payload_dtype(fmt), device=self.device)
        if v_out is None:
            v_out = torch.empty(n, dtype=torch.float64, device=self.device)
        scale = torch.zeros(1, dtype=torch.float64, device=self.device)
        self._check(self.lib.cbgmres_k_store(self.h, FORMAT_CODE[fmt], n, _ptr(w), float(hnorm), float(amax),
                                             _ptr(payload_col), _ptr(scale), _ptr(v_out)))
        return payload_col, scale, v_out

    def k_bj4_setup(self):
        """Inverted 4 x 4 diagonal blocks of the registered matrix, device tensor [ceil(n/4), 4, 4]."""
        torch = _torch()
        inv = torch.empty(((self.n + 3) // 4, 4, 4), dtype=torch.float64, device=self.device)
        self._check(self.lib.cbgmres_k_bj4_setup(self.h, _ptr(inv)))
        return inv

    def k_store_bj4(self, fmt: str, w, hnorm: float, amax: float, inv):
        """S4 with block-Jacobi(4): returns (payload, scale, z = M^-1 v)."""
        torch = _torch()
        n = w.numel()
        payload = torch.empty(n, dtype=payload_dtype(fmt), device=self.device)
        z = torch.empty(n, dtype=torch.float64, device=self.device)
        scale = torch.zeros(1, dtype=torch.float64, device=self.device)
        self._check(self.lib.cbgmres_k_store_bj4(self.h, FORMAT_CODE[fmt], n, _ptr(w), float(hnorm), float(amax),
                                                 _ptr(inv), _ptr(payload), _ptr(scale), _ptr(z)))
        return payload, scale, z

    def k_spmv(self, v, w=None, want_norm: bool = True):
        torch = _torch()
        if w is None:
            w = torch.empty(self.n, dtype=torch.float64, device=self.device)
        nrm = torch.zeros(1, dtype=torch.float64, device=self.device) if want_norm else None
        self._check(self.lib.cbgmres_k_spmv(self.h, _ptr(v), _ptr(w), _ptr(nrm)))
        return w, nrm


DEFAULT_ETA = 1.0 / math.sqrt(2.0)
