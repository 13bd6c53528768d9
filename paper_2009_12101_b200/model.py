"""Algorithmic-bytes model of the hot path (host logic only).

Each function returns the bytes the METHOD must move through HBM for one launch, from the paper's
memop model (eq. 4.1/4.2) extended with the vector traffic the paper assumes
cached -- SURVEY.md §8(d).  n = rows, nnz = nonzeros, k = basis vectors touched,
B = bytes per stored basis entry, f = index bytes / value bytes.
"""
from __future__ import annotations

FORMAT_BYTES = {"fp64": 8, "fp32": 4, "fp16": 2, "int32": 4, "int16": 2}


def spmv_bytes(n: int, nnz: int) -> int:
    """S1: 12 nnz (fp64 value + int32 column) + 4(n+1) row pointers + 8n (v once) + 8n (w)."""
    return 12 * nnz + 4 * (n + 1) + 16 * n


def multidot_bytes(n: int, k: int, fmt: str) -> int:
    """S2: k stored vectors + w once."""
    return k * n * FORMAT_BYTES[fmt] + 8 * n


def update_bytes(n: int, k: int, fmt: str) -> int:
    """S3: k stored vectors + w read and written."""
    return k * n * FORMAT_BYTES[fmt] + 16 * n


def store_bytes(n: int, fmt: str) -> int:
    """S4: read w, write the payload, write the fp64 v for the next SpMV."""
    return (16 + FORMAT_BYTES[fmt]) * n


def arnoldi_step_bytes(n: int, nnz: int, j: int, fmt: str, reorth: bool = False) -> int:
    """One Arnoldi step at basis size j (S1 + S2 + S3 [+ S2' + S3'] + S4)."""
    orth = multidot_bytes(n, j, fmt) + update_bytes(n, j, fmt)
    return spmv_bytes(n, nnz) + orth * (2 if reorth else 1) + store_bytes(n, fmt)


def memop_ratio_cycle(m: int, s: float, f: float = 0.5) -> float:
    """Eq. (4.2): memops of the two GEMVs over memops of the SpMV per restart
    cycle, m / (s (1 + f) + f), with the vectors assumed cached."""
    return m / (s * (1.0 + f) + f)


def memop_crossover_s(m: int, f: float = 0.5) -> float:
    """The nonzeros-per-row ratio at which eq. (4.2) equals 1."""
    return (m - f) / (1.0 + f)
