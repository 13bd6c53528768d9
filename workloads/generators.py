"""Synthetic stand-ins for the paper's SuiteSparse problems (Table 1).

The paper measures on 49 SuiteSparse matrices with n 5e5..3.5e6 and 4..82 nonzeros per row;
those files are not available here, so BASELINE.json's five seeded configs stand in
(readings Q15-Q19).  All draws use numpy.random.default_rng(seed) (PCG64)
in the order documented in each function.  CSR = fp64 values + int32 indices, columns
ascending inside each row (one integer per nonzero plus n+1 row pointers).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

CONFIG_NAMES = ("C1", "C2", "C4", "C5")


@dataclass
class CSR:
    n: int
    row_ptr: np.ndarray  # int32 [n+1]
    col_idx: np.ndarray  # int32 [nnz]
    vals: np.ndarray     # float64 [nnz]

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])

    def to_scipy(self):
        import scipy.sparse as sp

        return sp.csr_matrix((self.vals, self.col_idx, self.row_ptr), shape=(self.n, self.n))


@dataclass
class Problem:
    name: str
    A: CSR
    b: np.ndarray
    x0: np.ndarray
    restart: int
    rel_tol: float
    max_iters: int
    formats: tuple
    meta: dict = field(default_factory=dict)


def _stencil_csr(shape, offsets, coeffs=None):
    """CSR pattern of a stencil on a lexicographic grid (x fastest), Dirichlet truncation.

    offsets: list of (dz, dy, dx) sorted so that the flattened column offset ascends.
    coeffs : per-offset constant coefficient (or None -> caller fills values).
    Returns row_ptr, col_idx, off_id (which stencil offset each stored entry is).
    """
    nz, ny, nx = shape
    n = nz * ny * nx
    idx = np.arange(n, dtype=np.int64)
    ix = idx % nx
    iy = (idx // nx) % ny
    iz = idx // (nx * ny)
    noff = len(offsets)
    mask = np.empty((n, noff), dtype=bool)
    flat = np.empty(noff, dtype=np.int64)
    for o, (dz, dy, dx) in enumerate(offsets):
        mask[:, o] = (
            (ix + dx >= 0) & (ix + dx < nx) & (iy + dy >= 0) & (iy + dy < ny) & (iz + dz >= 0) & (iz + dz < nz)
        )
        flat[o] = (dz * ny + dy) * nx + dx
    assert np.all(np.diff(flat) > 0), "offsets must be given in ascending column order"
    counts = mask.sum(axis=1)
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(counts, out=row_ptr[1:])
    rows, offs = np.nonzero(mask)  # row-major order == CSR order
    col_idx = (rows + flat[offs]).astype(np.int32)
    assert row_ptr[-1] < 2**31
    return n, row_ptr.astype(np.int32), col_idx, offs.astype(np.int8)


def laplace2d_5pt(nx: int, ny: int) -> CSR:
    """C1: 5-point Laplacian, diagonal 4, neighbours -1, Dirichlet."""
    offsets = [(0, -1, 0), (0, 0, -1), (0, 0, 0), (0, 0, 1), (0, 1, 0)]
    n, rp, ci, off = _stencil_csr((1, ny, nx), offsets)
    coef = np.array([-1.0, -1.0, 4.0, -1.0, -1.0])
    return CSR(n, rp, ci, coef[off])


def convdiff3d_7pt(nx: int, ny: int, nz: int) -> CSR:
    """C2: 7-point convection-diffusion, diagonal 6, -1.3 on the (i - stride) neighbour and
    -0.7 on the (i + stride) neighbour of every axis (reading Q16: "-1 +- 0.3 upwind")."""
    offsets = [(-1, 0, 0), (0, -1, 0), (0, 0, -1), (0, 0, 0), (0, 0, 1), (0, 1, 0), (1, 0, 0)]
    n, rp, ci, off = _stencil_csr((nz, ny, nx), offsets)
    coef = np.array([-1.3, -1.3, -1.3, 6.0, -0.7, -0.7, -0.7])
    return CSR(n, rp, ci, coef[off])


def stencil3d_27pt(nx: int, rng: np.random.Generator, ny: int | None = None, nz: int | None = None) -> CSR:
    """C5: 27-point stencil, diagonal exactly 26, every stored off-diagonal -1 + 0.05*u with
    u ~ U[-1,1] drawn independently per entry in CSR order (reading Q18)."""
    ny = nx if ny is None else ny
    nz = nx if nz is None else nz
    offsets = [(dz, dy, dx) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1)]
    n, rp, ci, off = _stencil_csr((nz, ny, nx), offsets)
    diag = off == 13
    vals = np.empty(ci.shape[0], dtype=np.float64)
    u = rng.uniform(-1.0, 1.0, size=int((~diag).sum()))
    vals[~diag] = -1.0 + 0.05 * u
    vals[diag] = 26.0
    return CSR(n, rp, ci, vals)


def powerlaw_rows(n: int, rng: np.random.Generator, mean_shift: float = 3.139, kmax: int = 2000) -> CSR:
    """C4: off-diagonal count L_i ~ p(k) ∝ (k + 3.139)^-2 on k = 1..2000 (shifted Zipf with
    mean 20, reading Q17), uniform random columns != i, duplicates merged keeping the first
    drawn value, values U[-1,1], diagonal = 1.1 * sum |off-diagonals|, columns ascending.

    Draw order: (1) n uniforms for the row lengths, (2) sum(L) integers for the columns,
    (3) sum(L) uniforms for the values.
    """
    k = np.arange(1, kmax + 1, dtype=np.float64)
    p = (k + mean_shift) ** -2.0
    cdf = np.cumsum(p / p.sum())
    L = np.searchsorted(cdf, rng.random(n), side="right") + 1
    L = np.minimum(L, min(kmax, n - 1)).astype(np.int64)
    total = int(L.sum())
    rows = np.repeat(np.arange(n, dtype=np.int64), L)
    cols = rng.integers(0, n - 1, size=total, dtype=np.int64)
    cols += cols >= rows  # uniform on [0, n) \ {i}
    v = rng.uniform(-1.0, 1.0, size=total)
    key = rows * n + cols
    order = np.argsort(key, kind="stable")
    key = key[order]
    v = v[order]
    first = np.ones(total, dtype=bool)
    first[1:] = key[1:] != key[:-1]
    key = key[first]
    v = v[first]
    r_off = key // n
    abssum = np.bincount(r_off, weights=np.abs(v), minlength=n)
    dkey = np.arange(n, dtype=np.int64) * (n + 1)
    key = np.concatenate([key, dkey])
    v = np.concatenate([v, 1.1 * abssum])
    order = np.argsort(key, kind="stable")
    key = key[order]
    v = v[order]
    r = key // n
    c = key - r * n
    counts = np.bincount(r, minlength=n)
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(counts, out=row_ptr[1:])
    assert row_ptr[-1] < 2**31
    return CSR(n, row_ptr.astype(np.int32), c.astype(np.int32), np.ascontiguousarray(v))


ALL_FORMATS = ("fp64", "fp32", "fp16", "int32", "int16")


def make_config(name: str, grid: int | None = None, n: int | None = None) -> Problem:
    """BASELINE.json configs C1, C2, C4, C5.  `grid` / `n` shrink the problem for parity tests
    (same recipe, same seeds); None gives the full size."""
    if name == "C1":
        g = 64 if grid is None else grid
        A = laplace2d_5pt(g, g)
        rng = np.random.default_rng(0)
        xstar = rng.uniform(-1.0, 1.0, size=A.n)
        b = A.to_scipy() @ xstar  # input construction only (library routine)
        return Problem("C1", A, b, np.zeros(A.n), 50, 1e-10, 3000, ("fp64", "fp32"), {"grid": g, "xstar": xstar})
    if name == "C2":
        g = 100 if grid is None else grid
        A = convdiff3d_7pt(g, g, g)
        rng = np.random.default_rng(1)
        b = rng.uniform(-1.0, 1.0, size=A.n)
        return Problem("C2", A, b, np.zeros(A.n), 100, 1e-8, 20000, ALL_FORMATS, {"grid": g})
    if name == "C4":
        nn = 2_000_000 if n is None else n
        rng = np.random.default_rng(3)
        A = powerlaw_rows(nn, rng)
        b = rng.uniform(-1.0, 1.0, size=A.n)
        return Problem("C4", A, b, np.zeros(A.n), 50, 1e-9, 5000, ALL_FORMATS, {"n": nn})
    if name == "C5":
        g = 160 if grid is None else grid
        rng = np.random.default_rng(4)
        A = stencil3d_27pt(g, rng)
        b = rng.uniform(-1.0, 1.0, size=A.n)
        return Problem("C5", A, b, np.zeros(A.n), 100, 1e-8, 5000, ALL_FORMATS, {"grid": g})
    raise ValueError(f"unknown config {name!r}")


def ortho_basis(n: int, k: int, seed: int = 2):
    """C3: V = thin-QR Q factor of an n x k standard-normal matrix, then w standard normal,
    both from default_rng(seed) in that order.  Returns (V [k, n] C-contiguous: one basis vector
    per row, i.e. each vector contiguous in memory, and w [n])."""
    rng = np.random.default_rng(seed)
    G = rng.standard_normal((n, k))
    Q, _ = np.linalg.qr(G, mode="reduced")
    w = rng.standard_normal(n)
    return np.ascontiguousarray(Q.T), w


def random_dense_system(n: int, seed: int, density: float = 1.0):
    """Tiny well-conditioned nonsymmetric system for the dense-solve pins: A = n*I + G with
    G standard normal (optionally sparsified), b standard normal.  Returns (CSR, dense A, b)."""
    rng = np.random.default_rng(seed)
    G = rng.standard_normal((n, n))
    if density < 1.0:
        G *= rng.random((n, n)) < density
    Ad = G + n * np.eye(n)
    b = rng.standard_normal(n)
    import scipy.sparse as sp

    S = sp.csr_matrix(Ad)
    S.sort_indices()
    A = CSR(n, S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(np.float64))
    return A, Ad, b
