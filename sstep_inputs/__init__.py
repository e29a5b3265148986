"""Seeded synthetic inputs for the s-step PCG hot path (arxiv 2501.03743).

This module only *generates problems*: CSR matrices of 3-D Poisson-like
stencils and right-hand sides, in the shapes BASELINE.json's configs name.
It holds none of the solver's arithmetic (no CSR SpMV, no dot products, no
CG): the right-hand side b = A x* is evaluated by applying the *stencil
definition on the grid* (numpy slicing), which is the problem statement
itself ("discretization of the Poisson equation on a 3D cube,
with Dirichlet boundary conditions"), not the CSR kernel under test.

Both the oracle tests and the CUDA parity tests / bench.py import from here;
neither the oracle nor the CUDA library does.

Conventions:
  * grid index i = x + N*(y + N*z), x fastest;
  * CSR is 0-based, int32 indices, fp64 values, columns ascending in a row;
  * random numbers come from numpy.random.default_rng(seed).
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "poisson7", "poisson7_box", "apply_poisson7_box", "poisson27", "varcoef7", "varcoef_cells", "apply_poisson7", "apply_poisson27",
    "apply_varcoef7", "symmetric_permute", "random_spd_csr", "random_structure_spd_csr", "STRUCTURE_KINDS", "poisson1d",
    "make_config", "CONFIG_NAMES",
]


# --------------------------------------------------------------------------
# constant-coefficient stencils
# --------------------------------------------------------------------------
def _grid_coords(N, z0: int, z1: int):
    """x, y, z coordinates (int32) of the rows in the z-slab [z0, z1); N is an int (cube) or (nx, ny, nz)."""
    nx, ny, _ = (N, N, N) if isinstance(N, int) else N
    zz, yy, xx = np.meshgrid(np.arange(z0, z1, dtype=np.int32),
                             np.arange(ny, dtype=np.int32),
                             np.arange(nx, dtype=np.int32), indexing="ij")
    return xx.ravel(), yy.ravel(), zz.ravel()


def _stencil_csr(N, offsets, diag_value: float, off_value: float, slab: int = 16):
    """CSR of a constant-coefficient stencil on an N^3 grid (or an (nx, ny, nz) box) with homogeneous
    Dirichlet boundaries (neighbours outside the box are dropped).

    `offsets` is a list of (dx, dy, dz) in ascending column order.
    Built slab by slab in z to bound the temporary memory.
    """
    nx, ny, nz = (N, N, N) if isinstance(N, int) else N
    n = nx * ny * nz
    counts = np.empty(n, dtype=np.int32)
    col_parts, val_parts = [], []
    for z0 in range(0, nz, slab):
        z1 = min(nz, z0 + slab)
        x, y, z = _grid_coords((nx, ny, nz), z0, z1)
        rows = x.astype(np.int64) + nx * (y.astype(np.int64) + ny * z.astype(np.int64))
        m = rows.size
        cols = np.empty((m, len(offsets)), dtype=np.int32)
        mask = np.empty((m, len(offsets)), dtype=bool)
        vals = np.empty((m, len(offsets)), dtype=np.float64)
        for k, (dx, dy, dz) in enumerate(offsets):
            ok = ((x + dx >= 0) & (x + dx < nx) & (y + dy >= 0) & (y + dy < ny)
                  & (z + dz >= 0) & (z + dz < nz))
            mask[:, k] = ok
            cols[:, k] = (rows + dx + nx * (dy + ny * dz)).astype(np.int32)
            vals[:, k] = diag_value if (dx == 0 and dy == 0 and dz == 0) else off_value
        counts[rows[0]:rows[0] + m] = mask.sum(axis=1)
        col_parts.append(cols[mask])
        val_parts.append(vals[mask])
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(counts, out=rowptr[1:])
    assert rowptr[-1] < 2**31
    return rowptr.astype(np.int32), np.concatenate(col_parts), np.concatenate(val_parts)


_OFF7 = [(0, 0, -1), (0, -1, 0), (-1, 0, 0), (0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)]
_OFF27 = [(dx, dy, dz) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1)]


def poisson7(N: int):
    """7-point 3-D Poisson: 6 on the diagonal, -1 to the six face neighbours,
    Dirichlet (BASELINE.json configs 1, 2, 4; PAPER.md:259 — the paper says
    "five-point", its 514-iteration count fixes the 7-point stencil)."""
    return _stencil_csr(N, _OFF7, 6.0, -1.0)


def poisson7_box(nx: int, ny: int, nz: int):
    """The same 7-point operator on an nx x ny x nz box: a z-slab of the cube keeps the plane size and the
    nnz/row of the full problem (used for bounded CPU-baseline samples of config 4)."""
    return _stencil_csr((nx, ny, nz), _OFF7, 6.0, -1.0)


def apply_poisson7_box(nx: int, ny: int, nz: int, x: np.ndarray) -> np.ndarray:
    u = x.reshape(nz, ny, nx)
    out = 6.0 * u
    out[1:, :, :] -= u[:-1, :, :]
    out[:-1, :, :] -= u[1:, :, :]
    out[:, 1:, :] -= u[:, :-1, :]
    out[:, :-1, :] -= u[:, 1:, :]
    out[:, :, 1:] -= u[:, :, :-1]
    out[:, :, :-1] -= u[:, :, 1:]
    return out.ravel()


def poisson27(N: int):
    """27-point 3-D stencil: 26 on the diagonal, -1 to all 26 neighbours,
    Dirichlet (BASELINE.json config 3)."""
    return _stencil_csr(N, _OFF27, 26.0, -1.0)


def apply_poisson7(N: int, x: np.ndarray) -> np.ndarray:
    """(A x) for the 7-point stencil, evaluated on the grid by its definition."""
    u = x.reshape(N, N, N)  # [z, y, x]
    out = 6.0 * u
    out[1:, :, :] -= u[:-1, :, :]
    out[:-1, :, :] -= u[1:, :, :]
    out[:, 1:, :] -= u[:, :-1, :]
    out[:, :-1, :] -= u[:, 1:, :]
    out[:, :, 1:] -= u[:, :, :-1]
    out[:, :, :-1] -= u[:, :, 1:]
    return out.ravel()


def apply_poisson27(N: int, x: np.ndarray) -> np.ndarray:
    """(A x) for the 27-point stencil: 27*x minus the 3x3x3 box sum."""
    u = x.reshape(N, N, N)
    p = np.zeros((N + 2, N + 2, N + 2))
    p[1:-1, 1:-1, 1:-1] = u
    box = np.zeros_like(u)
    for dz in range(3):
        for dy in range(3):
            for dx in range(3):
                box += p[dz:dz + N, dy:dy + N, dx:dx + N]
    return (27.0 * u - box).ravel()


# --------------------------------------------------------------------------
# variable-coefficient diffusion (config 5)
# --------------------------------------------------------------------------
def _harmonic(a, b):
    return 2.0 * a * b / (a + b)


def _varcoef_faces(N: int, k: np.ndarray):
    """Face coefficients of the 7-point finite-volume diffusion operator.

    Interior faces: harmonic mean of the two cell coefficients.  A Dirichlet
    boundary face takes the cell's own k (ghost cell with equal k, reading
    A17 in SURVEY.md §8c).  Returns six [z,y,x] arrays: xm, xp, ym, yp, zm, zp.
    """
    kk = k.reshape(N, N, N)
    xm = kk.copy(); xp = kk.copy(); ym = kk.copy(); yp = kk.copy(); zm = kk.copy(); zp = kk.copy()
    hx = _harmonic(kk[:, :, :-1], kk[:, :, 1:]); xp[:, :, :-1] = hx; xm[:, :, 1:] = hx
    hy = _harmonic(kk[:, :-1, :], kk[:, 1:, :]); yp[:, :-1, :] = hy; ym[:, 1:, :] = hy
    hz = _harmonic(kk[:-1, :, :], kk[1:, :, :]); zp[:-1, :, :] = hz; zm[1:, :, :] = hz
    return xm, xp, ym, yp, zm, zp


def varcoef_cells(N: int, seed: int, sigma: float = 1.5) -> np.ndarray:
    """Per-cell diffusion coefficient k = exp(N(0, sigma^2)) (config 5)."""
    return np.exp(np.random.default_rng(seed).normal(0.0, sigma, N * N * N))


def varcoef7(N: int, k: np.ndarray):
    """CSR of the variable-coefficient 7-point operator in natural ordering:
    a_ii = sum of the six face coefficients, a_ij = -face coefficient."""
    n = N * N * N
    xm, xp, ym, yp, zm, zp = (f.ravel() for f in _varcoef_faces(N, k))
    diag = ((((xm + xp) + ym) + yp) + zm) + zp
    x, y, z = _grid_coords(N, 0, N)
    rows = np.arange(n, dtype=np.int64)
    # ascending column order: z-1, y-1, x-1, diag, x+1, y+1, z+1
    entries = [(-N * N, z > 0, -zm), (-N, y > 0, -ym), (-1, x > 0, -xm), (0, None, diag),
               (1, x < N - 1, -xp), (N, y < N - 1, -yp), (N * N, z < N - 1, -zp)]
    cols = np.empty((n, 7), dtype=np.int32)
    vals = np.empty((n, 7), dtype=np.float64)
    mask = np.ones((n, 7), dtype=bool)
    for j, (off, ok, v) in enumerate(entries):
        cols[:, j] = (rows + off).astype(np.int32)
        vals[:, j] = v
        if ok is not None:
            mask[:, j] = ok
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(mask.sum(axis=1), out=rowptr[1:])
    return rowptr.astype(np.int32), cols[mask], vals[mask]


def apply_varcoef7(N: int, k: np.ndarray, x: np.ndarray) -> np.ndarray:
    """(A x) of the variable-coefficient operator by its flux definition:
    sum over faces of coef * (u_cell - u_neighbour), boundary neighbour = 0."""
    xm, xp, ym, yp, zm, zp = _varcoef_faces(N, k)
    u = x.reshape(N, N, N)
    p = np.zeros((N + 2, N + 2, N + 2))
    p[1:-1, 1:-1, 1:-1] = u
    out = xm * (u - p[1:-1, 1:-1, 0:N]) + xp * (u - p[1:-1, 1:-1, 2:N + 2])
    out += ym * (u - p[1:-1, 0:N, 1:-1]) + yp * (u - p[1:-1, 2:N + 2, 1:-1])
    out += zm * (u - p[0:N, 1:-1, 1:-1]) + zp * (u - p[2:N + 2, 1:-1, 1:-1])
    return out.ravel()


def symmetric_permute(rowptr, colidx, vals, perm: np.ndarray):
    """A' = Pi A Pi^T with A'[i, j] = A[perm[i], perm[j]]; columns re-sorted in
    every row (reading A16: a row-only permutation would destroy symmetry)."""
    n = rowptr.size - 1
    inv = np.empty(n, dtype=np.int64)
    inv[perm] = np.arange(n, dtype=np.int64)
    counts = np.diff(rowptr.astype(np.int64))
    new_counts = counts[perm]
    new_rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(new_counts, out=new_rowptr[1:])
    nnz = int(new_rowptr[-1])
    # position of every new entry in the old arrays
    src = np.repeat(rowptr[:-1].astype(np.int64)[perm] - new_rowptr[:-1], new_counts) + np.arange(nnz, dtype=np.int64)
    new_cols = inv[colidx[src]]
    new_vals = vals[src]
    new_rows = np.repeat(np.arange(n, dtype=np.int64), new_counts)
    order = np.argsort(new_rows * n + new_cols, kind="stable")
    return new_rowptr.astype(np.int32), new_cols[order].astype(np.int32), new_vals[order]


# --------------------------------------------------------------------------
# tiny problems for the oracle pins
# --------------------------------------------------------------------------
def poisson1d(n: int):
    """tridiag(-1, 2, -1), Dirichlet: eigenvalues 2 - 2cos(k pi/(n+1))."""
    rowptr = [0]; cols = []; vals = []
    for i in range(n):
        if i > 0:
            cols.append(i - 1); vals.append(-1.0)
        cols.append(i); vals.append(2.0)
        if i < n - 1:
            cols.append(i + 1); vals.append(-1.0)
        rowptr.append(len(cols))
    return (np.array(rowptr, dtype=np.int32), np.array(cols, dtype=np.int32),
            np.array(vals, dtype=np.float64))


def random_spd_csr(n: int, density: float, seed: int, max_row: int | None = None):
    """Random sparse symmetric, strictly diagonally dominant (hence spd) matrix
    with an irregular row-length distribution; returns (rowptr, colidx, vals, dense).
    If max_row is given a few rows are made long (up to max_row entries)."""
    rng = np.random.default_rng(seed)
    B = np.zeros((n, n))
    m = rng.random((n, n)) < density
    B[m] = rng.uniform(-1.0, 1.0, int(m.sum()))
    if max_row:
        for i in rng.choice(n, size=max(1, n // 50), replace=False):
            js = rng.choice(n, size=min(n, max_row), replace=False)
            B[i, js] = rng.uniform(-1.0, 1.0, js.size)
    A = np.triu(B, 1)
    A = A + A.T
    A[np.arange(n), np.arange(n)] = np.abs(A).sum(axis=1) + rng.uniform(0.5, 1.5, n)
    rowptr = np.zeros(n + 1, dtype=np.int64)
    nzmask = A != 0.0
    np.cumsum(nzmask.sum(axis=1), out=rowptr[1:])
    cols = np.nonzero(nzmask)[1].astype(np.int32)
    return rowptr.astype(np.int32), cols, A[nzmask], A


STRUCTURE_KINDS = ("banded", "uniform_lengths", "stencil_long_rows", "box7", "box27", "power_law", "near_diagonal")


def random_structure_spd_csr(seed: int, kind: str | None = None, n: int | None = None):
    """Seeded symmetric, strictly diagonally dominant (hence spd) CSR matrix whose SPARSITY STRUCTURE is drawn from one of
    STRUCTURE_KINDS -- row lengths from 1 to thousands, banded or scattered columns, sizes from 1 row to 3e5 rows that are
    deliberately not multiples of any tile -- for the random-structure parity tests (every SpMV kernel, lane count and
    tile shape must either take the matrix and be right, or refuse it at setup).  Off-diagonal values U[-1, 0) (an
    M-matrix pattern like the paper's discretisations), diagonal = factor * sum|off-diagonal| + U[0.01, 1], constant over
    the rows with probability 0.3 where the structure allows it.  Returns (rowptr, colidx, vals, kind, n)."""
    rng = np.random.default_rng([seed, 0x5717])
    if kind is None:
        kind = STRUCTURE_KINDS[int(rng.integers(0, len(STRUCTURE_KINDS)))]
    if n is None:
        n = int(rng.choice([1, 2, 31, 32, 33, 255, 256, 257, 1000, 4097, 20000, 65537, 150001, 300000]))

    def band(offsets):
        offsets = np.array(sorted({int(o) for o in offsets if 0 < abs(int(o)) < n}), dtype=np.int64)
        rr = [np.arange(max(0, -o), min(n, n - o), dtype=np.int64) for o in offsets]
        return (np.concatenate(rr) if rr else np.zeros(0, np.int64),
                np.concatenate([r + o for r, o in zip(rr, offsets)]) if rr else np.zeros(0, np.int64))

    if kind == "banded":
        rows, cols = band(rng.integers(-min(n - 1, 3000), min(n - 1, 3000) + 1, int(rng.integers(0, 20))) if n > 1 else [])
    elif kind == "uniform_lengths":
        lens = rng.integers(0, int(rng.integers(1, 33)) + 1, n)
        rows = np.repeat(np.arange(n, dtype=np.int64), lens)
        cols = rng.integers(0, n, rows.size)
    elif kind == "stencil_long_rows":
        rows, cols = band([-1, 1])
        for i in rng.choice(n, size=min(n, 5), replace=False):
            js = rng.choice(n, size=int(rng.integers(1, min(n, 6000) + 1)), replace=False)
            rows = np.concatenate([rows, np.full(js.size, i, np.int64)]); cols = np.concatenate([cols, js])
    elif kind in ("box7", "box27"):
        lo, hi = (1, 40) if kind == "box7" else (2, 30)
        nx, ny, nz = (int(rng.integers(lo, hi)) for _ in range(3))
        n = nx * ny * nz
        i = np.arange(n, dtype=np.int64)
        x, y, z = i % nx, (i // nx) % ny, i // (nx * ny)
        rr, cc = [], []
        for dz in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dx in (-1, 0, 1):
                    if (dx, dy, dz) == (0, 0, 0) or (kind == "box7" and abs(dx) + abs(dy) + abs(dz) != 1):
                        continue
                    ok = (x + dx >= 0) & (x + dx < nx) & (y + dy >= 0) & (y + dy < ny) & (z + dz >= 0) & (z + dz < nz)
                    rr.append(i[ok]); cc.append(i[ok] + dx + nx * (dy + ny * dz))
        rows = np.concatenate(rr) if rr else np.zeros(0, np.int64)
        cols = np.concatenate(cc) if cc else np.zeros(0, np.int64)
    elif kind == "power_law":
        lens = np.minimum(np.minimum(n, 2000), np.maximum(0, (rng.pareto(1.2, n) * 2).astype(np.int64)))
        rows = np.repeat(np.arange(n, dtype=np.int64), lens)
        cols = rng.integers(0, n, rows.size)
    elif kind == "near_diagonal":
        k = n // 2 if n > 3 else 0
        rows, cols = rng.integers(0, n, k), rng.integers(0, n, k)
    else:
        raise ValueError(f"unknown structure kind {kind!r}")
    # symmetric pattern without the diagonal, one entry per (row, col)
    keep = rows != cols
    rows, cols = rows[keep], cols[keep]
    key = np.unique(np.concatenate([rows * n + cols, cols * n + rows]))
    rows, cols = key // n, key % n
    upper = rows < cols
    w = np.zeros(key.size)
    w[upper] = rng.uniform(-1.0, 0.0, int(upper.sum())) - 1e-3
    # the mirrored entry takes the same value: (c, r) sits at the position of key c * n + r
    w[np.searchsorted(key, cols[upper] * n + rows[upper])] = w[upper]
    offsum = np.bincount(rows, weights=np.abs(w), minlength=n)
    diag = offsum * rng.uniform(1.0, 1.3) + rng.uniform(0.01, 1.0, n)
    if rng.random() < 0.3:
        diag = np.full(n, float(diag.max()))
    allr = np.concatenate([rows, np.arange(n, dtype=np.int64)])
    allc = np.concatenate([cols, np.arange(n, dtype=np.int64)])
    allv = np.concatenate([w, diag])
    order = np.lexsort((allc, allr))
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(np.bincount(allr, minlength=n), out=rowptr[1:])
    return rowptr.astype(np.int32), allc[order].astype(np.int32), allv[order], kind, n


# --------------------------------------------------------------------------
# BASELINE.json configs
# --------------------------------------------------------------------------
CONFIG_NAMES = {
    1: "poisson7_32_s2", 2: "poisson7_128_s4", 3: "poisson27_160_s4",
    4: "poisson7_320_sweep", 5: "varcoef7_256_perm_s8", 6: "paper_poisson7_250_rhs1",
}


def make_config(cfg: int, N: int | None = None, s: int | None = None) -> dict:
    """Inputs of BASELINE.json config `cfg` (1-5) or the paper's own problem (6).

    `N` overrides the grid edge (parity tests run the same recipe at sizes the
    oracle finishes in seconds); `s` overrides the block size.  Returns a dict
    with rowptr, colidx, vals, b, x0 (None means zeros), xstar (or None), s,
    rtol, maxit, N, n, nnz, name.
    """
    if cfg == 1:
        N = N or 32; rp, ci, v = poisson7(N)
        xs = np.random.default_rng(0).uniform(-1.0, 1.0, N ** 3)
        b = apply_poisson7(N, xs); s_, rtol, maxit = 2, 1e-6, 2000
    elif cfg == 2:
        N = N or 128; rp, ci, v = poisson7(N)
        xs = np.random.default_rng(1).uniform(-1.0, 1.0, N ** 3)
        b = apply_poisson7(N, xs); s_, rtol, maxit = 4, 1e-8, 2000
    elif cfg == 3:
        N = N or 160; rp, ci, v = poisson27(N)
        xs = None
        b = np.random.default_rng(2).uniform(-1.0, 1.0, N ** 3); s_, rtol, maxit = 4, 1e-8, 2000
    elif cfg == 4:
        N = N or 320; rp, ci, v = poisson7(N)
        xs = np.random.default_rng(3).uniform(-1.0, 1.0, N ** 3)
        b = apply_poisson7(N, xs); s_, rtol, maxit = 4, 1e-8, 2000
    elif cfg == 5:
        N = N or 256
        k = varcoef_cells(N, 4)
        rp, ci, v = varcoef7(N, k)
        perm = np.random.default_rng(5).permutation(N ** 3)
        rp, ci, v = symmetric_permute(rp, ci, v, perm)
        xs = None
        b = np.random.default_rng(6).uniform(-1.0, 1.0, N ** 3); s_, rtol, maxit = 8, 1e-6, 2000
    elif cfg == 6:  # the paper's own workload
        N = N or 250; rp, ci, v = poisson7(N)
        xs = None
        b = np.ones(N ** 3); s_, rtol, maxit = 1, 1e-6, 2000
    else:
        raise ValueError(f"unknown config {cfg}")
    return dict(name=CONFIG_NAMES[cfg], cfg=cfg, N=N, n=N ** 3, nnz=int(rp[-1]), rowptr=rp, colidx=ci,
                vals=v, b=b, x0=None, xstar=xs, s=s or s_, rtol=rtol, maxit=maxit)
