"""Seeded synthetic SPD systems for AMP-PCG (arXiv 2505.04155) parity tests and benchmarks.

Recipe source: BASELINE.json ``configs`` (five synthetic systems) and SURVEY.md §8(d)
"Synthetic inputs"; the small dense systems are the paper's self-contained examples
(PAPER.md:48-53 Ex 1, :445-449 Ex 4, :473-481 Ex 6, :549-554 Ex 9, :570 Ex 10).

Everything here is input construction only: a counter-based RNG, stencil/graph assembly
into CSR (sorted columns, natural x-fastest ordering), and ``b = A x*`` through
scipy.sparse (a library mat-vec used to *define the input*, not part of the solver
under test).  No PCG arithmetic, no rounding emulation, no precision logic lives here.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, Dict, Optional, Sequence, Tuple

import numpy as np

BASE_SEED = 20250504  # seed_c = BASE_SEED + c

_U64 = np.uint64
_GOLD = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)


def _mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on uint64 arrays (wrapping arithmetic)."""
    z = np.asarray(z, dtype=_U64)
    z = (z ^ (z >> _U64(30))) * _M1
    z = (z ^ (z >> _U64(27))) * _M2
    return z ^ (z >> _U64(31))


def uniform01(seed: int, stream: int, idx: np.ndarray) -> np.ndarray:
    """Counter-based U[0,1) with 53 random bits: a pure function of (seed, stream, idx)."""
    with np.errstate(over="ignore"):
        key = _mix64(np.array([(seed * 0x2545F4914F6CDD1D + stream * 0x9E3779B97F4A7C15 + 1) % (1 << 64)], dtype=_U64))
        z = _mix64(key + np.asarray(idx, dtype=_U64) * _GOLD)
    return (z >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _normal(seed: int, stream: int, idx: np.ndarray) -> np.ndarray:
    """Box-Muller N(0,1) from two counter-based uniforms."""
    u1 = 1.0 - uniform01(seed, 2 * stream, idx)  # (0,1]
    u2 = uniform01(seed, 2 * stream + 1, idx)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


@dataclass
class CSRSystem:
    """One SPD system ``A x = b`` in CSR (int32 indices, float64 values, sorted columns)."""

    name: str
    n: int
    rowptr: np.ndarray
    colidx: np.ndarray
    vals: np.ndarray
    b: np.ndarray
    xstar: Optional[np.ndarray]
    tol: float
    maxit: int
    meta: Dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.rowptr[-1])

    def scipy(self):
        import scipy.sparse as sp

        return sp.csr_matrix((self.vals, self.colidx, self.rowptr), shape=(self.n, self.n))


def _spmv_for_rhs(rowptr, colidx, vals, x):
    import scipy.sparse as sp

    n = len(rowptr) - 1
    return np.asarray(sp.csr_matrix((vals, colidx, rowptr), shape=(n, n)) @ x, dtype=np.float64)


# ----------------------------------------------------------------------------------------
# structured-grid stencils
# ----------------------------------------------------------------------------------------
def _grid_coords(dims: Tuple[int, int, int]):
    nx, ny, nz = dims
    n = nx * ny * nz
    i = np.arange(n, dtype=np.int64)
    ix = (i % nx).astype(np.int32)
    iy = ((i // nx) % ny).astype(np.int32)
    iz = (i // (nx * ny)).astype(np.int32)
    return ix, iy, iz


def _stencil_csr(dims: Tuple[int, int, int], offsets: Sequence[Tuple[int, int, int]],
                 value_fn: Callable[[int, np.ndarray], "np.ndarray | float"]):
    """Assemble a stencil matrix on an nx*ny*nz grid (x fastest), dropping out-of-grid
    neighbours (homogeneous Dirichlet, boundary unknowns eliminated).

    ``offsets`` must be sorted by linear column offset so each CSR row has ascending columns.
    ``value_fn(k, rows)`` returns the value(s) of offset k on the given rows.
    """
    nx, ny, nz = dims
    n = nx * ny * nz
    ix, iy, iz = _grid_coords(dims)
    lin = [dx + nx * (dy + ny * dz) for (dx, dy, dz) in offsets]
    assert all(lin[k] < lin[k + 1] for k in range(len(lin) - 1)), "offsets must be column-sorted"
    masks = []
    counts = np.zeros(n, dtype=np.int64)
    for (dx, dy, dz) in offsets:
        m = np.ones(n, dtype=bool)
        if dx:
            m &= (ix + dx >= 0) & (ix + dx < nx)
        if dy:
            m &= (iy + dy >= 0) & (iy + dy < ny)
        if dz:
            m &= (iz + dz >= 0) & (iz + dz < nz)
        masks.append(m)
        counts += m
    rowptr64 = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(counts, out=rowptr64[1:])
    nnz = int(rowptr64[-1])
    assert nnz < 2**31
    colidx = np.empty(nnz, dtype=np.int32)
    vals = np.empty(nnz, dtype=np.float64)
    pos = rowptr64[:-1].copy()
    for k, m in enumerate(masks):
        rows = np.flatnonzero(m)
        dst = pos[rows]
        colidx[dst] = (rows + lin[k]).astype(np.int32)
        vals[dst] = value_fn(k, rows)
        pos[rows] += 1
    return rowptr64.astype(np.int32), colidx, vals


def poisson2d_5pt(N: int):
    """Unscaled 2-D 5-point FD Laplacian on an N*N interior grid: diag 4, off-diag -1 (config 1)."""
    offs = [(0, -1, 0), (-1, 0, 0), (0, 0, 0), (1, 0, 0), (0, 1, 0)]
    return _stencil_csr((N, N, 1), offs, lambda k, rows: 4.0 if offs[k] == (0, 0, 0) else -1.0)


def poisson3d_7pt(N: int):
    """Unscaled 3-D 7-point FD Laplacian on an N^3 interior grid: diag 6, off-diag -1 (config 2)."""
    offs = [(0, 0, -1), (0, -1, 0), (-1, 0, 0), (0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)]
    return _stencil_csr((N, N, N), offs, lambda k, rows: 6.0 if offs[k] == (0, 0, 0) else -1.0)


def vardiff3d_7pt(N: int, seed: int):
    """Cell-centred variable-coefficient diffusion, 7-point, N^3 cells (config 3).

    a_c = 10^(-3+6U) i.i.d. per cell; interior face coefficient = harmonic mean
    2 a_c a_c' / (a_c + a_c'); a Dirichlet boundary face has coefficient a_c (ghost cell of
    equal coefficient); A_cc' = -face, A_cc = sum of the six face coefficients.
    """
    n = N * N * N
    a = 10.0 ** (-3.0 + 6.0 * uniform01(seed, 0, np.arange(n, dtype=np.int64)))
    offs = [(0, 0, -1), (0, -1, 0), (-1, 0, 0), (0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)]
    lin = [dx + N * (dy + N * dz) for (dx, dy, dz) in offs]
    ix, iy, iz = _grid_coords((N, N, N))
    diag = np.zeros(n, dtype=np.float64)
    for (dx, dy, dz), l in zip(offs, lin):
        if l == 0:
            continue
        m = np.ones(n, dtype=bool)
        if dx:
            m &= (ix + dx >= 0) & (ix + dx < N)
        if dy:
            m &= (iy + dy >= 0) & (iy + dy < N)
        if dz:
            m &= (iz + dz >= 0) & (iz + dz < N)
        rows = np.flatnonzero(m)
        face = np.array(a, copy=True)  # boundary faces: coefficient a_c
        ac, an = a[rows], a[rows + l]
        face[rows] = 2.0 * ac * an / (ac + an)
        diag += face

    def value(k, rows):
        if lin[k] == 0:
            return diag[rows]
        ac, an = a[rows], a[rows + lin[k]]
        return -(2.0 * ac * an / (ac + an))

    return _stencil_csr((N, N, N), offs, value)


def fe27_laplacian(N: int, keep_zero_faces: bool = True):
    """Trilinear-FE Laplacian on N^3 interior nodes, h=1 (config 4):
    K(x)M(x)M + M(x)K(x)M + M(x)M(x)K with K=tridiag(-1,2,-1), M=tridiag(1,4,1)/6
    => centre 8/3, face 0, edge -1/6, corner -1/12.  All 27 pattern entries are stored
    (faces as explicit 0.0) unless ``keep_zero_faces`` is False.
    """
    offs = [(dx, dy, dz) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1)]
    table = {0: 8.0 / 3.0, 1: 0.0, 2: -1.0 / 6.0, 3: -1.0 / 12.0}
    if not keep_zero_faces:
        offs = [o for o in offs if sum(map(abs, o)) != 1]
    return _stencil_csr((N, N, N), offs, lambda k, rows: table[sum(map(abs, offs[k]))])


# ----------------------------------------------------------------------------------------
# random banded SPD (config 5)
# ----------------------------------------------------------------------------------------
def random_spd_banded(n: int, seed: int, draws: int = 16, width: int = 50_000, shift: float = 1e-2):
    """Row i: ``draws`` offsets o~U{1..width}, j=i+o (<n), first occurrence kept on duplicates,
    v = 0.1*N(0,1) (Box-Muller), mirrored to (j,i); diag_i = sum_j |a_ij| + shift."""
    width = min(width, max(n - 1, 1))
    e = np.arange(n * draws, dtype=np.int64)
    i = e // draws
    o = 1 + np.floor(uniform01(seed, 0, e) * width).astype(np.int64)
    o = np.minimum(o, width)
    j = i + o
    v = 0.1 * _normal(seed, 1, e)
    keep = j < n
    i, j, v, e = i[keep], j[keep], v[keep], e[keep]
    # dedupe (i,j): keep the first draw.  Sort by (i, j, draw index).
    key = (i * np.int64(n) + j)
    order = np.lexsort((e, key))
    key_s = key[order]
    first = np.ones(len(order), dtype=bool)
    first[1:] = key_s[1:] != key_s[:-1]
    sel = order[first]
    i, j, v = i[sel], j[sel], v[sel]
    absrow = np.bincount(i, weights=np.abs(v), minlength=n) + np.bincount(j, weights=np.abs(v), minlength=n)
    diag = absrow + shift
    rows = np.concatenate([i, j, np.arange(n, dtype=np.int64)])
    cols = np.concatenate([j, i, np.arange(n, dtype=np.int64)])
    data = np.concatenate([v, v, diag])
    order = np.argsort(rows * np.int64(n) + cols, kind="stable")
    rows, cols, data = rows[order], cols[order], data[order]
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(np.bincount(rows, minlength=n), out=rowptr[1:])
    assert rowptr[-1] < 2**31
    return rowptr.astype(np.int32), cols.astype(np.int32), data.astype(np.float64)


# ----------------------------------------------------------------------------------------
# BASELINE.json configs
# ----------------------------------------------------------------------------------------
CONFIGS = {
    # name: (description, full size parameter, tol, maxit)
    "c1": ("2D Poisson 5-pt 64x64", 64, 1e-8, 5000),
    "c2": ("3D Poisson 7-pt 128^3", 128, 1e-10, 20000),
    "c3": ("3D variable-coefficient diffusion 7-pt 160^3", 160, 1e-8, 20000),
    "c4": ("3D 27-pt trilinear FE Laplacian 200^3", 200, 1e-8, 20000),
    "c5": ("random banded SPD n=2e6, ~32 nnz/row", 2_000_000, 1e-9, 20000),
}


def make_config(name: str, size: Optional[int] = None) -> CSRSystem:
    """Build BASELINE.json config ``name`` ('c1'..'c5'); ``size`` overrides the grid edge
    (c1-c4) or the row count (c5) to make scaled-down parity cases with the same structure."""
    desc, full, tol, maxit = CONFIGS[name]
    size = full if size is None else int(size)
    c = int(name[1])
    seed = BASE_SEED + c
    if name == "c1":
        rowptr, colidx, vals = poisson2d_5pt(size)
    elif name == "c2":
        rowptr, colidx, vals = poisson3d_7pt(size)
    elif name == "c3":
        rowptr, colidx, vals = vardiff3d_7pt(size, seed)
    elif name == "c4":
        rowptr, colidx, vals = fe27_laplacian(size)
    elif name == "c5":
        rowptr, colidx, vals = random_spd_banded(size, seed, width=min(50_000, max(size // 40, 1)) if size != full else 50_000)
    else:
        raise KeyError(name)
    n = len(rowptr) - 1
    idx = np.arange(n, dtype=np.int64)
    if name == "c4":
        xstar = None
        b = 2.0 * uniform01(seed, 100, idx) - 1.0  # b ~ U[-1,1)
    else:
        xstar = 2.0 * uniform01(seed, 100, idx) - 1.0
        b = _spmv_for_rhs(rowptr, colidx, vals, xstar)
    return CSRSystem(name=f"{name}@{size}", n=n, rowptr=rowptr, colidx=colidx, vals=vals, b=b, xstar=xstar,
                     tol=tol, maxit=maxit, meta={"config": name, "size": size, "seed": seed, "desc": desc})


# ----------------------------------------------------------------------------------------
# the paper's self-contained dense examples, stored as dense CSR
# ----------------------------------------------------------------------------------------
def dense_spd_from_spectrum(lams: np.ndarray, seed: int, identity_q: bool = False):
    """A = Q diag(lams) Q^T with a seeded random orthonormal Q (QR of a Gaussian matrix), as
    a dense CSR matrix (all n^2 entries stored)."""
    lams = np.asarray(lams, dtype=np.float64)
    n = len(lams)
    if identity_q:
        A = np.diag(lams)
    else:
        G = _normal(seed, 7, np.arange(n * n, dtype=np.int64)).reshape(n, n)
        Q, R = np.linalg.qr(G)
        Q = Q * np.sign(np.diag(R))
        A = (Q * lams) @ Q.T
        A = 0.5 * (A + A.T)
    rowptr = (np.arange(n + 1, dtype=np.int64) * n).astype(np.int32)
    colidx = np.tile(np.arange(n, dtype=np.int32), n)
    return rowptr, colidx, A.reshape(-1).copy()


def _spectrum_55(n: int, rho: float) -> np.ndarray:
    """Eq. (5.5): lam_i = 1e-3 + (i-1)/(n-1) rho^(n-i), i=1..n-1; lam_n = 1."""
    i = np.arange(1, n + 1, dtype=np.float64)
    lam = 1e-3 + (i - 1.0) / (n - 1.0) * rho ** (n - i)
    lam[-1] = 1.0
    return lam


def paper_example(ex: int, seed: int = 1, identity_q: bool = False) -> CSRSystem:
    """Examples 1, 4, 6, 9, 10 of the paper (M = I, x0 = 0)."""
    if ex == 1:  # eq. (2.2)
        n = 100
        lam = np.empty(n)
        i = np.arange(95, 100, dtype=np.float64)  # i = 95..99
        lam[94:99] = 1e-3 + (i - 1.0) / 99.0 * (17.0 / 20.0) ** (100.0 - i)
        lam[99] = 1.0
        lam[:95] = np.linspace(1e-3, lam[94], 95)
        b = np.ones(n)
        tol = 1e-10
    elif ex in (4, 6):
        nn = 100
        i = np.arange(0, nn + 1, dtype=np.float64)
        small = 10.0 if ex == 4 else 1000.0
        lam = i / (small * nn) + (nn - i) / nn
        n = nn + 1
        b = 2.0 * uniform01(seed, 11, np.arange(n)) - 1.0  # "b is randomly generated" (:414)
        tol = 1e-10
    elif ex == 9:
        n = 10
        lam = _spectrum_55(n, 0.25)
        b = np.ones(n)
        tol = 1e-10
    elif ex == 10:
        n = 50
        lam = _spectrum_55(n, 0.9)
        b = np.ones(n)
        tol = 1e-10
    else:
        raise KeyError(ex)
    rowptr, colidx, vals = dense_spd_from_spectrum(lam, seed, identity_q=identity_q)
    return CSRSystem(name=f"ex{ex}", n=n, rowptr=rowptr, colidx=colidx, vals=vals, b=b, xstar=None,
                     tol=tol, maxit=10 * n, meta={"example": ex, "spectrum": lam, "seed": seed})
