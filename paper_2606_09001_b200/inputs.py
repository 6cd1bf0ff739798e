"""Seeded synthetic inputs: PDE matrices in CSR (fp64 values / int32 indices) and right-hand sides.

This module is the ONLY code shared by the CUDA path (`paper_2606_09001_b200.binding`) and the
CPU oracle (`oracle/`).  It holds no arithmetic of the method (no SpMV, no aggregation, no
solver): it only writes down the discretised operators and random vectors the paper's
workloads are made of, from integer seeds (numpy PCG64).

The matrices stand in for the paper's PDE workloads (2D Poisson examples, §3.1
and :243 §3.4; the tridiagonal inverse problem, §3.2; the pressure-Poisson system
of a 100x260x256 channel, §3.5).  The SuiteSparse matrices of PAPER.md:283 and the
in-house CFD matrix are not reproduced.  Recipes follow SURVEY.md §8(d) / BASELINE.json configs.

Conventions: unit stencil (diag 2d, neighbours -1), homogeneous Dirichlet,
rows lexicographic with x fastest, ascending unique columns in every row.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Csr:
    """CSR triple. rowptr int32[n+1], col int32[nnz], val float64[nnz]."""

    n: int
    rowptr: np.ndarray
    col: np.ndarray
    val: np.ndarray
    meta: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.rowptr[-1])

    def to_scipy(self):
        import scipy.sparse as sp

        return sp.csr_matrix((self.val, self.col, self.rowptr), shape=(self.n, self.n))

    def to_dense(self) -> np.ndarray:
        a = np.zeros((self.n, self.n))
        rows = np.repeat(np.arange(self.n), np.diff(self.rowptr))
        a[rows, self.col] = self.val
        return a


def _stencil_csr(shape, k_cell=None) -> Csr:
    """(2d+1)-point finite-volume operator  -div(k grad u)  on a box grid, Dirichlet.

    shape = (nx,), (ny, nx) or (nz, ny, nx); x is the fastest index.  k_cell=None means k == 1
    (the constant-coefficient Laplacian: diag 2d, neighbours -1).  Otherwise the coefficient
    of the face between cells a and b is the harmonic mean 2 k_a k_b / (k_a + k_b), computed
    once per face so that a_ij and a_ji carry the same bits; a boundary face uses k_face =
    k_cell (Dirichlet ghost); the diagonal is the sum of the 2d face coefficients of the cell
    (summed in the fixed order -z,-y,-x,+x,+y,+z), so k == 1 reproduces the Laplacian.
    """
    shape = tuple(int(s) for s in shape)
    d = len(shape)
    n = int(np.prod(shape))
    if n >= 2**31:
        raise ValueError("grid too large for int32 indices")
    idx = np.arange(n, dtype=np.int64).reshape(shape)
    strides = [int(np.prod(shape[a + 1:])) for a in range(d)]  # index stride per axis

    # per axis: face coefficient arrays "towards lower neighbour" and "towards upper neighbour"
    lo_coef, up_coef, lo_ok, up_ok = [], [], [], []
    for a in range(d):
        ok_lo = np.ones(shape, dtype=bool)
        ok_up = np.ones(shape, dtype=bool)
        sl_first = [slice(None)] * d
        sl_first[a] = slice(0, 1)
        sl_last = [slice(None)] * d
        sl_last[a] = slice(shape[a] - 1, shape[a])
        ok_lo[tuple(sl_first)] = False
        ok_up[tuple(sl_last)] = False
        if k_cell is None:
            c_lo = np.ones(shape)
            c_up = np.ones(shape)
        else:
            k = np.asarray(k_cell, dtype=np.float64).reshape(shape)
            sl_a = [slice(None)] * d
            sl_b = [slice(None)] * d
            sl_a[a] = slice(0, shape[a] - 1)
            sl_b[a] = slice(1, shape[a])
            ka, kb = k[tuple(sl_a)], k[tuple(sl_b)]
            face = 2.0 * ka * kb / (ka + kb)  # interior faces along axis a
            c_lo = k.copy()  # boundary face: k_face = k_cell
            c_up = k.copy()
            c_lo[tuple(sl_b)] = face
            c_up[tuple(sl_a)] = face
        lo_coef.append(c_lo)
        up_coef.append(c_up)
        lo_ok.append(ok_lo)
        up_ok.append(ok_up)

    return _assemble_stencil(shape, lo_coef, up_coef)


def _assemble_stencil(shape, lo_coef, up_coef, row_scale=None) -> Csr:
    """CSR of the (2d+1)-point operator with the given face coefficients per axis ("towards the lower
    neighbour" / "towards the upper neighbour", full-shape arrays; a boundary face has no neighbour
    entry but still counts in the diagonal: Dirichlet ghost).  row_scale (optional, full shape)
    multiplies every entry of a row (e.g. 1 / cell volume: a nonsymmetric matrix)."""
    d = len(shape)
    n = int(np.prod(shape))
    idx = np.arange(n, dtype=np.int64).reshape(shape)
    strides = [int(np.prod(shape[a + 1:])) for a in range(d)]
    lo_ok, up_ok = [], []
    for a in range(d):
        ok_lo = np.ones(shape, dtype=bool)
        ok_up = np.ones(shape, dtype=bool)
        sl_first = [slice(None)] * d
        sl_first[a] = slice(0, 1)
        sl_last = [slice(None)] * d
        sl_last[a] = slice(shape[a] - 1, shape[a])
        ok_lo[tuple(sl_first)] = False
        ok_up[tuple(sl_last)] = False
        lo_ok.append(ok_lo)
        up_ok.append(ok_up)
    # slots in ascending column order: lower neighbours from the slowest axis to the fastest,
    # the diagonal, upper neighbours from the fastest axis to the slowest.
    nslot = 2 * d + 1
    cols = np.empty((n, nslot), dtype=np.int64)
    vals = np.empty((n, nslot), dtype=np.float64)
    mask = np.empty((n, nslot), dtype=bool)
    flat = idx.reshape(-1)
    diag = np.zeros(n)
    s = 0
    for a in range(d):  # lower neighbours: axis 0 (slowest) first
        cols[:, s] = flat - strides[a]
        vals[:, s] = -lo_coef[a].reshape(-1)
        mask[:, s] = lo_ok[a].reshape(-1)
        diag += lo_coef[a].reshape(-1)
        s += 1
    sd = s
    s += 1
    for a in reversed(range(d)):  # upper neighbours: fastest axis first
        cols[:, s] = flat + strides[a]
        vals[:, s] = -up_coef[a].reshape(-1)
        mask[:, s] = up_ok[a].reshape(-1)
        diag += up_coef[a].reshape(-1)
        s += 1
    cols[:, sd] = flat
    vals[:, sd] = diag
    mask[:, sd] = True
    if row_scale is not None:
        vals = vals * np.asarray(row_scale, dtype=np.float64).reshape(-1, 1)

    rowlen = mask.sum(axis=1)
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(rowlen, out=rowptr[1:])
    if rowptr[-1] >= 2**31:
        raise ValueError("nnz too large for int32 indices")
    return Csr(n, rowptr.astype(np.int32), cols[mask].astype(np.int32), vals[mask],
               {"shape": shape})


def stretched_channel_csr(shape, stretch: float = 2.0) -> Csr:
    """Nonsymmetric "pressure-Poisson-like" system: the 7-point finite-volume Laplacian on a box grid
    whose axis 1 (wall-normal, shape = (nz, ny, nx)) is stretched by y_j = tanh(stretch (2j/ny - 1)) /
    tanh(stretch) (cells cluster at both walls; widths normalised to mean 1), the other axes uniform
    with width 1, Dirichlet ghost cells on every boundary, EVERY ROW DIVIDED BY ITS CELL VOLUME:
    A = D^-1 S with S symmetric, so a_ij != a_ji across the stretched axis while the pattern stays
    symmetric.  Stands in for the stretched-grid channel matrix of PAPER.md:293 (100 x 260 x 256,
    "nonsymmetric stored matrix"), which is not available.  Face coefficient = face area / distance
    between the cell centres (boundary face: distance to the wall = half a cell)."""
    shape = tuple(int(s) for s in shape)
    assert len(shape) == 3
    nz, ny, nx = shape
    edges = np.tanh(stretch * (2.0 * np.arange(ny + 1) / ny - 1.0)) / np.tanh(stretch)
    hy = np.diff(edges)
    hy = hy * (ny / hy.sum())
    widths = [np.ones(nz), hy, np.ones(nx)]
    vol = widths[0][:, None, None] * widths[1][None, :, None] * widths[2][None, None, :]
    lo_coef, up_coef = [], []
    for a in range(3):
        w = widths[a]
        sh = [1, 1, 1]
        sh[a] = shape[a]
        area = vol / w.reshape(sh)                       # face area normal to axis a
        d_lo = np.empty(shape[a])
        d_up = np.empty(shape[a])
        d_lo[0] = 0.5 * w[0]
        d_lo[1:] = 0.5 * (w[:-1] + w[1:])               # the same expression on both sides of a face
        d_up[-1] = 0.5 * w[-1]
        d_up[:-1] = 0.5 * (w[:-1] + w[1:])
        lo_coef.append(area / d_lo.reshape(sh))
        up_coef.append(area / d_up.reshape(sh))
    a_ = _assemble_stencil(shape, lo_coef, up_coef, row_scale=1.0 / vol)
    a_.meta["stretch"] = stretch
    a_.meta["hy_min"] = float(hy.min())
    a_.meta["hy_max"] = float(hy.max())
    return a_


def poisson_csr(shape) -> Csr:
    """Dirichlet Laplacian, unit stencil: 1D tridiag(-1,2,-1), 2D 5-point, 3D 7-point."""
    if isinstance(shape, int):
        shape = (shape,)
    return _stencil_csr(shape)


def tridiagonal_csr(n: int, diagonal_value: float = 2.0, off_value: float = -1.0) -> Csr:
    """Toeplitz tridiagonal matrix of the paper's inverse problem (§3.2)."""
    a = _stencil_csr((n,))
    row = np.repeat(np.arange(n), np.diff(a.rowptr))
    is_diag = a.col == row
    a.val = np.where(is_diag, float(diagonal_value), float(off_value))
    return a


def gaussian_random_field(shape, seed: int, sigma: float = 2.0, ell: float = 8.0) -> np.ndarray:
    """log k: white noise N(0,1) -> FFT -> * exp(-ell^2 |kappa|^2 / 4) -> inverse FFT (real part)
    -> subtract mean, divide by std, times sigma.  kappa = 2 pi fftfreq per axis.  Periodic
    field with correlation exp(-r^2 / (2 ell^2)) (SURVEY.md §8(d) cfg 4)."""
    rng = np.random.default_rng(seed)
    w = rng.standard_normal(shape)
    kap2 = np.zeros(shape)
    for a, m in enumerate(shape):
        kk = 2.0 * np.pi * np.fft.fftfreq(m)
        sh = [1] * len(shape)
        sh[a] = m
        kap2 = kap2 + (kk.reshape(sh)) ** 2
    f = np.fft.ifftn(np.fft.fftn(w) * np.exp(-(ell**2) * kap2 / 4.0)).real
    f -= f.mean()
    f /= f.std()
    return sigma * f


def variable_diffusion_csr(shape, seed: int, sigma: float = 2.0, ell: float = 8.0) -> Csr:
    """-div(k grad u), k = exp(gaussian_random_field), harmonic-mean faces, Dirichlet."""
    logk = gaussian_random_field(shape, seed, sigma, ell)
    a = _stencil_csr(shape, np.exp(logk))
    a.meta["k_min"] = float(np.exp(logk.min()))
    a.meta["k_max"] = float(np.exp(logk.max()))
    return a


def permute_symmetric(a: Csr, perm: np.ndarray) -> Csr:
    """A' = Pi A Pi^T : old row/column i becomes new row/column perm[i]; columns re-sorted."""
    n = a.n
    perm = np.asarray(perm, dtype=np.int64)
    inv = np.empty(n, dtype=np.int64)
    inv[perm] = np.arange(n, dtype=np.int64)
    rowlen = np.diff(a.rowptr).astype(np.int64)
    new_rowlen = rowlen[inv]
    new_rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(new_rowlen, out=new_rowptr[1:])
    # source position of every new entry (row-gather), then sort columns inside each new row
    old_start = a.rowptr[:-1].astype(np.int64)[inv]
    src = np.repeat(old_start - new_rowptr[:-1], new_rowlen) + np.arange(new_rowptr[-1])
    new_row = np.repeat(np.arange(n, dtype=np.int64), new_rowlen)
    new_col = perm[a.col[src]]
    order = np.argsort(new_row * n + new_col, kind="stable")
    meta = dict(a.meta)
    meta["permuted"] = True
    return Csr(n, new_rowptr.astype(np.int32), new_col[order].astype(np.int32),
               a.val[src][order], meta)


def rhs_uniform(n: int, seed: int) -> np.ndarray:
    """b ~ Uniform[-1, 1]."""
    return np.random.default_rng(seed).uniform(-1.0, 1.0, n)


def rhs_normal(n: int, seed: int) -> np.ndarray:
    """vector ~ N(0, 1) (x_true of cfg 2, x_target of cfg 5)."""
    return np.random.default_rng(seed).standard_normal(n)


def rhs_ones(n: int) -> np.ndarray:
    """The paper's rhs_ones."""
    return np.ones(n)


# ------------------------------------------------------------------------------------------
# The five BASELINE.json configurations.  `scale` shrinks the grid edge for tests (scale=1 is
# the full size); seeds as in SURVEY.md §8(d).
# ------------------------------------------------------------------------------------------
def config_matrix(cfg: int, edge: int | None = None) -> Csr:
    if cfg == 1:
        e = edge or 64
        return poisson_csr((e, e))
    if cfg == 2:
        e = edge or 1024
        return poisson_csr((e, e))
    if cfg == 3:
        e = edge or 128
        return poisson_csr((e, e, e))
    if cfg in (4, 5):
        e = edge or 192
        a = variable_diffusion_csr((e, e, e), seed=4001, sigma=2.0, ell=8.0)
        perm = np.random.default_rng(4002).permutation(a.n)
        return permute_symmetric(a, perm)
    raise ValueError(f"unknown config {cfg}")


def config_rhs(cfg: int, n: int, k: int = 0) -> np.ndarray:
    """k-th right-hand-side *seed vector* of a config.

    cfg 1: b ~ U[-1,1] [1001].  cfg 2: x_true,k ~ N(0,1) [2001+k] (the caller forms b = A x_true
    with whichever SpMV it is testing).  cfg 3: b ~ U[-1,1] [3001].  cfg 4: b ~ U[-1,1] [4003].
    cfg 5: b_k ~ U[-1,1] [5001+k]; targets from config_target.
    """
    if cfg == 1:
        return rhs_uniform(n, 1001)
    if cfg == 2:
        return rhs_normal(n, 2001 + k)
    if cfg == 3:
        return rhs_uniform(n, 3001)
    if cfg == 4:
        return rhs_uniform(n, 4003)
    if cfg == 5:
        return rhs_uniform(n, 5001 + k)
    raise ValueError(f"unknown config {cfg}")


def config_target(n: int, k: int) -> np.ndarray:
    """cfg 5: x_target,k ~ N(0,1) [5101+k] (one target per right-hand side)."""
    return rhs_normal(n, 5101 + k)
