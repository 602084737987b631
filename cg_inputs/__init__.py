"""Seeded synthetic inputs for the fp64 CSR conjugate-gradient path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_1107_0538_b200/``).  It imports neither and holds no CG arithmetic:
it only fabricates matrices and vectors.  The recipe is SURVEY.md section 8(d)
and BASELINE.json ``configs``; the paper itself only fixes the shape of the
workload ("CSR ... N=132651 and NNZ=3442951", PAPER.md:48 double
precision, PAPER.md:60 TOL=1E-10, "CGLoop is a 132651 loop").
The paper's FEM matrix is not public, so these inputs stand in for it
(DESIGN.md "Input recipe").

Everything is a pure function of (config, seed): no global RNG state.

Hash (frozen):
    mix(z)  : z ^= z >> 30; z *= 0xBF58476D1CE4E5B9;
              z ^= z >> 27; z *= 0x94D049BB133111EB;
              z ^= z >> 31                       (64-bit wrap-around)
    k       = mix(seed * 0x100000001B3 + stream)
    u       = (mix(k ^ key) >> 11) * 2**-53       in [0, 1)
    streams : 1 = edge weights, 2 = vectors, 3 = permutation keys
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

__all__ = [
    "CSRProblem", "hash_uniform", "stencil27", "laplacian7", "permute_symmetric",
    "seeded_vector", "rhs_from_solution", "make_config", "CONFIG_NAMES",
    "algorithmic_bytes_per_iteration", "flops_per_iteration",
]

_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_FNV = 0x100000001B3
_MASK64 = (1 << 64) - 1

STREAM_WEIGHT = 1
STREAM_VECTOR = 2
STREAM_PERM = 3


def _mix_scalar(z: int) -> int:
    z &= _MASK64
    z ^= z >> 30
    z = (z * 0xBF58476D1CE4E5B9) & _MASK64
    z ^= z >> 27
    z = (z * 0x94D049BB133111EB) & _MASK64
    z ^= z >> 31
    return z


def _mix_array(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array, in place on a private copy."""
    z = z.astype(np.uint64, copy=True)
    with np.errstate(over="ignore"):
        z ^= z >> np.uint64(30)
        z *= _M1
        z ^= z >> np.uint64(27)
        z *= _M2
        z ^= z >> np.uint64(31)
    return z


def hash_uniform(seed: int, stream: int, key) -> np.ndarray:
    """u(seed, stream, key): counter-based uniform doubles in [0, 1)."""
    k = np.uint64(_mix_scalar(seed * _FNV + stream))
    key = np.asarray(key).astype(np.uint64, copy=False)
    h = _mix_array(key ^ k)
    return (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


@dataclass
class CSRProblem:
    """One linear system A x = b in CSR (int32 indices, fp64 values)."""
    name: str
    n: int
    rowptr: np.ndarray          # int32[n+1]
    colind: np.ndarray          # int32[nnz], ascending inside each row
    vals: np.ndarray            # float64[nnz]
    b: np.ndarray               # float64[n]
    x0: np.ndarray              # float64[n]
    rtol: float
    maxit: int
    xstar: Optional[np.ndarray] = None   # known solution when b = A xstar
    meta: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.rowptr[-1])


def seeded_vector(seed: int, n: int) -> np.ndarray:
    """v_i = 2 u(seed, 2, i) - 1, i = 0..n-1."""
    return 2.0 * hash_uniform(seed, STREAM_VECTOR, np.arange(n, dtype=np.uint64)) - 1.0


def _offsets27():
    # (dz, dy, dx) ascending == ascending column index for node = x + n y + n^2 z
    return [(dz, dy, dx) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1)]


def stencil27(n: int, weight_seed: int = 0, contrast: float = 1.0,
              cyl_radius: float = 0.0):
    """Weighted 27-point stencil on an n^3 grid, natural ordering.

    a_ij = -w_ij, w_ij = 0.5 + u(weight_seed, 1, min(i,j) N + max(i,j)) for grid
    neighbours i != j; a_ii = sum_j |a_ij| (ascending j) + 0.01.  With
    ``contrast`` != 1 the weight of an edge whose two endpoints both lie inside
    the z-axis cylinder (x-c)^2 + (y-c)^2 <= cyl_radius^2, c = (n-1)/2, is
    multiplied by ``contrast`` (config 4).
    Returns (rowptr int32, colind int32, vals float64).
    """
    N = n * n * n
    if N * 27 >= 2**31:
        raise ValueError("nnz does not fit int32 indices")
    ids = np.arange(N, dtype=np.int64)
    x = ids % n
    y = (ids // n) % n
    z = ids // (n * n)
    if contrast != 1.0:
        c = (n - 1) / 2.0
        inside = (x - c) ** 2 + (y - c) ** 2 <= cyl_radius ** 2
    offs = _offsets27()
    V = np.zeros((N, 27), dtype=np.float64)
    C = np.zeros((N, 27), dtype=np.int32)
    M = np.zeros((N, 27), dtype=bool)
    diag = np.zeros(N, dtype=np.float64)
    Nu = np.uint64(N)
    for s, (dz, dy, dx) in enumerate(offs):
        if dx == 0 and dy == 0 and dz == 0:
            M[:, s] = True
            C[:, s] = ids
            continue
        valid = ((x + dx >= 0) & (x + dx < n) & (y + dy >= 0) & (y + dy < n)
                 & (z + dz >= 0) & (z + dz < n))
        i = ids[valid]
        j = i + (dx + n * dy + n * n * dz)
        lo = np.minimum(i, j).astype(np.uint64)
        hi = np.maximum(i, j).astype(np.uint64)
        with np.errstate(over="ignore"):
            key = lo * Nu + hi
        w = 0.5 + hash_uniform(weight_seed, STREAM_WEIGHT, key)
        if contrast != 1.0:
            both = inside[i] & inside[j]
            w = np.where(both, w * contrast, w)
        V[valid, s] = -w
        C[valid, s] = j
        M[:, s] = valid
        dcol = np.zeros(N, dtype=np.float64)
        dcol[valid] = w
        diag += dcol                 # ascending-j accumulation; + 0.0 is exact
    V[:, 13] = diag + 0.01
    counts = M.sum(axis=1, dtype=np.int64)
    rowptr = np.zeros(N + 1, dtype=np.int64)
    np.cumsum(counts, out=rowptr[1:])
    colind = C[M]
    vals = V[M]
    return rowptr.astype(np.int32), colind.astype(np.int32), vals


def laplacian7(n: int):
    """7-point Dirichlet Laplacian on an n^3 grid: diag 6, off-diagonals -1."""
    N = n * n * n
    ids = np.arange(N, dtype=np.int64)
    x = ids % n
    y = (ids // n) % n
    z = ids // (n * n)
    offs = [(-1, 0, 0), (0, -1, 0), (0, 0, -1), (0, 0, 0), (0, 0, 1), (0, 1, 0), (1, 0, 0)]
    V = np.zeros((N, 7), dtype=np.float64)
    C = np.zeros((N, 7), dtype=np.int32)
    M = np.zeros((N, 7), dtype=bool)
    for s, (dz, dy, dx) in enumerate(offs):
        valid = ((x + dx >= 0) & (x + dx < n) & (y + dy >= 0) & (y + dy < n)
                 & (z + dz >= 0) & (z + dz < n))
        C[:, s] = ids + (dx + n * dy + n * n * dz)
        V[:, s] = 6.0 if (dx, dy, dz) == (0, 0, 0) else -1.0
        M[:, s] = valid
    counts = M.sum(axis=1, dtype=np.int64)
    rowptr = np.zeros(N + 1, dtype=np.int64)
    np.cumsum(counts, out=rowptr[1:])
    return rowptr.astype(np.int32), C[M].astype(np.int32), V[M]


def permute_symmetric(rowptr, colind, vals, seed: int):
    """B = P A P^T with pi(i) = rank of i under a stable sort of u(seed, 3, i).

    B[pi(i), pi(j)] = A[i, j]; columns re-sorted ascending in every row.
    Returns (rowptr, colind, vals, pi).
    """
    n = len(rowptr) - 1
    keys = hash_uniform(seed, STREAM_PERM, np.arange(n, dtype=np.uint64))
    order = np.argsort(keys, kind="stable")
    pi = np.empty(n, dtype=np.int64)
    pi[order] = np.arange(n, dtype=np.int64)
    counts = np.diff(rowptr.astype(np.int64))
    rows_old = np.repeat(np.arange(n, dtype=np.int64), counts)
    rows_new = pi[rows_old]
    cols_new = pi[colind.astype(np.int64)]
    srt = np.lexsort((cols_new, rows_new))
    new_counts = np.zeros(n, dtype=np.int64)
    new_counts[pi] = counts
    rp = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(new_counts, out=rp[1:])
    return (rp.astype(np.int32), cols_new[srt].astype(np.int32),
            np.ascontiguousarray(vals[srt]), pi)


def rhs_from_solution(rowptr, colind, vals, xstar) -> np.ndarray:
    """Input recipe only: b = A xstar, each row summed left to right in stored order.

    Part of the definition of configs 0 and 2 (BASELINE.json: "b = A x*").  It
    is never used as an expected value for the method; the oracle's SpMV is
    checked against it as one more independent pin.
    """
    n = len(rowptr) - 1
    rp = rowptr.astype(np.int64)
    lens = np.diff(rp)
    b = np.zeros(n, dtype=np.float64)
    for k in range(int(lens.max()) if n else 0):
        rows = np.nonzero(lens > k)[0]
        idx = rp[rows] + k
        b[rows] = b[rows] + vals[idx] * xstar[colind[idx]]
    return b


CONFIG_NAMES = {
    0: "tiny_16^3_27pt",
    1: "laplacian_64^3_7pt",
    2: "fem_51^3_27pt",
    3: "fem_51^3_27pt_permuted",
    4: "contrast_160^3_27pt",
}


def make_config(cfg: int, grid: Optional[int] = None) -> CSRProblem:
    """Build BASELINE.json config ``cfg`` (0..4).

    ``grid`` overrides the grid edge n (tests use it for scaled-down variants
    of the same recipe; the cylinder radius of config 4 scales as n/4).
    """
    if cfg == 0:
        n = grid or 16
        rp, ci, va = stencil27(n)
        xs = seeded_vector(0, n ** 3)
        b = rhs_from_solution(rp, ci, va, xs)
        return CSRProblem(CONFIG_NAMES[0], n ** 3, rp, ci, va, b, np.zeros(n ** 3), 1e-10, 1000,
                          xstar=xs, meta={"grid": n, "stencil": 27})
    if cfg == 1:
        n = grid or 64
        rp, ci, va = laplacian7(n)
        b = seeded_vector(1, n ** 3)
        return CSRProblem(CONFIG_NAMES[1], n ** 3, rp, ci, va, b, np.zeros(n ** 3), 1e-8, 5000,
                          meta={"grid": n, "stencil": 7})
    if cfg == 2:
        n = grid or 51
        rp, ci, va = stencil27(n)
        xs = seeded_vector(2, n ** 3)
        b = rhs_from_solution(rp, ci, va, xs)
        return CSRProblem(CONFIG_NAMES[2], n ** 3, rp, ci, va, b, np.zeros(n ** 3), 1e-10, n ** 3,
                          xstar=xs, meta={"grid": n, "stencil": 27})
    if cfg == 3:
        n = grid or 51
        rp, ci, va = stencil27(n)
        rp, ci, va, pi = permute_symmetric(rp, ci, va, seed=3)
        b = seeded_vector(3, n ** 3)
        return CSRProblem(CONFIG_NAMES[3], n ** 3, rp, ci, va, b, np.zeros(n ** 3), 1e-10, n ** 3,
                          meta={"grid": n, "stencil": 27, "perm": pi})
    if cfg == 4:
        n = grid or 160
        radius = 40.0 * n / 160.0
        rp, ci, va = stencil27(n, contrast=1000.0, cyl_radius=radius)
        b = seeded_vector(4, n ** 3)
        return CSRProblem(CONFIG_NAMES[4], n ** 3, rp, ci, va, b, np.zeros(n ** 3), 1e-8, 20000,
                          meta={"grid": n, "stencil": 27, "contrast": 1000.0, "radius": radius})
    raise ValueError(f"unknown config {cfg}")


def algorithmic_bytes_per_iteration(n: int, nnz: int) -> int:
    """12 NNZ + 92 N + 4 bytes per CG iteration."""
    return 12 * nnz + 92 * n + 4


def flops_per_iteration(n: int, nnz: int) -> int:
    """The paper's own convention, fitted to Table I: 2 NNZ + 10 N."""
    return 2 * nnz + 10 * n
