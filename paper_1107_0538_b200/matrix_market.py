"""Matrix Market coordinate files -> the CSR arrays cg_create takes.

The paper's input is "resulting from a FEM model of an electrical machine ... stored in
Compressed Sparse Row (CSR) format" and is read by the "data reading" block of its task graph
(PAPER.md:34, :42).  That matrix is not public; FEM codes commonly export Matrix Market
`coordinate real symmetric` files (one triangle stored), which is what this host-side loader
reads.  It sits OUTSIDE libcg_b200: the library's contract stays "CSR arrays already on the
device" (include/cg.h); this module only produces those arrays on the host.

Supported: `%%MatrixMarket matrix coordinate {real|integer|pattern} {general|symmetric}`.
1-based indices become 0-based; a symmetric file is expanded to both triangles (the diagonal
once); `pattern` entries get the value 1.  Entries are sorted by (row, column) with a stable
sort; duplicates are kept as separate entries (CSR rows may hold duplicates: they add).
Complex, Hermitian, skew-symmetric and dense `array` files are rejected with ValueError.
"""
from __future__ import annotations

import io
from typing import Tuple

import numpy as np


def _open(path_or_file):
    if hasattr(path_or_file, "read"):
        return path_or_file, False
    return open(path_or_file, "r"), True


def read_matrix_market(path_or_file) -> Tuple[int, np.ndarray, np.ndarray, np.ndarray]:
    """Returns (n, rowptr int32[n+1], colind int32[nnz], vals float64[nnz]) of a square matrix."""
    f, close = _open(path_or_file)
    try:
        header = f.readline().split()
        if len(header) != 5 or header[0] != "%%MatrixMarket" or header[1].lower() != "matrix":
            raise ValueError("not a Matrix Market matrix file")
        fmt, field, sym = (h.lower() for h in header[2:5])
        if fmt != "coordinate":
            raise ValueError(f"unsupported format '{fmt}' (only sparse 'coordinate' files)")
        if field not in ("real", "integer", "pattern"):
            raise ValueError(f"unsupported field '{field}'")
        if sym not in ("general", "symmetric"):
            raise ValueError(f"unsupported symmetry '{sym}'")
        line = f.readline()
        while line and (line.startswith("%") or not line.strip()):
            line = f.readline()
        dims = line.split()
        if len(dims) != 3:
            raise ValueError("bad size line")
        nrows, ncols, nent = (int(d) for d in dims)
        if nrows != ncols or nrows <= 0 or nent < 0:
            raise ValueError("a square matrix with n > 0 is required")
        ncol_file = 2 if field == "pattern" else 3
        body = f.read()
    finally:
        if close:
            f.close()
    data = np.loadtxt(io.StringIO(body), dtype=np.float64, comments="%", ndmin=2) if nent else np.zeros((0, ncol_file))
    if data.shape[0] != nent or (nent and data.shape[1] != ncol_file):
        raise ValueError(f"expected {nent} entries of {ncol_file} fields, found {data.shape}")
    rows = data[:, 0].astype(np.int64) - 1
    cols = data[:, 1].astype(np.int64) - 1
    vals = data[:, 2].copy() if field != "pattern" else np.ones(nent, dtype=np.float64)
    if nent and (rows.min() < 0 or cols.min() < 0 or rows.max() >= nrows or cols.max() >= nrows):
        raise ValueError("index out of range")
    if sym == "symmetric":
        off = rows != cols
        rows, cols, vals = (np.concatenate([rows, cols[off]]), np.concatenate([cols, rows[off]]),
                            np.concatenate([vals, vals[off]]))
    if rows.size >= 2 ** 31 - 8:
        raise ValueError("too many entries for int32 CSR indices")
    order = np.lexsort((cols, rows))               # stable: duplicates keep their file order
    rows, cols, vals = rows[order], cols[order], vals[order]
    rowptr = np.zeros(nrows + 1, dtype=np.int64)
    np.add.at(rowptr, rows + 1, 1)
    np.cumsum(rowptr, out=rowptr)
    return nrows, rowptr.astype(np.int32), cols.astype(np.int32), np.ascontiguousarray(vals, dtype=np.float64)


def write_matrix_market(path_or_file, rowptr, colind, vals, symmetric: bool = False, comment: str = "") -> None:
    """Writes CSR arrays as `coordinate real general` (or `symmetric`: the lower triangle only;
    the caller vouches that the matrix is symmetric).  Values are written with 17 significant
    digits so that reading them back reproduces every bit."""
    rowptr = np.asarray(rowptr, dtype=np.int64)
    colind = np.asarray(colind, dtype=np.int64)
    vals = np.asarray(vals, dtype=np.float64)
    n = rowptr.size - 1
    rows = np.repeat(np.arange(n, dtype=np.int64), np.diff(rowptr))
    keep = rows >= colind if symmetric else np.ones(rows.size, dtype=bool)
    f, close = (path_or_file, False) if hasattr(path_or_file, "write") else (open(path_or_file, "w"), True)
    try:
        f.write(f"%%MatrixMarket matrix coordinate real {'symmetric' if symmetric else 'general'}\n")
        for c in comment.splitlines():
            f.write(f"% {c}\n")
        f.write(f"{n} {n} {int(keep.sum())}\n")
        for r, c, v in zip(rows[keep], colind[keep], vals[keep]):
            f.write(f"{r + 1} {c + 1} {v:.17g}\n")
    finally:
        if close:
            f.close()
