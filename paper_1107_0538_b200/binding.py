"""ctypes binding of libcg_b200 (include/cg.h).  Argument marshalling only.

The module-level functions mirror the C names one to one and take raw integers
(device pointers) exactly like the C ABI.  `CG` is a small convenience wrapper
that takes torch CUDA tensors, owns the workspace tensor and passes
``torch.cuda.current_stream().cuda_stream``; it adds no arithmetic.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional

from . import build as _build

_i64 = ctypes.c_int64
_f64 = ctypes.c_double
_vp = ctypes.c_void_p
_sz = ctypes.c_size_t

# name -> (restype, argtypes); must list every symbol include/cg.h declares
SIGNATURES = {
    "cg_workspace_bytes": (_sz, [_i64]),
    "cg_host_scratch_bytes": (_sz, [_i64, _i64]),
    "cg_create": (ctypes.c_int, [ctypes.POINTER(_vp), _i64, _i64, _vp, _vp, _vp, _vp, _sz]),
    "cg_index_bytes": (_sz, [_vp]),
    "cg_compress_index": (ctypes.c_int, [_vp, _vp, _sz, _vp]),
    "cg_reorder_bytes": (_sz, [_i64, _i64]),
    "cg_reorder": (ctypes.c_int, [_vp, _vp, _sz, _vp]),
    "cg_rcm_host": (ctypes.c_int, [_i64, _vp, _vp, _vp]),
    "cg_check_csr": (ctypes.c_int, [_vp, _vp]),
    "cg_spmv": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "cg_dot": (ctypes.c_int, [_vp, _vp, _vp, ctypes.POINTER(_f64), _vp]),
    "cg_dot_static": (ctypes.c_int, [_i64, _vp, _vp, _vp, _vp]),
    "cg_dot_static_max_n": (_i64, []),
    "cg_solve": (ctypes.c_int, [_vp, _vp, _vp, _f64, _i64, _vp, ctypes.POINTER(_i64),
                                ctypes.POINTER(_f64), _vp]),
    "cg_solve_jacobi": (ctypes.c_int, [_vp, _vp, _vp, _f64, _i64, _vp, ctypes.POINTER(_i64),
                                       ctypes.POINTER(_f64), _vp]),
    "cg_solve_host": (ctypes.c_int, [_vp, _vp, _vp, _f64, _i64, _vp, ctypes.POINTER(_i64),
                                     ctypes.POINTER(_f64), _vp, _sz, _vp]),
    "cg_probe_read_bandwidth": (ctypes.c_int, [_vp, _vp, _sz, ctypes.c_int, ctypes.POINTER(_f64), _vp]),
    "cg_probe_grid_sync": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, ctypes.POINTER(_f64), _vp]),
    "cg_set_trace": (ctypes.c_int, [_vp, _vp, _i64]),
    "cg_set_option": (ctypes.c_int, [_vp, ctypes.c_char_p, _i64]),
    "cg_get_info": (ctypes.c_int, [_vp, ctypes.c_char_p, ctypes.POINTER(_i64)]),
    "cg_destroy": (ctypes.c_int, [_vp]),
    "cg_strerror": (ctypes.c_char_p, [ctypes.c_int]),
}

_lib = None


def lib() -> ctypes.CDLL:
    """Load (building if stale) libcg_b200.so.  Raises when it cannot: no fallback."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if _build.is_stale():
            path = _build.build()
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing and could not be built")
        L = ctypes.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


class CGError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {cg_strerror(code)} (code {code})")


def cg_strerror(code: int) -> str:
    return lib().cg_strerror(int(code)).decode()


def cg_workspace_bytes(n: int) -> int:
    return int(lib().cg_workspace_bytes(n))


def cg_host_scratch_bytes(n: int, maxit: int) -> int:
    return int(lib().cg_host_scratch_bytes(n, maxit))


def cg_create(n: int, nnz: int, d_rowptr: int, d_colind: int, d_vals: int,
              d_workspace: int, workspace_bytes: int) -> int:
    """Returns the opaque handle (as int).  Raises CGError on a negative code."""
    out = _vp()
    rc = lib().cg_create(ctypes.byref(out), n, nnz, d_rowptr, d_colind, d_vals, d_workspace,
                         workspace_bytes)
    if rc != 0:
        raise CGError(rc, "cg_create")
    return out.value


def cg_destroy(h: int) -> None:
    lib().cg_destroy(h)


def cg_index_bytes(h: int) -> int:
    return int(lib().cg_index_bytes(h))


def cg_compress_index(h: int, d_index: int, index_bytes: int, stream: int = 0) -> int:
    """Returns 0 (compressed index in use) or 3 (CG_NOTCOMPRESSED); raises on errors."""
    rc = lib().cg_compress_index(h, d_index, index_bytes, stream)
    if rc < 0:
        raise CGError(rc, "cg_compress_index")
    return rc


def cg_reorder_bytes(n: int, nnz: int) -> int:
    return int(lib().cg_reorder_bytes(n, nnz))


def cg_reorder(h: int, d_buf: int, nbytes: int, stream: int = 0) -> int:
    """Returns 0 (solves now run on the renumbered matrix) or 4 (CG_NOTREORDERED); raises on errors."""
    rc = lib().cg_reorder(h, d_buf, nbytes, stream)
    if rc < 0:
        raise CGError(rc, "cg_reorder")
    return rc


def cg_rcm_host(n: int, h_rowptr: int, h_colind: int, h_perm: int) -> None:
    """Host arrays (raw addresses): int32 rowptr[n+1], colind[nnz] in, int32 perm[n] out."""
    rc = lib().cg_rcm_host(n, h_rowptr, h_colind, h_perm)
    if rc != 0:
        raise CGError(rc, "cg_rcm_host")


def cg_check_csr(h: int, stream: int = 0) -> int:
    return int(lib().cg_check_csr(h, stream))


def cg_spmv(h: int, d_x: int, d_y: int, stream: int = 0) -> None:
    rc = lib().cg_spmv(h, d_x, d_y, stream)
    if rc != 0:
        raise CGError(rc, "cg_spmv")


def cg_dot(h: int, d_a: int, d_b: int, stream: int = 0) -> float:
    out = _f64()
    rc = lib().cg_dot(h, d_a, d_b, ctypes.byref(out), stream)
    if rc != 0:
        raise CGError(rc, "cg_dot")
    return out.value


def cg_dot_static(n: int, d_a: int, d_b: int, d_result: int, stream: int = 0) -> None:
    """Handle-free, allocation-free dot product into DEVICE memory d_result; asynchronous on the stream."""
    rc = lib().cg_dot_static(n, d_a, d_b, d_result, stream)
    if rc != 0:
        raise CGError(rc, "cg_dot_static")


def cg_dot_static_max_n() -> int:
    return int(lib().cg_dot_static_max_n())


def _solve(fn_name, h, d_b, d_x, rtol, maxit, d_hist, stream):
    it, res = _i64(), _f64()
    rc = getattr(lib(), fn_name)(h, d_b, d_x, rtol, maxit, d_hist, ctypes.byref(it),
                                 ctypes.byref(res), stream)
    if rc < 0:
        raise CGError(rc, fn_name)
    return rc, it.value, res.value


def cg_solve(h: int, d_b: int, d_x: int, rtol: float, maxit: int, d_hist: Optional[int] = None,
             stream: int = 0):
    """Returns (status, iters, final_resnorm); status 0 converged, 1 maxit, 2 breakdown."""
    return _solve("cg_solve", h, d_b, d_x, rtol, maxit, d_hist, stream)


def cg_solve_jacobi(h: int, d_b: int, d_x: int, rtol: float, maxit: int,
                    d_hist: Optional[int] = None, stream: int = 0):
    return _solve("cg_solve_jacobi", h, d_b, d_x, rtol, maxit, d_hist, stream)


def cg_solve_host(h: int, h_b: int, h_x: int, rtol: float, maxit: int, h_hist: Optional[int],
                  d_scratch: int, scratch_bytes: int, stream: int = 0):
    it, res = _i64(), _f64()
    rc = lib().cg_solve_host(h, h_b, h_x, rtol, maxit, h_hist, ctypes.byref(it), ctypes.byref(res),
                             d_scratch, scratch_bytes, stream)
    if rc < 0:
        raise CGError(rc, "cg_solve_host")
    return rc, it.value, res.value


def cg_set_option(h: int, name: str, value: int) -> None:
    rc = lib().cg_set_option(h, name.encode(), value)
    if rc != 0:
        raise CGError(rc, f"cg_set_option({name}={value})")


def cg_probe_read_bandwidth(h: int, d_buf: int, nbytes: int, reps: int, stream: int = 0) -> float:
    out = _f64()
    rc = lib().cg_probe_read_bandwidth(h, d_buf, nbytes, reps, ctypes.byref(out), stream)
    if rc != 0:
        raise CGError(rc, "cg_probe_read_bandwidth")
    return out.value


def cg_probe_grid_sync(h: int, kind: int, reps: int, stream: int = 0) -> float:
    """Mean cycles per grid synchronisation of `kind` (0 counter barrier, 1 relaxed all-reduce mix, 2 fenced)."""
    out = _f64()
    rc = lib().cg_probe_grid_sync(h, kind, reps, ctypes.byref(out), stream)
    if rc != 0:
        raise CGError(rc, "cg_probe_grid_sync")
    return out.value


def cg_set_trace(h: int, d_trace: Optional[int], iters: int) -> None:
    rc = lib().cg_set_trace(h, d_trace, iters)
    if rc != 0:
        raise CGError(rc, "cg_set_trace")


def cg_get_info(h: int, name: str) -> int:
    out = _i64()
    rc = lib().cg_get_info(h, name.encode(), ctypes.byref(out))
    if rc != 0:
        raise CGError(rc, f"cg_get_info({name})")
    return out.value


# ---------------------------------------------------------------- torch convenience

@dataclass
class CGResult:
    status: int
    iters: int
    resnorm: float
    hist: "object"          # torch tensor on the device, ||r_j||_2 for j = 0..iters


class CG:
    """Handle bound to CSR arrays held in torch CUDA tensors (kept alive here)."""

    def __init__(self, rowptr, colind, vals, compress: bool = True, reorder: bool = True):
        import torch
        if not (rowptr.is_cuda and colind.is_cuda and vals.is_cuda):
            raise ValueError("CSR arrays must be CUDA tensors (there is no CPU path)")
        if rowptr.dtype != torch.int32 or colind.dtype != torch.int32 or vals.dtype != torch.float64:
            raise ValueError("expected int32 rowptr/colind and float64 vals")
        self.torch = torch
        self.rowptr, self.colind, self.vals = rowptr.contiguous(), colind.contiguous(), vals.contiguous()
        self.n = self.rowptr.numel() - 1
        self.nnz = self.colind.numel()
        self.device = vals.device
        wb = cg_workspace_bytes(self.n)
        self.workspace = torch.empty(wb, dtype=torch.uint8, device=self.device)
        torch.cuda.synchronize(self.device)          # cg_create reads rowptr on the legacy stream
        self.h = cg_create(self.n, self.nnz, self.rowptr.data_ptr(), self.colind.data_ptr(),
                           self.vals.data_ptr(), self.workspace.data_ptr(), wb)
        self._scratch = None
        self.index = None
        self.renumbered = None
        if compress:
            self.compress()
        # irregular gathers (more than 8 lines per warp-wide gather, the library's own threshold for
        # "irregular"): let the library renumber the matrix for the solves
        if reorder and self.info("lines_per_gather_x100") > 800:
            self.reorder()

    def compress(self) -> bool:
        """Build the compressed column index (cg_compress_index) in a tensor owned here.
        Returns True when the handle now uses it."""
        nb = cg_index_bytes(self.h)
        if nb == 0:
            return False
        buf = self.torch.empty(nb, dtype=self.torch.uint8, device=self.device)
        rc = cg_compress_index(self.h, buf.data_ptr(), nb, self._stream())
        self.index = buf if rc == 0 else None
        return rc == 0

    def reorder(self) -> bool:
        """Reverse Cuthill-McKee renumbering for the solves (cg_reorder) in a tensor owned here.
        Returns True when the handle now solves on the renumbered matrix."""
        nb = cg_reorder_bytes(self.n, self.nnz)
        buf = self.torch.empty(nb, dtype=self.torch.uint8, device=self.device)
        rc = cg_reorder(self.h, buf.data_ptr(), nb, self._stream())
        self.renumbered = buf if rc == 0 else None
        return rc == 0

    def close(self):
        if getattr(self, "h", None):
            cg_destroy(self.h)
            self.h = None

    __del__ = close

    def _stream(self):
        return self.torch.cuda.current_stream(self.device).cuda_stream

    def set_option(self, name, value):
        cg_set_option(self.h, name, value)

    def info(self, name):
        return cg_get_info(self.h, name)

    def trace(self, iters: int):
        """Switch the persistent loop's phase trace on (returns the uint64 device tensor
        [grid, iters + 1, 16] later solves fill (row `iters`: producer / wait statistics)) or, with iters = 0, off."""
        if iters <= 0:
            cg_set_trace(self.h, None, 0)
            self._trace = None
            return None
        self._trace = self.torch.zeros((self.info("grid"), iters + 1, 16), dtype=self.torch.int64,
                                       device=self.device)
        cg_set_trace(self.h, self._trace.data_ptr(), iters)
        return self._trace

    def probe_read_bandwidth(self, nbytes: int, reps: int = 20) -> float:
        """GB/s of a read-only sweep over a scratch buffer of nbytes (L2 if it fits, else HBM)."""
        buf = self.torch.ones(nbytes // 4, dtype=self.torch.int32, device=self.device)
        return cg_probe_read_bandwidth(self.h, buf.data_ptr(), buf.numel() * 4, reps, self._stream())

    def probe_grid_sync(self, kind: int, reps: int = 2000) -> float:
        return cg_probe_grid_sync(self.h, kind, reps, self._stream())

    def check_csr(self) -> bool:
        return cg_check_csr(self.h, self._stream()) == 0

    def spmv(self, x, out=None):
        if out is None:
            out = self.torch.empty_like(x)
        cg_spmv(self.h, x.data_ptr(), out.data_ptr(), self._stream())
        return out

    def dot(self, a, b) -> float:
        return cg_dot(self.h, a.data_ptr(), b.data_ptr(), self._stream())

    def solve(self, b, x0=None, rtol=1e-10, maxit=None, jacobi=False, want_hist=True) -> tuple:
        """Returns (x, CGResult).  x0 is copied; b is not modified."""
        torch = self.torch
        maxit = self.n if maxit is None else int(maxit)
        x = torch.zeros_like(b) if x0 is None else x0.clone()
        hist = torch.zeros(maxit + 1, dtype=torch.float64, device=self.device) if want_hist else None
        fn = cg_solve_jacobi if jacobi else cg_solve
        st, it, res = fn(self.h, b.data_ptr(), x.data_ptr(), float(rtol), maxit,
                         hist.data_ptr() if want_hist else None, self._stream())
        return x, CGResult(st, it, res, hist[:it + 1] if want_hist else None)

    def solve_host(self, b_host, x_host, rtol, maxit, hist_host=None):
        """End-to-end entry: pinned (or pageable) HOST torch tensors in, results copied back."""
        torch = self.torch
        sb = cg_host_scratch_bytes(self.n, maxit)
        if self._scratch is None or self._scratch.numel() < sb:
            self._scratch = torch.empty(sb, dtype=torch.uint8, device=self.device)
        return cg_solve_host(self.h, b_host.data_ptr(), x_host.data_ptr(), float(rtol), int(maxit),
                             None if hist_host is None else hist_host.data_ptr(),
                             self._scratch.data_ptr(), self._scratch.numel(), self._stream())
