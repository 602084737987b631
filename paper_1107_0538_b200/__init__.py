"""paper_1107_0538_b200: fp64 CSR conjugate gradient for one B200 (sm_100a).

Thin Python binding over the C-ABI library declared in include/cg.h.  Every step of
the path (SpMV, dots, AXPYs, scalar recurrences, the loop) runs in the CUDA kernels of
csrc/; Python only marshals pointers.  PyTorch supplies device memory and streams.
There is no CPU fallback: importing the binding without a built/buildable
libcg_b200.so raises.
"""
from .binding import (CG, CGError, CGResult, lib, cg_create, cg_destroy, cg_spmv, cg_dot, cg_solve,
                      cg_solve_jacobi, cg_solve_host, cg_check_csr, cg_workspace_bytes,
                      cg_host_scratch_bytes, cg_set_option, cg_get_info, cg_strerror, cg_set_trace,
                      cg_probe_read_bandwidth, cg_index_bytes, cg_compress_index, cg_probe_grid_sync,
                      cg_reorder_bytes, cg_reorder, cg_rcm_host, cg_dot_static, cg_dot_static_max_n)

__all__ = ["CG", "CGError", "CGResult", "lib", "cg_create", "cg_destroy", "cg_spmv", "cg_dot",
           "cg_solve", "cg_solve_jacobi", "cg_solve_host", "cg_check_csr", "cg_workspace_bytes",
           "cg_host_scratch_bytes", "cg_set_option", "cg_get_info", "cg_strerror", "cg_set_trace",
           "cg_probe_read_bandwidth", "cg_index_bytes", "cg_compress_index", "cg_probe_grid_sync",
           "cg_reorder_bytes", "cg_reorder", "cg_rcm_host", "cg_dot_static", "cg_dot_static_max_n"]
