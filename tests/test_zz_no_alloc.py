"""cg_dot_static (include/cg.h): the allocation-free dot product, against the existing cg_dot.

Collected last on purpose (the suite runs with pytest -x).  Self-contained: runs alone in a fresh
process as well as after the other tests (it builds its own handles and vectors).
"""
import math

import numpy as np
import pytest

import cg_inputs as gi


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _cg_dot(cg, a, b):
    """The existing path: cg_dot needs a handle of n rows (an identity matrix serves)."""
    n = len(a)
    A = cg.CG(_dev(np.arange(n + 1, dtype=np.int32)), _dev(np.arange(n, dtype=np.int32)), _dev(np.ones(n)),
              compress=False, reorder=False)
    try:
        return A.dot(_dev(a), _dev(b))
    finally:
        A.close()


@pytest.mark.gpu
def test_dot_static_matches_cg_dot_two_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    import paper_1107_0538_b200 as cg
    stream = torch.cuda.current_stream().cuda_stream
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    # two calls in a row on the shared scratch: a large one first, then a smaller one with other data, whose
    # result must not see what the first left behind; then sizes around the 8192-element block edge
    for n, seeds in ((1 << 20, (61, 62)), (132651, (63, 64)), (8193, (65, 66)), (8192, (67, 68)), (8191, (69, 70)), (1, (71, 72))):
        a, b = gi.seeded_vector(seeds[0], n), gi.seeded_vector(seeds[1], n)
        da, db = _dev(a), _dev(b)
        cg.cg_dot_static(n, da.data_ptr(), db.data_ptr(), out.data_ptr(), stream)
        got = float(out.cpu()[0])
        cg.cg_dot_static(n, da.data_ptr(), db.data_ptr(), out.data_ptr(), stream)      # again: same bits
        assert float(out.cpu()[0]) == got
        want = _cg_dot(cg, a, b)
        # the tolerance of test_dot_parity (two fixed-order fp64 sums with different grouping)
        assert abs(got - want) <= 1e-15 * np.sum(np.abs(a * b)) * max(1.0, math.log2(n)), (n, got, want)


@pytest.mark.gpu
def test_dot_static_limits_and_empty_input():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    import paper_1107_0538_b200 as cg
    out = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    v = torch.ones(16, dtype=torch.float64, device="cuda")
    nmax = cg.cg_dot_static_max_n()
    assert nmax == 4096 * 8192
    with pytest.raises(cg.CGError) as e:
        cg.cg_dot_static(nmax + 1, v.data_ptr(), v.data_ptr(), out.data_ptr(), 0)
    assert e.value.code == -6 and "exceeds" in str(e.value)
    with pytest.raises(cg.CGError):
        cg.cg_dot_static(-1, v.data_ptr(), v.data_ptr(), out.data_ptr(), 0)
    with pytest.raises(cg.CGError):
        cg.cg_dot_static(16, v.data_ptr(), v.data_ptr(), 0, 0)
    torch.cuda.synchronize()
    assert float(out.cpu()[0]) == 7.0                      # rejected calls wrote nothing
    cg.cg_dot_static(0, 0, 0, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    assert float(out.cpu()[0]) == 0.0
    cg.cg_dot_static(16, v.data_ptr(), v.data_ptr(), out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    assert float(out.cpu()[0]) == 16.0
