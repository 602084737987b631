"""cg_reorder (include/cg.h): reverse Cuthill-McKee renumbering for matrices with irregular gathers.

CPU part: cg_rcm_host is a pure host routine (no device needed): permutation validity, determinism,
bandwidth on the permuted stencil, disconnected components, empty rows, bad arguments.
GPU part: solves on the renumbered matrix are held to the same four parity bands against the oracle.
"""
import numpy as np
import pytest

import cg_inputs


def rcm(p_rowptr, p_colind):
    import paper_1107_0538_b200 as cg
    n = len(p_rowptr) - 1
    rp = np.ascontiguousarray(p_rowptr, dtype=np.int32)
    ci = np.ascontiguousarray(p_colind, dtype=np.int32)
    perm = np.full(n, -1, dtype=np.int32)
    cg.cg_rcm_host(n, rp.ctypes.data, ci.ctypes.data if len(ci) else 0, perm.ctypes.data)
    return perm


def bandwidth(rowptr, colind, inv):
    rows = np.repeat(np.arange(len(rowptr) - 1), np.diff(rowptr))
    return int(np.abs(inv[colind] - inv[rows]).max())


def test_rcm_is_a_permutation_and_cuts_the_bandwidth():
    p = cg_inputs.make_config(3, 14)                      # 14^3 27-point stencil, randomly permuted
    perm = rcm(p.rowptr, p.colind)
    assert np.array_equal(np.sort(perm), np.arange(p.n))
    assert np.array_equal(perm, rcm(p.rowptr, p.colind))  # a pure function of the pattern
    inv = np.empty(p.n, dtype=np.int64)
    inv[perm] = np.arange(p.n)
    before = bandwidth(p.rowptr, p.colind, np.arange(p.n))
    after = bandwidth(p.rowptr, p.colind, inv)
    # natural ordering of an n^3 27-point grid has bandwidth n^2 + n + 1 = 211; the level sets of the
    # search are at most 3 n^2 wide
    assert before > 2000 and after <= 3 * 14 * 14


def test_rcm_path_graph_gives_the_path_order():
    # a path 0-1-2-...-9 hidden under a permutation: RCM must number it end to end (bandwidth 1)
    n = 10
    rng = np.random.default_rng(5)
    lab = rng.permutation(n)
    rows = [[] for _ in range(n)]
    for a in range(n):
        for b in (a - 1, a, a + 1):
            if 0 <= b < n:
                rows[lab[a]].append(lab[b])
    rowptr = np.zeros(n + 1, dtype=np.int32)
    rowptr[1:] = np.cumsum([len(r) for r in rows])
    colind = np.array([c for r in rows for c in r], dtype=np.int32)
    perm = rcm(rowptr, colind)
    inv = np.empty(n, dtype=np.int64)
    inv[perm] = np.arange(n)
    assert bandwidth(rowptr, colind, inv) == 1


def test_rcm_components_and_empty_rows():
    # two triangles, one isolated node with a diagonal entry, one empty row
    edges = [(0, 1), (1, 2), (0, 2), (3, 4), (4, 5), (3, 5)]
    n = 8
    rows = [[i] if i != 7 else [] for i in range(n)]
    for a, b in edges:
        rows[a].append(b)
        rows[b].append(a)
    rowptr = np.zeros(n + 1, dtype=np.int32)
    rowptr[1:] = np.cumsum([len(r) for r in rows])
    colind = np.array([c for r in rows for c in r], dtype=np.int32)
    perm = rcm(rowptr, colind)
    assert np.array_equal(np.sort(perm), np.arange(n))
    inv = np.empty(n, dtype=np.int64)
    inv[perm] = np.arange(n)
    for comp in ([0, 1, 2], [3, 4, 5]):                   # every component is numbered contiguously
        assert inv[comp].max() - inv[comp].min() == 2


def test_rcm_rejects_bad_arguments():
    import paper_1107_0538_b200 as cg
    rp = np.array([0, 2, 1], dtype=np.int32)              # decreasing row pointer
    ci = np.array([0, 1], dtype=np.int32)
    perm = np.zeros(2, dtype=np.int32)
    with pytest.raises(cg.CGError):
        cg.cg_rcm_host(2, rp.ctypes.data, ci.ctypes.data, perm.ctypes.data)
    with pytest.raises(cg.CGError):
        cg.cg_rcm_host(0, rp.ctypes.data, ci.ctypes.data, perm.ctypes.data)
    assert cg.cg_reorder_bytes(0, 0) == 0
    assert cg.cg_reorder_bytes(1000, 27000) >= 12 * 27000 + 24 * 1000 + cg.cg_workspace_bytes(1000)


# ---------------------------------------------------------------- GPU: solves on the renumbered matrix

HIST_TOL, X_TOL = 1e-9, 1e-8


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _parity(res, x, ref):
    k = min(50, ref.iters, res.iters)
    h = res.hist.cpu().numpy()
    assert np.max(np.abs(h[:k + 1] - ref.hist[:k + 1]) / ref.hist[:k + 1]) <= HIST_TOL
    assert abs(res.iters - ref.iters) <= max(1, int(0.02 * ref.iters)), (res.iters, ref.iters)
    assert np.linalg.norm(x.cpu().numpy() - ref.x) / np.linalg.norm(ref.x) <= X_TOL
    assert res.status == ref.status and len(h) == res.iters + 1


@pytest.fixture(scope="module")
def cfg3(problems):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    import paper_1107_0538_b200 as cg
    from oracle import cg_oracle as orc
    p = problems(3)
    A = cg.CG(_dev(p.rowptr), _dev(p.colind), _dev(p.vals))
    ref = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit)
    yield cg, orc, p, A, ref
    A.close()


@pytest.mark.gpu
def test_reorder_is_used_on_the_permuted_matrix(cfg3):
    """Config 3: the binding asks for the renumbering (30 lines per warp-wide gather), the library takes
    it (fewer than 6 afterwards) and the solve runs gather + persistent kernel + scatter."""
    cg, orc, p, A, ref = cfg3
    assert A.info("lines_per_gather_x100") > 2000
    assert A.info("reordered") == 1 and A.info("solve_lines_per_gather_x100") < 600
    x, res = A.solve(_dev(p.b), rtol=p.rtol, maxit=p.maxit)
    assert A.info("launches") == 3
    _parity(res, x, ref)
    # the caller's matrix still serves cg_spmv, entry by entry
    xv = cg_inputs.seeded_vector(9, p.n)
    y = A.spmv(_dev(xv)).cpu().numpy()
    want = orc.spmv(p.rowptr, p.colind, p.vals, xv)
    assert np.all(np.abs(y - want) <= 1e-13 * orc.absrow(p.rowptr, p.colind, p.vals, xv))


@pytest.mark.gpu
@pytest.mark.parametrize("loop,algo,jacobi", [(0, 0, False), (1, 0, False), (2, 0, False), (0, 1, False),
                                              (0, 2, False), (0, 0, True)])
def test_reorder_parity_all_loops(cfg3, loop, algo, jacobi):
    cg, orc, p, A, ref = cfg3
    A.set_option("loop", loop)
    A.set_option("algo", algo)
    try:
        if jacobi:
            dinv = 1.0 / p.vals[[np.searchsorted(p.colind[p.rowptr[i]:p.rowptr[i + 1]], i) + p.rowptr[i]
                                 for i in range(p.n)]]
            refj = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit, dinv=dinv)
            x, res = A.solve(_dev(p.b), rtol=p.rtol, maxit=p.maxit, jacobi=True)
            _parity(res, x, refj)
        else:
            x, res = A.solve(_dev(p.b), rtol=p.rtol, maxit=p.maxit)
            _parity(res, x, ref)
        # run twice: same bits
        x2, res2 = A.solve(_dev(p.b), rtol=p.rtol, maxit=p.maxit, jacobi=jacobi)
        import torch
        assert torch.equal(x, x2) and torch.equal(res.hist, res2.hist)
    finally:
        A.set_option("loop", 0)
        A.set_option("algo", 0)


@pytest.mark.gpu
def test_reorder_switch_nonzero_x0_and_host_entry(cfg3):
    """"reorder" = 0 goes back to the caller's numbering; a non-zero x0 travels through the gather;
    cg_solve_host runs on the renumbered matrix too; "values_changed" drops the copy."""
    import torch
    cg, orc, p, A, ref = cfg3
    b = _dev(p.b)
    A.set_option("reorder", 0)
    assert A.info("reordered") == 0
    x0, r0 = A.solve(b, rtol=p.rtol, maxit=p.maxit)
    assert A.info("launches") == 1
    _parity(r0, x0, ref)
    A.set_option("reorder", 1)
    start = cg_inputs.seeded_vector(11, p.n)
    refs = orc.cg(p.rowptr, p.colind, p.vals, p.b, x0=start, rtol=p.rtol, maxit=p.maxit)
    x, res = A.solve(b, x0=_dev(start), rtol=p.rtol, maxit=p.maxit)
    _parity(res, x, refs)
    hb = torch.from_numpy(p.b.copy()).pin_memory()
    hx = torch.zeros(p.n, dtype=torch.float64).pin_memory()
    hh = torch.zeros(p.maxit + 1, dtype=torch.float64).pin_memory()
    st, it, rn = A.solve_host(hb, hx, p.rtol, p.maxit, hh)
    assert st == 0 and abs(it - ref.iters) <= max(1, int(0.02 * ref.iters))
    assert np.linalg.norm(hx.numpy() - ref.x) / np.linalg.norm(ref.x) <= X_TOL
    A.set_option("values_changed", 1)
    assert A.info("reordered") == 0
    assert A.reorder() and A.info("reordered") == 1


@pytest.mark.gpu
def test_reorder_declined_on_a_well_numbered_matrix(problems):
    """Natural ordering (config 0): the renumbering cannot cut the lines per gather by a third, the
    library says so (CG_NOTREORDERED) and keeps solving in the caller's numbering."""
    import paper_1107_0538_b200 as cg
    p = problems(0)
    A = cg.CG(_dev(p.rowptr), _dev(p.colind), _dev(p.vals))
    assert A.info("reordered") == 0                       # the binding did not even ask
    assert A.reorder() is False and A.info("reordered") == 0
    x, res = A.solve(_dev(p.b), rtol=p.rtol, maxit=p.maxit)
    assert res.status == 0 and A.info("launches") == 1
    A.close()


@pytest.mark.gpu
def test_reorder_with_rows_longer_than_the_sorting_limit(problems):
    """A 14^3 stencil plus one node coupled to the 400 nodes around it (a local 'arrow'), then randomly
    permuted: that row (and no other) is longer than the 256 entries cg_reorder sorts in registers, so it
    keeps its stored order; the renumbering is still taken, and the solve must match the oracle within the
    bands in both numberings."""
    import scipy.sparse as sp
    import paper_1107_0538_b200 as cg
    from oracle import cg_oracle as orc
    p = problems(2, 14)
    n = p.n
    A0 = sp.csr_matrix((p.vals, p.colind, p.rowptr), shape=(n, n))
    rng = np.random.default_rng(7)
    hub = n // 2
    others = np.setdiff1d(np.arange(hub - 200, hub + 201), [hub])
    w = 1e-3 * (1.0 + rng.random(len(others)))
    arrow = sp.coo_matrix((np.concatenate([-w, -w]), (np.concatenate([np.full(len(others), hub), others]),
                                                       np.concatenate([others, np.full(len(others), hub)]))), shape=(n, n))
    diag = np.zeros(n)
    diag[hub] = w.sum()
    diag[others] = w
    A = (A0 + arrow + sp.diags(diag)).tocsr()                 # still symmetric and strictly diagonally dominant
    perm = rng.permutation(n)
    A = A[perm][:, perm].tocsr()
    A.sort_indices()
    rp, ci, va = A.indptr.astype(np.int32), A.indices.astype(np.int32), A.data.astype(np.float64)
    assert np.diff(rp).max() > 256
    b = cg_inputs.seeded_vector(21, n)
    ref = orc.cg(rp, ci, va, b, rtol=1e-10, maxit=n)
    H = cg.CG(_dev(rp), _dev(ci), _dev(va), reorder=False)
    x0, r0 = H.solve(_dev(b), rtol=1e-10, maxit=n)
    _parity(r0, x0, ref)
    assert H.reorder() and H.info("reordered") == 1           # kept: the gathers become more local
    x1, r1 = H.solve(_dev(b), rtol=1e-10, maxit=n)
    _parity(r1, x1, ref)
    assert H.info("launches") == 3
    H.close()
