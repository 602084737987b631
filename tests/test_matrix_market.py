"""Matrix Market loader (PAPER.md:34 / :42 "data reading"): CPU tests of the
parser, and one -m gpu test that runs a loaded matrix through cg_solve against the oracle."""
import io
import os

import numpy as np
import pytest

import cg_inputs as gi
from paper_1107_0538_b200.matrix_market import read_matrix_market, write_matrix_market

HERE = os.path.dirname(os.path.abspath(__file__))
FIXTURE = os.path.join(HERE, "golden", "fem_4cubed_27pt_symmetric.mtx")


def dense(n, rp, ci, va):
    A = np.zeros((n, n))
    for i in range(n):
        for k in range(rp[i], rp[i + 1]):
            A[i, ci[k]] += va[k]
    return A


def test_general_real_file():
    txt = """%%MatrixMarket matrix coordinate real general
% a comment
3 3 5
3 1 -1.5
1 1 2
2 2 4e0
1 3 0.25
3 3 1
"""
    n, rp, ci, va = read_matrix_market(io.StringIO(txt))
    assert n == 3 and rp.dtype == np.int32 and ci.dtype == np.int32 and va.dtype == np.float64
    assert rp.tolist() == [0, 2, 3, 5] and ci.tolist() == [0, 2, 1, 0, 2]
    np.testing.assert_array_equal(dense(n, rp, ci, va), [[2, 0, 0.25], [0, 4, 0], [-1.5, 0, 1]])


def test_symmetric_expansion_pattern_and_duplicates():
    sym = "%%MatrixMarket matrix coordinate integer symmetric\n3 3 4\n1 1 2\n2 1 -1\n3 2 -1\n3 3 5\n"
    n, rp, ci, va = read_matrix_market(io.StringIO(sym))
    A = dense(n, rp, ci, va)
    np.testing.assert_array_equal(A, [[2, -1, 0], [-1, 0, -1], [0, -1, 5]])
    assert np.array_equal(A, A.T) and len(va) == 6                     # the diagonal is not doubled
    pat = "%%MatrixMarket matrix coordinate pattern general\n2 2 2\n1 2\n2 1\n"
    n, rp, ci, va = read_matrix_market(io.StringIO(pat))
    np.testing.assert_array_equal(dense(n, rp, ci, va), [[0, 1], [1, 0]])
    dup = "%%MatrixMarket matrix coordinate real general\n2 2 3\n1 1 1.0\n1 1 2.5\n2 2 1\n"
    n, rp, ci, va = read_matrix_market(io.StringIO(dup))
    assert rp.tolist() == [0, 2, 3] and va.tolist() == [1.0, 2.5, 1.0]  # kept, in file order: CSR duplicates add


@pytest.mark.parametrize("bad", [
    "%%MatrixMarket matrix array real general\n2 2\n1\n2\n3\n4\n",
    "%%MatrixMarket matrix coordinate complex general\n1 1 1\n1 1 1 0\n",
    "%%MatrixMarket matrix coordinate real hermitian\n1 1 1\n1 1 1\n",
    "%%MatrixMarket matrix coordinate real general\n2 3 1\n1 1 1\n",
    "%%MatrixMarket matrix coordinate real general\n2 2 1\n3 1 1\n",
    "%%MatrixMarket matrix coordinate real general\n2 2 2\n1 1 1\n",
    "not a header\n",
])
def test_rejects_what_it_does_not_support(bad):
    with pytest.raises(ValueError):
        read_matrix_market(io.StringIO(bad))


def test_fixture_round_trip_bitwise():
    """The committed fixture is the lower triangle of cg_inputs.stencil27(4); expanding it gives
    the generator's CSR arrays back bit for bit, and writing + reading the full matrix too."""
    rp, ci, va = gi.stencil27(4)
    n, rp2, ci2, va2 = read_matrix_market(FIXTURE)
    assert n == 64 and np.array_equal(rp, rp2) and np.array_equal(ci, ci2) and np.array_equal(va, va2)
    buf = io.StringIO()
    write_matrix_market(buf, rp, ci, va)
    buf.seek(0)
    n3, rp3, ci3, va3 = read_matrix_market(buf)
    assert np.array_equal(rp, rp3) and np.array_equal(ci, ci3) and np.array_equal(va, va3)


@pytest.mark.gpu
def test_loaded_matrix_through_cg_solve():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    import paper_1107_0538_b200 as cg
    from oracle import cg_oracle as orc
    n, rp, ci, va = read_matrix_market(FIXTURE)
    b = gi.seeded_vector(11, n)
    ref = orc.cg(rp, ci, va, b, rtol=1e-8, maxit=n)     # (a 64-row system: below ~1e-10 its residual norms are rounding noise)
    A = cg.CG(*(torch.from_numpy(a).cuda() for a in (rp, ci, va)))
    assert A.check_csr()
    for loop in (0, 1):
        A.set_option("loop", loop)
        x, res = A.solve(torch.from_numpy(b).cuda(), rtol=1e-8, maxit=n)
        assert res.status == 0 and abs(res.iters - ref.iters) <= 1
        k = min(50, ref.iters, res.iters)
        h = res.hist.cpu().numpy()
        assert np.max(np.abs(h[:k + 1] - ref.hist[:k + 1]) / ref.hist[:k + 1]) <= 1e-9
        assert np.linalg.norm(x.cpu().numpy() - ref.x) / np.linalg.norm(ref.x) <= 1e-8
    A.close()
