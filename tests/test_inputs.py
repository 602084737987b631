"""Structure checks of the seeded generator (SURVEY.md 8(c) "Generator" pins, 8(d) recipe)."""
import numpy as np
import pytest

import cg_inputs as gi


def _to_dense(rp, ci, va):
    n = len(rp) - 1
    A = np.zeros((n, n))
    for i in range(n):
        for k in range(rp[i], rp[i + 1]):
            A[i, ci[k]] += va[k]
    return A


def test_hash_reference_values():
    # frozen hash: splitmix64 finaliser, values computed by hand-rolled Python ints
    def mix(z):
        m = (1 << 64) - 1
        z &= m
        z ^= z >> 30; z = z * 0xBF58476D1CE4E5B9 & m
        z ^= z >> 27; z = z * 0x94D049BB133111EB & m
        z ^= z >> 31
        return z
    for seed, stream, key in [(0, 1, 0), (2, 2, 17), (3, 3, 132650), (0, 1, 132651 * 132650 + 7)]:
        k = mix(seed * 0x100000001B3 + stream)
        want = (mix(k ^ key) >> 11) * 2.0 ** -53
        got = gi.hash_uniform(seed, stream, np.array([key], dtype=np.uint64))[0]
        assert got == want
        assert 0.0 <= got < 1.0


def test_hash_is_roughly_uniform():
    u = gi.hash_uniform(5, 2, np.arange(200000, dtype=np.uint64))
    assert abs(u.mean() - 0.5) < 5e-3
    assert abs(u.var() - 1 / 12) < 2e-3
    assert u.min() >= 0 and u.max() < 1


@pytest.mark.parametrize("n", [2, 3, 5, 16])
def test_stencil27_structure(n):
    rp, ci, va = gi.stencil27(n)
    N = n ** 3
    assert rp.dtype == np.int32 and ci.dtype == np.int32 and va.dtype == np.float64
    assert rp[0] == 0 and rp[-1] == len(ci) == len(va) == (3 * n - 2) ** 3
    lens = np.diff(rp)
    allowed = {8, 12, 18, 27} if n >= 3 else {8}
    assert set(lens.tolist()) <= allowed
    for i in range(N):                       # ascending unique columns
        row = ci[rp[i]:rp[i + 1]]
        assert np.all(np.diff(row) > 0)
        assert i in row


def test_config_sizes_match_paper():
    # PAPER.md:34 / :60: N = 132651, NNZ = 3442951
    p = gi.make_config(2)
    assert p.n == 132651 and p.nnz == 3442951
    assert p.rtol == 1e-10 and p.maxit == 132651
    lens = np.diff(p.rowptr)
    vals, cnt = np.unique(lens, return_counts=True)
    assert dict(zip(vals.tolist(), cnt.tolist())) == {8: 8, 12: 588, 18: 14406, 27: 117649}
    assert gi.make_config(0).nnz == 97336
    assert gi.make_config(1).nnz == 1810432


def test_symmetry_and_diagonal_rule_small():
    rp, ci, va = gi.stencil27(4)
    A = _to_dense(rp, ci, va)
    assert np.array_equal(A, A.T)                       # bitwise symmetric
    off = A - np.diag(np.diag(A))
    assert np.all(off <= 0) and np.all(np.diag(A) > 0)
    w = -off[off != 0]
    assert w.min() >= 0.5 and w.max() < 1.5
    np.testing.assert_allclose(A.sum(axis=1), 0.01, rtol=0, atol=1e-13 * np.abs(A).sum(axis=1).max())
    ev = np.linalg.eigvalsh(A)
    gersh = 2 * np.abs(off).sum(axis=1).max() + 0.01
    assert ev.min() >= 0.01 - 1e-12 and ev.max() <= gersh


def test_contrast_rule_small():
    n = 8
    rp, ci, va = gi.stencil27(n, contrast=1000.0, cyl_radius=2.0)
    rp1, ci1, va1 = gi.stencil27(n)
    assert np.array_equal(rp, rp1) and np.array_equal(ci, ci1)
    A, A1 = _to_dense(rp, ci, va), _to_dense(rp1, ci1, va1)
    assert np.array_equal(A, A.T)
    ids = np.arange(n ** 3)
    c = (n - 1) / 2
    inside = ((ids % n) - c) ** 2 + (((ids // n) % n) - c) ** 2 <= 4.0
    both = np.outer(inside, inside)
    offmask = (A1 != 0) & ~np.eye(n ** 3, dtype=bool)
    np.testing.assert_array_equal(A[offmask & both], A1[offmask & both] * 1000.0)
    np.testing.assert_array_equal(A[offmask & ~both], A1[offmask & ~both])
    assert inside.any() and (~inside).any()


def test_laplacian7_small_matches_kron():
    n = 4
    rp, ci, va = gi.laplacian7(n)
    T = 2 * np.eye(n) - np.eye(n, k=1) - np.eye(n, k=-1)
    I = np.eye(n)
    K = np.kron(np.kron(I, I), T) + np.kron(np.kron(I, T), I) + np.kron(np.kron(T, I), I)
    assert np.array_equal(_to_dense(rp, ci, va), K)


def test_permutation_is_similarity():
    rp, ci, va = gi.stencil27(4)
    rp2, ci2, va2, pi = gi.permute_symmetric(rp, ci, va, seed=3)
    A, B = _to_dense(rp, ci, va), _to_dense(rp2, ci2, va2)
    assert sorted(pi.tolist()) == list(range(64))
    assert np.array_equal(B[np.ix_(pi, pi)], A)
    for i in range(64):
        assert np.all(np.diff(ci2[rp2[i]:rp2[i + 1]]) > 0)


def test_config3_is_config2_permuted(problems):
    p2, p3 = problems(2), problems(3)
    pi = p3.meta["perm"]
    assert np.array_equal(np.diff(p3.rowptr)[pi], np.diff(p2.rowptr))
    # diagonal entries travel with the permutation
    d2 = p2.vals[np.searchsorted(p2.colind[:p2.rowptr[1]], 0)]
    d3row = pi[0]
    seg = slice(p3.rowptr[d3row], p3.rowptr[d3row + 1])
    assert d2 == p3.vals[seg][p3.colind[seg] == d3row][0]
    assert sorted(p3.vals.tolist()) == sorted(p2.vals.tolist())


def test_vectors_and_rhs():
    v = gi.seeded_vector(2, 1000)
    assert v.min() >= -1 and v.max() < 1 and abs(v.mean()) < 0.1
    p = gi.make_config(0)
    A = _to_dense(*gi.stencil27(4))
    xs = gi.seeded_vector(0, 64)
    b = gi.rhs_from_solution(*gi.stencil27(4), xs)
    np.testing.assert_allclose(b, A @ xs, rtol=0, atol=1e-13)
    assert p.xstar is not None and np.all(p.x0 == 0)


def test_byte_and_flop_models():
    # SURVEY.md 8 table; flops fit Table I of the paper
    assert gi.algorithmic_bytes_per_iteration(132651, 3442951) == 53519308
    assert gi.flops_per_iteration(132651, 3442951) == 8212412
    for iters, t, gf in [(117, 3.17, 0.303), (116, 0.659, 1.45), (116, 0.461, 2.07), (116, 0.380, 2.50)]:
        assert abs(8212412 * iters / t / 1e9 - gf) < 0.01
