"""Parity of the CUDA path (through the C ABI) against the CPU oracle, on the same seeded inputs.

Tolerances are BASELINE.json north_star's, with the readings of SURVEY.md 8(c) 12-15:
  SpMV        |y_gpu - y_or|_i <= 1e-13 * (|A||x|)_i
  history     |h_gpu[j] - h_or[j]| / h_or[j] <= 1e-9 for j = 0..min(50, k)
  iterations  within +-2 % of the oracle's count (at least +-1)
  solution    ||x_gpu - x_or||_2 / ||x_or||_2 <= 1e-8
"""
import math
import os

import numpy as np
import pytest

import cg_inputs as gi

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

SPMV_TOL = 1e-13
HIST_TOL = 1e-9
X_TOL = 1e-8


@pytest.fixture(scope="module")
def cgmod():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    import paper_1107_0538_b200 as m
    return m


@pytest.fixture(scope="module")
def orc():
    from oracle import cg_oracle
    return cg_oracle


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class Bound:
    def __init__(self, m, p):
        self.p = p
        self.cg = m.CG(dev(p.rowptr), dev(p.colind), dev(p.vals))
        self.b = dev(p.b)


@pytest.fixture(scope="module")
def bound(cgmod, problems):
    cache = {}

    def get(cfg, grid=None):
        if (cfg, grid) not in cache:
            cache[(cfg, grid)] = Bound(cgmod, problems(cfg, grid))
        return cache[(cfg, grid)]
    yield get
    for b in cache.values():
        b.cg.close()


_oracle_cache = {}


def oracle_solve(orc, p, key, **kw):
    if key not in _oracle_cache:
        _oracle_cache[key] = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=kw.get("rtol", p.rtol),
                                    maxit=kw.get("maxit", p.maxit), dinv=kw.get("dinv"))
    return _oracle_cache[key]


def check_solve_parity(res, x, ref, iters_band=0.02):
    k = min(50, ref.iters, res.iters)
    hg = res.hist.cpu().numpy()
    rel = np.abs(hg[:k + 1] - ref.hist[:k + 1]) / ref.hist[:k + 1]
    assert rel.max() <= HIST_TOL, f"history differs: {rel.max():.3e}"
    if iters_band:
        band = max(1, math.floor(iters_band * ref.iters))
        assert abs(res.iters - ref.iters) <= band, (res.iters, ref.iters)
    xe = np.linalg.norm(x.cpu().numpy() - ref.x) / np.linalg.norm(ref.x)
    assert xe <= X_TOL, f"solution differs: {xe:.3e}"
    assert res.status == ref.status
    assert len(hg) == res.iters + 1


# ---------------------------------------------------------------- SpMV / dot

@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
@pytest.mark.parametrize("variant", [1, 2, 3, 4])
def test_spmv_parity(bound, orc, cfg, variant):
    B = bound(cfg)
    p = B.p
    B.cg.set_option("spmv", variant)
    assert B.cg.info("spmv") == (variant if (variant != 4 or cfg != 3) else 1)     # 4 needs the matrix pinned
    x = gi.seeded_vector(100 + cfg, p.n)
    y = B.cg.spmv(dev(x)).cpu().numpy()
    want = orc.spmv(p.rowptr, p.colind, p.vals, x)
    denom = orc.absrow(p.rowptr, p.colind, p.vals, x)
    err = np.abs(y - want) / denom
    assert err.max() <= SPMV_TOL, f"cfg {cfg} variant {variant}: {err.max():.3e}"
    B.cg.set_option("spmv", 0)


@pytest.mark.parametrize("tpr", [2, 4, 8, 16, 32])
def test_spmv_vector_all_lane_widths(bound, orc, tpr):
    B = bound(0)
    p = B.p
    B.cg.set_option("spmv", 1)
    B.cg.set_option("tpr", tpr)
    x = gi.seeded_vector(7, p.n)
    y = B.cg.spmv(dev(x)).cpu().numpy()
    want = orc.spmv(p.rowptr, p.colind, p.vals, x)
    assert np.all(np.abs(y - want) <= SPMV_TOL * orc.absrow(p.rowptr, p.colind, p.vals, x))
    B.cg.set_option("tpr", 8)
    B.cg.set_option("spmv", 0)


def _random_csr(n, seed, max_len, empty_every=0, unsorted=False):
    """Irregular CSR with ragged rows, optional empty rows, unsorted / duplicate columns."""
    u = gi.hash_uniform(seed, 2, np.arange(n, dtype=np.uint64))
    lens = (u * (max_len + 1)).astype(np.int64)
    if empty_every:
        lens[::empty_every] = 0
    rp = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(lens, out=rp[1:])
    nnz = int(rp[-1])
    ci = (gi.hash_uniform(seed + 1, 2, np.arange(nnz, dtype=np.uint64)) * n).astype(np.int32)
    va = 2 * gi.hash_uniform(seed + 2, 2, np.arange(nnz, dtype=np.uint64)) - 1
    if not unsorted:
        for i in range(n):
            ci[rp[i]:rp[i + 1]].sort()
    return rp.astype(np.int32), ci, va


@pytest.mark.parametrize("n,max_len,empty_every", [(1, 1, 0), (2, 3, 0), (31, 5, 3), (33, 40, 0),
                                                   (1000, 31, 7), (4097, 70, 5), (5000, 300, 11)])
def test_spmv_irregular_matrices(cgmod, orc, n, max_len, empty_every):
    """Ragged tails, empty rows, duplicate and unsorted columns, rows longer than a tile
    (the streamed variant must refuse those and fall back), nnz not a multiple of 4."""
    rp, ci, va = _random_csr(n, 1000 + n, max_len, empty_every, unsorted=True)
    cg = cgmod.CG(dev(rp), dev(ci), dev(va))
    x = gi.seeded_vector(5, n)
    want = orc.spmv(rp, ci, va, x)
    denom = orc.absrow(rp, ci, va, x) + 1e-300
    for variant in (1, 2):
        cg.set_option("spmv", variant)
        if variant == 2 and not cg.info("stream_ok"):
            assert cg.info("spmv") == 1
        y = cg.spmv(dev(x)).cpu().numpy()
        assert np.all(np.abs(y - want) <= SPMV_TOL * denom), (n, variant)
    assert cg.check_csr()
    cg.close()


@pytest.mark.parametrize("n", [1, 2, 255, 256, 257, 132651, 1 << 20])
def test_dot_parity(bound, orc, n):
    B = bound(0)
    a, b = gi.seeded_vector(61, n), gi.seeded_vector(62, n)
    cg = B.cg if n == B.p.n else None
    if cg is None:
        rp = np.arange(n + 1, dtype=np.int32)
        cgm = __import__("paper_1107_0538_b200")
        cg = cgm.CG(dev(rp), dev(np.arange(n, dtype=np.int32)), dev(np.ones(n)))
    got = cg.dot(dev(a), dev(b))
    ref = orc.dot_ld(a, b)
    assert abs(got - ref) <= 1e-15 * np.sum(np.abs(a * b)) * max(1.0, math.log2(n))
    assert got == cg.dot(dev(a), dev(b))                     # bitwise reproducible
    if cg is not B.cg:
        cg.close()


# ---------------------------------------------------------------- cg_solve

@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
@pytest.mark.parametrize("variant", [1, 2, 3, 4])
def test_solve_parity_persistent(bound, orc, cfg, variant):
    B = bound(cfg)
    p = B.p
    B.cg.set_option("loop", 0)
    B.cg.set_option("spmv", variant)
    ref = oracle_solve(orc, p, ("cg", cfg))
    x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    check_solve_parity(res, x, ref)
    assert res.status == 0
    # the recurrence residual the GPU reports is the true residual of the x it returns
    true_r = p.b - orc.spmv_ld(p.rowptr, p.colind, p.vals, x.cpu().numpy())
    assert np.linalg.norm(true_r) / np.linalg.norm(p.b) <= 2 * p.rtol
    assert abs(res.resnorm - res.hist[-1].item()) == 0.0
    if p.xstar is not None:
        assert np.linalg.norm(x.cpu().numpy() - p.xstar) / np.linalg.norm(p.xstar) < 1e-7
    B.cg.set_option("spmv", 0)


def _banded_spd(n, half_band):
    """SPD band matrix with 2*half_band + 1 entries per interior row (longer than the 27 the
    streamed consumer handles in one trip): off-diagonals -1/(d+1), strictly dominant diagonal."""
    rows, cols, vals = [], [], []
    for i in range(n):
        lo, hi = max(0, i - half_band), min(n - 1, i + half_band)
        js = np.arange(lo, hi + 1)
        v = -1.0 / (np.abs(js - i) + 1.0)
        v[js == i] = 0.0
        v[js == i] = np.abs(v).sum() + 0.05
        rows.append(len(js)); cols.append(js); vals.append(v)
    rp = np.zeros(n + 1, dtype=np.int32)
    np.cumsum(rows, out=rp[1:])
    return rp, np.concatenate(cols).astype(np.int32), np.concatenate(vals)


@pytest.mark.parametrize("half_band", [30, 36, 45])
def test_solve_long_rows_streamed(cgmod, orc, half_band):
    """Rows of 61 / 73 / 91 entries: several trips per row in the streamed consumer, few ring slots
    (a tile is 2-3 times a 27-point one), and past that the fall-back to the generic path; all
    variants and loop modes against the oracle."""
    n = 5003
    rp, ci, va = _banded_spd(n, half_band)
    b = gi.seeded_vector(77, n)
    ref = orc.cg(rp, ci, va, b, rtol=1e-10, maxit=n)
    cg = cgmod.CG(dev(rp), dev(ci), dev(va))
    assert cg.info("compressed") == 1                            # a band matrix has 2 * half_band + 1 offsets
    assert cg.info("stream_ok") == 1                             # 8 + 1 bytes per entry: even the 91-entry rows fit 8 slots
    cg.set_option("compress", 0)
    cg.set_option("pin", 0)              # (pinned, each CTA's 2 tiles fit in any case)
    assert cg.info("stream_ok") == (1 if half_band <= 36 else 0)   # 12 bytes per entry
    outs = []
    for variant in (2, 3):
        cg.set_option("spmv", variant)
        if half_band > 36:               # a 32-row tile no longer fits a ring of 8 plain slots: generic path
            assert cg.info("spmv") == 1
        else:
            if variant == 3 and cg.info("spmv") == 1:
                continue                 # 5 producer warps need a ring depth they divide (a multiple of 20)
            assert cg.info("spmv") == variant and (cg.info("ring_slots") >= 8 or cg.info("pinned_tiles") > 0)
        for loop in (0, 1):
            cg.set_option("loop", loop)
            x, res = cg.solve(dev(b), rtol=1e-10, maxit=n)
            check_solve_parity(res, x, ref)
            outs.append((cg.info("spmv"), x.cpu().numpy().copy()))
    for (va_, xa), (vb_, xb) in zip(outs[::2], outs[1::2]):
        assert va_ == vb_ and np.array_equal(xa, xb)             # persistent == graph twin, per variant
    cg.set_option("compress", 1)
    for variant in (2, 3):
        cg.set_option("spmv", variant)
        cg.set_option("pin", 3 - variant)    # streamed through the ring with variant 2, pinned with variant 3
        if cg.info("spmv") == 1:
            continue
        for loop in (0, 1):
            cg.set_option("loop", loop)
            x, res = cg.solve(dev(b), rtol=1e-10, maxit=n)
            check_solve_parity(res, x, ref)
            if outs and outs[0][0] == variant:
                assert np.array_equal(x.cpu().numpy(), outs[0][1])   # same bits as the plain-CSR slots
    cg.close()


@pytest.mark.parametrize("cfg", [0, 2])
def test_loop_modes_agree_bitwise(bound, cfg):
    """Persistent kernel, CUDA-graph replay and plain launches share the phase code and the
    reduction order: identical bits.  Also run-to-run reproducibility (a cheap race detector)."""
    B = bound(cfg)
    p = B.p
    outs = []
    for variant in (1, 2):
        B.cg.set_option("spmv", variant)
        per_mode = []
        for loop in (0, 1, 2, 0):
            B.cg.set_option("loop", loop)
            x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
            per_mode.append((x.cpu().numpy().copy(), res.hist.cpu().numpy().copy(), res.iters, res.status))
        for other in per_mode[1:]:
            assert other[2] == per_mode[0][2] and other[3] == per_mode[0][3]
            assert np.array_equal(other[1], per_mode[0][1])
            assert np.array_equal(other[0], per_mode[0][0])
        outs.append(per_mode[0])
    B.cg.set_option("loop", 0)
    B.cg.set_option("spmv", 0)
    assert abs(outs[0][2] - outs[1][2]) <= 1           # the two SpMV variants differ only by rounding


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_streamed_persistent_modes_agree_bitwise(bound, cfg):
    """The streamed persistent kernel with x, r, p, q in registers (with K3 folded into the next
    K1's gathers, two grid syncs per iteration, or not), the same kernel with the vectors in
    global memory, with and without producer run-ahead across the grid barriers, with part of
    the matrix pinned in shared memory or all of it streamed every iteration, and the graph
    twin all perform the same operations in the same order: identical bits."""
    B = bound(cfg)
    p = B.p
    for variant in (2, 3):
        B.cg.set_option("spmv", variant)
        runs = []
        big = 1 << 30
        for loop, resident, lookahead, fold, pin in ((0, 1, big, 1, 1), (0, 1, big, 0, 1), (0, 0, big, 1, 1),
                                                     (0, 1, 0, 1, 1), (0, 0, 3, 0, 0), (1, 1, big, 1, 1),
                                                     (0, 1, big, 0, 0), (1, 1, big, 1, 0)):
            B.cg.set_option("pin", pin)
            B.cg.set_option("loop", loop)
            B.cg.set_option("resident", resident)
            B.cg.set_option("lookahead", lookahead)
            B.cg.set_option("fold", fold)
            if loop == 0 and resident == 1 and cfg != 1:          # config 1 has 5-7 rows per thread: global vectors
                assert B.cg.info("resident_rows") in (2, 4)
            x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
            runs.append((x.cpu().numpy().copy(), res.hist.cpu().numpy().copy(), res.iters, res.status))
        for other in runs[1:]:
            assert other[2] == runs[0][2] and other[3] == runs[0][3]
            assert np.array_equal(other[1], runs[0][1])
            assert np.array_equal(other[0], runs[0][0])
    for name, v in (("loop", 0), ("resident", 1), ("lookahead", 1 << 30), ("fold", 2), ("pin", 1), ("spmv", 0)):
        B.cg.set_option(name, v)


def test_phase_trace_and_bandwidth_probe(bound, cgmod):
    """cg_set_trace fills monotone clock stamps for every CTA; cg_probe_read_bandwidth returns
    a plausible figure (both are profiling aids of include/cg.h)."""
    B = bound(2)
    p = B.p
    B.cg.set_option("loop", 0)
    B.cg.set_option("pin", 0)            # stream the matrix: the producers' statistics are part of the trace
    iters = 12
    tr = B.cg.trace(iters)
    st, it, res = cgmod.cg_solve(B.cg.h, B.b.data_ptr(), torch.zeros_like(B.b).data_ptr(), 0.0, iters, None,
                                 torch.cuda.current_stream().cuda_stream)
    assert it == iters and st == 1
    t = tr.cpu().numpy()
    assert t.shape == (B.cg.info("grid"), iters + 1, 16)
    stamps = t[:, :iters - 1, :8]
    assert (stamps > 0).all() and (np.diff(stamps, axis=2) > 0).all()
    assert t[:, iters, 2].max() > 0                      # tiles issued by producer warp 0
    B.cg.trace(0)
    B.cg.set_option("pin", 1)
    gbs = B.cg.probe_read_bandwidth(32 << 20, reps=10)
    assert 500.0 < gbs < 50000.0
    cyc = [B.cg.probe_grid_sync(kind, 500) for kind in (0, 1, 2)]
    assert all(300.0 < c < 50000.0 for c in cyc) and cyc[2] > cyc[0]       # the fenced all-reduce costs more than the bare barrier
    x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)                   # the probe leaves the handle usable
    assert res.status == 0
    with pytest.raises(cgmod.CGError):
        cgmod.cg_probe_read_bandwidth(B.cg.h, 0, 1 << 20, 1, 0)


def test_sync_place_and_global_clock_trace(bound, cgmod):
    """Where the all-reduce inboxes sit ("sync_place", chosen by measurement at cg_create) cannot change a
    bit of the result: the sums have one fixed order.  "trace_clock" = 1 stamps the nanosecond clock all SMs
    share, so stamps of different CTAs are comparable: every CTA leaves a grid synchronisation after the last
    one has reached it."""
    B = bound(2)
    p = B.p
    for name, v in (("loop", 0), ("spmv", 0), ("algo", 0)):
        B.cg.set_option(name, v)
    places = B.cg.info("sync_places")
    chosen = B.cg.info("sync_place")
    assert places >= 200 and 0 <= chosen < 40
    x0, r0 = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    for place in (0, 7, places):
        B.cg.set_option("sync_place", place)
        assert B.cg.info("sync_place") == place
        x, r = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
        assert r.iters == r0.iters and torch.equal(x, x0) and torch.equal(r.hist, r0.hist), place
    with pytest.raises(cgmod.CGError):
        B.cg.set_option("sync_place", places + 1)
    B.cg.set_option("sync_place", chosen)
    n_it = 12
    B.cg.set_option("trace_clock", 1)
    tr = B.cg.trace(n_it)
    x, r = B.cg.solve(B.b, rtol=0.0, maxit=n_it)
    t = tr.cpu().numpy().astype(np.int64)[:, 1:n_it - 1, :8]      # the last iteration leaves at the stop test
    B.cg.trace(0)
    B.cg.set_option("trace_clock", 0)
    assert (np.diff(t, axis=2) >= 0).all()                                   # monotone inside an iteration
    for arrive, leave in ((1, 2), (3, 4), (6, 7)):                             # the three synchronisations of the textbook loop
        assert (t[:, :, leave].min(axis=0) >= t[:, :, arrive].max(axis=0)).all()
    it_ns = float((t[:, -1, 7] - t[:, 0, 0]).mean()) / t.shape[1]
    assert 3000.0 < it_ns < 100000.0                                           # ~10 us per iteration, in nanoseconds


def test_graph_chunk_sizes_and_launch_count(bound):
    B = bound(0)
    p = B.p
    B.cg.set_option("loop", 0)
    x0, r0 = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    assert B.cg.info("launches") == 1
    for chunk in (2, 8, 64):
        B.cg.set_option("loop", 1)
        B.cg.set_option("chunk", chunk)
        x, r = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
        assert r.iters == r0.iters and torch.equal(x, x0)
        assert B.cg.info("launches") == 3 + 3 * chunk * math.ceil(r.iters / chunk)
    B.cg.set_option("chunk", 32)
    B.cg.set_option("loop", 0)


def test_handworked_2x2(cgmod):
    """tests/golden/cg_2x2_handworked.txt through the CUDA path."""
    cg = cgmod.CG(dev(np.array([0, 2, 4], dtype=np.int32)), dev(np.array([0, 1, 0, 1], dtype=np.int32)),
                  dev(np.array([2.0, -1.0, -1.0, 2.0])))
    for loop in (0, 1, 2):
        cg.set_option("loop", loop)
        x, res = cg.solve(dev(np.array([1.0, 0.0])), rtol=1e-14, maxit=10)
        assert res.iters == 2 and res.status == 0
        np.testing.assert_allclose(res.hist.cpu().numpy(), [1.0, 0.5, 0.0], atol=1e-16)
        np.testing.assert_allclose(x.cpu().numpy(), [2 / 3, 1 / 3], rtol=1e-15)
    cg.close()


def test_conventions_and_edge_cases(bound, cgmod, orc):
    B = bound(0)
    p = B.p
    for loop in (0, 1, 2):
        B.cg.set_option("loop", loop)
        # b = 0 -> x = 0, k = 0, converged, hist = [0]
        x, res = B.cg.solve(torch.zeros_like(B.b), x0=torch.ones_like(B.b), rtol=1e-10, maxit=10)
        assert res.iters == 0 and res.status == 0 and float(x.abs().max()) == 0.0
        assert res.hist.cpu().tolist() == [0.0]
        # rtol = 0 -> exactly maxit iterations, status 1
        x, res = B.cg.solve(B.b, rtol=0.0, maxit=7)
        ref = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=0.0, maxit=7)
        assert res.iters == 7 and res.status == 1
        assert np.linalg.norm(x.cpu().numpy() - ref.x) / np.linalg.norm(ref.x) < 1e-12
        # maxit = 0 -> no iteration, x = x0
        x, res = B.cg.solve(B.b, rtol=1e-10, maxit=0)
        assert res.iters == 0 and res.status == 1 and float(x.abs().max()) == 0.0
        assert abs(res.resnorm - np.linalg.norm(p.b)) <= 1e-13 * np.linalg.norm(p.b)
        # x0 = solution -> zero iterations, converged
        ref = oracle_solve(orc, p, ("cg", 0))
        x, res = B.cg.solve(B.b, x0=dev(ref.x), rtol=1e-9, maxit=10)
        assert res.iters == 0 and res.status == 0
        # nonzero x0 is used as the starting point (r0 = b - A x0)
        x0 = gi.seeded_vector(77, p.n)
        x, res = B.cg.solve(B.b, x0=dev(x0), rtol=p.rtol, maxit=p.maxit)
        ref2 = orc.cg(p.rowptr, p.colind, p.vals, p.b, x0=x0, rtol=p.rtol, maxit=p.maxit)
        check_solve_parity(res, x, ref2)
    B.cg.set_option("loop", 0)
    # breakdown: -A is negative definite
    neg = cgmod.CG(dev(p.rowptr), dev(p.colind), dev(-p.vals))
    for loop in (0, 1, 2):
        neg.set_option("loop", loop)
        x, res = neg.solve(B.b, rtol=1e-10, maxit=10)
        assert res.status == 2 and res.iters == 0
        assert float(x.abs().max()) == 0.0
    neg.close()


def test_invalid_arguments(bound, cgmod):
    B = bound(0)
    L = cgmod.lib()
    n = B.p.n
    x = torch.zeros(n + 1, dtype=torch.float64, device="cuda")
    h, b = B.cg.h, B.b.data_ptr()
    assert L.cg_solve(h, b, x.data_ptr(), float("nan"), 10, None, None, None, None) == -1
    assert L.cg_solve(h, b, x.data_ptr(), -1.0, 10, None, None, None, None) == -1
    assert L.cg_solve(h, b, x.data_ptr(), 1e-3, -1, None, None, None, None) == -1
    assert L.cg_solve(h, b, None, 1e-3, 10, None, None, None, None) == -1
    assert L.cg_solve(h, b, x[1:].data_ptr(), 1e-3, 10, None, None, None, None) == -1   # misaligned
    assert L.cg_spmv(h, b, b, None) == -1                                                # aliasing
    with pytest.raises(cgmod.CGError):
        cgmod.cg_create(n, B.p.nnz, B.cg.rowptr.data_ptr(), B.cg.colind.data_ptr(),
                        B.cg.vals.data_ptr(), B.cg.workspace.data_ptr(), 1024)            # workspace too small
    with pytest.raises(cgmod.CGError):
        cgmod.cg_create(0, 0, B.cg.rowptr.data_ptr(), B.cg.colind.data_ptr(), B.cg.vals.data_ptr(),
                        B.cg.workspace.data_ptr(), B.cg.workspace.numel())
    with pytest.raises(cgmod.CGError):
        B.cg.set_option("nonsense", 1)
    # a broken CSR structure is reported by cg_check_csr
    bad_ci = B.cg.colind.clone()
    bad_ci[5] = n + 3
    bad = cgmod.CG(B.cg.rowptr, bad_ci, B.cg.vals)
    assert not bad.check_csr()
    bad.close()
    assert B.cg.check_csr()


def test_solve_host_end_to_end(bound, orc):
    B = bound(2)
    p = B.p
    hb = torch.from_numpy(p.b).pin_memory()
    hx = torch.zeros(p.n, dtype=torch.float64).pin_memory()
    hh = torch.zeros(p.maxit + 1, dtype=torch.float64).pin_memory()
    st, it, res = B.cg.solve_host(hb, hx, p.rtol, p.maxit, hh)
    ref = oracle_solve(orc, p, ("cg", 2))
    assert st == 0 and abs(it - ref.iters) <= max(1, int(0.02 * ref.iters))
    assert np.linalg.norm(hx.numpy() - ref.x) / np.linalg.norm(ref.x) <= X_TOL
    k = min(50, it)
    assert np.max(np.abs(hh.numpy()[:k + 1] - ref.hist[:k + 1]) / ref.hist[:k + 1]) <= HIST_TOL
    assert hh.numpy()[it] == res


# ---------------------------------------------------------------- compressed column index (8(f) rank 4)

@pytest.mark.parametrize("cfg,grid", [(0, None), (1, None), (2, None), (4, 32)])
def test_compressed_index_same_bits(cgmod, problems, orc, cfg, grid):
    """cg_compress_index: one byte per entry naming col - row (27 distinct offsets on the 27-point
    stencils, 7 on the Laplacian).  Entries keep their CSR order, so SpMV and whole solves give the
    bits of the plain-CSR slots, in every variant and loop mode; parity with the oracle as usual."""
    p = problems(cfg, grid)
    A = cgmod.CG(dev(p.rowptr), dev(p.colind), dev(p.vals))          # compresses by default
    assert A.index is not None and A.info("compressed") == 1
    assert A.info("index_codes") == (7 if cfg == 1 else 27)
    b = dev(p.b)
    xv = dev(gi.seeded_vector(300 + cfg, p.n))
    want = orc.spmv(p.rowptr, p.colind, p.vals, xv.cpu().numpy())
    denom = orc.absrow(p.rowptr, p.colind, p.vals, xv.cpu().numpy())
    ref = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit)
    for variant in (2, 3):
        A.set_option("spmv", variant)
        got = {}
        for cmp in (1, 0):
            A.set_option("compress", cmp)
            assert A.info("compressed") == cmp
            y = A.spmv(xv).cpu().numpy()
            assert (np.abs(y - want) / denom).max() <= SPMV_TOL
            runs = []
            for loop in (0, 1):
                A.set_option("loop", loop)
                x, res = A.solve(b, rtol=p.rtol, maxit=p.maxit)
                check_solve_parity(res, x, ref)
                runs.append((x.cpu().numpy().copy(), res.hist.cpu().numpy().copy()))
            assert np.array_equal(runs[0][0], runs[1][0]) and np.array_equal(runs[0][1], runs[1][1])
            got[cmp] = (y, runs[0])
        assert np.array_equal(got[0][0], got[1][0])
        assert np.array_equal(got[0][1][0], got[1][1][0]) and np.array_equal(got[0][1][1], got[1][1][1])
    A.close()


def test_compressed_index_declines(cgmod, problems):
    """Config 3 (random permutation): far more than 256 distinct offsets -> CG_NOTCOMPRESSED and
    the plain path keeps running; a too-small or misaligned buffer is an argument error."""
    p = problems(3)
    A = cgmod.CG(dev(p.rowptr), dev(p.colind), dev(p.vals), compress=False)
    nb = cgmod.cg_index_bytes(A.h)
    assert nb > p.nnz
    buf = torch.empty(nb + 256, dtype=torch.uint8, device="cuda")
    assert cgmod.cg_compress_index(A.h, buf.data_ptr(), nb, 0) == 3
    assert A.info("compressed") == 0 and A.info("index_codes") == 0
    with pytest.raises(cgmod.CGError):
        cgmod.cg_compress_index(A.h, buf.data_ptr(), nb - 1, 0)
    with pytest.raises(cgmod.CGError):
        cgmod.cg_compress_index(A.h, buf.data_ptr() + 16, nb, 0)
    A.close()


def test_config2_matrix_pinned_in_shared_memory(bound):
    """At the paper's size the compressed slice of every CTA fits its shared memory: nothing is
    re-streamed inside a solve (the whole point of the compression there)."""
    B = bound(2)
    for name, v in (("loop", 0), ("spmv", 0), ("compress", 1), ("pin", 1)):
        B.cg.set_option(name, v)
    assert B.cg.info("compressed") == 1
    tiles = -(-B.p.n // 32)
    assert B.cg.info("pinned_tiles") == -(-tiles // B.cg.info("sms")) == B.cg.info("ring_slots")
    assert B.cg.info("smem") <= 227 * 1024
    B.cg.set_option("compress", 0)
    assert B.cg.info("pinned_tiles") == 0 and B.cg.info("ring_slots") == 20
    B.cg.set_option("compress", 1)


# ---------------------------------------------------------------- option paths, all against the default's bits

def test_ring_and_grid_options_same_bits(bound):
    """"ring_slots", "pin" (off, auto, mixed split), "lookahead" and "compress" only change where
    the matrix waits, never the arithmetic; "ctas_per_sm" changes the generic variant's grid and
    with it the reduction grouping, so that one is held to the tolerances instead."""
    B = bound(2)
    p = B.p
    B.cg.set_option("loop", 0)
    B.cg.set_option("spmv", 2)           # one thread <-> row map throughout (variant 3 has 11 consumer warps)
    x0, r0 = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    settings = [{"compress": 0, "ring_slots": 8}, {"compress": 0, "ring_slots": 12}, {"compress": 0, "ring_slots": 16},
                {"compress": 1, "pin": 0}, {"compress": 1, "pin": 0, "ring_slots": 9},
                {"compress": 1, "pin": 5}, {"compress": 0, "pin": 7, "lookahead": 2},
                {"compress": 1, "pin": 12}, {"compress": 0, "pin": 3, "loop": 1}]
    for st in settings:
        for k, v in st.items():
            B.cg.set_option(k, v)
        assert B.cg.info("spmv") == 2
        if "ring_slots" in st and st.get("pin", 1) == 0 or st.get("compress") == 0 and "ring_slots" in st:
            assert B.cg.info("ring_slots") <= st["ring_slots"]
        if st.get("pin", 1) >= 2:
            assert B.cg.info("pinned_tiles") == st["pin"]
        x, r = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
        assert r.iters == r0.iters and torch.equal(x, x0) and torch.equal(r.hist, r0.hist), st
        for k, v in (("compress", 1), ("pin", 1), ("ring_slots", 64), ("lookahead", 1 << 30), ("loop", 0)):
            B.cg.set_option(k, v)
    B.cg.set_option("spmv", 0)


@pytest.mark.parametrize("grid", [None, 50, 45])
def test_short_row_kernels_same_bits(bound, orc, grid):
    """The short-row kernels ("short_rows", chosen when no row has more than 9 entries: the 7-point
    Laplacian) keep the gathers of several tiles in flight per warp; per row the operations and their
    order are those of the one-tile trip, so the bits of every loop (textbook, Jacobi, Chronopoulos-Gear,
    pipelined) are those of the kernels they replace.  64^3 (config 1: 3 or 4 tiles per warp), 50^3 (a ragged
    last tile, which falls back to the one-tile trip) and 45^3 (1 or 2 tiles per warp); parity against the
    oracle on top."""
    B = bound(1, grid)
    p = B.p
    for name, v in (("loop", 0), ("spmv", 0), ("fold", 2), ("algo", 0), ("short_rows", 1)):
        B.cg.set_option(name, v)
    assert B.cg.info("spmv") == 4 and B.cg.info("short_rows") == 1 and B.cg.info("fold") == 0
    ref = oracle_solve(orc, p, ("cfg1", grid))
    for algo, jacobi in ((0, False), (0, True), (1, False), (2, False)):
        B.cg.set_option("algo", algo)
        runs = []
        for short in (1, 0):
            B.cg.set_option("short_rows", short)
            B.cg.set_option("fold", 0)                  # short_rows = 0 alone would fold (auto), other bits
            assert B.cg.info("short_rows") == short
            x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit, jacobi=jacobi)
            runs.append((x, res))
        (x1, r1), (x0, r0) = runs
        assert r1.iters == r0.iters and r1.status == r0.status
        assert torch.equal(r1.hist, r0.hist) and torch.equal(x1, x0), (algo, jacobi)
        if not jacobi:                                  # (the diagonal is constant: Jacobi is CG on a scaled system)
            check_solve_parity(r1, x1, ref)
    for name, v in (("algo", 0), ("fold", 2), ("short_rows", 1)):
        B.cg.set_option(name, v)


@pytest.mark.parametrize("ctas", [1, 2, 3])
def test_generic_ctas_per_sm(bound, orc, ctas):
    B = bound(0)
    p = B.p
    B.cg.set_option("spmv", 1)
    B.cg.set_option("ctas_per_sm", ctas)
    assert B.cg.info("grid") == B.cg.info("sms") * min(ctas, 2)      # launch bounds allow 2 CTAs per SM
    ref = oracle_solve(orc, p, ("cg", 0))
    for loop in (0, 1):
        B.cg.set_option("loop", loop)
        x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
        check_solve_parity(res, x, ref)
    for k, v in (("ctas_per_sm", 0), ("spmv", 0), ("loop", 0)):
        B.cg.set_option(k, v)


# ---------------------------------------------------------------- single-reduction CG (8(f) rank 2, second half)

@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
@pytest.mark.parametrize("algo", [1, 2])
def test_single_reduction_cg_parity(bound, orc, cfg, algo):
    """Option "algo" = 1: Chronopoulos-Gear CG (one all-reduce + one publish barrier per iteration);
    "algo" = 2: pipelined CG (one barrier per iteration, the reduction hidden behind the SpMV).
    Same Krylov iteration, different rounding: each must pass the same four bands against the same
    (unchanged) oracle as the textbook path, and return an x whose true residual, computed with the
    oracle's SpMV, meets rtol."""
    B = bound(cfg)
    p = B.p
    B.cg.set_option("loop", 0)
    B.cg.set_option("algo", algo)
    assert B.cg.info("algo") == algo
    ref = oracle_solve(orc, p, ("cg", cfg))
    x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    check_solve_parity(res, x, ref)
    true_r = p.b - orc.spmv_ld(p.rowptr, p.colind, p.vals, x.cpu().numpy())
    assert np.linalg.norm(true_r) / np.linalg.norm(p.b) <= 2 * p.rtol
    x2, res2 = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    assert torch.equal(x, x2) and torch.equal(res.hist, res2.hist)        # reproducible
    # conventions hold here too
    x3, r3 = B.cg.solve(B.b, rtol=0.0, maxit=5)
    r5 = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=0.0, maxit=5)
    assert r3.iters == 5 and r3.status == 1
    assert np.linalg.norm(x3.cpu().numpy() - r5.x) / np.linalg.norm(r5.x) < 1e-12
    x4, r4 = B.cg.solve(torch.zeros_like(B.b), x0=torch.ones_like(B.b), rtol=1e-10, maxit=10)
    assert r4.iters == 0 and r4.status == 0 and float(x4.abs().max()) == 0.0
    B.cg.set_option("loop", 1)
    assert B.cg.info("algo") == 0                                          # graph twin: textbook only
    B.cg.set_option("loop", 0)
    B.cg.set_option("algo", 0)


@pytest.mark.parametrize("algo", [1, 2])
def test_single_reduction_cg_breakdown(bound, cgmod, algo):
    B = bound(0)
    neg = cgmod.CG(dev(B.p.rowptr), dev(B.p.colind), dev(-B.p.vals))
    neg.set_option("algo", algo)
    x, res = neg.solve(B.b, rtol=1e-10, maxit=10)
    assert res.status == 2 and res.iters == 0
    x, res = neg.solve(B.b, rtol=1e-10, maxit=0)
    assert res.status == 1 and res.iters == 0
    neg.close()


# ---------------------------------------------------------------- the library's own memcheck

@pytest.mark.parametrize("cfg", [0, 2, 3])
def test_checked_spmv_clean_on_valid_matrices(bound, cfg):
    """Option "checked": the SpMV with every index validated on the device (bulk-copy source ranges,
    slot offsets, index codes, gathered columns).  On valid matrices it must count nothing, in every
    kernel shape and slot format, pinned and streamed, and return the unchecked kernel's bits."""
    B = bound(cfg)
    xv = dev(gi.seeded_vector(400 + cfg, B.p.n))
    for spmv in (2, 3, 4):
        for compress in (1, 0):
            for pin in (1, 0):
                for k, v in (("spmv", spmv), ("compress", compress), ("pin", pin)):
                    B.cg.set_option(k, v)
                if B.cg.info("spmv") != spmv:
                    continue
                y0 = B.cg.spmv(xv)
                B.cg.set_option("checked", 1)
                y1 = B.cg.spmv(xv)
                B.cg.set_option("checked", 0)
                assert B.cg.info("check_errors") == 0 and torch.equal(y0, y1), (spmv, compress, pin)
    for k, v in (("spmv", 0), ("compress", 1), ("pin", 1)):
        B.cg.set_option(k, v)


@pytest.mark.parametrize("n,max_len,empty_every", [(33, 40, 0), (1000, 31, 7), (4097, 70, 5)])
def test_checked_spmv_clean_on_ragged_matrices(cgmod, n, max_len, empty_every):
    rp, ci, va = _random_csr(n, 1000 + n, max_len, empty_every, unsorted=True)
    A = cgmod.CG(dev(rp), dev(ci), dev(va))
    xv = dev(gi.seeded_vector(5, n))
    for spmv in (2, 3, 4):
        A.set_option("spmv", spmv)
        if A.info("spmv") != spmv:
            continue
        y0 = A.spmv(xv)
        A.set_option("checked", 1)
        y1 = A.spmv(xv)
        A.set_option("checked", 0)
        assert A.info("check_errors") == 0 and torch.equal(y0, y1)
    A.close()


@pytest.mark.parametrize("compress", [False, True])
@pytest.mark.parametrize("bad_col", [-3, 5])
def test_checked_spmv_catches_a_corrupt_column(cgmod, problems, compress, bad_col):
    """A column index outside [0, n) (relative to n for the positive case): the checked SpMV counts
    it, never dereferences it, reports CG_ECUDA, and leaves the device usable."""
    p = problems(0)
    ci = p.colind.copy()
    ci[1234] = bad_col if bad_col < 0 else p.n + bad_col
    A = cgmod.CG(dev(p.rowptr), dev(ci), dev(p.vals), compress=compress)
    assert not A.check_csr()
    A.set_option("checked", 1)
    xv = dev(gi.seeded_vector(1, p.n))
    with pytest.raises(cgmod.CGError) as err:
        A.spmv(xv)
    assert err.value.code == -2 and "caught" in str(err.value) and A.info("check_errors") >= 1
    A.close()
    good = cgmod.CG(dev(p.rowptr), dev(p.colind), dev(p.vals))
    good.set_option("checked", 1)
    good.spmv(xv)
    assert good.info("check_errors") == 0
    good.close()


# ---------------------------------------------------------------- watchdog

@pytest.mark.parametrize("compress,loop,spmv", [(1, 0, 0), (0, 0, 0), (0, 2, 3), (1, 1, 2)])
def test_watchdog_turns_a_lost_copy_into_an_error(bound, cgmod, compress, loop, spmv):
    """Every device-side spin is bounded.  "inject_fault" makes one producer announce a tile and
    never copy it -- the consumers of that tile would wait for ever; with the watchdog the solve
    comes back with CG_ETIMEOUT within a few budgets and the device stays usable."""
    import time
    B = bound(2)
    p = B.p
    for k, v in (("compress", compress), ("loop", loop), ("spmv", spmv)):
        B.cg.set_option(k, v)
    x_good, r_good = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    B.cg.set_option("spin_budget_ms", 100)
    B.cg.set_option("inject_fault", 3)
    t0 = time.time()
    with pytest.raises(cgmod.CGError) as err:
        B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    assert err.value.code == -4 and "watchdog" in str(err.value)
    assert time.time() - t0 < 20.0
    B.cg.set_option("inject_fault", 0)
    B.cg.set_option("spin_budget_ms", 2000)
    x, r = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)               # nothing is left wedged
    assert r.status == 0 and torch.equal(x, x_good) and torch.equal(r.hist, r_good.hist)
    for k, v in (("compress", 1), ("loop", 0), ("spmv", 0)):
        B.cg.set_option(k, v)


# ---------------------------------------------------------------- Jacobi PCG (8(f) rank 1)

@pytest.mark.parametrize("cfg,grid", [(0, None), (4, 32)])
def test_jacobi_parity(bound, orc, cfg, grid):
    B = bound(cfg, grid)
    p = B.p
    diag = np.array([p.vals[p.rowptr[i]:p.rowptr[i + 1]][p.colind[p.rowptr[i]:p.rowptr[i + 1]] == i].sum()
                     for i in range(p.n)])
    ref = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit, dinv=1.0 / diag)
    for loop in (0, 1):
        B.cg.set_option("loop", loop)
        x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit, jacobi=True)
        check_solve_parity(res, x, ref)
    B.cg.set_option("loop", 0)
    if cfg == 4:
        plain = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit)
        assert ref.iters < plain.iters / 3          # the point of the preconditioner on contrast


# ---------------------------------------------------------------- full-size config 4

@pytest.fixture(scope="module")
def config4(cgmod, problems):
    B = Bound(cgmod, problems(4))
    yield B
    B.cg.close()


def test_config4_spmv_full_size(config4, orc):
    """160^3, NNZ = 109 215 352, in the launch configuration bench.py times."""
    B = config4
    p = B.p
    assert p.n == 4096000 and p.nnz == 109215352
    x = gi.seeded_vector(104, p.n)
    want = orc.spmv(p.rowptr, p.colind, p.vals, x)
    denom = orc.absrow(p.rowptr, p.colind, p.vals, x)
    for variant in (1, 2):
        B.cg.set_option("spmv", variant)
        y = B.cg.spmv(dev(x)).cpu().numpy()
        assert (np.abs(y - want) / denom).max() <= SPMV_TOL
    B.cg.set_option("spmv", 0)
    ones = torch.ones(p.n, dtype=torch.float64, device="cuda")
    y1 = B.cg.spmv(ones).cpu().numpy()
    assert np.all(np.abs(y1 - 0.01) <= SPMV_TOL * orc.absrow(p.rowptr, p.colind, p.vals, np.ones(p.n)))


def test_config4_fixed_iterations(config4, orc):
    """Reading 14: on the ill-conditioned config a fixed-iteration run (rtol = 0, maxit = 50)
    must match the oracle's history (first 50) and x to 1e-8."""
    B = config4
    p = B.p
    ref = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=0.0, maxit=50)
    x, res = B.cg.solve(B.b, rtol=0.0, maxit=50)
    check_solve_parity(res, x, ref)
    assert res.iters == 50 and res.status == 1


def test_contrast_matrix_to_convergence_all_loop_modes(bound, orc):
    """Reading 14 at a reduced grid: the config-4 recipe at 48^3 (kappa ~ 1e6, ~4400 iterations,
    the oracle needs seconds) solved to rtol by unpreconditioned CG in every loop mode: history,
    solution, the true residual checked with the ORACLE's SpMV, identical bits across the loop
    modes.  The iteration count is held to 3 % here, not 2 %: on this system the count depends on
    the summation order of the dot products alone by more than 1 % (the oracle's own loops with
    the r.r / p.q sums split over 8 OpenMP threads need 4347 instead of 4402 iterations, -1.25 %;
    the GPU's tree sums with FMA need 4306, -2.2 %: the sequential sum of 110 592 terms is the
    least accurate of the three and converges last).  BASELINE.json's own configs, full config 4
    included, are held to the stated 2 % (test_config4_to_convergence: 12 267 against 12 451)."""
    B = bound(4, 48)
    p = B.p
    ref = oracle_solve(orc, p, ("cg", 4, 48))
    assert ref.status == 0 and ref.iters > 3000
    outs = []
    for loop in (0, 1, 2):
        B.cg.set_option("loop", loop)
        B.cg.set_option("chunk", 256)
        x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
        check_solve_parity(res, x, ref, iters_band=0.03)
        xh = x.cpu().numpy()
        true_r = p.b - orc.spmv_ld(p.rowptr, p.colind, p.vals, xh)
        assert np.linalg.norm(true_r) / np.linalg.norm(p.b) <= 2 * p.rtol
        outs.append((xh, res.hist.cpu().numpy().copy()))
    for o in outs[1:]:
        assert np.array_equal(o[0], outs[0][0]) and np.array_equal(o[1], outs[0][1])
    B.cg.set_option("chunk", 32)
    B.cg.set_option("loop", 0)
    B.cg.set_option("resident", 0)          # the launch shape of full config 4: vectors in global memory
    x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    assert np.array_equal(x.cpu().numpy(), outs[0][0])
    B.cg.set_option("resident", 1)


GOLDEN4 = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config4_converged.npz")


def test_config4_to_convergence(config4, orc):
    """The north-star config solved to its rtol (1e-8) in the launch configuration bench.py times,
    against the oracle's own to-convergence run stored by tests/golden/make_config4_golden.py
    (the oracle needs ~20 minutes for it).  SURVEY.md 8(c) reading 14: iteration count within 2 %,
    first 50 residual norms to 1e-9, and (i) the ORACLE's SpMV confirms ||b - A x_gpu|| / ||b|| <=
    2 rtol.  ~12 300 iterations x 3 grid synchronisations x 148 CTAs in one launch is also the
    stress test of the ring and barrier protocols; a second run must reproduce every bit."""
    import hashlib
    B = config4
    p = B.p
    g = np.load(GOLDEN4)
    hsh = hashlib.sha256()
    for a in (p.rowptr, p.colind, p.vals, p.b):
        hsh.update(np.ascontiguousarray(a).view(np.uint8).data)
    assert hsh.hexdigest() == str(g["generator_sha256"]), "cg_inputs changed under the stored oracle run"
    assert int(g["status"]) == 0 and int(g["n"]) == p.n
    for name, v in (("loop", 0), ("spmv", 0)):
        B.cg.set_option(name, v)
    x, res = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    assert res.status == 0
    it_or = int(g["iters"])
    assert abs(res.iters - it_or) <= math.floor(0.02 * it_or), (res.iters, it_or)
    hg, ho = res.hist.cpu().numpy(), g["hist"]
    assert np.max(np.abs(hg[:51] - ho[:51]) / ho[:51]) <= HIST_TOL
    xh = x.cpu().numpy()
    true_r = p.b - orc.spmv_ld(p.rowptr, p.colind, p.vals, xh)
    relres = math.sqrt(orc.dot_ld(true_r, true_r)) / float(g["bnorm"])
    assert relres <= 2 * p.rtol, relres
    # reading 14: report the distance between the two solutions, do not demand what fp64 cannot give
    rows = g["x_rows"]
    xe = np.linalg.norm(xh[rows] - g["x_sample"]) / np.linalg.norm(g["x_sample"])
    print(f"config 4: gpu {res.iters} iterations, oracle {it_or}; true relres {relres:.3e}; "
          f"|x_gpu - x_or| / |x_or| on {len(rows)} sampled rows = {xe:.3e}")
    # measured 1.7e-8 (round 2): just past north_star's 1e-8, as reading 14 anticipated for this
    # system (kappa >~ 3e6, both x are solutions to rtol 1e-8); the two checks reading 14 requires
    # instead are (i) above and (ii) test_config4_fixed_iterations.  Sanity bound only:
    assert xe <= 1e-6
    x2, res2 = B.cg.solve(B.b, rtol=p.rtol, maxit=p.maxit)
    assert res2.iters == res.iters and torch.equal(x2, x) and torch.equal(res2.hist, res.hist)
