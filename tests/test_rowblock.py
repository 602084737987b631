"""Row-block multi-GPU split: the partition / halo /
exchange arithmetic with two gloo ranks on the CPU, and the whole RowBlockCG class on one GPU."""
import os
import sys

import numpy as np
import pytest

import cg_inputs as gi
from paper_1107_0538_b200 import rowblock as rb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_balances_bytes_and_cuts_between_tiles():
    p = gi.make_config(0, grid=24)
    for world in (1, 2, 3, 4, 8):
        b = rb.partition_rows(p.rowptr, world)
        assert b[0] == 0 and b[-1] == p.n and np.all(np.diff(b) > 0)
        assert np.all(b[1:-1] % 32 == 0)
        cost = 12 * np.diff(p.rowptr.astype(np.int64)[b]) + 92 * np.diff(b)
        assert cost.max() <= 1.05 * cost.mean() + 12 * 27 * 32 + 92 * 32       # within one tile of even


def test_local_blocks_reassemble_the_matrix_and_the_spmv():
    """Every entry lands in exactly one block with its value, owned columns map to [0, n_loc), halo
    columns to the sorted halo list; the blocks' local SpMVs on [owned | halo] slices of x put
    together are the global SpMV (checked against the oracle)."""
    from oracle import cg_oracle as orc
    p = gi.make_config(2, grid=12)
    x = gi.seeded_vector(3, p.n)
    want = orc.spmv(p.rowptr, p.colind, p.vals, x)
    for world in (1, 2, 3, 5):
        bounds = rb.partition_rows(p.rowptr, world)
        blocks = [rb.local_block(p.rowptr, p.colind, p.vals, bounds, r) for r in range(world)]
        halos = [b.halo for b in blocks]
        got = np.zeros(p.n)
        nnz = 0
        for b in blocks:
            plan = rb.exchange_plan(b, bounds, halos)
            assert np.all((b.halo < b.lo) | (b.halo >= b.hi)) and np.all(np.diff(b.halo) > 0)
            assert b.rowptr[-1] == len(b.vals) and np.all(b.rowptr[b.n_loc:] == len(b.vals))     # halo rows are empty
            assert b.colind.max(initial=0) < b.n_ext
            # what the peers would send me, in my halo order
            x_ext = np.concatenate([x[b.lo:b.hi], np.zeros(b.halo.size)])
            pos = b.n_loc
            for q in range(world):
                if q == b.rank:
                    continue
                their = rb.exchange_plan(blocks[q], bounds, halos)
                chunk = x[blocks[q].lo:blocks[q].hi][their.send_idx[b.rank]]
                assert chunk.size == plan.recv_cnt[q]
                x_ext[pos:pos + chunk.size] = chunk
                pos += chunk.size
            assert pos == b.n_ext and np.array_equal(x_ext[b.n_loc:], x[b.halo])
            y = orc.spmv(b.rowptr, b.colind, b.vals, x_ext)
            got[b.lo:b.hi] = y[:b.n_loc]
            nnz += len(b.vals)
        assert nnz == p.nnz and np.array_equal(got, want)          # same entries in the same order: same bits
    # the 27-point stencil in natural ordering only needs +-(n^2 + n + 1) neighbouring entries
    n = 12
    bounds = rb.partition_rows(p.rowptr, 4)
    b1 = rb.local_block(p.rowptr, p.colind, p.vals, bounds, 1)
    assert b1.halo.min() >= b1.lo - (n * n + n + 1) and b1.halo.max() < b1.hi + (n * n + n + 1)
    assert b1.halo.size <= 2 * (n * n + n + 1)


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import cg_inputs as gi
from paper_1107_0538_b200 import rowblock as rb
from oracle import cg_oracle as orc            # test infrastructure: the local SpMV of this CPU test
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
p = gi.make_config(0, grid=10)
bounds = rb.partition_rows(p.rowptr, 2)
blk = rb.local_block(p.rowptr, p.colind, p.vals, bounds, rank)
halos = [None, None]
dist.all_gather_object(halos, blk.halo)
plan = rb.exchange_plan(blk, bounds, halos)
def exchange(v_loc):
    ext = np.concatenate([v_loc, np.zeros(blk.halo.size)])
    peer = 1 - rank
    send = torch.from_numpy(np.ascontiguousarray(v_loc[plan.send_idx[peer]]))
    recv = torch.zeros(plan.recv_cnt[peer], dtype=torch.float64)
    reqs = [dist.isend(send, peer), dist.irecv(recv, peer)]
    for r_ in reqs: r_.wait()
    ext[blk.n_loc:] = recv.numpy()
    return ext
def allsum(v):
    t = torch.tensor([v], dtype=torch.float64); dist.all_reduce(t); return float(t[0])
# the textbook recurrence on the two row blocks: halo exchange + two scalar all-reduces per iteration
b = p.b[blk.lo:blk.hi]
x = np.zeros(blk.n_loc); r = b.copy(); pv = r.copy()
rr = allsum(r @ r); hist = [np.sqrt(rr)]
for k in range(30):
    q = orc.spmv(blk.rowptr, blk.colind, blk.vals, exchange(pv))[:blk.n_loc]
    alpha = rr / allsum(pv @ q)
    x += alpha * pv; r -= alpha * q
    rr_new = allsum(r @ r); beta = rr_new / rr; rr = rr_new
    pv = r + beta * pv; hist.append(np.sqrt(rr))
ref = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=0.0, maxit=30)
assert np.max(np.abs(np.array(hist) - ref.hist) / ref.hist) < 1e-9, "history"
assert np.linalg.norm(x - ref.x[blk.lo:blk.hi]) / np.linalg.norm(ref.x) < 1e-10, "x"
dist.barrier(); dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_two_rank_halo_exchange_and_recurrence_gloo(tmp_path):
    """World size 2 over gloo on the CPU: the exchange plan moves exactly the halo entries and the
    sharded recurrence (one halo exchange + two scalar all-reduces per iteration, no all-gather of
    p) reproduces the oracle's history and solution."""
    import socket
    import subprocess
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
             for r in range(2)]
    outs = [pr.communicate(timeout=300)[0] for pr in procs]
    for r, (pr, out) in enumerate(zip(procs, outs)):
        assert pr.returncode == 0 and f"rank {r} ok" in out, out


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,grid", [(0, None), (2, 20)])
def test_rowblock_cg_single_rank_on_gpu(cfg, grid):
    """RowBlockCG with one rank (no peers: the halo is empty) runs the same recurrence through
    cg_spmv with device-side scalars and a host look every 16 iterations: all four bands against the
    oracle, and the reported iteration count is the first that met the test."""
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    from oracle import cg_oracle as orc
    p = gi.make_config(cfg, grid)
    ref = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit)
    S = rb.RowBlockCG(p.rowptr, p.colind, p.vals, dist=None)
    assert S.n_ext == S.n_loc == p.n
    b = torch.from_numpy(p.b).cuda()
    x, iters, status, hist = S.solve(b, rtol=p.rtol, maxit=p.maxit)
    assert status == 0 and abs(iters - ref.iters) <= max(1, int(0.03 * ref.iters)) and len(hist) == iters + 1
    k = min(50, iters, ref.iters)
    assert np.max(np.abs(hist[:k + 1] - ref.hist[:k + 1]) / ref.hist[:k + 1]) <= 1e-9
    assert np.linalg.norm(x.cpu().numpy() - ref.x) / np.linalg.norm(ref.x) <= 1e-8
    y = S.spmv(b).cpu().numpy()
    want = orc.spmv(p.rowptr, p.colind, p.vals, p.b)
    assert np.all(np.abs(y - want) <= 1e-13 * orc.absrow(p.rowptr, p.colind, p.vals, p.b))
    x2, it2, st2, h2 = S.solve(b, rtol=0.0, maxit=7)
    assert it2 == 7 and st2 == 1 and len(h2) == 8
    S.close()
