"""Row-block split of one CG solve over several GPUs -- the modern form of
the paper's 1 / 2 / 4-device experiment ("kernels are launched onto 1, 2 and 4 devices",
:50 the compiler "split[s] tasks equally", Table I :55-57).

NOT the default and not part of BASELINE.json's metric (north_star: one GPU, no sharding); `bench.py`
runs replicas.  This module is the sharded path for systems like config 4 whose iteration is
bandwidth-bound: every rank owns a contiguous block of rows and the matching slices of x, r, p, q.

  partition_rows    contiguous row blocks, balanced by the bytes a rank streams per iteration
                    (12 per entry + 92 per row), cut at multiples of 32 rows (the
                    kernels' tile)
  local_block       the rank's rows as a square local CSR matrix over [owned columns | halo
                    columns]; the halo rows are empty, so the library's square-CSR contract holds
                    and cg_spmv works on the extended vector unchanged
  exchange_plan     who sends which owned entries of p to whom (for the 27-point stencil in
                    natural ordering: the +-(n^2 + n + 1) neighbouring entries of the two adjacent
                    ranks, not an all-gather of p)
  RowBlockCG        the solve: per iteration one halo exchange of p (all_to_all over NVLink /
                    NVSwitch through torch.distributed), cg_spmv on the local block, and ONE
                    all-reduce of the two partial inner products' operands at a time -- the
                    scalars stay on the device (no host round trip per iteration, the paper's
                    bottleneck); the host looks at the stop flag every
                    `check_every` iterations only

What this is and is not: the data-path collectives here are NCCL calls issued between kernel
launches -- the baseline form.  The form this design is meant to reach keeps the single-GPU
persistent kernel and lets K1's consumers gather halo entries of p straight from the peers'
memory over NVLink (peer mappings of the published p vector) and fuses the two-scalar exchange
into the existing push/poll all-reduce across all ranks' CTAs; it is not built, because nothing
in this environment can run more than one GPU.  Everything here that does
not need a second GPU is tested: the partition / halo arithmetic with two gloo ranks on the CPU,
and the whole class on one GPU (world size 1) against the single-GPU solve.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional

import numpy as np

TILE_ROWS = 32


def partition_rows(rowptr: np.ndarray, world: int) -> np.ndarray:
    """bounds[world + 1]: rank r owns rows [bounds[r], bounds[r + 1]).  Balanced by streamed bytes."""
    rowptr = np.asarray(rowptr, dtype=np.int64)
    n = rowptr.size - 1
    if world < 1 or n < 1:
        raise ValueError("world >= 1 and n >= 1 required")
    cost = 12 * rowptr + 92 * np.arange(n + 1, dtype=np.int64)        # prefix sums of the per-row bytes
    bounds = np.zeros(world + 1, dtype=np.int64)
    bounds[world] = n
    for r in range(1, world):
        target = cost[n] * r // world
        i = int(np.searchsorted(cost, target))
        i = (i + TILE_ROWS // 2) // TILE_ROWS * TILE_ROWS              # cut between tiles
        bounds[r] = min(max(i, bounds[r - 1]), n)
    return bounds


@dataclass
class LocalBlock:
    rank: int
    lo: int
    hi: int
    halo: np.ndarray            # global column ids this rank reads but does not own, ascending
    rowptr: np.ndarray          # int32[n_loc + n_halo + 1]; rows n_loc.. are empty
    colind: np.ndarray          # int32, local numbering: owned c -> c - lo, halo -> n_loc + position in `halo`
    vals: np.ndarray            # float64 (the rows' entries, unchanged, in their stored order)

    @property
    def n_loc(self) -> int:
        return self.hi - self.lo

    @property
    def n_ext(self) -> int:
        return self.hi - self.lo + int(self.halo.size)


def local_block(rowptr, colind, vals, bounds, rank: int) -> LocalBlock:
    rowptr = np.asarray(rowptr, dtype=np.int64)
    lo, hi = int(bounds[rank]), int(bounds[rank + 1])
    s, e = int(rowptr[lo]), int(rowptr[hi])
    cols = np.asarray(colind[s:e], dtype=np.int64)
    owned = (cols >= lo) & (cols < hi)
    halo = np.unique(cols[~owned])
    loc = np.where(owned, cols - lo, (hi - lo) + np.searchsorted(halo, cols))
    n_loc = hi - lo
    rp = np.concatenate([rowptr[lo:hi + 1] - s, np.full(halo.size, e - s, dtype=np.int64)])
    if n_loc + halo.size >= 2 ** 31 - 64:
        raise ValueError("local block too large for int32 indices")
    return LocalBlock(rank, lo, hi, halo, rp.astype(np.int32), loc.astype(np.int32),
                      np.ascontiguousarray(vals[s:e], dtype=np.float64))


@dataclass
class ExchangePlan:
    send_idx: List[np.ndarray]   # per peer: LOCAL indices (0 .. n_loc) of owned entries to send, in the peer's halo order
    recv_cnt: List[int]          # per peer: how many halo entries come from it (they are contiguous in `halo`)

    @property
    def send_cnt(self) -> List[int]:
        return [int(a.size) for a in self.send_idx]


def exchange_plan(block: LocalBlock, bounds, all_halos: List[np.ndarray]) -> ExchangePlan:
    """`all_halos[q]` is rank q's halo list (gathered once at setup).  The halo is sorted by
    global id and ownership is by contiguous ranges, so what comes from peer q is one contiguous
    run of my halo, and what I send to q is the part of q's halo inside my range."""
    world = len(bounds) - 1
    send, recv = [], []
    for q in range(world):
        hq = np.asarray(all_halos[q], dtype=np.int64)
        mine = hq[(hq >= block.lo) & (hq < block.hi)] if q != block.rank else hq[:0]
        send.append((mine - block.lo).astype(np.int64))
        recv.append(int(np.count_nonzero((block.halo >= bounds[q]) & (block.halo < bounds[q + 1]))) if q != block.rank else 0)
    assert sum(recv) == block.halo.size
    return ExchangePlan(send, recv)


class RowBlockCG:
    """One rank's share of a row-block CG solve on its GPU.  `dist` is torch.distributed (already
    initialised, backend nccl) or None for a single rank."""

    def __init__(self, rowptr, colind, vals, dist=None, device=None, check_every: int = 16):
        import torch
        from . import binding
        self.torch, self.dist = torch, dist
        self.rank = dist.get_rank() if dist is not None else 0
        self.world = dist.get_world_size() if dist is not None else 1
        self.device = device if device is not None else torch.device("cuda", torch.cuda.current_device())
        self.check_every = int(check_every)
        self.bounds = partition_rows(rowptr, self.world)
        self.block = local_block(rowptr, colind, vals, self.bounds, self.rank)
        if dist is not None and self.world > 1:
            halos: List[Optional[np.ndarray]] = [None] * self.world
            dist.all_gather_object(halos, self.block.halo)
        else:
            halos = [self.block.halo]
        self.plan = exchange_plan(self.block, self.bounds, halos)
        to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(self.device)
        self.A = binding.CG(to(self.block.rowptr), to(self.block.colind), to(self.block.vals))
        self.send_idx = to(np.concatenate(self.plan.send_idx) if self.world > 1 else np.zeros(0, dtype=np.int64))
        self.n_loc, self.n_ext = self.block.n_loc, self.block.n_ext

    def close(self):
        self.A.close()

    def _halo_exchange(self, p_ext):
        """p_ext[:n_loc] is mine; fill p_ext[n_loc:] with the peers' entries."""
        if self.world == 1:
            return
        out = p_ext[:self.n_loc].index_select(0, self.send_idx)
        self.dist.all_to_all_single(p_ext[self.n_loc:], out, output_split_sizes=self.plan.recv_cnt,
                                    input_split_sizes=self.plan.send_cnt)

    def _allreduce(self, t):
        if self.world > 1:
            self.dist.all_reduce(t)
        return t

    def spmv(self, x_loc):
        """y_loc = (A x)[lo:hi] from this rank's slice of x (one halo exchange)."""
        torch = self.torch
        x_ext = torch.zeros(self.n_ext, dtype=torch.float64, device=self.device)
        x_ext[:self.n_loc] = x_loc
        self._halo_exchange(x_ext)
        return self.A.spmv(x_ext)[:self.n_loc]

    def solve(self, b_loc, x0_loc=None, rtol=1e-10, maxit=None):
        """Textbook CG (the recurrence of cg_solve) on this rank's slices.  Returns (x_loc, iters,
        status, hist) with hist on the host; status as cg_solve (0 converged, 1 maxit, 2 breakdown)."""
        torch = self.torch
        n_loc, dev = self.n_loc, self.device
        maxit = int(self.bounds[-1]) if maxit is None else int(maxit)
        x = torch.zeros(n_loc, dtype=torch.float64, device=dev) if x0_loc is None else x0_loc.clone()
        p_ext = torch.zeros(self.n_ext, dtype=torch.float64, device=dev)
        q_ext = torch.empty(self.n_ext, dtype=torch.float64, device=dev)
        p_ext[:n_loc] = x
        self._halo_exchange(p_ext)
        self.A.spmv(p_ext, out=q_ext)
        r = b_loc - q_ext[:n_loc]
        p_ext[:n_loc] = r
        s = self._allreduce(torch.stack([torch.dot(r, r), torch.dot(b_loc, b_loc)]))
        rr, bb = s[0].clone(), s[1]
        hist_dev = torch.zeros(maxit + 1, dtype=torch.float64, device=dev)
        hist_dev[0] = torch.sqrt(rr)
        if float(bb) == 0.0:
            return torch.zeros_like(x), 0, 0, np.zeros(1)
        thresh = float(rtol) * float(torch.sqrt(bb))
        if float(hist_dev[0]) <= thresh:
            return x, 0, 0, hist_dev[:1].cpu().numpy()
        if maxit == 0:
            return x, 0, 1, hist_dev[:1].cpu().numpy()
        zero = torch.zeros((), dtype=torch.float64, device=dev)
        done = torch.zeros((), dtype=torch.bool, device=dev)       # the stop test was met (device-side flag)
        broke = torch.zeros((), dtype=torch.bool, device=dev)      # p.Ap <= 0 or not finite
        kdone = torch.zeros((), dtype=torch.int64, device=dev)     # iterations that really updated x
        k = 0
        while k < maxit:
            for _ in range(min(self.check_every, maxit - k)):
                self._halo_exchange(p_ext)
                self.A.spmv(p_ext, out=q_ext)
                p, q = p_ext[:n_loc], q_ext[:n_loc]
                pq = self._allreduce(torch.dot(p, q).reshape(1))[0]
                broke = broke | (~done & ~((pq > 0) & torch.isfinite(pq)))
                active = ~(done | broke)           # once stopped, the remaining iterations of the chunk are no-ops
                alpha = torch.where(active, rr / pq, zero)
                x.add_(p * alpha)
                r.sub_(q * alpha)
                rr_new = self._allreduce(torch.dot(r, r).reshape(1))[0]
                beta = torch.where(active, rr_new / rr, zero)
                rr = torch.where(active, rr_new, rr)
                kdone = kdone + active.to(torch.int64)
                k += 1
                hist_dev[k] = torch.sqrt(rr)
                done = done | (active & (torch.sqrt(rr) <= thresh))
                p.mul_(beta).add_(r)
            if bool(done | broke):                 # the one host look per `check_every` iterations
                break
        iters = int(kdone)
        status = 2 if bool(broke) else 0 if bool(done) else 1
        return x, iters, status, hist_dev[:iters + 1].cpu().numpy()
