"""Writes tests/golden/config4_converged.npz: the ORACLE's solve of config 4 (160^3 contrast
matrix, rtol 1e-8, maxit 20000) to convergence.

Calls only oracle/ and cg_inputs/ -- never the CUDA path.  SURVEY.md 8(c) reading 14 and
8(d) ("run it once, cache hist and x on disk keyed by the generator hash"): the oracle needs
10-25 minutes on one core for this solve, too long for a test, so its result is stored.

Stored: iters, status, resnorm, the whole residual history hist[0..iters] (the
quantity the continue-condition tests; :60 TOL), the oracle's x on a fixed sample of rows and
||x||_2 (the full x is 32 MB, too big for the repository; a second file, config4_x_full.npy,
is written next to it only with --full-x and is git-ignored), and a hash of the generator output
so that a test can tell when cg_inputs changed under the stored values.

Also writes the same for the 48^3 and 64^3 reduced grids of the same recipe (seconds each),
which the parity tests recompute live; they are stored only as a cross-check of this script.

Usage:  python tests/golden/make_config4_golden.py [--grid 160] [--full-x]
"""
from __future__ import annotations

import argparse
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import cg_inputs                      # noqa: E402
from oracle import cg_oracle as orc   # noqa: E402

SAMPLE_ROWS = 4096                    # rows of x stored (fixed stride over the whole vector)


def generator_hash(p) -> str:
    """sha256 over the CSR arrays and b: identifies the generator output the values belong to."""
    h = hashlib.sha256()
    for a in (p.rowptr, p.colind, p.vals, p.b):
        h.update(np.ascontiguousarray(a).view(np.uint8).data)
    return h.hexdigest()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--grid", type=int, default=160)
    ap.add_argument("--full-x", action="store_true")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()

    t0 = time.time()
    p = cg_inputs.make_config(4, grid=args.grid) if args.grid != 160 else cg_inputs.make_config(4)
    print(f"generated config 4 at grid {args.grid}: N={p.n} NNZ={p.nnz} in {time.time() - t0:.1f} s", flush=True)
    ghash = generator_hash(p)
    t0 = time.time()
    ref = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit)
    dt = time.time() - t0
    print(f"oracle: iters={ref.iters} status={ref.status} resnorm={ref.resnorm:.6e} in {dt:.1f} s", flush=True)
    # true residual of the oracle's own x, with the oracle's long-double SpMV
    r = p.b - orc.spmv_ld(p.rowptr, p.colind, p.vals, ref.x)
    bnorm = float(np.sqrt(orc.dot_ld(p.b, p.b)))
    true_relres = float(np.sqrt(orc.dot_ld(r, r))) / bnorm
    print(f"oracle true relres = {true_relres:.3e}", flush=True)
    rows = np.linspace(0, p.n - 1, SAMPLE_ROWS).astype(np.int64)
    name = "config4_converged.npz" if args.grid == 160 else f"config4_grid{args.grid}_converged.npz"
    out = args.out or os.path.join(HERE, name)
    np.savez_compressed(
        out,
        grid=np.int64(args.grid), n=np.int64(p.n), nnz=np.int64(p.nnz), rtol=np.float64(p.rtol),
        maxit=np.int64(p.maxit), iters=np.int64(ref.iters), status=np.int64(ref.status),
        resnorm=np.float64(ref.resnorm), hist=ref.hist, bnorm=np.float64(bnorm),
        true_relres=np.float64(true_relres), x_rows=rows, x_sample=ref.x[rows],
        x_norm=np.float64(np.sqrt(orc.dot_ld(ref.x, ref.x))),
        generator_sha256=np.array(ghash), oracle_seconds=np.float64(dt))
    print("wrote", out, flush=True)
    if args.full_x:
        np.save(os.path.join(HERE, f"config4_grid{args.grid}_x_full.npy"), ref.x)


if __name__ == "__main__":
    main()
