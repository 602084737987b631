#!/usr/bin/env python
"""bench.py -- fp64 CG iterations/s on the paper-shaped workload (BASELINE.json metric).

One "step" is one whole cg_solve (prologue a0, then K1/K2/K3 with the device-side scalar
steps until the continue-condition stops the loop) on config 2: the
27-point 51^3 matrix with exactly the paper's N = 132651, NNZ = 3442951, TOL = 1e-10
(PAPER.md:34, :60).  Timed like the paper times it ("just computing and data
transfer times in CG loop"): generation, the one-off upload of the matrix and cg_create
are outside the timed region.

  value      iterations/s, inputs already resident in HBM, CUDA events per step on the
             launching stream, L2 flushed between steps (inside one solve the 41.9 MB matrix
             is L2-resident by design -- north_star asks for exactly that to be reported)
  e2e        same metric through cg_solve_host: pinned HOST b / x0 in, x and the residual
             history back, copies inside the timed region
  roofline   the persistent kernel (the one launch of a step) against measured HBM peak
  north_star_160   the HBM-bound 160^3 config (config 4): fixed-work run, roofline fraction
  cpu_baseline     the oracle as it stands, on the host, on a bounded sample

`--impl reference` times the CPU oracle (this tier's reference arm) on the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import cg_inputs  # noqa: E402

METRIC = "fp64_cg_iterations_per_s"
UNIT = "iterations/s"
WORKLOAD_CFG = 2


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md, MEASURED_PEAKS.json absent)"


class ClockSampler:
    """Samples SM clocks and throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, reasons = [], None, set()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.1] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax = float(f[1])
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


def reduce_over_ranks(dist, value, op, device):
    """MAX or SUM of one float over the ranks of the job (identity when dist is None).
    Replicas only: the only cross-rank traffic of the bench is this bookkeeping."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_value(dist, device, iterations_this_rank, seconds_this_rank):
    """iterations of ALL ranks / MAX over ranks of the device time (weak scaling, replicas)."""
    t = reduce_over_ranks(dist, seconds_this_rank, "max", device)
    n = reduce_over_ranks(dist, iterations_this_rank, "sum", device)
    return n / t, n, t


def describe(A):
    """Launch configuration of the handle the solves run on, from cg_get_info ("solve_*": the renumbered
    matrix's handle after cg_reorder, else the handle itself)."""
    info = lambda name: A.info("solve_" + name)
    v = info("spmv")
    d = {"loop": {0: "persistent cooperative kernel", 1: "cuda graph", 2: "stepwise launches"}[info("loop")],
         "grid": info("grid"), "block": info("block"), "smem_bytes": info("smem")}
    if A.info("reordered"):
        d["numbering"] = (f"reverse Cuthill-McKee (cg_reorder): {A.info('lines_per_gather_x100') / 100:.1f} -> "
                          f"{info('lines_per_gather_x100') / 100:.1f} lines per warp-wide gather; b, x0 gathered and x "
                          "scattered by two small kernels inside the timed region")
    if v == 1:
        d["spmv"] = f"generic: {info('tpr')} lanes per row from global memory"
    else:
        npw, pin, slots = info("producer_warps"), info("pinned_tiles"), info("ring_slots")
        who = (f"{npw} TMA producer warps + {info('consumer_warps')} consumer warps" if npw
               else f"{info('consumer_warps')} consumer warps, each copying its own tiles once per launch (TMA bulk copies)")
        where = (f"{slots} x {info('slot_bytes')} B tiles pinned in shared memory" if pin >= slots
                 else f"ring of {slots} x {info('slot_bytes')} B tiles" + (f", {pin} of them pinned" if pin else ""))
        flight = ("9 gathers per tile, 2-3 tiles in flight per lane (short-row kernel)" if info("short_rows")
                  else f"{info('in_flight')} gathers in flight per lane")
        d["spmv"] = (f"streamed: {who}, one lane per row, {flight}, {where}, "
                     + ("compressed column index (9 B per entry)" if info("compressed") else "plain CSR slots (12 B per entry)"))
        rr = info("resident_rows")
        d["vectors"] = (f"x, r, p, q in registers ({4 if info('short_rows') else rr} rows per thread)" if rr and info("loop") == 0
                        else "x, r, p, q in global memory")
    return d


def workload_string(p):
    """The one description of the metric's workload, shared by both arms (the driver compares them)."""
    return (f"config{WORKLOAD_CFG} {p.name} N={p.n} NNZ={p.nnz} rtol={p.rtol:g} x0=0 maxit=N, "
            "one step = one full cg_solve to convergence")


def kernel_name(A):
    """Which instantiation of the persistent kernel a handle launches, from cg_get_info."""
    info = lambda name: A.info("solve_" + name)
    if info("spmv") == 1:
        return "k_persistent (generic)"
    if info("short_rows"):
        return f"ks_persistent<W={info('consumer_warps')},NP=0,U=9,R=4,fold=0,cmp=1> (short rows)"
    return (f"ks_persistent<W={info('consumer_warps')},NP={info('producer_warps')},U={info('in_flight')},"
            f"R={info('resident_rows')},fold={info('fold')},cmp={info('compressed')}>"
            + (" (renumbered)" if A.info("reordered") else ""))


def traffic_entry(cfg, kernel, iterations):
    """DRAM bytes per launch of `kernel` on config `cfg` from the committed ncu capture list
    profiles/r02_traffic.json (written by hand from `ncu --set full` captures, each entry names its
    file).  None, with the reason, when no capture of this very kernel and iteration count exists:
    a stale figure is worse than none."""
    path = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        with open(path) as f:
            entries = json.load(f)["entries"]
    except (OSError, ValueError, KeyError):
        return {"traffic": None, "traffic_note": "profiles/r02_traffic.json missing"}
    for e in entries:
        if e["config"] == cfg and e["kernel"] == kernel and abs(e["iterations"] - iterations) <= 0.02 * iterations:
            return {"traffic": e["dram_bytes"], "traffic_source": e["source"]}
    return {"traffic": None, "traffic_note": f"no ncu capture of {kernel} on config{cfg} with {iterations:g} iterations on file"}


def per_config_leg(cg, torch, dev, cfg, p, args, peak, l2_gbs, flush_l2, with_cpu):
    """Fixed-work throughput, the SpMV alone, the solve to convergence and the oracle's fixed work
    for one BASELINE.json config."""
    p = p if p is not None else cg_inputs.make_config(cfg)
    A = cg.CG(*(torch.from_numpy(a).to(dev) for a in (p.rowptr, p.colind, p.vals)))
    A.set_option("loop", args.loop)
    A.set_option("spmv", args.spmv)
    b = torch.from_numpy(p.b).to(dev)
    x = torch.zeros(p.n, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream().cuda_stream
    bytes_it = cg_inputs.algorithmic_bytes_per_iteration(p.n, p.nnz)
    flops_it = cg_inputs.flops_per_iteration(p.n, p.nnz)
    K = args.fixed_iters_160 if cfg == 4 else 2000

    def timed_solve(rtol, maxit, flush):
        x.zero_()
        if flush:
            flush_l2()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        st, it, res = cg.cg_solve(A.h, b.data_ptr(), x.data_ptr(), rtol, maxit, None, stream)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3, it, st

    timed_solve(0.0, K, False)
    ts = []
    for _ in range(5):
        t, it, st = timed_solve(0.0, K, cfg != 4)           # config 4's 1.33 GB of inputs exceed the L2 anyway
        assert it == K
        ts.append(t / K)
    med, mn = float(np.median(ts)), float(min(ts))
    rec = {
        "workload": f"config{cfg} {p.name} N={p.n} NNZ={p.nnz}, fixed work: rtol=0, maxit={K}"
                    + (" (inputs 1.33 GB >> L2)" if cfg == 4 else " (L2 flushed between solves)"),
        "us_per_iteration": {"median": med * 1e6, "min": mn * 1e6, "reps": len(ts)},
        "iterations_per_s": 1.0 / med,
        "effective_gbs": bytes_it / med / 1e9,
        "cg_gflops": flops_it / med / 1e9,
        "roofline": {"bound": "hbm", "achieved": bytes_it / med / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": bytes_it / med / 1e9 / peak,
                     "bytes_model": "12 NNZ + 92 N + 4 per iteration (SURVEY.md 8(d): plain CSR, the method's bytes)"
                                    + ("; the compressed index moves 9.1 NNZ + 92 N" if A.info("solve_compressed") else ""),
                     **traffic_entry(cfg, kernel_name(A), K)},
        "launch": describe(A),
    }
    if cfg != 4:
        rec["frac_of_l2_read_peak"] = bytes_it / med / 1e9 / l2_gbs
    # the SpMV alone through the ABI ("DGEMV(sparse)"; gflops = 2 NNZ / t)
    xv = torch.from_numpy(cg_inputs.seeded_vector(50 + cfg, p.n)).to(dev)
    y = torch.empty_like(xv)
    for _ in range(3):
        A.spmv(xv, out=y)
    reps = 20 if cfg == 4 else 100
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        A.spmv(xv, out=y)
    e1.record()
    torch.cuda.synchronize()
    t_spmv = e0.elapsed_time(e1) * 1e-3 / reps
    spmv_bytes = 12 * p.nnz + 4 * (p.n + 1) + 16 * p.n
    rec["spmv"] = {"us": t_spmv * 1e6, "gflops": 2 * p.nnz / t_spmv / 1e9, "effective_gbs": spmv_bytes / t_spmv / 1e9,
                   "frac_of_hbm_peak": spmv_bytes / t_spmv / 1e9 / peak,
                   "what": f"cg_spmv, {reps} back-to-back launches (each one refills its shared-memory slots"
                           + (" from the L2" if cfg != 4 else " from HBM") + ")"}
    # K1 inside the persistent loop, from the phase trace (slowest CTA per iteration)
    if A.info("loop") == 0 and A.info("solve_spmv") >= 2:
        n_tr = 24
        tr = A.trace(n_tr)
        timed_solve(0.0, n_tr, False)
        tt = tr.cpu().numpy().astype(np.int64)[:, 2:n_tr - 1, :8]
        A.trace(0)
        k1 = float((tt[:, :, 1] - tt[:, :, 0]).max(axis=0).mean())
        it_cyc = float((np.diff(tt[:, :, 0], axis=1)).mean())
        sync = float(((tt[:, :, 2] - tt[:, :, 1]) + (tt[:, :, 4] - tt[:, :, 3]) + (tt[:, :, 7] - tt[:, :, 6])).mean())
        t_k1 = med * k1 / it_cyc
        rec["k1_in_loop"] = {"cycles": k1, "share_of_iteration": k1 / it_cyc, "us": t_k1 * 1e6,
                             "spmv_gflops": 2 * p.nnz / t_k1 / 1e9,
                             "grid_sync_share_of_iteration": sync / it_cyc,
                             "what": "cg_set_trace over 24 iterations: K1 of the slowest CTA per iteration, scaled to the untraced iteration time"}
    if cfg != 4 and A.info("loop") == 0:
        # the reduced-synchronisation recurrences, reported BESIDE the textbook path (options, never the
        # metric).  Timed on the solve to convergence: past the accuracy the arithmetic can reach their
        # denominators lose positivity (CG_BREAKDOWN), so a fixed 2000 iterations is not a workload for them.
        var = {}
        for algo, name in ((1, "chronopoulos_gear"), (2, "pipelined")):
            A.set_option("algo", algo)
            if A.info("solve_algo") == algo:
                timed_solve(p.rtol, p.maxit, True)
                runs = sorted((timed_solve(p.rtol, p.maxit, True) for _ in range(3)), key=lambda r: r[0])
                t, it, st = runs[1]
                var[name] = {"iterations": it, "status": st, "us_per_iteration": t / max(it, 1) * 1e6,
                             "frac_of_hbm_roofline": bytes_it * it / t / 1e9 / peak,
                             "what": "solve to convergence, prologue (two SpMVs) included"}
        A.set_option("algo", 0)
        rec["reduced_sync_variants"] = var
    if A.info("reordered"):
        # the same fixed work in the caller's numbering: the gather-bound regime the config stands for
        A.set_option("reorder", 0)
        timed_solve(0.0, K, False)
        t0s = [timed_solve(0.0, K, True)[0] / K for _ in range(3)]
        m0 = float(np.median(t0s))
        rec["callers_numbering"] = {"us_per_iteration": m0 * 1e6, "frac_of_hbm_roofline": bytes_it / m0 / 1e9 / peak,
                                    "launch": describe(A), **traffic_entry(cfg, kernel_name(A), K),
                                    "what": 'cg_set_option "reorder" = 0: same handle, same kernels, rows as the caller numbered them'}
        A.set_option("reorder", 1)
    if cfg != 4:
        timed_solve(p.rtol, p.maxit, True)
        tc = [timed_solve(p.rtol, p.maxit, True) for _ in range(3)]
        t_med = float(np.median([t for t, _, _ in tc]))
        rec["to_convergence"] = {"iterations": tc[0][1], "status": tc[0][2], "ms": t_med * 1e3,
                                 "iterations_per_s": tc[0][1] / t_med, "rtol": p.rtol}
    A.close()
    if with_cpu:
        from oracle import cg_oracle as orc
        K_or = 20 if cfg == 4 else 200
        t0 = time.perf_counter()
        r = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=0.0, maxit=K_or)
        dt = time.perf_counter() - t0
        rec["oracle_fixed_work"] = {"iterations_per_s": r.iters / dt, "us_per_iteration": dt / r.iters * 1e6,
                                    "cores": 1, "kind": "oracle", "sample": f"rtol=0, maxit={K_or} ({dt:.2f} s)"}
    return rec


def time_oracle(problem, seconds_budget, fixed_iters=None):
    """The CPU oracle as it stands, single thread, on a bounded sample of the workload."""
    from oracle import cg_oracle as orc
    p = problem
    total_it, t0 = 0, time.perf_counter()
    solves = 0
    while True:
        if fixed_iters is None:
            r = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit)
        else:
            r = orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=0.0, maxit=fixed_iters)
        total_it += r.iters
        solves += 1
        dt = time.perf_counter() - t0
        if dt >= seconds_budget:
            break
    return total_it / dt, solves, total_it, dt


def time_oracle_omp(problem, seconds_budget):
    """oracle/cg_oracle_omp.c (row-parallel OpenMP build of the oracle's loops; checked against
    the oracle in tests/test_oracle_pins.py) on all host cores and on half of them (containers
    often expose more CPUs than they may use); the faster of the two is reported."""
    from oracle import cg_oracle as orc
    p = problem
    ncpu = os.cpu_count() or 1
    best = None
    for threads in sorted({ncpu, max(1, ncpu // 2)}, reverse=True):
        orc.omp_set_threads(threads)
        orc.cg_omp(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit)       # warm-up
        its, solves, t0 = 0, 0, time.perf_counter()
        while True:
            its += orc.cg_omp(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit).iters
            solves += 1
            dt = time.perf_counter() - t0
            if dt >= seconds_budget / 2:
                break
        rec = {"value": its / dt, "unit": UNIT, "cores": threads, "kind": "oracle loops + OpenMP (cg_oracle_omp.c)",
               "sample": f"{solves} full solves of config{WORKLOAD_CFG} ({its} iterations, {dt:.1f} s)"}
        if best is None or rec["value"] > best["value"]:
            best = rec
    return best


def run_reference(args):
    """--impl reference: this tier's reference arm is the CPU oracle (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    p = cg_inputs.make_config(WORKLOAD_CFG)
    from oracle import cg_oracle as orc
    for _ in range(args.warmup):
        orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit)
    iters, t0 = 0, time.perf_counter()
    for _ in range(args.steps):
        iters += orc.cg(p.rowptr, p.colind, p.vals, p.b, rtol=p.rtol, maxit=p.maxit).iters
    dt = time.perf_counter() - t0
    v = iters / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload_string(p),
                   "sample": "each step is the whole workload (one full solve), no sub-sampling"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"{args.steps} full solves of config{WORKLOAD_CFG} ({iters} iterations)"},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-160", action="store_true", help="skip the 160^3 north-star leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config legs (configs 0-4, fixed work)")
    ap.add_argument("--loop", type=int, default=0)
    ap.add_argument("--spmv", type=int, default=0)
    ap.add_argument("--fixed-iters-160", type=int, default=200)
    ap.add_argument("--profile", type=int, default=None, metavar="CFG",
                    help="profiling aid (ncu): only run 3 fixed-work solves of config CFG and exit")
    ap.add_argument("--profile-iters", type=int, default=6)
    ap.add_argument("--ctas-per-sm", type=int, default=0)
    ap.add_argument("--lookahead", type=int, default=None)
    ap.add_argument("--resident", type=int, default=None)
    ap.add_argument("--ring-slots", type=int, default=None)
    ap.add_argument("--fold", type=int, default=None)
    ap.add_argument("--pin", type=int, default=None)
    ap.add_argument("--compress", type=int, default=None)
    ap.add_argument("--algo", type=int, default=None, help="with --profile: 1 = Chronopoulos-Gear, 2 = pipelined CG")
    ap.add_argument("--reorder", type=int, default=None, help="with --profile: 0 = solve in the caller's numbering")
    ap.add_argument("--short-rows", type=int, default=None, dest="short_rows", help="with --profile: 0 = no short-row kernels")
    ap.add_argument("--trace-clock", type=int, default=0, dest="trace_clock",
                    help="with --trace: 1 = stamp %%globaltimer (ns, comparable across CTAs) and print the skew at each synchronisation")
    ap.add_argument("--trace", action="store_true",
                    help="with --profile and --loop 0: print the per-phase cycle breakdown (cg_set_trace)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)

    import torch
    import paper_1107_0538_b200 as cg   # raises if libcg_b200.so is missing: no CPU fallback

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product has no CPU path)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(v):
        return reduce_over_ranks(dist, v, "max", "cuda")

    def sum_over_ranks(v):
        return reduce_over_ranks(dist, v, "sum", "cuda")

    peak, peak_src = measured_peaks()
    dev = torch.device("cuda", local)
    flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device=dev)     # 4x the 126 MB L2

    def flush_l2():
        flush_buf.fill_(1)

    def bind(p):
        rp, ci, va = (torch.from_numpy(a).to(dev) for a in (p.rowptr, p.colind, p.vals))
        return cg.CG(rp, ci, va)

    if args.profile is not None:
        pp = cg_inputs.make_config(args.profile)
        Ap = bind(pp)
        Ap.set_option("loop", args.loop)
        Ap.set_option("spmv", args.spmv)
        if args.profile_iters % 2 == 0:
            Ap.set_option("chunk", args.profile_iters)      # no no-op launches after the stop flag
        if args.ctas_per_sm:
            Ap.set_option("ctas_per_sm", args.ctas_per_sm)
        if args.lookahead is not None:
            Ap.set_option("lookahead", args.lookahead)
        if args.resident is not None:
            Ap.set_option("resident", args.resident)
        if args.ring_slots is not None:
            Ap.set_option("ring_slots", args.ring_slots)
        if args.fold is not None:
            Ap.set_option("fold", args.fold)
        if args.pin is not None:
            Ap.set_option("pin", args.pin)
        if args.compress is not None:
            Ap.set_option("compress", args.compress)
        if args.algo is not None:
            Ap.set_option("algo", args.algo)
        if args.reorder is not None:
            Ap.set_option("reorder", args.reorder)
        if args.short_rows is not None:
            Ap.set_option("short_rows", args.short_rows)
        bp = torch.from_numpy(pp.b).to(dev)
        xp = torch.zeros(pp.n, dtype=torch.float64, device=dev)
        out = []
        Ap.set_option("trace_clock", args.trace_clock)
        tr = Ap.trace(args.profile_iters) if (args.trace and args.loop == 0) else None
        for rep in range(3):
            xp.zero_()
            flush_l2()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            st, it, res = cg.cg_solve(Ap.h, bp.data_ptr(), xp.data_ptr(), 0.0, args.profile_iters, None,
                                      torch.cuda.current_stream().cuda_stream)
            e1.record()
            torch.cuda.synchronize()
            out.append(e0.elapsed_time(e1) * 1e3 / max(it, 1))
        rec = {"profile_config": args.profile, "iters": args.profile_iters, "us_per_iteration": out,
               "loop": Ap.info("solve_loop"), "spmv": Ap.info("solve_spmv"), "grid": Ap.info("solve_grid"),
               "compressed": Ap.info("solve_compressed"), "pinned_tiles": Ap.info("solve_pinned_tiles"),
               "ring_slots": Ap.info("solve_ring_slots"), "fold": Ap.info("solve_fold"), "resident_rows": Ap.info("solve_resident_rows"),
               "algo": Ap.info("solve_algo"), "short_rows": Ap.info("solve_short_rows"), "reordered": Ap.info("reordered"),
               "kernel": kernel_name(Ap)}
        if tr is not None:
            # [cta, iter, slot] clock64 stamps -> cycles per interval; skip the first 2 iterations
            full = tr.cpu().numpy().astype(np.int64)
            st = full[:, args.profile_iters, :]
            rec["ring_stats"] = {"producer_wait_cycles": float(st[:, 0].mean()), "producer_total_cycles": float(st[:, 1].mean()),
                                 "tiles_issued": float(st[:, 2].mean()), "consumer_warp0_full_wait_cycles": float(st[:, 3].mean())}
            t = full[:, 2:args.profile_iters - 1, :]
            names = {0: ["K1 work", "barrier 1", "alpha + K2 work", "barrier 2", "beta", "K3 work", "barrier 3"],
                     1: ["vector updates", "publish barrier", "K1 work", "all-reduce", "scalars", "(unused a)", "(unused b)"],
                     2: ["K1 work", "partials read + sum", "scalars", "(unused a)", "(unused b)", "vector updates", "barrier"]}[Ap.info("solve_algo")]
            d = np.diff(t[:, :, :8], axis=2)
            if t.shape[2] >= 16 and t[:, :, 8:].any():
                dd = np.diff(t[:, :, 8:], axis=2)
                rec["barrier3_detail_cycles"] = {nm: float(dd[:, :, i].mean()) for i, nm in enumerate(
                    ["cta reduce", "publish", "poll", "syncwarp", "fence", "totals", "final sync"])}
            rec["trace_cycles"] = {nm: {"mean": float(d[:, :, i].mean()), "max_cta": float(d[:, :, i].max(axis=0).mean()),
                                        "min_cta": float(d[:, :, i].min(axis=0).mean())} for i, nm in enumerate(names)}
            rec["trace_cycles"]["iteration"] = float((t[:, :, 7] - t[:, :, 0]).mean())
            if args.trace_clock:
                # one clock for all SMs: the stamps of different CTAs can be compared.  Per synchronisation of the
                # textbook loop: how far apart the CTAs arrive, and how long after the LAST arrival the first, the
                # average and the last CTA leave (nanoseconds, means over the iterations).
                rec["trace_unit"] = "ns (%globaltimer)"
                g = (t[:, :, :8] - t[:, :, :8].min()).astype(np.float64)      # int64 first: 1.7e18 ns does not fit a double's 53 bits
                sk = {}
                for a, b_, nm in ((1, 2, "sync 1"), (3, 4, "sync 2"), (6, 7, "sync 3")):
                    last_in = g[:, :, a].max(axis=0)
                    sk[nm] = {"arrival_spread": float((last_in - g[:, :, a].min(axis=0)).mean()),
                              "last_arrival_to_first_release": float((g[:, :, b_].min(axis=0) - last_in).mean()),
                              "last_arrival_to_mean_release": float((g[:, :, b_].mean(axis=0) - last_in).mean()),
                              "last_arrival_to_last_release": float((g[:, :, b_].max(axis=0) - last_in).mean())}
                rec["sync_skew_ns"] = sk
        print(json.dumps(rec))
        Ap.close()
        return

    # ------------------------------------------------------------ the metric's workload (config 2)
    p = cg_inputs.make_config(WORKLOAD_CFG)
    A = bind(p)
    A.set_option("loop", args.loop)
    A.set_option("spmv", args.spmv)
    if args.ctas_per_sm:
        A.set_option("ctas_per_sm", args.ctas_per_sm)
    b = torch.from_numpy(p.b).to(dev)
    x = torch.zeros(p.n, dtype=torch.float64, device=dev)
    hist = torch.zeros(p.maxit + 1, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream().cuda_stream
    bytes_it = cg_inputs.algorithmic_bytes_per_iteration(p.n, p.nnz)
    flops_it = cg_inputs.flops_per_iteration(p.n, p.nnz)
    prologue_bytes = 12 * p.nnz + 4 * (p.n + 1) + 16 * p.n + 40 * p.n     # a0: one SpMV + r, p init

    def one_solve():
        x.zero_()
        return cg.cg_solve(A.h, b.data_ptr(), x.data_ptr(), p.rtol, p.maxit, hist.data_ptr(), stream)

    for _ in range(args.warmup):
        flush_l2()
        one_solve()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)
    barrier()
    t_wall0 = time.time()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    iters_total, launches = 0, 0
    for s in range(args.steps):
        flush_l2()                      # outside the timed pair
        x.zero_()
        ev[s][0].record()
        st, it, res = cg.cg_solve(A.h, b.data_ptr(), x.data_ptr(), p.rtol, p.maxit, hist.data_ptr(), stream)
        ev[s][1].record()
        iters_total += it
        launches += A.info("launches")
        assert st == 0, f"solve did not converge: status {st}"
    barrier()
    t_wall1 = time.time()
    ms = [a.elapsed_time(b_) for a, b_ in ev]
    value, iters_all, t_dev = whole_job_value(dist, "cuda", iters_total, sum(ms) / 1e3)
    clocks = sampler.stop(t_wall0, t_wall1)
    it_per_solve = iters_total / args.steps
    kernel_ms = float(np.mean(ms))
    achieved = (bytes_it * it_per_solve + prologue_bytes) / (kernel_ms * 1e-3) / 1e9
    # sanity: the solve we just timed is the right answer (residual check through the C ABI)
    r_true = b - A.spmv(x)
    relres = float(torch.linalg.norm(r_true) / torch.linalg.norm(b))
    assert relres <= 2 * p.rtol, relres

    # ------------------------------------------------------------ e2e: host buffers through cg_solve_host
    hb = torch.from_numpy(p.b).pin_memory()
    hx = torch.zeros(p.n, dtype=torch.float64).pin_memory()
    hh = torch.zeros(p.maxit + 1, dtype=torch.float64).pin_memory()
    for _ in range(2):
        hx.zero_()
        A.solve_host(hb, hx, p.rtol, p.maxit, hh)
    barrier()
    e2e_it, t0 = 0, time.perf_counter()
    for s in range(args.steps):
        hx.zero_()
        st, it, res = A.solve_host(hb, hx, p.rtol, p.maxit, hh)
        e2e_it += it
    torch.cuda.synchronize()
    t_e2e = max_over_ranks(time.perf_counter() - t0)
    e2e_value = sum_over_ranks(e2e_it) / t_e2e
    h2d = 2 * 8 * p.n
    d2h = 8 * p.n + 8 * (e2e_it // args.steps + 1) + 192

    # measured read rooflines on this box (cg_probe_read_bandwidth): 40 MB sweeps stay in the L2,
    # 2 GiB sweeps come from HBM
    l2_gbs = A.probe_read_bandwidth(40 << 20, reps=50)
    hbm_read_gbs = A.probe_read_bandwidth(2 << 30, reps=5)
    sync_probe = {name: A.probe_grid_sync(kind, 3000) for kind, name in
                  ((0, "counter_barrier"), (1, "relaxed_allreduce_x2_plus_counter_barrier_mean"), (2, "fenced_allreduce"))}
    t_iter = t_dev / iters_total if world == 1 else None
    launch2 = describe(A)
    kernel2 = kernel_name(A)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_dev / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {
            "workload": workload_string(p),
            "iterations_per_solve": it_per_solve,
            "l2": "flushed (512 MiB write) between steps, outside the timed event pairs; inside a solve the "
                  "matrix stays on chip by design (shared memory when it fits, else the L2)",
            **launch2,
            "parallelism": "replicas only (north_star: one GPU, no sharding, no collectives)",
        },
        "us_per_iteration": t_dev / iters_total * 1e6 if world == 1 else None,
        "effective_gbs": bytes_it * iters_all / t_dev / 1e9,
        "cg_gflops": flops_it * iters_all / t_dev / 1e9,
        "relres_check": relres,
        "clocks": clocks,
        "gpu_launches": launches,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "api": "cg_solve_host (pinned host b, x0 in; x, hist out); matrix upload and cg_create are "
                       "setup, as in PAPER.md:48"},
        "roofline": {
            "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            **traffic_entry(WORKLOAD_CFG, kernel2, it_per_solve),
            "kernel": f"{kernel2} (one launch = one solve)",
            "bytes_per_launch": bytes_it * it_per_solve + prologue_bytes,
            "peak_source": peak_src,
            "note": "the 53.5 MB working set never leaves the chip inside a solve (matrix slice pinned in shared "
                    "memory, vectors in registers, gathers from the L2): the iteration is bound by grid-synchronisation "
                    "latency and the SM's load/store pipe, the HBM fraction is reported as north_star asks; "
                    "see north_star_160 for the HBM-bound case",
        },
        "roofline_l2": {"bound": "l2", "achieved": bytes_it / t_iter / 1e9 if t_iter else None, "peak": l2_gbs,
                        "unit": "GB/s", "frac": (bytes_it / t_iter / 1e9 / l2_gbs) if t_iter else None,
                        "peak_source": "measured here: cg_probe_read_bandwidth over a 40 MiB buffer (L2-resident), 50 sweeps",
                        "hbm_read_gbs_measured_here": hbm_read_gbs,
                        "us_per_iteration": t_iter * 1e6 if t_iter else None,
                        "us_at_l2_peak": bytes_it / l2_gbs / 1e3, "us_at_hbm_peak": bytes_it / peak / 1e3},
        "grid_sync_probe_cycles": {**sync_probe, "what": "cg_probe_grid_sync: mean cycles per synchronisation, 148 CTAs, "
                                   "back to back with nothing in between (the floor; inside a solve they also absorb the CTAs' skew)"},
        "paper_context": {"source": "PAPER.md:52-57 Table I (Tesla T10 / Core 2 Duo, the paper's own FEM matrix)",
                          "opencl_1gpu_iters_per_s": 116 / 0.659, "matlab_pcg_iters_per_s": 117 / 3.17,
                          "opencl_4gpu_iters_per_s": 116 / 0.380, "opencl_1gpu_gflops": 1.45, "matlab_gflops": 0.303},
    }
    A.close()
    del A

    # ------------------------------------------------------------ every config, fixed work
    # rtol = 0, maxit = K (2000 for configs 0-3, 200 for config 4): throughput that does not depend on
    # where convergence falls; plus the SpMV alone (cg_spmv), the to-convergence solve of configs 0-3,
    # and the oracle on the same fixed work (K = 200 / 20) on one host core.
    if rank == 0 and world == 1 and not args.no_per_config:
        per = {}
        for cfg in (0, 1, 2, 3, 4):
            if cfg == 4 and args.no_160:
                continue
            try:
                per[f"config{cfg}"] = per_config_leg(cg, torch, dev, cfg, p if cfg == WORKLOAD_CFG else None, args,
                                                     peak, l2_gbs, flush_l2, not args.no_cpu and world == 1)
            except Exception as e:  # the main line must still print
                per[f"config{cfg}"] = {"error": repr(e)}
        line["per_config"] = per
        c4 = per.get("config4")
        if c4 and "error" not in c4:
            line["north_star_160"] = {
                "workload": c4["workload"],
                "iterations_per_s": c4["iterations_per_s"], "us_per_iteration": c4["us_per_iteration"]["median"],
                "roofline": {**c4["roofline"], "target_frac": 0.70},
                "cg_gflops": c4["cg_gflops"], "launch": c4["launch"],
            }

    # ------------------------------------------------------------ the oracle timed beside it
    if not args.no_cpu and rank == 0 and world == 1:
        v, solves, its, dt = time_oracle(p, seconds_budget=8.0)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{solves} full solves of config{WORKLOAD_CFG} ({its} iterations, {dt:.1f} s)"}
        try:        # the same loops with OpenMP on the host's cores, beside the oracle
            line["cpu_allcores"] = time_oracle_omp(p, seconds_budget=4.0)
        except Exception as e:
            line["cpu_allcores"] = {"error": repr(e)}
    elif rank == 0:
        line["cpu_baseline"] = None

    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
