"""Throughput sweep of the swept and per-step variants over problem x N x tile width (BASELINE.json configs 2-5).

    python -m paper_1705_03162_b200.sweep [--problems heat,ks,euler] [--logn 11,14,17,20] [--widths 32,...,1024]
                                          [--dtype f64|f32] [--steps K] [--csv out.csv]

For every (problem, N) it times the per-step variant (best of 128 / 256 threads per block) and, for every tile
width n, every admissible swept flavour (FLOW, CHAR with 32/16/8 lanes per tile, TIER), and prints one CSV row per
(problem, N, n) with the best flavour: point-timestep updates per second, speed-up over per-step, and the fraction
of the bound that applies: FP64/FP32 ALU pipe for swept, L2/HBM bytes for per-step.  Timing: CUDA
events around `swept_run`, best of `--reps`, state resident on the device (the paper's figures include allocation
and transfers, PAPER.md:236 — bench.py's `e2e` is the inclusive number).  Argument marshalling and timing only:
all arithmetic runs in the library's kernels.
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import paper_1705_03162_b200 as sw  # noqa: E402

FLAVOR_NAME = {sw.FLAVOR_TIER: "tier", sw.FLAVOR_CHAR: "char", sw.FLAVOR_FLOW: "flow"}
# FP64-pipe instructions per point and timestep of the canonical expression trees
FP64_INSTR = {sw.HEAT: 3, sw.KS: 22}
BYTES_PER_STEP = {sw.HEAT: 16, sw.KS: 16, sw.EULER: 120}  # per-step algorithmic traffic, FP64


def _time(torch, st, u0_dev, nsteps, n, variant, flavor, group, reps):
    lib = sw.load()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best = float("inf")
    for r in range(reps + 1):  # first run warms up (graph capture, attribute setting)
        lib.swept_write_device(st._h, u0_dev.data_ptr())
        e0.record()
        st.run(nsteps, n, variant, flavor, group)
        e1.record()
        e1.synchronize()
        if r:
            best = min(best, e0.elapsed_time(e1))
    return best


def main(argv=None):
    import torch
    import swept_inputs as si

    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--problems", default="heat,ks,euler")
    ap.add_argument("--logn", default="11,14,17,20")
    ap.add_argument("--widths", default="32,64,128,256,512,1024")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--steps", type=int, default=0, help="timesteps per run (0 = the config's own count)")
    ap.add_argument("--reps", type=int, default=2)
    ap.add_argument("--bc", default="periodic", choices=["periodic", "paper"],
                    help="paper = insulated heat ends (B.5) / Dirichlet Euler tube (PAPER.md:377); TIER flavour only")
    ap.add_argument("--csv", default="")
    args = ap.parse_args(argv)
    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device: the swept library has no CPU fallback")
    dtype = np.float64 if args.dtype == "f64" else np.float32
    props = torch.cuda.get_device_properties(0)
    sm_mhz = getattr(props, "clock_rate", 1965000) / 1e3  # max SM clock
    sms = props.multi_processor_count
    lanes = 64 if args.dtype == "f64" else 128
    alu_peak = sms * lanes * sm_mhz * 1e6  # pipe instructions (lanes) per second

    out = open(args.csv, "w") if args.csv else None

    def emit(line):
        print(line, flush=True)
        if out:
            out.write(line + "\n")
            out.flush()

    if args.bc == "paper":
        emit("# boundary conditions: the paper's own (insulated heat ends, Dirichlet Euler tube)")
    emit("problem,dtype,N,nsteps,variant,tile_width,flavor,group,ms,updates_per_s,speedup_vs_per_step,bound,frac_of_bound")
    for pname in args.problems.split(","):
        problem = {"heat": si.HEAT, "ks": si.KS, "euler": si.EULER}[pname]
        if problem != si.HEAT and args.dtype == "f32":
            continue
        for logn in [int(x) for x in args.logn.split(",")]:
            N = 1 << logn
            cfg = {si.HEAT: 2, si.KS: 3, si.EULER: 4}[problem]
            w = si.config(cfg, N=N) if problem != si.EULER else si.config(4, N=N, rk2=si.RK2_HEUN)
            if args.bc == "paper":
                if problem == si.KS:
                    continue
                w = si.heat_insulated(N, 16, si.BASE_SEED + 6, w.nsteps) if problem == si.HEAT else \
                    si.euler_sod(N, w.nsteps)
            nsteps = args.steps or w.nsteps
            st = sw.Swept.from_workload(w, dtype=dtype)
            u0_dev = torch.from_numpy(np.ascontiguousarray(w.u0, dtype=dtype)).cuda()
            ps_ms, ps_thr = min((_time(torch, st, u0_dev, nsteps, thr, sw.PER_STEP, 0, 0, args.reps), thr)
                                for thr in (128, 256))
            ups = N * nsteps / (ps_ms * 1e-3)
            gbs = ups * BYTES_PER_STEP[problem] * (1 if args.dtype == "f64" else 0.5) / 1e9
            emit(f"{pname},{args.dtype},{N},{nsteps},per_step,{ps_thr},,,{ps_ms:.4f},{ups:.4e},1.0,"
                 f"bytes(L2/HBM) {gbs:.0f} GB/s,")
            for n in [int(x) for x in args.widths.split(",")]:
                if N % n:
                    continue
                best = None
                cands = [(sw.FLAVOR_FLOW, 0), (sw.FLAVOR_CHAR, 32), (sw.FLAVOR_CHAR, 16), (sw.FLAVOR_CHAR, 8),
                         (sw.FLAVOR_TIER, 0)]
                for fl, grp in cands:
                    try:
                        ms = _time(torch, st, u0_dev, nsteps, n, sw.SWEPT, fl, grp, args.reps)
                    except sw.SweptError:
                        continue
                    if best is None or ms < best[0]:
                        best = (ms, fl, grp)
                if best is None:
                    continue
                ms, fl, grp = best
                ups = N * nsteps / (ms * 1e-3)
                frac = ups * FP64_INSTR[problem] / alu_peak if problem in FP64_INSTR else float("nan")
                emit(f"{pname},{args.dtype},{N},{nsteps},swept,{n},{FLAVOR_NAME[fl]},{grp},{ms:.4f},{ups:.4e},"
                     f"{ps_ms / ms:.3f},alu,{frac:.3f}")
            st.close()
    if out:
        out.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
