"""Throughput sweep of the swept and per-step variants over problem x N x tile width (BASELINE.json configs 2-5).

    python -m paper_1705_03162_b200.sweep [--problems heat,ks,euler,ks3] [--logn 11,14,17,20] [--widths 32,...,1024]
                                          [--dtype f64|f32] [--steps K] [--csv out.csv]
    python -m paper_1705_03162_b200.sweep --probes [--csv out.csv]     (roofline denominators and the sweep model)
    python -m paper_1705_03162_b200.sweep --flow-profile [--logn 20,24] [--csv out.csv]
                                          (where the warps of the FLOW flavour spend their cycles; heat FP64)

For every (problem, N) it times the per-step variant (best of 128 / 256 threads per block) and, for every tile
width n, every admissible swept flavour (FLOW, CHAR with 32/16/8 lanes per tile, TIER, CLUSTER), and prints one CSV row per
(problem, N, n) with the best flavour: point-timestep updates per second, speed-up over per-step, and the fraction
of the bound that applies: FP64/FP32 ALU pipe for swept, L2/HBM bytes for per-step.  Timing: CUDA
events around `swept_run`, best of `--reps`, state resident on the device (the paper's figures include allocation
and transfers, PAPER.md:236 — bench.py's `e2e` is the inclusive number).  The last column is the fraction of the
dependent-chain latency bound, which is what governs small N: a sub-timestep cannot finish before the FP64
operations on its critical path have (heat 2: DADD -> DFMA; KS 6 per stage), whatever the parallelism, so
time >= sub-timesteps x depth x (FP64 dependent-issue latency, measured by `swept_probe_chain`).
This is the measurement tool behind profiles/*_sweep_*.csv — argument marshalling and timing only, no library code:
all arithmetic runs in the library's kernels.
"""
from __future__ import annotations

import argparse
import os
import sys
import threading

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import paper_1705_03162_b200 as sw  # noqa: E402

FLAVOR_NAME = {sw.FLAVOR_TIER: "tier", sw.FLAVOR_CHAR: "char", sw.FLAVOR_FLOW: "flow", sw.FLAVOR_CLUSTER: "cluster"}
# FP64-pipe instructions per point and timestep of the canonical expression trees.  Euler: counted
# from the SASS of per_step_lane_kernel (profiles/r2_sass.md): 194 DADD/DMUL/DFMA/DSETP + 14 MUFU seeds per cell and
# stage with every pressure and interface flux computed once, two stages.  KS3: 11 + 13 + 13 for the three stages.
FP64_INSTR = {sw.HEAT: 3, sw.KS: 22, sw.EULER: 416, sw.KS3: 37}
# per-step algorithmic traffic per point and timestep, FP64: heat one launch; KS both stages fused in
# one launch; Euler and KS3 one launch per stage, the later stages also read u^n
BYTES_PER_STEP = {sw.HEAT: 16, sw.KS: 16, sw.EULER: 120, sw.KS3: 64}
# FP64 operations on the critical path of one sub-timestep (dependent chain), and sub-timesteps per timestep
CHAIN_DEPTH = {sw.HEAT: 2, sw.KS: 6, sw.KS3: 7}
SIGMA = {sw.HEAT: 1, sw.KS: 2, sw.EULER: 2, sw.KS3: 3}


def probes(emit):
    """Roofline denominators measured by the library's probes, and the issue-rate table of the characteristic sweep
    (DESIGN.md §5.6, §7)."""
    import torch
    props = torch.cuda.get_device_properties(0)
    emit(f"# device: {props.name}, {props.multi_processor_count} SMs, max SM clock {props.clock_rate / 1e3:.0f} MHz")
    # SM clock and throttle reasons sampled WHILE the FP64 probe runs (NVML, from a thread), so that "of nominal" can be
    # read against the clock actually held
    clocks, reasons, stop = [], set(), threading.Event()

    def poll():
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(torch.cuda.current_device())
            while not stop.is_set():
                clocks.append(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                reasons.add(int(pynvml.nvmlDeviceGetCurrentClocksEventReasons(h)))
                stop.wait(0.002)
        except Exception:
            pass

    thr = threading.Thread(target=poll, daemon=True)
    thr.start()
    fp64 = max(sw.swept_probe_fp64() for _ in range(3))
    stop.set()
    thr.join(timeout=5)
    emit(f"probe,fp64_pipe_lane_instr_per_s,{fp64:.4e},TFLOP/s (FMA=2) {2 * fp64 / 1e12:.2f},of nominal "
         f"{fp64 / (props.multi_processor_count * 64 * props.clock_rate * 1e3):.3f}")
    if clocks:
        med = sorted(clocks)[len(clocks) // 2]
        emit(f"probe,sm_clock_mhz_during_fp64_probe,{med},min {min(clocks)} max {max(clocks)} over {len(clocks)} samples,"
             f"clock event reason masks {sorted(reasons)} (0 = none; 1 = gpu idle; 4 = sw power cap),"
             f"of the pipe at the held clock {fp64 / (props.multi_processor_count * 64 * med * 1e6):.3f}")
    emit(f"probe,launch_us,{sw.swept_probe_launch(2000):.3f}")
    pair = sw.swept_probe_chain()
    emit(f"probe,dadd_dfma_pair_cycles,{pair:.2f},ns at max clock {pair / (props.clock_rate / 1e6):.2f}")
    t = sw.swept_probe_tier()
    emit(f"probe,register_tier_chain_cycles,{t[2]:.1f},shuffle->shuffle {t[0]:.1f},two 64-bit shuffles->DADD->DFMA {t[1]:.1f},"
         f"DFMA->select {t[3]:.1f},[2] = one heat tier of the CLUSTER flavour (one point per lane) with nothing else in the way")
    bps, bpc = sw.swept_probe_smem()
    emit(f"probe,smem_read_bytes_per_s,{bps:.4e},bytes/clk/SM {bpc:.1f},of nominal 128 {bpc / 128:.3f}")
    emit("sweep_probe,problem,lines_per_lane,warps_per_scheduler,cycles_per_superstep,fp64_pipe_busy")
    for problem, name in ((sw.HEAT, "heat"), (sw.KS, "ks")):
        for B in (8, 16, 32):
            for wps in (1, 2, 3, 4, 6, 8):
                try:
                    cyc, busy = sw.swept_probe_sweep(problem, B, wps)
                except sw.SweptError:
                    continue
                emit(f"sweep_probe,{name},{B},{wps},{cyc:.1f},{busy:.3f}")


def flow_profile(emit, logns, widths):
    """Per-part cycle shares of the persistent FLOW launch (instrumented kernel, `swept_flow_profile`), next to the
    throughput of the plain kernel in the same configuration."""
    import torch
    import swept_inputs as si
    emit("N,tile_width,group,plain_updates_per_s,instrumented_updates_per_s,tiles,cycles_per_tile,ticket,wait_parents,"
         "stage,sweep,publish")
    for logn in logns:
        N = 1 << logn
        w = si.config(2, N=N, nsteps=10000)
        st = sw.Swept.from_workload(w)
        u0_dev = torch.from_numpy(np.ascontiguousarray(w.u0)).cuda()
        for n in widths:
            for grp in (2, 3, 4, 6, 16 + 2, 16 + 3, 16 + 4, 16 + 6):  # resident CTAs per SM; +16 = TMA staging
                try:
                    plain = _time(torch, st, u0_dev, w.nsteps, n, sw.SWEPT, sw.FLAVOR_FLOW, grp, 2)
                    sw.swept_flow_profile(st._h, True)
                    inst = _time(torch, st, u0_dev, w.nsteps, n, sw.SWEPT, sw.FLAVOR_FLOW, grp, 1)
                    c = sw.swept_flow_profile(st._h, False)
                except sw.SweptError:
                    sw.swept_flow_profile(st._h, False)
                    continue
                tot = sum(c[k] for k in ("ticket", "wait_parents", "stage", "sweep", "publish")) or 1
                emit(f"{N},{n},{grp},{N * w.nsteps / (plain * 1e-3):.4e},{N * w.nsteps / (inst * 1e-3):.4e},{c['tiles']},"
                     f"{tot / max(c['tiles'], 1):.0f}," + ",".join(f"{c[k] / tot:.4f}" for k in
                                                                   ("ticket", "wait_parents", "stage", "sweep", "publish")))
        st.close()


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
                    help="paper = insulated heat ends (B.5) / Dirichlet Euler tube (PAPER.md:377): every flavour that applies "
                         "walls (heat: TIER, hybrid CHAR, FLOW, CLUSTER; Euler: TIER)")
    ap.add_argument("--csv", default="")
    ap.add_argument("--probes", action="store_true", help="print the probe measurements instead of a sweep")
    ap.add_argument("--flow-profile", action="store_true", help="cycle shares of the FLOW kernel's task parts")
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

    if args.probes or args.flow_profile:
        if args.probes:
            probes(emit)
        else:
            flow_profile(emit, [int(x) for x in args.logn.split(",")],
                         [int(x) for x in args.widths.split(",") if int(x) in (256, 512, 1024)])
        if out:
            out.close()
        return 0
    # dependent-issue latency of one FP64 operation (half a DADD -> DFMA pair), seconds
    fp64_latency_s = sw.swept_probe_chain() / 2 / (sm_mhz * 1e6)
    if args.bc == "paper":
        emit("# boundary conditions: the paper's own (insulated heat ends, Dirichlet Euler tube)")
    emit("problem,dtype,N,nsteps,variant,tile_width,flavor,group,ms,updates_per_s,speedup_vs_per_step,bound,frac_of_bound,"
         "frac_of_latency_bound")
    for pname in args.problems.split(","):
        problem = {"heat": si.HEAT, "ks": si.KS, "euler": si.EULER, "ks3": si.KS3}[pname]
        if problem != si.HEAT and args.dtype == "f32":
            continue
        for logn in [int(x) for x in args.logn.split(",")]:
            N = 1 << logn
            cfg = {si.HEAT: 2, si.KS: 3, si.EULER: 4, si.KS3: 3}[problem]
            w = si.config(cfg, N=N) if problem != si.EULER else si.config(4, N=N, rk2=si.RK2_HEUN)
            if problem == si.KS3:
                w = si.ks3_cos(N, si.BASE_SEED + 3, w.nsteps)
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

            def lat(ms):  # fraction of the dependent-chain latency bound (1 = nothing but the critical path)
                if problem not in CHAIN_DEPTH:
                    return ""
                return f"{nsteps * SIGMA[problem] * CHAIN_DEPTH[problem] * fp64_latency_s / (ms * 1e-3):.4f}"

            emit(f"{pname},{args.dtype},{N},{nsteps},per_step,{ps_thr},,,{ps_ms:.4f},{ups:.4e},1.0,"
                 f"bytes(L2/HBM) {gbs:.0f} GB/s,,{lat(ps_ms)}")
            for n in [int(x) for x in args.widths.split(",")]:
                if N % n:
                    continue
                best = None
                cands = [(sw.FLAVOR_FLOW, 0), (sw.FLAVOR_FLOW, 3), (sw.FLAVOR_CHAR, 32), (sw.FLAVOR_CHAR, 16),
                         (sw.FLAVOR_CHAR, 8), (sw.FLAVOR_TIER, 0),   # FLOW group 0 = defaults (TMA staging); 3 = 16-byte copies, 3 CTAs/SM
                         (sw.FLAVOR_CLUSTER, 0), (sw.FLAVOR_CLUSTER, 8), (sw.FLAVOR_CLUSTER, 16)]  # group = warps per CTA
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
                     f"{ps_ms / ms:.3f},alu,{frac:.3f},{lat(ms)}")
            st.close()
    if out:
        out.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
