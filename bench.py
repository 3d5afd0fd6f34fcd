#!/usr/bin/env python
"""bench.py — headline benchmark of the swept hot path on B200 (contract: see DESIGN.md §8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Workload (BASELINE.json `metric`: "point-timestep updates/sec (swept vs per-step, FP64, N=2^20)", quoted on
configs[1]): 1-D heat, FTCS, FP64, periodic, N = 2^20, r = 0.25, 10 000 timesteps, seeded 16-mode sine data.
One bench "step" = one pass of the whole hot path over that batch = one `swept_run(state, 10000, n, SWEPT)`
(UpTriangle, SplitDiamond/WholeDiamond ..., DownTriangle, per-step remainder).

`value`   : N * nsteps * K / (device time of K steps), state resident in HBM, L2 flushed between steps.
`e2e`     : the same metric through the C ABI with HOST buffers: swept_write (H2D from pinned memory) +
            swept_run + swept_read (D2H) inside the timed region, every step.
`roofline`: the dominant kernel is the persistent FLOW launch (or the Split/WholeDiamond launches of the CHAR
            flavour); it is bound by the FP64 ALU pipe ("alu").  achieved = FP64-pipe lane-instructions per
            second = 3 per update (DADD, DMUL, DFMA) x updates per launch / measured duration;
            peak = 148 SMs x 64 FP64 lanes/clk x SM clock: `frac` is the useful share of the pipe's
            issue slots.  The live DFMA-chain probe is reported beside the nominal peak, and the true flop rate
            (4 flops per update: one add, one multiply, one fused multiply-add) separately.
`cpu_baseline`: the oracle (oracle/, plain per-step C++) timed on this host's cores on a bounded sample.

N > 1 (torchrun): the path does not shard (single GPU) — "replicas only": every rank runs the
same workload on its own GPU, no data-path collective; value = total updates / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import swept_inputs as si  # noqa: E402

N_HEADLINE = 1 << 20
NSTEPS_HEADLINE = 10000
METRIC = "point-timestep updates/sec (swept, heat FTCS FP64, N=2^20, 10000 steps)"
UNIT = "updates/s"
FP64_LANES_PER_CLK_PER_SM = 64  # B200: 40 TFLOP/s FP64 class part = 148 SM x 64 FMA lanes x 2 x ~2 GHz


# ----------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (pynvml, else nvidia-smi)."""

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nvml = None

    _BITS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
             0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}

    def _poll(self):
        nv = self._nvml
        while not self._stop.is_set():
            try:
                if nv is not None:
                    self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                    for bit, name in self._BITS.items():
                        if mask & bit:
                            self.reasons.add(name)
                else:
                    import subprocess
                    out = subprocess.run(
                        ["nvidia-smi", f"--id={self.index}", "--format=csv,noheader,nounits",
                         "--query-gpu=clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
                         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
                         "clocks_event_reasons.sw_power_cap"], capture_output=True, text=True, timeout=5).stdout
                    f = [x.strip() for x in out.strip().split(",")]
                    self.samples.append(int(f[0]))
                    self.max_mhz = int(f[1])
                    for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown",
                                        "sw_power_cap"), f[2:]):
                        if v.lower().startswith("active"):
                            self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.01)

    def __enter__(self):
        self._thr = threading.Thread(target=self._poll, daemon=True)
        self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._thr.join(timeout=5)

    def summary(self):
        med = statistics.median(self.samples) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# ----------------------------------------------------------------------------------------------------
def max_over_ranks(ms: float, dist, device) -> float:
    """Replicas only: the job's time is the slowest rank's device time.  `dist` is
    torch.distributed (initialised) or None for a single process."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_value(updates_per_step: int, steps: int, world: int, max_ms: float) -> float:
    """Whole-job throughput: every rank advanced `updates_per_step * steps` point-timesteps."""
    return world * updates_per_step * steps / (max_ms * 1e-3)


# ----------------------------------------------------------------------------------------------------
def oracle_sample(w, budget_s: float = 12.0):
    """Time the oracle, as it stands, on a bounded sample of workload `w` (same N, fewer steps)."""
    import oracle
    probe_steps = 4
    t0 = time.perf_counter()
    oracle.run_workload(w, nsteps=probe_steps)
    t1 = time.perf_counter() - t0
    steps = int(max(8, min(w.nsteps, budget_s / max(t1 / probe_steps, 1e-9))))
    t0 = time.perf_counter()
    oracle.run_workload(w, nsteps=steps)
    dt = time.perf_counter() - t0
    return {"value": w.N * steps / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{w.name}: N={w.N}, first {steps} of {w.nsteps} timesteps, {dt:.2f} s wall"}, steps, dt


def run_reference(args):
    """--impl reference: for this tier the reference arm is the CPU oracle (bounded sample per step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    w = si.config(2, N=N_HEADLINE)
    # size one step to ~2 s of CPU work
    t0 = time.perf_counter()
    oracle.run_workload(w, nsteps=4)
    per = (time.perf_counter() - t0) / 4
    steps_per = int(max(4, min(w.nsteps, 2.0 / max(per, 1e-9))))
    for _ in range(args.warmup):
        oracle.run_workload(w, nsteps=steps_per)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.run_workload(w, nsteps=steps_per)
    dt = time.perf_counter() - t0
    value = w.N * steps_per * args.steps / dt
    sample = f"{w.name}: N={w.N}, {steps_per} of {w.nsteps} timesteps per bench step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[1]: heat FTCS FP64 N=2^20 r=0.25 (bounded sample)",
                       "N": w.N, "nsteps_per_step": steps_per},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------------
def time_runs(torch, sw, state, w, nsteps, tile, variant, flavor, group, reps, flush, warm=1):
    """Median / best device time (ms) of `reps` runs of nsteps, each from the same initial data."""
    u0_dev = torch.from_numpy(np.ascontiguousarray(w.u0)).cuda()
    lib = sw.load()
    ms = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for r in range(warm + reps):
        lib.swept_write_device(state._h, u0_dev.data_ptr())
        if flush is not None:
            flush.add_(1.0)
        e0.record()
        state.run(nsteps, tile, variant, flavor, group)
        e1.record()
        e1.synchronize()
        if r >= warm:
            ms.append(e0.elapsed_time(e1))
    return ms


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-detail", action="store_true", help="skip the per-problem detail table")
    ap.add_argument("--tile", type=int, default=0, help="force the swept tile width (0 = autotune)")
    ap.add_argument("--flavor", type=int, default=0)
    ap.add_argument("--group", type=int, default=0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_1705_03162_b200 as sw

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the swept library has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    w = si.config(2, N=N_HEADLINE)  # heat FP64, N = 2^20, 10 000 steps, 16 sine modes
    nsteps = w.nsteps
    state = sw.Swept.from_workload(w)
    lib = sw.load()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda").view(torch.float32)  # > 126 MB L2

    # ---- tile width: autotune (excluded from timing, as SURVEY.md §8(d) says) or forced
    if args.tile:
        tile, flavor, group = args.tile, args.flavor, args.group
    else:
        tile = state.autotune(sw.SWEPT)
        _, flavor, group = state.tuned(sw.SWEPT)

    u0_dev = torch.from_numpy(np.ascontiguousarray(w.u0)).cuda()
    e_pairs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
               for _ in range(args.steps)]

    def one_step(ev=None):
        lib.swept_write_device(state._h, u0_dev.data_ptr())
        flush.add_(1.0)  # L2 flush between timed iterations (untimed)
        if ev:
            ev[0].record()
        state.run(nsteps, tile, sw.SWEPT, flavor, group)
        if ev:
            ev[1].record()

    for _ in range(args.warmup):
        one_step()
    state.phase_times()
    state.set_phase_timing(True)  # CUDA-event pair around every swept launch, on the library's stream
    barrier()
    with ClockSampler(local) as clk:
        t_wall0 = time.perf_counter()
        for k in range(args.steps):
            one_step(e_pairs[k])
        barrier()
        t_wall = time.perf_counter() - t_wall0
    step_ms = [a.elapsed_time(b) for a, b in e_pairs]
    total_ms = sum(step_ms)
    launches_per_step = state.last_launches
    phase = state.phase_times()  # per-kind device time of this rank's launches inside the timed region
    state.set_phase_timing(False)
    total_ms = max_over_ranks(total_ms, dist, "cuda")
    updates_per_step = w.N * nsteps
    value = replica_value(updates_per_step, args.steps, world, total_ms)

    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region
    host_in = torch.from_numpy(np.ascontiguousarray(w.u0)).pin_memory()
    host_out = torch.empty_like(host_in).pin_memory()
    import ctypes
    e2e_ms = []
    for r in range(2 + args.steps):
        flush.add_(1.0)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        lib.swept_write(state._h, ctypes.c_void_p(host_in.data_ptr()))
        state.run(nsteps, tile, sw.SWEPT, flavor, group)
        lib.swept_read(state._h, ctypes.c_void_p(host_out.data_ptr()))
        b.record()
        b.synchronize()
        if r >= 2:
            e2e_ms.append(a.elapsed_time(b))
    # what the end-to-end figure is bound by: the two 8 MiB copies over PCIe, measured here with the same pinned buffers
    copy_ms = {}
    dev_tmp = torch.empty_like(u0_dev)
    for name, dst, src in (("h2d", dev_tmp, host_in), ("d2h", host_out, dev_tmp)):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        dst.copy_(src, non_blocking=True)
        a.record()
        for _ in range(10):
            dst.copy_(src, non_blocking=True)
        b.record()
        b.synchronize()
        copy_ms[name] = a.elapsed_time(b) / 10
    e2e_total = sum(e2e_ms)
    e2e_total = max_over_ranks(e2e_total, dist, "cuda")
    e2e_value = replica_value(updates_per_step, args.steps, world, e2e_total)
    final_field = host_out.numpy().copy()

    if rank != 0:
        state.close()
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel family (Split/WholeDiamond)
    peaks, peak_src = read_peaks()
    clocks = clk.summary()
    sm_max = float(peaks.get("sm_max_mhz") or clocks["sm_max_mhz"] or 1965.0)
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    peak_tinstr = sms * FP64_LANES_PER_CLK_PER_SM * sm_max * 1e6 / 1e12  # FP64-pipe lane-instructions per second / 1e12
    probe = sw.swept_probe_fp64()
    plan = sw.swept_plan(nsteps * state.sigma, tile, state.h)
    m_top = tile // (2 * state.h)
    # dominant kernel = the Split/WholeDiamond launches of the top-level cycle: N * m updates per launch,
    # 3 FP64-pipe instructions per update (DADD, DMUL, DFMA) = 6 FMA-equivalent flops
    d_ms = phase["SplitDiamond"][0] + phase["WholeDiamond"][0]
    d_cnt = phase["SplitDiamond"][1] + phase["WholeDiamond"][1]
    n_diamonds_top = sum(1 for p in plan if p[0] in (1, 2) and p[4] == tile)
    n_diamonds_all = sum(1 for p in plan if p[0] in (1, 2))
    fp64_instr_per_update = 3
    flow_ms, flow_cnt = phase["FlowCycle"]
    kernel_name = "swept Split/WholeDiamond (heat FP64)"
    if flow_cnt:
        # FLOW flavour: the dominant kernel is the persistent launch that runs whole Up..Down cycles; the
        # sub-timesteps it covers = sum over the cycles of widths 256/512/1024 of (D+1) * m (swept_plan)
        t_flow = 0
        for p in plan:
            if p[4] in (256, 512, 1024) and p[0] in (1, 2, 3):   # each diamond row and the Down row close m tiers
                t_flow += p[4] // (2 * state.h)
        avg_launch_ms = flow_ms / flow_cnt
        upd_per_s = w.N * t_flow * args.steps / (flow_ms * 1e-3)
        kernel_name = "swept_flow_kernel: persistent launch running whole Up..Down cycles (heat FP64)"
        how = "CUDA events around every FLOW launch of the timed region (swept_phase_times)"
    elif d_cnt and n_diamonds_all == n_diamonds_top:
        avg_launch_ms = d_ms / d_cnt
        upd_per_s = w.N * m_top / (avg_launch_ms * 1e-3)
        how = "CUDA events around every Split/WholeDiamond launch of the timed region (swept_phase_times)"
    else:  # flavours without per-launch phases, or diamonds of several widths: whole-step figure
        avg_launch_ms = total_ms / args.steps
        upd_per_s = updates_per_step / (avg_launch_ms * 1e-3)
        how = "whole swept_run (all phases) timed with CUDA events"
    ach_tinstr = fp64_instr_per_update * upd_per_s / 1e12
    step_tinstr = fp64_instr_per_update * updates_per_step / (total_ms / args.steps * 1e-3) / 1e12
    units = (f"N x {t_flow} timesteps per FLOW launch (the cycles of widths 256-1024 of swept_plan)" if flow_cnt
             else f"N x m = N x {m_top} updates per diamond launch")
    roofline = {"bound": "alu", "achieved": ach_tinstr, "peak": peak_tinstr,
                "unit": "Tinstr/s (FP64-pipe lane-instructions; x2 = FMA-equivalent TFLOP/s)",
                "frac": ach_tinstr / peak_tinstr, "traffic": None,
                "kernel": kernel_name, "timed_by": how,
                "note": "FP64 pipe issue utilisation: 3 FP64-pipe instructions per update (DADD, DMUL, DFMA), "
                        f"{units}; peak = {sms} SM x 64 lanes x {sm_max:.0f} MHz (nominal unit count, max clock); "
                        "probe = live DFMA-chain measurement of the same quantity",
                "peak_probe": probe / 1e12,
                "frac_of_probe": ach_tinstr / (probe / 1e12) if probe else None,
                "true_tflops": 4 * upd_per_s / 1e12,
                "true_tflops_note": "4 floating-point operations per update (add, multiply, fused multiply-add); the "
                                    f"FMA peak 2 x {peak_tinstr:.1f} TFLOP/s is not reachable by this instruction mix",
                "avg_launch_ms": avg_launch_ms, "diamond_launches_timed": d_cnt,
                "whole_step": step_tinstr, "whole_step_frac": step_tinstr / peak_tinstr,
                "phase_ms_per_step": {k: v[0] / args.steps for k, v in phase.items()},
                "phase_launches_per_step": {k: v[1] / args.steps for k, v in phase.items()}}
    try:  # DRAM bytes per launch of the dominant kernel, from the committed ncu --set full capture
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            want = "swept_flow_kernel" if flow_cnt else "swept_char_kernel"
            for row in csv.DictReader(f):
                if row["kernel"].startswith(want):
                    roofline["traffic"] = int(row["dram_bytes_per_launch"])
                    roofline["traffic_source"] = row["source"]
                    break
    except Exception:
        pass

    # ---- per-step variant on the same workload (the "vs per-step" half of the metric)
    hbm = float(peaks["hbm_gbs"])
    detail = {}
    if not args.no_detail:
        ps_threads = state.autotune(sw.PER_STEP)
        ps_ms = time_runs(torch, sw, state, w, nsteps, ps_threads, sw.PER_STEP, 0, 0, reps=3, flush=flush)
        ps_value = updates_per_step / (min(ps_ms) * 1e-3)
        detail = {"per_step": {"value": ps_value, "ms": min(ps_ms), "threads": ps_threads,
                               "bytes_per_update": 16, "achieved_gbs": ps_value * 16 / 1e9,
                               "note": "N=2^20 FP64 working set (16 MiB) is L2-resident: launch/L2-bound, "
                                       "not HBM-bound (SURVEY.md §7 H7)"},
                  "swept_over_per_step": (updates_per_step / (statistics.median(step_ms) * 1e-3)) / ps_value,
                  "launch_us": sw.swept_probe_launch(2000)}
        try:  # launch-free per-step baseline (PS_RESIDENT): same sub-timesteps, one persistent launch
            rs_ms = time_runs(torch, sw, state, w, nsteps, 0, sw.PER_STEP, sw.PS_RESIDENT, 0, reps=3, flush=flush)
            detail["per_step_resident"] = {"value": updates_per_step / (min(rs_ms) * 1e-3), "ms": min(rs_ms),
                                           "us_per_substep": min(rs_ms) * 1e3 / (nsteps * state.sigma),
                                           "note": "field in registers, neighbour-only flags between CTAs "
                                                   "(DESIGN.md §5.7); bound by the L2 round trips of the edge exchange"}
            detail["swept_over_per_step_resident"] = (updates_per_step / (statistics.median(step_ms) * 1e-3)) \
                / detail["per_step_resident"]["value"]
        except sw.SweptError as e:
            detail["per_step_resident"] = {"unsupported": str(e)}
        detail["problems"] = problem_table(torch, sw, flush, hbm)

    cpu_base, _, _ = oracle_sample(w) if not args.no_detail else ({"value": None, "unit": UNIT, "cores": 0, "kind": "oracle", "sample": "skipped (--no-detail)"}, 0, 0)
    # sanity: the benchmarked field equals the oracle's on a prefix-sized rerun is covered by tests;
    # here just make sure the run produced finite numbers
    assert np.all(np.isfinite(final_field))

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[1]: 1-D heat FTCS FP64 periodic, N=2^20, r=0.25, "
                                   "10000 steps, seeded 16-mode sine data",
                       "N": w.N, "nsteps": nsteps, "variant": "swept", "tile_width": tile, "flavor": flavor,
                       "group": group, "l2": "flushed between timed steps (256 MiB write); the 8 MiB field is "
                                              "L2-resident within a step by nature of the workload",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "clocks": clocks, "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(w.u0.nbytes),
                                      "d2h_bytes_per_step": int(w.u0.nbytes),
                                      "ms_per_step": e2e_total / args.steps,
                                      "h2d_ms": copy_ms["h2d"], "d2h_ms": copy_ms["d2h"],
                                      "h2d_gbs": w.u0.nbytes / copy_ms["h2d"] / 1e6,
                                      "d2h_gbs": w.u0.nbytes / copy_ms["d2h"] / 1e6,
                                      "note": "device time of the step + the two pinned-memory copies over PCIe "
                                              "(measured beside it) + two host synchronisations"},
            "gpu_launches": int(launches_per_step * args.steps), "roofline": roofline,
            "cpu_baseline": cpu_base, "peaks_source": peak_src, "wall_s_timed_region": t_wall,
            "detail": detail}
    print(json.dumps(line))
    state.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


def problem_table(torch, sw, flush, hbm):
    """Swept vs per-step for the three PDEs at N = 2^20 (configs 2-4 shapes, shortened runs), config 1 (N = 2048) and
    the HBM-bound per-step regime at N = 2^26 (config 5's largest size)."""
    rows = []
    cases = [("heat", si.config(2, N=1 << 20, nsteps=10000)), ("ks", si.config(3, N=1 << 20, nsteps=4000)),
             ("euler_heun", si.config(4, N=1 << 20, nsteps=1000))]
    for name, w in cases:
        st = sw.Swept.from_workload(w)
        tile = st.autotune(sw.SWEPT)
        _, fl, grp = st.tuned(sw.SWEPT)
        thr = st.autotune(sw.PER_STEP)
        sx = min(time_runs(torch, sw, st, w, w.nsteps, tile, sw.SWEPT, fl, grp, reps=2, flush=flush))
        ps = min(time_runs(torch, sw, st, w, w.nsteps, thr, sw.PER_STEP, 0, 0, reps=2, flush=flush))
        rows.append({"problem": name, "N": w.N, "nsteps": w.nsteps, "tile_width": tile, "flavor": fl, "group": grp,
                     "swept_updates_per_s": w.N * w.nsteps / (sx * 1e-3),
                     "per_step_updates_per_s": w.N * w.nsteps / (ps * 1e-3), "speedup": ps / sx})
        st.close()
    # BASELINE.json configs[0] (heat N = 2048, 20 000 steps): the latency-bound end, library defaults (CLUSTER flavour)
    w = si.config(1)
    st = sw.Swept.from_workload(w)
    sx = min(time_runs(torch, sw, st, w, w.nsteps, 0, sw.SWEPT, sw.FLAVOR_AUTO, 0, reps=2, flush=flush))
    ps = min(time_runs(torch, sw, st, w, w.nsteps, 0, sw.PER_STEP, 0, 0, reps=2, flush=flush))
    rows.append({"problem": "heat_config1", "N": w.N, "nsteps": w.nsteps, "tile_width": 0, "flavor": sw.FLAVOR_AUTO,
                 "note": "untuned library default: one thread-block cluster, a warp per tile in registers (DESIGN.md 5.10)",
                 "swept_updates_per_s": w.N * w.nsteps / (sx * 1e-3), "swept_ns_per_timestep": sx * 1e6 / w.nsteps,
                 "per_step_updates_per_s": w.N * w.nsteps / (ps * 1e-3), "speedup": ps / sx})
    st.close()
    # HBM-bound per-step: N = 2^26 heat FP64 (512 MiB per array > L2)
    w = si.heat_sines(1 << 26, 16, si.BASE_SEED + 5, 200)
    st = sw.Swept.from_workload(w)
    ps = min(time_runs(torch, sw, st, w, w.nsteps, 256, sw.PER_STEP, 0, 0, reps=2, flush=None))
    ups = w.N * w.nsteps / (ps * 1e-3)
    rows.append({"problem": "heat_per_step_hbm", "N": w.N, "nsteps": w.nsteps,
                 "per_step_updates_per_s": ups, "achieved_gbs": ups * 16 / 1e9, "hbm_peak_gbs": hbm,
                 "frac_hbm": ups * 16 / 1e9 / hbm})
    st.close()
    return rows


if __name__ == "__main__":
    sys.exit(main())
