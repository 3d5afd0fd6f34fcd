"""Small runs of every kernel family, sized for compute-sanitizer:

    compute-sanitizer --tool memcheck|racecheck|synccheck|initcheck python tests/sanitizer_cases.py

The GPU pool this build ran on refuses compute-sanitizer ("closed on this pool and stays closed", recorded in
profiles/r2_sanitizer.md), so there the script only runs as it is: every case is compared bit for bit with the CPU
oracle, and `SWEPT_POISON=1` (the default here) makes the library fill every slab and scratch buffer with NaNs /
0xFF before use, so that a read of memory no kernel wrote shows up as a wrong result.  Not collected by pytest.
`--only NAME` runs the cases whose label contains NAME.
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

os.environ.setdefault("SWEPT_POISON", "1")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import paper_1705_03162_b200 as sw  # noqa: E402
import swept_inputs as si  # noqa: E402


def cases():
    heat = si.heat_sines(2048, 8, 31, 150)
    heat_flow = si.heat_sines(4096, 8, 32, 300)
    ks = si.ks_cos(2048, 33, 40)
    ks_flow = si.ks_cos(4096, 34, 80)
    ks3 = si.ks3_cos(1024, 35, 30)
    eul = si.euler_double_sod(512, 24)
    eul_mid = si.euler_double_sod(512, 24, rk2=si.RK2_MIDPOINT)
    wall = si.heat_insulated(2048, 6, 36, 150)
    tube = si.euler_sod(512, 24)
    T, C, F = sw.FLAVOR_TIER, sw.FLAVOR_CHAR, sw.FLAVOR_FLOW
    yield "heat per_step", heat, sw.PER_STEP, 0, 0, 0
    yield "heat per_step resident", heat, sw.PER_STEP, 0, sw.PS_RESIDENT, 0
    yield "heat TIER n=64 P=1", heat, sw.SWEPT, 64, T, 1
    yield "heat TIER n=256 P=2", heat, sw.SWEPT, 256, T, 2
    yield "heat TIER n=1024 P=4", heat, sw.SWEPT, 1024, T, 4
    yield "heat CHAR n=256 L=8", heat, sw.SWEPT, 256, C, 8
    yield "heat CHAR n=256 L=16", heat, sw.SWEPT, 256, C, 16
    yield "heat CHAR n=512 L=32", heat, sw.SWEPT, 512, C, 32
    yield "heat FLOW n=256", heat_flow, sw.SWEPT, 256, F, 0
    yield "heat FLOW n=512 TMA", heat_flow, sw.SWEPT, 512, F, 16
    yield "heat CLUSTER n=64", heat, sw.SWEPT, 64, sw.FLAVOR_CLUSTER, 0
    yield "heat CLUSTER n=256 (one CTA)", heat, sw.SWEPT, 256, sw.FLAVOR_CLUSTER, 8
    yield "heat CLUSTER n=32 (16 CTAs)", heat, sw.SWEPT, 32, sw.FLAVOR_CLUSTER, 4
    yield "heat CLUSTER n=64 one tile", si.heat_sines(64, 4, 38, 150), sw.SWEPT, 64, sw.FLAVOR_CLUSTER, 0
    yield "heat walls TIER n=256", wall, sw.SWEPT, 256, T, 1
    yield "heat walls hybrid CHAR n=256", wall, sw.SWEPT, 256, C, 32
    yield "heat walls FLOW n=256", si.heat_insulated(4096, 6, 37, 300), sw.SWEPT, 256, F, 0
    yield "heat walls CLUSTER n=128", wall, sw.SWEPT, 128, sw.FLAVOR_CLUSTER, 0
    yield "heat walls CLUSTER n=64 (source lanes)", wall, sw.SWEPT, 64, sw.FLAVOR_CLUSTER, 0
    yield "heat walls CLUSTER n=32 (source lanes)", wall, sw.SWEPT, 32, sw.FLAVOR_CLUSTER, 0
    yield "heat walls per_step", wall, sw.PER_STEP, 0, 0, 0
    yield "heat walls per_step resident", wall, sw.PER_STEP, 0, sw.PS_RESIDENT, 0
    yield "ks per_step (fused stages)", ks, sw.PER_STEP, 0, 0, 0
    yield "ks per_step resident", ks, sw.PER_STEP, 0, sw.PS_RESIDENT, 0
    yield "ks TIER n=128 P=1", ks, sw.SWEPT, 128, T, 1
    yield "ks CHAR n=256 L=16", ks, sw.SWEPT, 256, C, 16
    yield "ks CHAR n=256 L=32", ks, sw.SWEPT, 256, C, 32
    yield "ks FLOW n=256", ks_flow, sw.SWEPT, 256, F, 0
    yield "ks FLOW n=512 TMA", ks_flow, sw.SWEPT, 512, F, 16
    yield "ks CLUSTER n=128", ks, sw.SWEPT, 128, sw.FLAVOR_CLUSTER, 0
    yield "ks CLUSTER n=64 two warps per scheduler", ks, sw.SWEPT, 64, sw.FLAVOR_CLUSTER, 8
    yield "ks3 per_step", ks3, sw.PER_STEP, 0, 0, 0
    yield "ks3 TIER n=128 P=1", ks3, sw.SWEPT, 128, T, 1
    yield "ks3 TIER n=256 P=2", ks3, sw.SWEPT, 256, T, 2
    yield "ks3 CLUSTER n=128", ks3, sw.SWEPT, 128, sw.FLAVOR_CLUSTER, 0
    yield "euler per_step (Heun)", eul, sw.PER_STEP, 0, 0, 0
    yield "euler per_step resident", eul, sw.PER_STEP, 0, sw.PS_RESIDENT, 0
    yield "euler TIER n=128 P=1 (Heun)", eul, sw.SWEPT, 128, T, 1
    yield "euler TIER n=256 P=2 (midpoint)", eul_mid, sw.SWEPT, 256, T, 2
    yield "euler CHAR n=64 L=8", eul, sw.SWEPT, 64, C, 8
    yield "euler tube per_step", tube, sw.PER_STEP, 0, 0, 0
    yield "euler tube TIER n=128", tube, sw.SWEPT, 128, T, 1


def main() -> int:
    only = sys.argv[sys.argv.index("--only") + 1] if "--only" in sys.argv else ""
    bad = 0
    for label, w, variant, n, flavor, group in cases():
        if only and only not in label:
            continue
        t0 = time.perf_counter()
        ref = oracle.run_workload(w)
        s = sw.Swept.from_workload(w)
        try:
            s.run(w.nsteps, n, variant, flavor, group)
            got = s.read()
        finally:
            s.close()
        ok = bool(np.array_equal(got, ref))
        bad += not ok
        print(f"{'ok  ' if ok else 'FAIL'} {label:36s} N={w.N:5d} steps={w.nsteps:4d}  {time.perf_counter() - t0:6.1f} s",
              flush=True)
    print("cases failed:", bad, flush=True)
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
