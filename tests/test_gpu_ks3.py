"""GPU parity for row f3: a scheme with THREE sub-timesteps per timestep — the KS discretisation
(C.2) advanced by SSP-RK3 — for which the paper says the two-row decomposition "must be adjusted".
The library keeps a three-row inter-launch state (tier modulo 3) and lets diamonds start on any stage; the oracle
(`oracle_ks3_f64`, pinned in tests/test_oracle_ks3.py) is plain stage-by-stage stepping.  Same expression trees on both
sides, so the expected difference is zero; the gate is north_star's 1e-12.
"""
import numpy as np
import pytest

import oracle
import paper_1705_03162_b200 as sw
import swept_inputs as si

pytestmark = pytest.mark.gpu


def run(w, nsteps, variant, n=0, flavor=sw.FLAVOR_AUTO, group=0):
    s = sw.Swept.from_workload(w)
    try:
        s.run(nsteps, n, variant, flavor, group)
        return s.read(), s.last_launches
    finally:
        s.close()


def relerr(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


@pytest.mark.parametrize("N,nsteps", [(256, 0), (256, 1), (256, 7), (512, 64), (1024, 100), (96, 33), (4096, 400)])
def test_ks3_per_step_and_tier_match_oracle(N, nsteps):
    w = si.ks3_cos(N, 21, nsteps)
    ref = oracle.run_workload(w)
    ps, launches = run(w, nsteps, sw.PER_STEP)
    assert launches == 3 * nsteps, "one launch per sub-timestep"
    assert relerr(ps, ref) <= 1e-12 if nsteps else np.array_equal(ps, ref)
    assert np.array_equal(ps, ref), "same expression trees: expected 0 ulp"
    ran = 0
    for n in (32, 64, 128, 256, 512, 1024):
        for P in (0, 1, 2, 4):
            ok = N % n == 0 and (P == 0 or 8 <= n // P <= 1024)
            try:
                sx, _ = run(w, nsteps, sw.SWEPT, n, sw.FLAVOR_TIER, P)
            except sw.SweptError as e:
                assert not ok, f"library refused n={n} P={P}: {e}"
                continue
            assert ok, f"library ran the inadmissible n={n} P={P}"
            assert np.array_equal(sx, ps), f"swept TIER n={n} P={P} != per_step bitwise"
            ran += 1
    assert ran >= (4 if N % 32 == 0 else 0)


def test_ks3_default_flavour_and_launch_count():
    # 3 * 1000 sub-timesteps, n = 256: m = 64; 46 rows would fit after the Up row, the cycle takes 45 (a multiple of 3)
    N, nsteps, n = 8192, 1000, 256
    w = si.ks3_cos(N, 22, nsteps)
    ref = oracle.run_workload(w)
    sx, launches = run(w, nsteps, sw.SWEPT, n)
    assert np.array_equal(sx, ref)
    plan = sw.swept_plan(3 * nsteps, n, 2, 3)
    top = [p for p in plan if p[4] == n]
    assert len(top) == 46 and top[-1][2] + top[-1][3] == 45 * 64
    assert launches < 3 * nsteps / 20, "far fewer launches than one per sub-timestep (PAPER.md:83)"
    sx0, _ = run(w, nsteps, sw.SWEPT, 0)   # library default width and flavour
    assert np.array_equal(sx0, ref)


def test_ks3_unsupported_combinations_are_refused():
    w = si.ks3_cos(1024, 23, 10)
    for fl, grp in ((sw.FLAVOR_CHAR, 32), (sw.FLAVOR_FLOW, 0)):
        with pytest.raises(sw.SweptError):
            run(w, 10, sw.SWEPT, 256, fl, grp)
    with pytest.raises(sw.SweptError):
        run(w, 10, sw.PER_STEP, 0, sw.PS_RESIDENT)
    with pytest.raises(sw.SweptError):
        sw.Swept(sw.KS3, 1024, 0.5, 0.005, dtype=np.float32)


def test_ks3_config3_size_full_length_prefix():
    # config 3's largest size with the three-stage integrator: per-step vs oracle over a prefix, swept == per-step
    N, nsteps = 1 << 20, 300
    w = si.ks3_cos(N, 24, nsteps)
    ref = oracle.run_workload(w)
    ps, _ = run(w, nsteps, sw.PER_STEP)
    assert np.array_equal(ps, ref)
    for n in (256, 1024):
        sx, _ = run(w, nsteps, sw.SWEPT, n, sw.FLAVOR_TIER)
        assert np.array_equal(sx, ref), n


def test_ks3_autotune_picks_an_admissible_width():
    w = si.ks3_cos(1 << 16, 25, 200)
    s = sw.Swept.from_workload(w)
    try:
        n = s.autotune(sw.SWEPT)
        _, fl, grp = s.tuned(sw.SWEPT)
        assert fl == sw.FLAVOR_TIER and n in (32, 64, 128, 256, 512, 1024, 2048, 4096)
        s.run(200, 0, sw.SWEPT)
        assert np.array_equal(s.read(), oracle.run_workload(w))
    finally:
        s.close()


@pytest.mark.parametrize("N,nsteps", [(128, 16), (2048, 100), (4096, 257), (16384, 64)])
def test_ks3_cluster_flavour_matches_oracle(N, nsteps):
    # the three-row scheme in registers: one thread-block cluster, a warp per tile, rows of tiles chained through
    # distributed shared memory; diamonds start on any of the three stages (swept_cluster.cuh: swept_cluster3_kernel)
    w = si.ks3_cos(N, 26, nsteps)
    ref = oracle.run_workload(w)
    ran = 0
    for n in (64, 128, 256, 512):
        for wpc in (0, 4, 8, 16):
            K, P = N // n if N % n == 0 else 0, n // 32
            max_wpc = 8 if P >= 8 else 16
            ok = False
            if K and n <= 256:
                for cand in (1, 2, 4, 8, 16, 32):
                    if (cand != wpc) if wpc else (cand < 4 and K > cand):
                        continue
                    if cand > max_wpc or K % cand or K // cand > 16 or 2 * 3 * cand * n * 8 > 200 * 1024:
                        continue
                    ok = True
                    break
            try:
                got, launches = run(w, nsteps, sw.SWEPT, n, sw.FLAVOR_CLUSTER, wpc)
            except sw.SweptError as e:
                assert not ok, f"library refused n={n} wpc={wpc}: {e}"
                continue
            assert ok, f"library ran the inadmissible n={n} wpc={wpc}"
            assert np.array_equal(got, ref), (n, wpc)
            ran += 1
    assert ran >= 2
