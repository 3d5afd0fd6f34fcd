"""GPU parity (run with -m gpu on the B200): the CUDA path, called through the C ABI, against the CPU oracle
on the same seeded inputs, and swept against per-step bit for bit.

Tolerances (north_star): max relative error <= 1e-12 in FP64 and <= 1e-5 in FP32 after the full run, where
"relative" is ||gpu - oracle||_inf / ||oracle||_inf per component (reading X14) and the FP32 path is gated
against the FP32 instantiation of the oracle (reading X15).  Because both sides evaluate the same IEEE
expression trees the expected difference is exactly zero; the tests record that too.
"""
import numpy as np
import pytest

import oracle
import paper_1705_03162_b200 as sw
import swept_inputs as si

pytestmark = pytest.mark.gpu

TOL = {np.dtype(np.float64): 1e-12, np.dtype(np.float32): 1e-5}


def relerr(got, ref, C):
    got = got.reshape(C, -1).astype(np.float64)
    ref = ref.reshape(C, -1).astype(np.float64)
    return max(np.max(np.abs(g - r)) / max(np.max(np.abs(r)), 1e-300) for g, r in zip(got, ref))


def gpu_run(w, nsteps, variant, tile_width=0, flavor=sw.FLAVOR_AUTO, group=0, dtype=np.float64):
    s = sw.Swept.from_workload(w, dtype=dtype)
    try:
        s.run(nsteps, tile_width, variant, flavor, group)
        out = s.read()
        launches = s.last_launches
    finally:
        s.close()
    return out, launches


CHAR = tuple((sw.FLAVOR_CHAR, L) for L in (8, 16, 32))
FLOW = ((sw.FLAVOR_FLOW, 0), (sw.FLAVOR_FLOW, 16))   # heat / KS, n in {256, 512, 1024}; group 16 = TMA staging
TIER12 = ((sw.FLAVOR_TIER, 1), (sw.FLAVOR_TIER, 2))


def admissible(w, n, flavor, group, dtype=np.float64):
    """Which (tile width, flavour, group) the library must accept for workload `w` — the rules of include/swept.h and
    DESIGN.md §5, restated here independently of the library, so that a regression which makes a flavour
    inadmissible (or silently admits one it has no kernel for) fails the tests instead of being skipped."""
    N, problem, bc = w.N, w.problem, getattr(w, "bc", 0)
    h, _, C = si.PROBLEM_SHAPE[problem]
    size = np.dtype(dtype).itemsize
    if n < 32 or n & (n - 1) or N % n:
        return False
    if flavor == sw.FLAVOR_TIER:  # one CTA per tile, P points per thread, rows (+ Euler pressures/fluxes) in shared memory
        P = group
        if P == 0:
            P = (1 if n <= 256 else 2 if n <= 2048 else 4) if problem == si.EULER else \
                {32: 1, 64: 1, 128: 1, 256: 1, 512: 2, 1024: 4, 2048: 4, 4096: 4}.get(n, 0)
        row = (n + 4 * (16 // size)) * size
        smem = 2 * C * row + 16 + (4 * row if problem == si.EULER else 0)
        return n <= 4096 and P in (1, 2, 4) and 8 <= n // P <= 1024 and smem <= 227 * 1024
    if flavor == sw.FLAVOR_CHAR:  # L lanes per tile, B = n/L lines per lane in registers, 32 or 64 threads per CTA
        if bc and not (problem == si.HEAT and n <= 1024):  # walls: hybrid with TIER wall tiles, heat only
            return False
        Ls = (group,) if group else (32, 16, 8)
        for L in Ls:
            if L not in (8, 16, 32) or n % L:
                continue
            B = n // L
            if B not in ((4, 8, 16, 32) if h == 1 else (8, 16, 32)) or B > (8 if problem == si.EULER else 32):
                continue
            T = 64 if N % (64 * B) == 0 else 32 if N % (32 * B) == 0 else 0
            if T >= L:
                return True
        return False
    if flavor == sw.FLAVOR_FLOW:  # persistent launch: periodic heat / KS, 32 lanes per tile, B = n/32 in {8, 16, 32}
        if bc and problem != si.HEAT:   # walls inside the persistent launch: insulated heat ends only
            return False
        return problem != si.EULER and n in (256, 512, 1024) and N % 256 == 0 and (group & 15) <= 12 and group < 32
    raise ValueError(flavor)


def run_or_refusal(w, nsteps, n, fl, grp, dtype=np.float64):
    """The swept result, or None when the library refuses the configuration — and it must refuse exactly the
    inadmissible ones (no silent skip: the expected set is `admissible`)."""
    want = admissible(w, n, fl, grp, dtype)
    try:
        sx, _ = gpu_run(w, nsteps, sw.SWEPT, n, fl, grp, dtype=dtype)
    except sw.SweptError as e:
        assert not want, f"library refused an admissible configuration (n={n}, flavor={fl}, group={grp}): {e}"
        assert "not admissible" in str(e) or "no FLOW kernel" in str(e), str(e)
        return None
    assert want, f"library ran a configuration this table calls inadmissible (n={n}, flavor={fl}, group={grp})"
    return sx


def check(w, nsteps, tile_widths, dtype=np.float64, flavors=((sw.FLAVOR_TIER, 0),) + CHAR + FLOW, exact=True,
          min_ran=None):
    C = w.components
    ref = oracle.run_workload(w, nsteps=nsteps, dtype=dtype)
    ps, _ = gpu_run(w, nsteps, sw.PER_STEP, dtype=dtype)
    tol = TOL[np.dtype(dtype)]
    assert np.all(np.isfinite(ps))
    assert relerr(ps, ref, C) <= tol, f"per_step vs oracle: {relerr(ps, ref, C)}"
    if exact:
        assert np.array_equal(ps, ref), "same expression trees: expected 0 ulp"
    ran = []
    for n in tile_widths:
        for fl, grp in flavors:
            sx = run_or_refusal(w, nsteps, n, fl, grp, dtype)
            if sx is None:
                continue
            ran.append((n, fl, grp))
            assert np.array_equal(sx, ps), f"swept(n={n}, flavor={fl}, group={grp}) != per_step bitwise"
            assert relerr(sx, ref, C) <= tol
    expected = [(n, fl, grp) for n in tile_widths for fl, grp in flavors if admissible(w, n, fl, grp, dtype)]
    assert ran == expected
    if min_ran is not None:  # the caller's own count of what this case is meant to exercise
        assert len(ran) >= min_ran, (len(ran), min_ran)
    return ran


# ---------------------------------------------------------------- small cases spanning several tiles
@pytest.mark.parametrize("N,nsteps", [(256, 0), (256, 7), (256, 64), (512, 333), (96, 50)])
def test_heat_small(N, nsteps):
    w = si.heat_sines(N, 8, 11, nsteps)
    widths = [n for n in (32, 64, 128, 256) if N % n == 0]
    check(w, nsteps, widths, flavors=TIER12 + CHAR + FLOW)


@pytest.mark.parametrize("rk2", [si.RK2_MIDPOINT, si.RK2_HEUN])
@pytest.mark.parametrize("N,nsteps", [(256, 5), (512, 100), (1024, 77)])
def test_ks_small(N, nsteps, rk2):
    w = si.ks_cos(N, 5, nsteps)
    w.rk2 = rk2
    check(w, nsteps, [32, 64, 128, 256], flavors=TIER12 + ((sw.FLAVOR_TIER, 4),) + CHAR + FLOW)


@pytest.mark.parametrize("rk2", [si.RK2_MIDPOINT, si.RK2_HEUN])
@pytest.mark.parametrize("N,nsteps", [(256, 3), (512, 150)])
def test_euler_small(N, nsteps, rk2):
    w = si.euler_double_sod(N, nsteps, rk2=rk2)
    check(w, nsteps, [32, 64, 128, 256], flavors=TIER12 + CHAR + FLOW)


def test_euler_random_data():
    N = 384
    w = si.euler_double_sod(N, 40)
    w.u0 = si.random_smooth(si.EULER, N, 123)
    w.dt = 0.1 * w.dx
    check(w, 40, [32, 64, 128])


def test_single_tile_wraps_onto_itself():
    # N == n: the one shifted tile is split across the periodic boundary
    for w in (si.heat_sines(64, 4, 3, 200), si.ks_cos(64, 3, 60)):
        check(w, w.nsteps, [64])


def test_heat_fp32():
    w = si.heat_sines(1024, 16, 21, 500)
    check(w, 500, [32, 128, 256, 1024], dtype=np.float32, flavors=((sw.FLAVOR_TIER, 1), (sw.FLAVOR_TIER, 4)) + CHAR + FLOW)


def test_wide_tiles():
    w = si.heat_sines(8192, 16, 5, 3000)
    check(w, 3000, [2048, 4096], flavors=((sw.FLAVOR_TIER, 4),))
    w = si.ks_cos(8192, 5, 700)
    check(w, 700, [2048, 4096], flavors=((sw.FLAVOR_TIER, 4),))
    # Euler: the TIER kernel with shared pressures / fluxes, up to 1024 threads per tile
    w = si.euler_double_sod(8192, 600)
    check(w, 600, [1024, 2048], flavors=((sw.FLAVOR_TIER, 1), (sw.FLAVOR_TIER, 2), (sw.FLAVOR_TIER, 4)))


@pytest.mark.parametrize("warps", [0, 1, 3, 16, 18])  # resident CTAs per SM (0 = default policy); +16 = TMA staging
def test_flow_flavour_many_cycles_and_small_grids(warps):
    # FLOW: one persistent launch per Up..Down cycle, rows chained by per-tile flags.  K = N/n = 1, 2 and
    # many tiles per row; D = 0 (Up + Down only), odd and even D; remainder levels; both RK2 flavours
    for w, widths in ((si.heat_sines(1024, 8, 3, 1500), (256, 512, 1024)),
                      (si.heat_sines(1 << 15, 8, 4, 700), (256, 512, 1024)),
                      (si.ks_cos(2048, 6, 333), (256, 512, 1024)),
                      (si.ks_cos(1 << 14, 7, 200), (256, 512))):
        ref = oracle.run_workload(w)
        for n in widths:
            got, launches = gpu_run(w, w.nsteps, sw.SWEPT, n, sw.FLAVOR_FLOW, warps)
            assert np.array_equal(got, ref), (w.name, n, warps)
    w = si.heat_sines(4096, 8, 2, 0)
    s = sw.Swept.from_workload(w)
    s.run(128 * 5, 256, sw.SWEPT, sw.FLAVOR_FLOW)     # exactly 5 rows of m = 128: one launch
    assert s.last_launches == 1
    s.close()


def test_per_step_resident_matches_oracle():
    # per-step sub-timesteps in one persistent cooperative launch (PS_RESIDENT): single CTA (no global exchange),
    # several CTAs (neighbour flags), a ragged last CTA, N not a power of two, both RK2 flavours, FP32
    cases = [(si.heat_sines(2048, 8, 3, 700), np.float64), (si.heat_sines(1 << 16, 8, 4, 300), np.float64),
             (si.heat_sines(1 << 20, 16, 5, 150), np.float64), (si.heat_sines(3000, 4, 6, 200), np.float64),
             (si.heat_sines(100000, 4, 7, 120), np.float64), (si.heat_sines(1 << 17, 8, 8, 200), np.float32),
             (si.ks_cos(4096, 9, 150), np.float64), (si.ks_cos(1 << 18, 10, 60), np.float64),
             (si.euler_double_sod(2048, 80), np.float64), (si.euler_double_sod(1 << 15, 40), np.float64)]
    w = si.ks_cos(1 << 14, 11, 90)
    w.rk2 = si.RK2_HEUN
    cases.append((w, np.float64))
    cases.append((si.euler_double_sod(4096, 50, rk2=si.RK2_MIDPOINT), np.float64))
    for w, dtype in cases:
        ref = oracle.run_workload(w, dtype=dtype)
        got, launches = gpu_run(w, w.nsteps, sw.PER_STEP, 0, sw.PS_RESIDENT, dtype=dtype)
        assert launches == 1
        assert np.array_equal(got, ref), (w.name, w.N, dtype)
    # continues from a swept run and into a launch-per-step run on the same state
    w = si.heat_sines(8192, 8, 2, 0)
    s = sw.Swept.from_workload(w)
    s.run(300, 256, sw.SWEPT)
    s.run(77, 0, sw.PER_STEP, sw.PS_RESIDENT)
    s.run(23, 0, sw.PER_STEP)
    got = s.read()
    s.close()
    assert np.array_equal(got, oracle.run_workload(w, nsteps=400))
    # too large for a co-resident register-resident grid: a clean error, no fallback
    w = si.heat_sines(1 << 26, 4, 2, 0)
    s = sw.Swept.from_workload(w)
    with pytest.raises(sw.SweptError):
        s.run(10, 0, sw.PER_STEP, sw.PS_RESIDENT)
    s.close()


def test_heat_insulated_ends_bc_paper():
    # the paper's own heat boundary condition (B.5): per-step and swept (TIER flavour; the tile split across the
    # boundary applies the walls at its centre) against the oracle, bit for bit
    for N, steps in ((64, 100), (256, 333), (1024, 1500), (4096, 700)):
        w = si.heat_insulated(N, 6, 31, steps)
        ref = oracle.run_workload(w)
        ps, _ = gpu_run(w, steps, sw.PER_STEP)
        assert np.array_equal(ps, ref), ("per_step", N)
        for n in (32, 64, 256, 1024):
            if N % n:
                continue
            for P in (1, 2, 4):
                sx = run_or_refusal(w, steps, n, sw.FLAVOR_TIER, P)
                if sx is not None:
                    assert np.array_equal(sx, ref), ("swept", N, n, P)
        sx, _ = gpu_run(w, steps, sw.SWEPT)          # library default: must pick an admissible (TIER) configuration
        assert np.array_equal(sx, ref)
        rs, _ = gpu_run(w, steps, sw.PER_STEP, 0, sw.PS_RESIDENT)   # launch-free per-step, walls at the two end threads
        assert np.array_equal(rs, ref), ("resident", N)
    w = si.heat_insulated(2048, 4, 32, 300)
    assert np.array_equal(gpu_run(w, 300, sw.SWEPT, 128, dtype=np.float32)[0],
                          oracle.run_workload(w, dtype=np.float32))
    # hybrid: CHAR on every tile that touches no wall, the wall tiles by the TIER kernels on a second stream
    for N, steps in ((1024, 900), (1 << 15, 700), (1 << 20, 1300)):
        w2 = si.heat_insulated(N, 6, 33, steps)
        ref2 = oracle.run_workload(w2)
        ran = 0
        for n in (64, 256, 512, 1024):
            for L in (8, 16, 32):
                sx = run_or_refusal(w2, steps, n, sw.FLAVOR_CHAR, L)
                if sx is None:
                    continue
                ran += 1
                assert np.array_equal(sx, ref2), ("hybrid", N, n, L)
        assert ran == sum(admissible(w2, n, sw.FLAVOR_CHAR, L) for n in (64, 256, 512, 1024) for L in (8, 16, 32)) >= 8
        # FLOW with walls: the one or two wall tiles of a row advance tier by tier inside the persistent launch
        ran = 0
        for n in (256, 512, 1024):
            for grp in (0, 2, 16 + 3):
                sx = run_or_refusal(w2, steps, n, sw.FLAVOR_FLOW, grp)
                if sx is None:
                    continue
                ran += 1
                assert np.array_equal(sx, ref2), ("flow walls", N, n, grp)
        assert ran == sum(admissible(w2, n, sw.FLAVOR_FLOW, g) for n in (256, 512, 1024) for g in (0, 2, 19)) >= 3
    w3 = si.heat_insulated(1 << 14, 6, 34, 777)
    assert np.array_equal(gpu_run(w3, 777, sw.SWEPT, 256, sw.FLAVOR_FLOW, dtype=np.float32)[0],
                          oracle.run_workload(w3, dtype=np.float32))
    e = si.euler_sod(2048, 10)
    with pytest.raises(sw.SweptError):               # walls in the persistent flavour: heat only
        gpu_run(e, 10, sw.SWEPT, 256, sw.FLAVOR_FLOW)
    s = sw.Swept.from_workload(w)
    best = s.autotune(sw.SWEPT)
    s.run(300, 0, sw.SWEPT)
    assert np.array_equal(s.read(), oracle.run_workload(w)) and best >= 32
    s.close()
    with pytest.raises(sw.SweptError):
        sw.swept_create(sw.KS, 4096, 0.5, 0.005, bc=sw.BC_PAPER)


@pytest.mark.parametrize("rk2", [si.RK2_MIDPOINT, si.RK2_HEUN])
def test_euler_dirichlet_ends_bc_paper(rk2):
    # the paper's Sod tube: end states held; long enough for the waves to reach and leave the ends
    for N, steps in ((256, 40), (512, 700), (2048, 300)):
        w = si.euler_sod(N, steps, rk2=rk2)
        ref = oracle.run_workload(w)
        ps, _ = gpu_run(w, steps, sw.PER_STEP)
        assert np.array_equal(ps, ref), ("per_step", N)
        ran = 0
        for n in (32, 128, 512):
            for P in (1, 2):
                sx = run_or_refusal(w, steps, n, sw.FLAVOR_TIER, P)   # refused only where n > N
                if sx is None:
                    continue
                ran += 1
                assert np.array_equal(sx, ref), ("swept", N, n, P)
        assert ran == 2 * sum(1 for n in (32, 128, 512) if n <= N) >= 4
        assert np.array_equal(gpu_run(w, steps, sw.SWEPT)[0], ref)
        assert np.array_equal(gpu_run(w, steps, sw.PER_STEP, 0, sw.PS_RESIDENT)[0], ref), ("resident", N)


def test_euler_dirichlet_rewrite_discards_cached_graphs():
    # The per-step CUDA graphs hold the Dirichlet end states as kernel arguments: writing a field with other end
    # states must not replay graphs captured for the old ones.  300 steps = one 256-step graph + 44 launches
    wA = si.euler_sod(2048, 300)
    wB = si.euler_sod(2048, 300)
    N = wB.N
    u = wB.u0.reshape(3, N).copy()
    u[0, : N // 2] *= 1.5          # other left state (density, energy) ...
    u[2, : N // 2] *= 1.25
    u[0, N // 2:] *= 0.8           # ... and other right state
    wB.u0 = u.reshape(-1)
    s = sw.Swept.from_workload(wA)
    s.run(300, 0, sw.PER_STEP)
    assert np.array_equal(s.read(), oracle.run_workload(wA))
    s.write(wB.u0)
    s.run(300, 0, sw.PER_STEP)
    assert np.array_equal(s.read(), oracle.run_workload(wB))
    s.write(wA.u0)                 # and back, through the device-to-device entry point
    import torch
    dev = torch.from_numpy(wA.u0).cuda()
    sw.load().swept_write_device(s._h, dev.data_ptr())
    s.run(300, 0, sw.PER_STEP)
    s.run(300, 128, sw.SWEPT)
    assert np.array_equal(s.read(), oracle.run_workload(wA, nsteps=600))
    s.close()


def test_swept_run_neither_allocates_nor_synchronises():
    # "swept_run never synchronises", device memory comes from the allocator hooks at creation.
    # Proof by capture: under a GLOBAL-mode stream capture any cudaMalloc / cudaFree / synchronisation made by the
    # capturing thread is an error that invalidates the capture.  Each variant is recorded into a CUDA graph,
    # replayed and checked against the oracle; a last case replays twice (the persistent launch must leave its
    # scratch as it found it).
    import torch
    w = si.heat_sines(1 << 14, 8, 2, 0)
    wk = si.ks_cos(1 << 13, 4, 0)
    wb = si.heat_insulated(1 << 13, 4, 5, 0)
    cases = [(w, sw.SWEPT, 256, sw.FLAVOR_FLOW, 0, 128 * 6 + 20), (w, sw.SWEPT, 256, sw.FLAVOR_CHAR, 32, 128 * 3 + 5),
             (w, sw.SWEPT, 64, sw.FLAVOR_TIER, 1, 200), (w, sw.SWEPT, 0, sw.FLAVOR_AUTO, 0, 500),
             (wk, sw.SWEPT, 256, sw.FLAVOR_FLOW, 0, 150), (wk, sw.PER_STEP, 0, sw.PS_LAUNCH, 0, 70),
             (wb, sw.SWEPT, 256, sw.FLAVOR_CHAR, 32, 300),          # hybrid: wall tiles on the second stream
             (w, sw.PER_STEP, 0, sw.PS_LAUNCH, 0, 100), (w, sw.PER_STEP, 0, sw.PS_RESIDENT, 0, 60)]
    for wl, variant, n, fl, grp, steps in cases:
        s = sw.Swept.from_workload(wl)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, capture_error_mode="global"):
            s.run(steps, n, variant, fl, grp)
        assert s.last_launches >= 1
        g.replay()
        got = s.read()
        assert np.array_equal(got, oracle.run_workload(wl, nsteps=steps)), (wl.name, variant, n, fl)
        s.close()
    # replay-safety of the FLOW scratch proper: capture write + run together, replay twice
    s = sw.Swept.from_workload(w)
    dev = torch.from_numpy(w.u0).cuda()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    lib = sw.load()
    with torch.cuda.graph(g, capture_error_mode="global"):
        sw.swept_set_stream(s._h, int(torch.cuda.current_stream().cuda_stream))
        assert lib.swept_write_device(s._h, dev.data_ptr()) == 0
        s.run(128 * 4, 256, sw.SWEPT, sw.FLAVOR_FLOW)
    ref = oracle.run_workload(w, nsteps=512)
    for _ in range(2):
        g.replay()
        assert np.array_equal(s.read(), ref)
    s.close()


def test_per_step_non_power_of_two_N():
    # the paper's `& lastidx` wrap needs N = 2^k; ours does not
    for N in (1000, 1001, 1002):
        w = si.heat_sines(N, 4, 9, 120)
        ref = oracle.run_workload(w)
        got, _ = gpu_run(w, 120, sw.PER_STEP)
        assert np.array_equal(got, ref)
    w = si.ks_cos(1001, 9, 30)
    assert np.array_equal(gpu_run(w, 30, sw.PER_STEP)[0], oracle.run_workload(w))
    # Euler's interface-per-lane kernel: 28 cells per warp, ragged last warp, wrap inside a warp
    for N in (30, 57, 1000, 1023):
        w = si.euler_double_sod(N, 25)
        w.u0 = si.random_smooth(si.EULER, N, 77)
        w.dt = 0.1 * w.dx
        assert np.array_equal(gpu_run(w, 25, sw.PER_STEP)[0], oracle.run_workload(w)), N
    w = si.euler_sod(999, 40)
    assert np.array_equal(gpu_run(w, 40, sw.PER_STEP)[0], oracle.run_workload(w))


def test_repeated_runs_accumulate_and_launch_counts():
    w = si.heat_sines(4096, 8, 2, 0)
    s = sw.Swept.from_workload(w)
    s.run(1000, 64, sw.SWEPT)
    # m = 32: D = 1000/32 - 1 = 30 diamonds + Up + Down, remainder 8 per-step launches
    assert s.last_launches == 32 + 8
    s.run(300, 0, sw.PER_STEP)
    assert s.last_launches == 300
    s.run(500, 512, sw.SWEPT)
    got = s.read()
    s.close()
    assert np.array_equal(got, oracle.run_workload(w, nsteps=1800))


def test_phase_timing_and_fully_default_run():
    # swept_set_phase_timing / swept_phase_times: one CUDA-event pair per launch, reported per phase kind
    w = si.heat_sines(1 << 14, 8, 2, 0)
    s = sw.Swept.from_workload(w)
    s.set_phase_timing(True)
    s.run(128 * 6, 256, sw.SWEPT, sw.FLAVOR_CHAR, 32)      # Up, 5 diamonds (3 split, 2 whole), Down
    t = s.phase_times()
    assert [t[k][1] for k in ("UpTriangle", "SplitDiamond", "WholeDiamond", "DownTriangle")] == [1, 3, 2, 1]
    assert all(t[k][0] > 0 for k in ("UpTriangle", "SplitDiamond", "WholeDiamond", "DownTriangle"))
    s.run(128 * 6, 256, sw.SWEPT, sw.FLAVOR_FLOW)
    t = s.phase_times()
    assert t["FlowCycle"][1] == 1 and t["FlowCycle"][0] > 0 and t["SplitDiamond"][1] == 0
    s.set_phase_timing(False)
    s.run(10, 256, sw.SWEPT)
    assert sum(v[1] for v in s.phase_times().values()) == 0
    s.close()
    # swept_run(state, nsteps, 0, SWEPT) with nothing tuned on a large problem: FLOW at the measured-best width
    for w in (si.heat_sines(1 << 19, 8, 3, 600), si.ks_cos(1 << 19, 3, 300)):
        s = sw.Swept.from_workload(w)
        s.run(w.nsteps, 0, sw.SWEPT)
        got = s.read()
        s.close()
        ps, _ = gpu_run(w, w.nsteps, sw.PER_STEP)
        assert np.array_equal(got, ps)


def test_default_run_with_insulated_ends_medium_and_large():
    # swept_run(state, nsteps, 0, SWEPT) with nothing tuned on the heat problem with the paper's own ends (B.5): the
    # persistent FLOW launch from N = 2^15 up (wall tiles inside the launch), i.e. a handful of launches, not one per row
    for N, steps in ((1 << 15, 700), (1 << 19, 300), (1 << 21, 520)):
        w = si.heat_insulated(N, 6, 71, steps)
        got, launches = gpu_run(w, steps, sw.SWEPT)
        ref = oracle.run_workload(w) if N <= (1 << 19) else gpu_run(w, steps, sw.PER_STEP)[0]
        assert np.array_equal(got, ref), N
        assert launches <= 24, (N, launches)


def test_error_codes():
    w = si.heat_sines(4096, 8, 2, 0)
    s = sw.Swept.from_workload(w)
    with pytest.raises(sw.SweptError):
        s.run(10, 48, sw.SWEPT)          # not a power of two
    with pytest.raises(sw.SweptError):
        s.run(10, 8192, sw.SWEPT)        # does not divide N
    with pytest.raises(sw.SweptError):
        s.run(-1, 64, sw.SWEPT)
    with pytest.raises(sw.SweptError):
        s.run(10, 100, sw.PER_STEP)      # threads per block not a power of two
    with pytest.raises(sw.SweptError):
        sw.swept_create(sw.KS, 4096, 0.5, 0.005, dtype=sw.F32)  # FP32 is heat only
    s.run(10, 64, sw.SWEPT)              # still usable after errors
    assert np.array_equal(s.read(), oracle.run_workload(w, nsteps=10))
    s.close()


# ---------------------------------------------------------------- the five configs
def test_config1_full():
    w = si.config(1)  # heat FP64 N=2048, 20000 steps
    check(w, w.nsteps, [32, 64, 128, 256, 512, 1024], flavors=TIER12 + CHAR + FLOW)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_config2_full_length(dtype):
    for N in (1 << 11, 1 << 16):  # full 10000 steps against the oracle
        w = si.config(2, N=N)
        check(w, w.nsteps, [32, 256, 1024], dtype=dtype, flavors=((sw.FLAVOR_TIER, 2),) + CHAR + FLOW)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_config2_large_N(dtype):
    # oracle over a reduced step count covering > 2 swept cycles + remainder; full run swept == per_step
    for N in (1 << 20, 1 << 22):
        w = si.config(2, N=N)
        check(w, 1100, [256, 1024], dtype=dtype, flavors=((sw.FLAVOR_TIER, 2),) + CHAR + FLOW)
    w = si.config(2, N=1 << 20)
    ps, _ = gpu_run(w, w.nsteps, sw.PER_STEP, dtype=dtype)
    sx, _ = gpu_run(w, w.nsteps, sw.SWEPT, 256, dtype=dtype)
    assert np.array_equal(ps, sx)


def test_headline_full_size_in_the_bench_configuration():
    # BASELINE.json's metric workload at full size (heat FP64, N = 2^20, 10 000 steps) in the launch configuration
    # bench.py times: the autotuned (n, flavour, group), and the FLOW configuration it reports on B200.  The oracle
    # runs the full length (a few seconds on the host cores), so every one of the 2^20 outputs is compared
    w = si.config(2, N=1 << 20)
    ref = oracle.run_workload(w)
    s = sw.Swept.from_workload(w)
    n = s.autotune(sw.SWEPT)
    _, fl, grp = s.tuned(sw.SWEPT)
    s.run(w.nsteps, n, sw.SWEPT, fl, grp)
    got = s.read()
    s.close()
    assert np.array_equal(got, ref), (n, fl, grp)
    assert relerr(got, ref, 1) <= 1e-12
    got, launches = gpu_run(w, w.nsteps, sw.SWEPT, 512, sw.FLAVOR_FLOW, 3)
    assert np.array_equal(got, ref) and launches == 3   # one persistent launch + Up/Down of the 16-step tail
    got, _ = gpu_run(w, w.nsteps, sw.PER_STEP, 0, sw.PS_RESIDENT)
    assert np.array_equal(got, ref)


def test_config3_ks():
    w = si.config(3, N=1 << 14)  # full 20000 steps
    check(w, w.nsteps, [64, 256, 1024], flavors=((sw.FLAVOR_TIER, 2),) + CHAR + FLOW)
    w = si.config(3, N=1 << 20)
    check(w, 300, [256], flavors=((sw.FLAVOR_TIER, 2),) + CHAR + FLOW)
    ps, _ = gpu_run(w, 4000, sw.PER_STEP)
    sx, _ = gpu_run(w, 4000, sw.SWEPT, 512)
    assert np.array_equal(ps, sx) and np.all(np.isfinite(ps)) and np.max(np.abs(ps)) < 10


@pytest.mark.parametrize("rk2", [si.RK2_HEUN, si.RK2_MIDPOINT])
def test_config4_euler(rk2):
    for N in (1 << 11, 1 << 14):  # full 5000 steps
        w = si.config(4, N=N, rk2=rk2)
        check(w, w.nsteps, [64, 256], flavors=((sw.FLAVOR_TIER, 2),) + CHAR + FLOW)
    w = si.config(4, N=1 << 20, rk2=rk2)
    check(w, 70, [256], flavors=((sw.FLAVOR_TIER, 2),) + CHAR + FLOW)


def test_config5_sampled_grid():
    # swept == per_step bit for bit over the (problem, N, n) grid; oracle on the smallest N of each
    for problem, steps in ((si.HEAT, 2000), (si.KS, 600), (si.EULER, 150)):
        for N in (1 << 11, 1 << 17, 1 << 22):
            w = si.config(5, N=N, problem=problem, nsteps=steps)
            ps, _ = gpu_run(w, steps, sw.PER_STEP)
            if N == 1 << 11:
                assert np.array_equal(ps, oracle.run_workload(w, nsteps=steps))
            for n in (32, 128, 512, 1024):
                for fl, grp in ((sw.FLAVOR_TIER, 0), (sw.FLAVOR_CHAR, 16), (sw.FLAVOR_CHAR, 32), (sw.FLAVOR_FLOW, 0)):
                    sx = run_or_refusal(w, steps, n, fl, grp)
                    if sx is not None:
                        assert np.array_equal(ps, sx), (problem, N, n, fl, grp)


def test_autotune_picks_admissible_width_and_keeps_state():
    w = si.heat_sines(1 << 16, 8, 2, 0)
    s = sw.Swept.from_workload(w)
    s.run(100, 64, sw.SWEPT)
    best = s.autotune(sw.SWEPT)
    assert best in (32, 64, 128, 256, 512, 1024, 2048, 4096) and (1 << 16) % best == 0
    bt = s.autotune(sw.PER_STEP)
    assert 32 <= bt <= 1024
    s.run(100, 0, sw.SWEPT)  # uses the tuned width; the field was restored after tuning
    got = s.read()
    tuned = s.tuned(sw.SWEPT)
    s.close()
    assert np.array_equal(got, oracle.run_workload(w, nsteps=200))
    s2 = sw.Swept.from_workload(w)   # same (problem, dtype, N): the process-wide cache hands the result over
    assert s2.tuned(sw.SWEPT) == tuned and tuned[0] == best
    s2.close()
