"""GPU parity at BASELINE.json config 5's top sizes (N = 2^24, 2^26) and at the full lengths of configs 3 and 4
(run with -m gpu on the B200).

What is compared at sizes where a full-length oracle run would take minutes (SURVEY.md §8(d) "Oracle timing"):
  (i)   per-step and every swept flavour against the oracle, element by element over ALL N outputs, on a reduced
        step count that still covers Up, several diamonds, Down and a multi-level remainder at every tile width;
  (ii)  swept == per-step bit for bit over the config's full step count;
  (iii) for heat, where the method has a closed form (pin P1: g_k = 1 - 4 r sin^2(pi k / N), north_star), the
        full-length result against that closed form at every point.
These are the sizes whose launch shapes exist nowhere else in the suite: 65 536-CTA CHAR grids, FLOW rows of 2^18
tiles, 64-bit element offsets (3 x 2^26 x 8 B per Euler slab), HBM-resident per-step arrays.
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
        return s.read()
    finally:
        s.close()


def closed_form_heat(w, M):
    """u_i^M = sum_k a_k g_k^M sin(2 pi k i / N) (pin P1; g^M as exp(M log1p(.)) to avoid an M*eps error)."""
    i = np.arange(w.N, dtype=np.float64)
    u = np.zeros(w.N)
    for k, a in enumerate(w.meta["amps"], start=1):
        g_pow = np.exp(M * np.log1p(-4.0 * w.meta["r"] * np.sin(np.pi * k / w.N) ** 2))
        u += a * g_pow * np.sin(2.0 * np.pi * k * i / w.N)
    return u


@pytest.mark.parametrize("logn,oracle_steps", [(24, 1700), (26, 1100)])
def test_config5_heat_top_sizes(logn, oracle_steps):
    w = si.config(5, N=1 << logn, problem=si.HEAT)          # 5000 steps beyond 2^20 (BASELINE.json configs[4])
    assert w.nsteps == 5000
    ref = oracle.run_workload(w, nsteps=oracle_steps)
    ps = run(w, oracle_steps, sw.PER_STEP)
    assert np.array_equal(ps, ref), "per_step vs oracle"
    # n = 256: D >= 7 diamonds; 512: D >= 3; 1024: Up, one or two diamonds, Down; each followed by remainder cycles
    cases = [(256, sw.FLAVOR_FLOW, 0), (512, sw.FLAVOR_FLOW, 0), (1024, sw.FLAVOR_FLOW, 0),
             (256, sw.FLAVOR_CHAR, 32), (512, sw.FLAVOR_CHAR, 32), (1024, sw.FLAVOR_CHAR, 32),
             (512, sw.FLAVOR_CHAR, 16), (1024, sw.FLAVOR_TIER, 4)]
    for n, fl, grp in cases:
        got = run(w, oracle_steps, sw.SWEPT, n, fl, grp)
        assert np.array_equal(got, ref), (logn, n, fl, grp)
    del ref
    # full length: swept == per_step bitwise, and both against the closed form at every point
    ps = run(w, w.nsteps, sw.PER_STEP)
    exact = closed_form_heat(w, w.nsteps)
    assert np.max(np.abs(ps - exact)) <= 1e-11 * np.max(np.abs(w.u0))
    for n, fl, grp in ((512, sw.FLAVOR_FLOW, 0), (512, sw.FLAVOR_CHAR, 32), (0, sw.FLAVOR_AUTO, 0)):
        sx = run(w, w.nsteps, sw.SWEPT, n, fl, grp)
        assert np.array_equal(sx, ps), (logn, n, fl, grp)


def test_config5_ks_2p24():
    w = si.config(5, N=1 << 24, problem=si.KS)
    steps = 230   # 460 sub-timesteps: n = 256 (m = 64): Up, 6 diamonds, Down + 12; n = 1024 (m = 256): Up, Down + levels
    ref = oracle.run_workload(w, nsteps=steps)
    assert np.array_equal(run(w, steps, sw.PER_STEP), ref)
    for n, fl, grp in ((256, sw.FLAVOR_FLOW, 0), (1024, sw.FLAVOR_FLOW, 0), (512, sw.FLAVOR_CHAR, 32),
                       (1024, sw.FLAVOR_CHAR, 32), (256, sw.FLAVOR_TIER, 2)):
        assert np.array_equal(run(w, steps, sw.SWEPT, n, fl, grp), ref), (n, fl, grp)
    del ref
    ps = run(w, 2000, sw.PER_STEP)
    assert np.all(np.isfinite(ps)) and np.max(np.abs(ps)) < 10
    for n, fl, grp in ((1024, sw.FLAVOR_FLOW, 0), (1024, sw.FLAVOR_CHAR, 32)):
        assert np.array_equal(run(w, 2000, sw.SWEPT, n, fl, grp), ps), (n, fl, grp)


@pytest.mark.parametrize("logn,oracle_steps,long_steps", [(24, 24, 300), (26, 8, 80)])
def test_config5_euler_top_sizes(logn, oracle_steps, long_steps):
    w = si.config(5, N=1 << logn, problem=si.EULER)          # midpoint RK2, the paper's integrator
    ref = oracle.run_workload(w, nsteps=oracle_steps)
    ps = run(w, oracle_steps, sw.PER_STEP)
    assert np.array_equal(ps, ref), "per_step vs oracle"
    # 2 x oracle_steps sub-timesteps: n = 32 (m = 8) gives Up, diamonds, Down at 2^26 too
    for n, grp in ((32, 1), (64, 1)):
        assert np.array_equal(run(w, oracle_steps, sw.SWEPT, n, sw.FLAVOR_TIER, grp), ref), (n, grp)
    del ref
    ps = run(w, long_steps, sw.PER_STEP)
    for n, grp in ((256, 1), (512, 2)):
        assert np.array_equal(run(w, long_steps, sw.SWEPT, n, sw.FLAVOR_TIER, grp), ps), (n, grp)


def test_config3_ks_full_length_2p20():
    # BASELINE.json configs[2] at its largest N and full 20 000 steps: swept == per_step bit for bit (the oracle
    # covers the first 300 steps of the same run in test_gpu_parity.py::test_config3_ks)
    w = si.config(3, N=1 << 20)
    assert w.nsteps == 20000
    ps = run(w, w.nsteps, sw.PER_STEP)
    assert np.all(np.isfinite(ps)) and np.max(np.abs(ps)) < 10
    for n, fl, grp in ((1024, sw.FLAVOR_FLOW, 0), (512, sw.FLAVOR_CHAR, 32), (0, sw.FLAVOR_AUTO, 0)):
        assert np.array_equal(run(w, w.nsteps, sw.SWEPT, n, fl, grp), ps), (n, fl, grp)


@pytest.mark.parametrize("rk2", [si.RK2_HEUN, si.RK2_MIDPOINT])
def test_config4_euler_full_length_2p20(rk2):
    # BASELINE.json configs[3] at its largest N and full 5 000 steps (Heun as the config names it; midpoint = the
    # paper's scheme, reading X6): swept == per_step bit for bit
    w = si.config(4, N=1 << 20, rk2=rk2)
    assert w.nsteps == 5000
    ps = run(w, w.nsteps, sw.PER_STEP)
    assert np.all(np.isfinite(ps))
    rho = ps[:w.N]
    assert rho.min() > 0.1 and rho.max() < 1.1             # the double tube stays physical
    for n, grp in ((512, 2), (128, 1), (0, 0)):
        fl = sw.FLAVOR_TIER if n else sw.FLAVOR_AUTO
        assert np.array_equal(run(w, w.nsteps, sw.SWEPT, n, fl, grp), ps), (n, grp)
