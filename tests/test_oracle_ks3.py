"""Pins for the three-sub-timestep KS oracle ("more than two sub-timesteps per
timestep"): Eq. (C.2) advanced by the three-stage Shu-Osher SSP Runge-Kutta method.

growth   : a tiny Fourier mode is multiplied per step by 1 + z + z^2/2 + z^3/6, z = dt (16 s^2 - 256 s^4) at dx = 0.5
           (pins the stage weights 3/4, 1/4, 1/3, 2/3 and the order of the stages; a two-stage or mis-weighted
           scheme gives another polynomial),
order    : third-order convergence in dt on a fixed grid (independent of the polynomial: it also involves the
           nonlinear term),
mean     : conservation of the mean (each stage is a convex combination of conservative Euler steps),
pde      : one tiny step reproduces -(u u_x + u_xx + u_xxxx) of Eq. (C.1),
rational : exact-rational evaluation of the three stages as written above on 9 points,
same f   : with dt -> 0 the step agrees with the two-stage oracle's to O(dt^3) (same spatial operator).
"""
from fractions import Fraction

import numpy as np
import pytest

import oracle
import swept_inputs as si


@pytest.mark.parametrize("k,N", [(3, 64), (10, 64), (32, 64), (7, 100)])
def test_growth_polynomial_third_order(k, N):
    dx, dt, M, eps = 0.5, 0.005, 40, 1e-8
    i = np.arange(N)
    u0 = eps * np.sin(2 * np.pi * k * i / N + 0.3)
    s = np.sin(np.pi * k / N)
    z = dt * (4.0 * s * s / dx ** 2 - 16.0 * s ** 4 / dx ** 4)
    G = 1.0 + z + z * z / 2.0 + z ** 3 / 6.0
    if abs(G) < 0.5:
        M = 8                                        # strongly damped mode: stay above the round-off floor
    u = oracle.run(oracle.KS3, u0, N, M, dx, dt)
    kk = k if k <= N // 2 else N - k
    ratio = np.fft.rfft(u)[kk] / np.fft.rfft(u0)[kk]
    assert abs(ratio - G ** M) < 1e-6 * abs(G ** M)
    G2 = 1.0 + z + z * z / 2.0                       # what a two-stage scheme would give: must be told apart
    if abs(z) > 0.3:
        assert abs(ratio - G2 ** M) > 1e-3 * abs(G2 ** M)


def test_third_order_in_dt():
    # smooth nonlinear solution on a fixed coarse grid; reference = the same scheme at dt/32
    N, dx, T = 64, 1.0, 3.2                            # dt = 0.05 and 0.025: |z| <= 12 dt, inside the stability region
    x = np.arange(N) * dx
    u0 = np.cos(2 * np.pi * x / (N * dx)) * (1.0 + 0.5 * np.sin(4 * np.pi * x / (N * dx)))

    def solve(nsteps):
        return oracle.run(oracle.KS3, u0, N, nsteps, dx, T / nsteps)

    ref = solve(64 * 32)
    e1 = np.max(np.abs(solve(64) - ref))
    e2 = np.max(np.abs(solve(128) - ref))
    assert e1 > 1e-9                                   # above round-off, so the ratio means something
    assert 6.5 < e1 / e2 < 9.5                         # 2^3 = 8
    # the two-stage midpoint scheme on the same problem converges with order 2: different scheme, told apart
    r1 = np.max(np.abs(oracle.run(oracle.KS, u0, N, 64, dx, T / 64) - ref))
    r2 = np.max(np.abs(oracle.run(oracle.KS, u0, N, 128, dx, T / 128) - ref))
    assert 3.3 < r1 / r2 < 4.7


def test_mean_conserved_and_bounded():
    w = si.ks3_cos(1 << 12, si.BASE_SEED + 3, 3000)
    u = oracle.run_workload(w)
    assert np.all(np.isfinite(u)) and np.max(np.abs(u)) < 10.0
    assert abs(u.mean() - w.u0.mean()) < 1e-14
    assert np.max(np.abs(u)) > 0.5 and np.max(np.abs(u - w.u0)) > 0.1


def test_pde_consistency():
    errs = []
    for N in (64, 128):
        dx = 2 * np.pi / N
        x = np.arange(N) * dx
        u0 = np.sin(x) + 0.5 * np.cos(2 * x)
        f = -(u0 * (np.cos(x) - np.sin(2 * x)) + (-np.sin(x) - 2.0 * np.cos(2 * x)) + (np.sin(x) + 8.0 * np.cos(2 * x)))
        dt = 1e-10
        u1 = oracle.run(oracle.KS3, u0, N, 1, dx, dt)
        errs.append(np.max(np.abs((u1 - u0) / dt - f)))
    assert errs[1] < 0.02 * np.max(np.abs(f)) and 3.0 < errs[0] / errs[1] < 5.0


def test_rational_brute_force():
    rng = np.random.default_rng(17)
    N, steps = 9, 2
    u0 = rng.uniform(-1, 1, N)
    dx, dt = 0.5, 0.005
    DX, DT = Fraction(dx), Fraction(dt)

    def f(u, i):  # right-hand side of (C.2) with reading X2
        p1, m1, p2, m2 = u[(i + 1) % N], u[(i - 1) % N], u[(i + 2) % N], u[(i - 2) % N]
        return -((p1 * p1 - m1 * m1) / (4 * DX) + (p1 + m1 - 2 * u[i]) / DX ** 2
                 + (p2 - 4 * p1 + 6 * u[i] - 4 * m1 + m2) / DX ** 4)

    u = [Fraction(x) for x in u0]
    for _ in range(steps):
        u1 = [u[i] + DT * f(u, i) for i in range(N)]
        u2 = [Fraction(3, 4) * u[i] + Fraction(1, 4) * (u1[i] + DT * f(u1, i)) for i in range(N)]
        u = [Fraction(1, 3) * u[i] + Fraction(2, 3) * (u2[i] + DT * f(u2, i)) for i in range(N)]
    got = oracle.run(oracle.KS3, u0, N, steps, dx, dt)
    assert np.max(np.abs(got - np.array([float(v) for v in u]))) < 64 * np.finfo(float).eps


def test_same_spatial_operator_as_two_stage_oracle():
    # u + dt f + dt^2/2 f'f is common to both schemes; they differ at O(dt^3)
    N, dx = 128, 0.5
    w = si.ks_cos(N, 5, 1)
    d = []
    for dt in (1e-3, 5e-4):
        a = oracle.run(oracle.KS, w.u0, N, 1, dx, dt)
        b = oracle.run(oracle.KS3, w.u0, N, 1, dx, dt)
        d.append(np.max(np.abs(a - b)))
    assert d[0] > 0 and 6.0 < d[0] / d[1] < 10.0


def test_thread_count_does_not_change_bits():
    w = si.ks3_cos(1 << 15, 3, 10)
    nt = oracle.num_threads()
    try:
        oracle.set_num_threads(1)
        a = oracle.run_workload(w)
        oracle.set_num_threads(max(2, nt))
        b = oracle.run_workload(w)
    finally:
        oracle.set_num_threads(nt)
    assert np.array_equal(a, b)
