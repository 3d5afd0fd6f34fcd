"""Pins for the Kuramoto-Sivashinsky oracle (Eqs. C.1-C.4).

P4 conservation of the mean (each term of C.2 telescopes on a periodic grid),
P5 linear growth factor 1 + z + z^2/2 of a tiny Fourier mode (pins the u_xx / u_xxxx terms, their
   signs (reading X2) and the two RK2 stages),
PDE consistency: one tiny step reproduces the continuous right-hand side of Eq. (C.1),
   -(u u_x + u_xx + u_xxxx), for a smooth field, with second-order convergence in dx
   (pins the nonlinear term's coefficient 1/(4 dx) and sign, independent of the discrete formula),
P6 brute-force rational evaluation of Eq. (C.2) with (C.3)/(C.4) as printed, N <= 16.
"""
from fractions import Fraction

import numpy as np
import pytest

import oracle
import swept_inputs as si


def test_p4_mean_conserved_config3_shape():
    w = si.config(3, N=1 << 12, nsteps=4000)
    u = oracle.run_workload(w)
    assert np.all(np.isfinite(u)) and np.max(np.abs(u)) < 10.0
    assert abs(u.mean() - w.u0.mean()) < 1e-14
    # chaotic, not decayed to nothing and not the initial field
    assert np.max(np.abs(u)) > 0.5 and np.max(np.abs(u - w.u0)) > 0.1


@pytest.mark.parametrize("rk2", [oracle.RK2_MIDPOINT, oracle.RK2_HEUN])
@pytest.mark.parametrize("k,N", [(3, 64), (10, 64), (32, 64), (7, 100)])
def test_p5_linear_growth_factor(rk2, k, N):
    dx, dt, M, eps = 0.5, 0.005, 50, 1e-8
    i = np.arange(N)
    u0 = eps * np.sin(2 * np.pi * k * i / N + 0.3)
    u = oracle.run(oracle.KS, u0, N, M, dx, dt, rk2=rk2)
    s = np.sin(np.pi * k / N)
    z = dt * (4.0 * s * s / dx ** 2 - 16.0 * s ** 4 / dx ** 4)
    G = 1.0 + z + 0.5 * z * z
    # amplitude of mode k by projection
    ck0 = np.fft.rfft(u0)[k if k <= N // 2 else N - k]
    ck = np.fft.rfft(u)[k if k <= N // 2 else N - k]
    assert abs(ck / ck0 - G ** M) < 1e-6 * abs(G ** M)


@pytest.mark.parametrize("rk2", [oracle.RK2_MIDPOINT, oracle.RK2_HEUN])
def test_pde_consistency_second_order(rk2):
    # u = sin x + 0.5 cos 2x on [0, 2 pi): all three terms of (C.1) are O(1..10)
    errs = []
    for N in (64, 128):
        dx = 2 * np.pi / N
        x = np.arange(N) * dx
        u0 = np.sin(x) + 0.5 * np.cos(2 * x)
        ux = np.cos(x) - np.sin(2 * x)
        uxx = -np.sin(x) - 2.0 * np.cos(2 * x)
        uxxxx = np.sin(x) + 8.0 * np.cos(2 * x)
        f = -(u0 * ux + uxx + uxxxx)
        dt = 1e-10  # dt * 16/dx^4 << 1: one RK2 step is u + dt f(u) to O(dt^2 f' f)
        u1 = oracle.run(oracle.KS, u0, N, 1, dx, dt, rk2=rk2)
        errs.append(np.max(np.abs((u1 - u0) / dt - f)))
    assert errs[1] < 0.02 * np.max(np.abs(f))
    assert 3.0 < errs[0] / errs[1] < 5.0  # second-order central differences


def test_nonlinear_term_alone():
    # dx huge: u_xx and u_xxxx terms vanish (1/dx^2, 1/dx^4), only (u_{+1}^2 - u_{-1}^2)/(4 dx) remains
    N, dx, dt = 12, 1.0e6, 1.0
    rng = np.random.default_rng(5)
    u0 = rng.uniform(-1, 1, N)
    # Heun stage 1 is a plain forward-Euler step u + dt f(u); run one full Heun step with dt so small
    # relative to dx that stage 2 changes nothing beyond O(dt^2): compare with first-order expectation
    u1 = oracle.run(oracle.KS, u0, N, 1, dx, dt, rk2=oracle.RK2_MIDPOINT)
    f = -(np.roll(u0, -1) ** 2 - np.roll(u0, 1) ** 2) / (4 * dx)
    assert np.max(np.abs((u1 - u0) / dt - f)) < 1e-10


@pytest.mark.parametrize("rk2", [oracle.RK2_MIDPOINT, oracle.RK2_HEUN])
def test_p6_rational_brute_force(rk2):
    rng = np.random.default_rng(13)
    N, steps = 9, 2
    u0 = rng.uniform(-1, 1, N)
    dx, dt = 0.5, 0.005
    DX, DT = Fraction(dx), Fraction(dt)

    def f(u, i):  # right-hand side of (C.2) as printed (with reading X2 for the sign of 2u_i)
        p1, m1 = u[(i + 1) % N], u[(i - 1) % N]
        p2, m2 = u[(i + 2) % N], u[(i - 2) % N]
        return -((p1 * p1 - m1 * m1) / (4 * DX) + (p1 + m1 - 2 * u[i]) / DX ** 2
                 + (p2 - 4 * p1 + 6 * u[i] - 4 * m1 + m2) / DX ** 4)

    u = [Fraction(x) for x in u0]
    for _ in range(steps):
        if rk2 == oracle.RK2_MIDPOINT:
            us = [u[i] + DT / 2 * f(u, i) for i in range(N)]       # (C.3)
            u = [u[i] + DT * f(us, i) for i in range(N)]           # (C.4)
        else:
            us = [u[i] + DT * f(u, i) for i in range(N)]
            u = [(u[i] + us[i] + DT * f(us, i)) / 2 for i in range(N)]
    got = oracle.run(oracle.KS, u0, N, steps, dx, dt, rk2=rk2)
    ref = np.array([float(x) for x in u])
    # the largest term is 6 u / dx^4 * dt ~ 0.5: a few ulp of that
    assert np.max(np.abs(got - ref)) < 64 * np.finfo(float).eps


def test_fp32_instantiation_tracks_fp64():
    w = si.ks_cos(512, 3, 50)
    u64 = oracle.run_workload(w)
    u32 = oracle.run_workload(w, dtype=np.float32)
    assert 0 < np.max(np.abs(u32 - u64)) < 1e-3


def test_periodic_initial_data_variant():
    # ADVICE r1 / reading X12: the literal config's smooth part jumps by O(1) at the wrap; the periodic variant does not
    lit = si.ks_cos(4096, 1, 10, noise=0.0)
    per = si.ks_cos(4096, 1, 10, noise=0.0, periodic=True)
    assert abs(lit.u0[0] - lit.u0[-1]) > 1.0
    assert abs(per.u0[0] - per.u0[-1]) < 0.05
    for w in (lit, per):   # both stay bounded under the scheme (the jump is damped, |G| = 0.52 at Nyquist)
        out = oracle.run_workload(w, nsteps=400)
        assert np.all(np.isfinite(out)) and np.max(np.abs(out)) < 5.0
