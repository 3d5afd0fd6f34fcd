"""Pins of the oracle's Euler stepping with Dirichlet ends: the end states of the tube are held at
their initial values.  None re-types the oracle: (1) while no disturbance has reached an end, the run must equal the
PERIODIC oracle (pinned in test_oracle_euler.py) on the double tube, bit for bit; (2) a uniform state is a fixed
point; (3) mass and energy are conserved and the momentum grows by exactly dt/dx (p_left - p_right) per step while
the ends are undisturbed (flux balance of the conservation law D.1 with the end fluxes (0, p, 0))."""
import numpy as np
import pytest

import oracle
import swept_inputs as si


@pytest.mark.parametrize("rk2", [si.RK2_MIDPOINT, si.RK2_HEUN])
def test_equals_periodic_double_tube_while_ends_undisturbed(rk2):
    # periodic double Sod on 2N cells: (1,1) on [N/2, 3N/2).  Its cells [N, 2N) are a single Sod tube (high left, low
    # right).  The scheme moves information 4 cells per timestep (two stages x 2 cells), the nearest other
    # diaphragm is N/2 cells from either end of that range: identical bits for fewer than N/8 steps
    N = 256
    steps = N // 8 - 2
    w = si.euler_sod(N, steps, rk2=rk2)
    dbl = si.euler_double_sod(2 * N, steps, rk2=rk2)
    assert np.array_equal(dbl.u0.reshape(3, -1)[:, N:], w.u0.reshape(3, -1))
    got = oracle.run_workload(w).reshape(3, N)
    per = oracle.run(oracle.EULER, dbl.u0, 2 * N, steps, w.dx, w.dt, gamma=w.gamma, rk2=rk2).reshape(3, 2 * N)
    assert np.array_equal(got, per[:, N:])
    assert not np.array_equal(got, w.u0.reshape(3, N))        # something did happen at the diaphragm


def test_uniform_state_is_a_fixed_point():
    N = 64
    q = np.concatenate([np.full(N, 0.7), np.full(N, 0.21), np.full(N, 2.3)])
    out = oracle.run(oracle.EULER, q, N, 25, 1.0 / N, 0.1 / N, bc=1)
    assert np.array_equal(out, q)


@pytest.mark.parametrize("rk2", [si.RK2_MIDPOINT, si.RK2_HEUN])
def test_flux_balance_at_the_ends(rk2):
    N, steps = 512, 50
    w = si.euler_sod(N, steps, rk2=rk2)
    q0 = w.u0.reshape(3, N)
    q = oracle.run_workload(w).reshape(3, N)
    lam = w.dt / w.dx
    assert abs(q[0].sum() - q0[0].sum()) <= 1e-12 * q0[0].sum()
    assert abs(q[2].sum() - q0[2].sum()) <= 1e-12 * q0[2].sum()
    assert abs(q[1].sum() - steps * lam * (1.0 - 0.1)) <= 1e-12 * steps
    # the ends themselves have not moved yet
    assert np.array_equal(q[:, :8], q0[:, :8]) and np.array_equal(q[:, -8:], q0[:, -8:])


def test_late_time_stays_physical_and_ends_hold():
    # long after the waves reached the ends: finite, positive density/pressure, ghost states still imposed
    N = 128
    w = si.euler_sod(N, 600)
    q = oracle.run_workload(w).reshape(3, N)
    assert np.all(np.isfinite(q)) and q[0].min() > 0
    p = 0.4 * (q[2] - 0.5 * q[1] ** 2 / q[0])
    assert p.min() > 0
