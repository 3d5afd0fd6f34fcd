"""Pins of the oracle's insulated-end heat stepping, Eq. (B.5) PAPER.md:328-331 (T_{-1} = T_1, T_N = T_{N-2}).

None of them re-types the oracle's loop: (1) the even extension turns the problem into the PERIODIC one (already
pinned in test_oracle_heat.py) on 2(N-1) points; (2) cosines are eigenmodes with a closed-form factor; (3) the
trapezoid-weighted sum is conserved; (4) exact rational hand expansion on 5 points; (5) a delta at the wall."""
from fractions import Fraction

import numpy as np

import oracle
import swept_inputs as si


def test_even_extension_equals_periodic_problem_bitwise():
    # mirror about the end points: period 2(N-1); u_{-j} = u_j.  The stencil sum um + up is commutative, so the
    # two computations agree bit for bit, for any data (no symmetry of the data needed beyond the extension)
    rng = np.random.default_rng(7)
    for N, steps in ((5, 3), (9, 20), (33, 100), (257, 300)):
        u0 = rng.uniform(-1, 1, N)
        ext = np.concatenate([u0, u0[-2:0:-1]])            # 0..N-1, N-2..1
        assert ext.size == 2 * (N - 1)
        dx = 1.0 / (N - 1)
        dt = 0.25 * dx * dx
        got = oracle.run(oracle.HEAT, u0, N, steps, dx, dt, bc=1)
        per = oracle.run(oracle.HEAT, ext, ext.size, steps, dx, dt)
        assert np.array_equal(got, per[:N])
        assert np.array_equal(per[N:], per[N - 2:0:-1])    # the periodic run stays mirror symmetric


def test_cosine_modes_closed_form():
    # cos(pi k i/(N-1)) is an eigenvector of the mirrored FTCS matrix with g = 1 - 4 r sin^2(pi k/(2(N-1)))
    w = si.heat_insulated(129, 6, 11, 4000)
    i = np.arange(w.N)
    amps, r = w.meta["amps"], w.meta["r"]
    exact = np.full(w.N, amps[0])
    for k in range(1, len(amps)):
        g = 1.0 - 4.0 * r * np.sin(np.pi * k / (2 * (w.N - 1))) ** 2
        exact += amps[k] * np.exp(w.nsteps * np.log(g)) * np.cos(np.pi * k * i / (w.N - 1))
    got = oracle.run_workload(w)
    assert np.max(np.abs(got - exact)) <= 1e-11 * np.max(np.abs(w.u0))


def test_trapezoid_sum_conserved_and_constant_fixed():
    rng = np.random.default_rng(3)
    N = 100
    u0 = rng.uniform(0, 1, N)
    dx = 1.0 / (N - 1)
    got = oracle.run(oracle.HEAT, u0, N, 5000, dx, 0.25 * dx * dx, bc=1)
    trap = lambda u: u[1:-1].sum() + 0.5 * (u[0] + u[-1])   # noqa: E731
    assert abs(trap(got) - trap(u0)) <= 1e-12 * N
    assert u0.min() <= got.min() and got.max() <= u0.max()   # maximum principle, r <= 1/2
    c = np.full(N, 0.375)
    assert np.array_equal(oracle.run(oracle.HEAT, c, N, 50, dx, 0.25 * dx * dx, bc=1), c)


def test_hand_expansion_exact_rationals_N5():
    # two steps on 5 points, r = 1/4, written out point by point with the mirrored neighbours of (B.5)
    u = [Fraction(x) for x in (3, -1, 4, 1, -5)]
    r = Fraction(1, 4)

    def step(v):
        return [r * (v[1] + v[1]) + (1 - 2 * r) * v[0],
                r * (v[0] + v[2]) + (1 - 2 * r) * v[1],
                r * (v[1] + v[3]) + (1 - 2 * r) * v[2],
                r * (v[2] + v[4]) + (1 - 2 * r) * v[3],
                r * (v[3] + v[3]) + (1 - 2 * r) * v[4]]
    ref = step(step(u))
    dx = 0.25
    got = oracle.run(oracle.HEAT, np.array([float(x) for x in u]), 5, 2, dx, 0.25 * dx * dx, bc=1)
    assert [Fraction(float(g)) for g in got] == ref          # dyadic rationals: exact in binary


def test_delta_at_the_wall_reflects():
    # a unit delta at point 0 with r = 1/4: after one step (1/2, 1/4, 0, ...): the wall keeps 1 - 2r, gives r to its
    # single neighbour; the mirrored stencil doubles what comes back: step 2 at point 0 = 1/2 * 1/2 + 1/4 * (1/4 + 1/4)
    N = 8
    u0 = np.zeros(N)
    u0[0] = 1.0
    dx = 1.0 / (N - 1)
    one = oracle.run(oracle.HEAT, u0, N, 1, dx, 0.25 * dx * dx, bc=1)
    assert one[0] == 0.5 and one[1] == 0.25 and not one[2:].any()
    two = oracle.run(oracle.HEAT, u0, N, 2, dx, 0.25 * dx * dx, bc=1)
    assert two[0] == 0.375 and two[1] == 0.25 and two[2] == 0.0625
