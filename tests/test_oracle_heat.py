"""Pins for the heat oracle (Eq. B.4) against things that are NOT the oracle.

P1 closed form (north_star: exact discrete FTCS amplification factor g = 1 - 4 r sin^2(k dx / 2)),
P2 exact binomial response of a unit delta at r = 1/4 (bit-exact, also pins the periodic wrap),
P3 Nyquist / constant modes, P4 conservation of the mean + discrete maximum principle,
P6 brute-force rational evaluation of Eq. (B.4) as printed, N <= 16.
"""
from fractions import Fraction
from math import comb

import numpy as np
import pytest

import oracle
import swept_inputs as si


def closed_form_heat(amps, N, M, r):
    i = np.arange(N, dtype=np.float64)
    u = np.zeros(N)
    for k, a in enumerate(amps, start=1):
        s2 = np.sin(np.pi * k / N) ** 2
        g_pow = np.exp(M * np.log1p(-4.0 * r * s2))  # g^M without M*eps error
        u += a * g_pow * np.sin(2.0 * np.pi * k * i / N)
    return u


def test_p1_config1_closed_form():
    w = si.config(1)  # N=2048, 8 modes, 20000 steps: the whole of config 1
    u = oracle.run_workload(w)
    ref = closed_form_heat(w.meta["amps"], w.N, w.nsteps, w.meta["r"])
    assert np.max(np.abs(u - ref)) <= 1e-11 * np.max(np.abs(w.u0))
    # the solution must actually have decayed by a non-trivial, mode-dependent amount
    assert 0.05 < np.max(np.abs(u)) / np.max(np.abs(w.u0)) < 0.999


@pytest.mark.parametrize("N,modes,steps", [(64, 16, 500), (4096, 16, 3000)])
def test_p1_closed_form_other_sizes(N, modes, steps):
    w = si.heat_sines(N, modes, si.BASE_SEED + 2, steps)
    u = oracle.run_workload(w)
    ref = closed_form_heat(w.meta["amps"], N, steps, 0.25)
    assert np.max(np.abs(u - ref)) <= 1e-11 * np.max(np.abs(w.u0))


def test_p1_single_mode_general_r():
    # a value of r that is not a power of two, one mode: per-step factor g exactly as north_star states
    N, k, r, M = 128, 5, 0.2, 40
    i = np.arange(N)
    u0 = np.sin(2 * np.pi * k * i / N)
    dx = 1.0 / N
    u = oracle.run(oracle.HEAT, u0, N, M, dx, r * dx * dx, alpha=1.0)
    g = 1.0 - 4.0 * r * np.sin(np.pi * k / N) ** 2
    assert np.max(np.abs(u - g ** M * u0)) < 1e-13


@pytest.mark.parametrize("N", [5, 8, 16])
@pytest.mark.parametrize("s", [1, 2, 7, 26])
def test_p2_delta_binomial_bit_exact(N, s):
    # r = 1/4: one step convolves with (1/4, 1/2, 1/4); s steps give C(2s, s+j)/4^s, wrapped mod N
    pos = 3
    u0 = np.zeros(N)
    u0[pos] = 1.0
    dx = 1.0 / N
    u = oracle.run(oracle.HEAT, u0, N, s, dx, 0.25 * dx * dx)
    exp = np.zeros(N)
    for j in range(-s, s + 1):
        exp[(pos + j) % N] += comb(2 * s, s + j) / 4.0 ** s  # dyadic: exact in binary64 for s <= 26
    assert np.array_equal(u, exp)


def test_p3_nyquist_and_constant_exact():
    N = 32
    dx = 1.0 / N
    ny = (-1.0) ** np.arange(N)
    assert np.array_equal(oracle.run(oracle.HEAT, ny, N, 1, dx, 0.25 * dx * dx), np.zeros(N))
    const = np.full(N, 0.3)
    assert np.array_equal(oracle.run(oracle.HEAT, const, N, 100, dx, 0.25 * dx * dx), const)


def test_p4_mean_conserved_and_max_principle():
    rng = np.random.default_rng(7)
    N = 1000  # not a power of two: the periodic wrap is not a mask
    u0 = rng.uniform(-1, 1, N)
    dx = 1.0 / N
    u = oracle.run(oracle.HEAT, u0, N, 300, dx, 0.4 * dx * dx)
    assert abs(u.mean() - u0.mean()) < 1e-15 * np.sqrt(N)
    assert u.min() >= u0.min() and u.max() <= u0.max()


def test_p6_rational_brute_force():
    # Eq. (B.4) literally, in exact rationals, with periodic indexing
    rng = np.random.default_rng(11)
    N, steps = 11, 3
    u0 = rng.uniform(-1, 1, N)
    alpha, dx = 0.7, 0.1
    dt = 0.3 * dx * dx / alpha
    Fo = Fraction(alpha) * Fraction(dt) / (Fraction(dx) * Fraction(dx))
    u = [Fraction(x) for x in u0]
    for _ in range(steps):
        u = [Fo * (u[(i + 1) % N] + u[(i - 1) % N]) + (1 - 2 * Fo) * u[i] for i in range(N)]
    got = oracle.run(oracle.HEAT, u0, N, steps, dx, dt, alpha=alpha)
    assert np.max(np.abs(got - np.array([float(x) for x in u]))) < 8 * np.finfo(float).eps


# ---- FP32 instantiation (the checker of north_star's 1e-5 gate, reading X15): pinned to the BIT, not to "close to FP64"
def round_to_binary32(fr):
    """Nearest-even rounding of an exact rational to IEEE binary32 (normal range), by integer arithmetic."""
    fr = Fraction(fr)
    if fr == 0:
        return np.float32(0.0)
    sign, a = (-1 if fr < 0 else 1), abs(fr)
    e = a.numerator.bit_length() - a.denominator.bit_length()
    if Fraction(2) ** e > a:
        e -= 1
    assert Fraction(2) ** e <= a < Fraction(2) ** (e + 1) and -126 <= e <= 127
    q = a / Fraction(2) ** (e - 23)          # in [2^23, 2^24)
    n = q.numerator // q.denominator
    rem = q - n
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and n % 2 == 1):
        n += 1
    return np.float32(sign * float(Fraction(n) * Fraction(2) ** (e - 23)))   # exact in double, exact in float


@pytest.mark.parametrize("N", [5, 8, 16])
@pytest.mark.parametrize("s", [1, 2, 7, 11])
def test_p2_delta_binomial_bit_exact_fp32(N, s):
    # C(2s, s+j) < 2^24 for s <= 11 (and every partial sum of a step is such a dyadic), so binary32 is exact too
    pos = 2
    u0 = np.zeros(N, dtype=np.float32)
    u0[pos] = 1.0
    dx = 1.0 / N
    u = oracle.run(oracle.HEAT, u0, N, s, dx, 0.25 * dx * dx, dtype=np.float32)
    exp = np.zeros(N)
    for j in range(-s, s + 1):
        exp[(pos + j) % N] += comb(2 * s, s + j) / 4.0 ** s
    assert u.dtype == np.float32 and np.array_equal(u.astype(np.float64), exp)


def test_p3_nyquist_and_constant_exact_fp32():
    N = 32
    dx = 1.0 / N
    ny = ((-1.0) ** np.arange(N)).astype(np.float32)
    assert np.array_equal(oracle.run(oracle.HEAT, ny, N, 1, dx, 0.25 * dx * dx, dtype=np.float32), np.zeros(N, np.float32))
    const = np.full(N, 0.3, dtype=np.float32)
    assert np.array_equal(oracle.run(oracle.HEAT, const, N, 100, dx, 0.25 * dx * dx, dtype=np.float32), const)


def test_p6_fp32_rational_and_bit_level_emulation():
    # Eq. (B.4) with r != 2^-k on 11 points, three steps, float data:
    # (a) against the exact rational value of B.4 applied to the float inputs with the once-rounded constants:
    #     within a few binary32 ulps — a wrong sign, term, index or a constant built from rounded pieces fails;
    # (b) bit for bit against B.4 evaluated with correctly rounded binary32 operations built from integer
    #     arithmetic (sum, product, ONE rounding for the fused multiply-add, SURVEY.md §8(c) F-heat): a double
    #     intermediate, a missing fusion or a twice-rounded constant in the float instantiation fails.
    rng = np.random.default_rng(12)
    N, steps = 11, 3
    u0 = rng.uniform(-1, 1, N).astype(np.float32)
    alpha, dx = 0.7, 0.1
    dt = 0.3 * dx * dx / alpha
    Fo_d = alpha * dt / (dx * dx)                       # double, as the F-rules say; rounded ONCE to float
    Fo, c0 = Fraction(float(np.float32(Fo_d))), Fraction(float(np.float32(1.0 - 2.0 * Fo_d)))
    exact = [Fraction(float(x)) for x in u0]
    emu = [Fraction(float(x)) for x in u0]
    for _ in range(steps):
        exact = [Fo * (exact[(i + 1) % N] + exact[(i - 1) % N]) + c0 * exact[i] for i in range(N)]
        nxt = []
        for i in range(N):
            ssum = Fraction(float(round_to_binary32(emu[(i - 1) % N] + emu[(i + 1) % N])))
            t = Fraction(float(round_to_binary32(c0 * emu[i])))
            nxt.append(Fraction(float(round_to_binary32(Fo * ssum + t))))
        emu = nxt
    got = oracle.run(oracle.HEAT, u0, N, steps, dx, dt, alpha=alpha, dtype=np.float32)
    assert got.dtype == np.float32
    ulp = np.finfo(np.float32).eps
    assert np.max(np.abs(got.astype(np.float64) - np.array([float(x) for x in exact]))) < 6 * ulp
    assert np.array_equal(got.astype(np.float64), np.array([float(x) for x in emu]))


def test_fp32_instantiation_tracks_fp64():
    w = si.heat_sines(256, 16, 3, 200)
    u64 = oracle.run_workload(w)
    u32 = oracle.run_workload(w, dtype=np.float32)
    assert u32.dtype == np.float32
    assert np.max(np.abs(u32 - u64)) < 1e-4 * np.max(np.abs(u64))
    assert np.max(np.abs(u32 - u64)) > 0  # really computed in float


def test_thread_count_does_not_change_bits():
    w = si.heat_sines(1 << 15, 16, 5, 20)
    nt = oracle.num_threads()
    try:
        oracle.set_num_threads(1)
        a = oracle.run_workload(w)
        oracle.set_num_threads(max(2, nt))
        b = oracle.run_workload(w)
    finally:
        oracle.set_num_threads(nt)
    assert np.array_equal(a, b)
