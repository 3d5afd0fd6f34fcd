"""Seeded synthetic input generators (shared by the oracle tests, the GPU parity tests and bench.py).

This module holds NONE of the method's arithmetic: it only builds initial data and the
(dx, dt, params) of a workload.  Both the CPU oracle (``oracle/``) and the CUDA library
(``paper_1705_03162_b200/``) are fed the *same host buffer* produced here, so no
PRNG or ``sin`` has to be bit-matched in two languages.

The paper (§6) runs three PDEs on N = 2^11..2^20 points, 50 000 steps, FP64, with
initial data it does not print (heat: unstated; KS "periodic initial condition" PAPER.md:356; Sod
PAPER.md:377 with Eq. D.5 missing from the text).  BASELINE.json's five configs fix shapes and
value distributions; the recipes below are those configs verbatim (readings X8, X11, X12, X13 in
DESIGN.md).  No public dataset is involved.

Base seed 170503162; config k uses seed + k.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 170503162

HEAT, KS, EULER, KS3 = 0, 1, 2, 3
RK2_MIDPOINT, RK2_HEUN = 0, 1
PROBLEM_NAMES = {HEAT: "heat", KS: "ks", EULER: "euler", KS3: "ks3"}
#: stencil half-width h, sub-timesteps per timestep sigma, components C
#: (KS3 = the KS discretisation advanced with three sub-timesteps per timestep)
PROBLEM_SHAPE = {HEAT: (1, 1, 1), KS: (2, 2, 1), EULER: (2, 2, 3), KS3: (2, 3, 1)}


@dataclass
class Workload:
    """One problem instance: everything `swept_create` / the oracle need, plus the initial data."""

    problem: int
    N: int
    dx: float
    dt: float
    nsteps: int
    u0: np.ndarray  # float64, shape (C*N,), component-major (Euler: rho[N], rho*u[N], E[N])
    alpha: float = 1.0
    gamma: float = 1.4
    rk2: int = RK2_MIDPOINT
    name: str = ""
    meta: dict = field(default_factory=dict)
    bc: int = 0  # 0 periodic (BASELINE.json configs); 1 = the paper's insulated heat ends, Eq. (B.5)

    @property
    def components(self) -> int:
        return PROBLEM_SHAPE[self.problem][2]


def heat_sines(N: int, nmodes: int, seed: int, nsteps: int, r: float = 0.25, alpha: float = 1.0,
               name: str = "") -> Workload:
    """Configs 1, 2 (reading X13): u0_i = sum_{k=1..K} a_k sin(2 pi k i / N), a_k ~ U(-1, 1).

    L = 1, dx = 1/N, dt = r dx^2 / alpha (so Fo = r; r = 0.25 is exact in binary).
    The amplitudes are returned in ``meta['amps']`` for the closed-form pin (P1).
    """
    rng = np.random.default_rng(seed)
    amps = rng.uniform(-1.0, 1.0, size=nmodes)
    i = np.arange(N, dtype=np.float64)
    u0 = np.zeros(N, dtype=np.float64)
    for k in range(1, nmodes + 1):
        u0 += amps[k - 1] * np.sin(2.0 * np.pi * k * i / N)
    dx = 1.0 / N
    dt = r * dx * dx / alpha
    return Workload(HEAT, N, dx, dt, nsteps, u0, alpha=alpha, name=name or f"heat_N{N}",
                    meta={"amps": amps, "r": r})


BC_PERIODIC, BC_PAPER = 0, 1


def heat_insulated(N: int, nmodes: int, seed: int, nsteps: int, r: float = 0.25, name: str = "") -> Workload:
    """The paper's own heat set-up: N points 0..N-1 with insulated ends (B.5), here with
    u0_i = a_0 + sum_{k=1..K} a_k cos(pi k i / (N-1)), a_k ~ U(-1, 1) — cosines are the eigenmodes of the
    mirrored stencil, so the closed form of the pin is g_k = 1 - 4 r sin^2(pi k / (2 (N-1))).  dx = 1/(N-1)."""
    rng = np.random.default_rng(seed)
    amps = rng.uniform(-1.0, 1.0, size=nmodes + 1)
    i = np.arange(N, dtype=np.float64)
    u0 = np.full(N, amps[0], dtype=np.float64)
    for k in range(1, nmodes + 1):
        u0 += amps[k] * np.cos(np.pi * k * i / (N - 1))
    dx = 1.0 / (N - 1)
    return Workload(HEAT, N, dx, r * dx * dx, nsteps, u0, name=name or f"heat_insulated_N{N}",
                    meta={"amps": amps, "r": r}, bc=BC_PAPER)


def ks_cos(N: int, seed: int, nsteps: int, dx: float = 0.5, dt: float = 0.005,
           noise: float = 1e-3, name: str = "", periodic: bool = False) -> Workload:
    """Config 3 (reading X12): u0 = cos(x/16)(1 + sin(x/16)) + noise * N(0,1), x_i = i dx.

    With the config's literal 1/16 the smooth part is NOT periodic over L = N dx (L / (32 pi) is not an integer): u0 has
    an O(1) jump at the wrap, which the scheme damps, whereas the paper speaks of a periodic initial condition
    (PAPER.md:356).  `periodic=True` replaces 1/16 by the nearest wavenumber 2 pi j / L, so that u0 is continuous
    across the boundary; the literal config stays the default (it is what BASELINE.json names)."""
    rng = np.random.default_rng(seed)
    x = np.arange(N, dtype=np.float64) * dx
    kappa = 1.0 / 16.0
    if periodic:
        L = N * dx
        kappa = 2.0 * np.pi * max(1, round(L / (32.0 * np.pi))) / L
    u0 = np.cos(kappa * x) * (1.0 + np.sin(kappa * x)) + noise * rng.standard_normal(N)
    return Workload(KS, N, dx, dt, nsteps, u0, rk2=RK2_MIDPOINT, name=name or f"ks_N{N}")


def ks3_cos(N: int, seed: int, nsteps: int, dx: float = 0.5, dt: float = 0.005, noise: float = 1e-3,
            name: str = "") -> Workload:
    """Row f3 (a scheme with three sub-timesteps per timestep): config 3's KS field and steps, advanced with the
    three-stage SSP Runge-Kutta method instead of the midpoint rule."""
    w = ks_cos(N, seed, nsteps, dx, dt, noise, name or f"ks3_N{N}")
    w.problem = KS3
    return w


def euler_double_sod(N: int, nsteps: int, rk2: int = RK2_HEUN, gamma: float = 1.4,
                     cfl: float = 0.4, lam_ref: float = 2.2, name: str = "") -> Workload:
    """Config 4 (readings X8, X11): periodic double Sod tube.

    (rho, u, p) = (1, 0, 1) on N/4 <= j < 3N/4 and (0.125, 0, 0.1) elsewhere; E = p/(gamma-1) at rest;
    dx = 1/N, dt = cfl * dx / lam_ref with the literal lam_ref = 2.2.  Deterministic (no RNG).
    """
    j = np.arange(N)
    mid = (j >= N // 4) & (j < 3 * N // 4)
    rho = np.where(mid, 1.0, 0.125)
    p = np.where(mid, 1.0, 0.1)
    mom = np.zeros(N)
    E = p / (gamma - 1.0)
    u0 = np.concatenate([rho, mom, E]).astype(np.float64)
    dx = 1.0 / N
    dt = cfl * dx / lam_ref
    return Workload(EULER, N, dx, dt, nsteps, u0, gamma=gamma, rk2=rk2, name=name or f"euler_N{N}")


def euler_sod(N: int, nsteps: int, rk2: int = RK2_MIDPOINT, gamma: float = 1.4, cfl: float = 0.4,
              lam_ref: float = 2.2, name: str = "") -> Workload:
    """The paper's own Sod tube (readings X8, X11): one diaphragm at N/2, (rho, u, p) = (1, 0, 1) left
    and (0.125, 0, 0.1) right, Dirichlet ends (bc = BC_PAPER), midpoint RK2."""
    j = np.arange(N)
    lft = j < N // 2
    rho = np.where(lft, 1.0, 0.125)
    p = np.where(lft, 1.0, 0.1)
    u0 = np.concatenate([rho, np.zeros(N), p / (gamma - 1.0)]).astype(np.float64)
    dx = 1.0 / N
    return Workload(EULER, N, dx, cfl * dx / lam_ref, nsteps, u0, gamma=gamma, rk2=rk2,
                    name=name or f"euler_sod_N{N}", bc=BC_PAPER)


def config(k: int, N: int | None = None, nsteps: int | None = None, problem: int | None = None,
           rk2: int | None = None) -> Workload:
    """BASELINE.json config k (1-based, as numbered in SURVEY.md §8(d)); N / nsteps may be overridden
    to pick one point of a config's sweep (or a reduced-length parity case)."""
    seed = BASE_SEED + k
    if k == 1:
        return heat_sines(N or 2048, 8, seed, 20000 if nsteps is None else nsteps, name="config1_heat")
    if k == 2:
        return heat_sines(N or (1 << 20), 16, seed, 10000 if nsteps is None else nsteps,
                          name="config2_heat")
    if k == 3:
        return ks_cos(N or (1 << 20), seed, 20000 if nsteps is None else nsteps, name="config3_ks")
    if k == 4:
        return euler_double_sod(N or (1 << 20), 5000 if nsteps is None else nsteps,
                                rk2=RK2_HEUN if rk2 is None else rk2, name="config4_euler")
    if k == 5:
        p = HEAT if problem is None else problem
        n_ = N or (1 << 20)
        ns = (50000 if n_ <= (1 << 20) else 5000) if nsteps is None else nsteps
        if p == HEAT:
            return heat_sines(n_, 16, seed, ns, name="config5_heat")
        if p == KS:
            return ks_cos(n_, seed, ns, name="config5_ks")
        return euler_double_sod(n_, ns, rk2=RK2_MIDPOINT if rk2 is None else rk2, name="config5_euler")
    raise ValueError(f"unknown config {k}")


def random_smooth(problem: int, N: int, seed: int) -> np.ndarray:
    """Generic bounded, positive-density random data for small parity / property cases."""
    rng = np.random.default_rng(seed)
    if problem == EULER:
        rho = 0.5 + rng.uniform(0.0, 1.0, N)
        vel = rng.uniform(-0.3, 0.3, N)
        p = 0.5 + rng.uniform(0.0, 1.0, N)
        E = p / 0.4 + 0.5 * rho * vel * vel
        return np.concatenate([rho, rho * vel, E])
    return rng.uniform(-1.0, 1.0, N)
