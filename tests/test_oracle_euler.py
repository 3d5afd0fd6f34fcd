"""Pins for the Euler oracle (Eqs. D.1-D.12; RK2 per PAPER.md:418).

P7 conservation of total mass / momentum / energy, uniform-state fixed point, exact mirror symmetry of the
   double Sod tube;
P8 the star region of the Sod problem (the paper's canonical case) against an independent
   textbook exact Riemann solver (pins flux, sign of (D.12) = reading X1, pressure law = X4, wave speeds);
advected density wave: convergence to the exact solution rho0(x - u t) (pins mass flux and dt/dx);
pressure-jump special case of the Roe-averaged spectral radius (reading X3, partial pin);
P9 50-digit evaluation of (D.4)-(D.12) as printed on N <= 16 including limiter-off and r > 1 cells.
"""
import mpmath as mp
import numpy as np
import pytest

import oracle
import swept_inputs as si

G = 1.4


def split(q, N):
    return q[:N], q[N:2 * N], q[2 * N:]


def prim(q, N):
    rho, M, E = split(q, N)
    u = M / rho
    return rho, u, (G - 1) * (E - 0.5 * M * u)


@pytest.mark.parametrize("rk2", [oracle.RK2_MIDPOINT, oracle.RK2_HEUN])
def test_p7_conservation_and_mirror(rk2):
    w = si.config(4, N=1 << 11, nsteps=3000, rk2=rk2)  # long enough for the waves to collide
    q = oracle.run_workload(w)
    N = w.N
    for a, b in zip(split(q, N), split(w.u0, N)):
        assert abs(a.sum() - b.sum()) <= 4e-15 * N * max(1.0, np.max(np.abs(b)))
    rho, M, E = split(q, N)
    assert np.array_equal(rho, rho[::-1])
    assert np.array_equal(M, -M[::-1])
    assert np.array_equal(E, E[::-1])
    r, u, p = prim(q, N)
    assert r.min() > 0.1 and p.min() > 0.05 and np.max(np.abs(u)) > 0.3
    # reading X11: realised CFL stays well below 1
    assert np.max(np.abs(u) + np.sqrt(G * p / r)) * w.dt / w.dx < 0.6


def test_p7_uniform_state_is_fixed_point():
    N = 16
    q0 = np.concatenate([np.full(N, 0.7), np.full(N, 0.7 * 0.3), np.full(N, 2.0)])
    q = oracle.run(oracle.EULER, q0, N, 25, 1.0 / N, 0.1 / N)
    assert np.array_equal(q, q0)


def exact_riemann_star(rl, ul, pl, rr, ur, pr, g=G):
    """Textbook exact Riemann solver (two-shock/rarefaction pressure function, Newton iteration)."""
    cl, cr = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)

    def fk(p, rk, pk, ck):
        if p > pk:  # shock
            A, B = 2.0 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            return (p - pk) * np.sqrt(A / (p + B)), np.sqrt(A / (p + B)) * (1 - 0.5 * (p - pk) / (p + B))
        return (2 * ck / (g - 1)) * ((p / pk) ** ((g - 1) / (2 * g)) - 1), (1.0 / (rk * ck)) * (p / pk) ** (-(g + 1) / (2 * g))

    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dfl = fk(p, rl, pl, cl)
        fr, dfr = fk(p, rr, pr, cr)
        dp = (fl + fr + (ur - ul)) / (dfl + dfr)
        p -= dp
        if abs(dp) < 1e-14:
            break
    fl, _ = fk(p, rl, pl, cl)
    fr, _ = fk(p, rr, pr, cr)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    # densities either side of the contact
    rsl = rl * (p / pl) ** (1 / g) if p <= pl else rl * ((p / pl + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * p / pl + 1))
    rsr = rr * (p / pr) ** (1 / g) if p <= pr else rr * ((p / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * p / pr + 1))
    shock_speed = ur + cr * np.sqrt((g + 1) / (2 * g) * p / pr + (g - 1) / (2 * g))
    return p, u, rsl, rsr, shock_speed


@pytest.mark.parametrize("rk2", [oracle.RK2_MIDPOINT, oracle.RK2_HEUN])
def test_p8_sod_star_region(rk2):
    N = 4096
    t_end = 0.1  # before the shocks meet at x = 0 (t = 0.143) and the rarefactions at x = 0.5 (t = 0.211)
    w = si.config(4, N=N, nsteps=0, rk2=rk2)
    nsteps = int(round(t_end / w.dt))
    q = oracle.run_workload(w, nsteps=nsteps)
    t = nsteps * w.dt
    ps, us, rsl, rsr, ss = exact_riemann_star(1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    assert abs(ps - 0.30313) < 1e-4 and abs(us - 0.92745) < 1e-4 and abs(rsr - 0.26557) < 1e-4
    r, u, p = prim(q, N)
    x = (np.arange(N) + 0.5) / N
    x0 = 0.75  # right diaphragm: cell faces at j = 3N/4
    # between contact and shock
    sel = (x > x0 + us * t + 0.02) & (x < x0 + ss * t - 0.02)
    assert sel.sum() > 50
    assert np.max(np.abs(p[sel] - ps)) < 2e-3
    assert np.max(np.abs(u[sel] - us)) < 3e-3
    assert np.max(np.abs(r[sel] - rsr)) < 3e-3
    # between rarefaction tail and contact
    c_star_l = np.sqrt(G * ps / rsl)
    sel = (x > x0 + (us - c_star_l) * t + 0.02) & (x < x0 + us * t - 0.02)
    assert sel.sum() > 20
    assert np.max(np.abs(r[sel] - rsl)) < 3e-3 and np.max(np.abs(p[sel] - ps)) < 2e-3
    # shock location: density crosses the mid value within a few cells of the exact position
    right = x > x0 + us * t + 0.03
    xs = x[right][np.argmin(np.abs(r[right] - 0.5 * (rsr + 0.125)))]
    assert abs(xs - (x0 + ss * t)) < 6.0 / N + 1e-3
    # undisturbed states remain
    assert abs(r[np.argmin(np.abs(x - 0.97))] - 0.125) < 1e-12
    assert abs(r[np.argmin(np.abs(x - 0.5))] - 1.0) < 1e-12


@pytest.mark.parametrize("rk2", [oracle.RK2_MIDPOINT, oracle.RK2_HEUN])
def test_advected_density_wave_converges(rk2):
    errs = []
    for N in (64, 128, 256):
        x = (np.arange(N) + 0.5) / N
        rho = 1.0 + 0.2 * np.sin(2 * np.pi * x)
        vel, p = 1.0, 1.0
        q0 = np.concatenate([rho, rho * vel, p / (G - 1) + 0.5 * rho * vel * vel])
        dx = 1.0 / N
        dt = 0.2 * dx
        steps = int(round(0.25 / dt))
        q = oracle.run(oracle.EULER, q0, N, steps, dx, dt, gamma=G, rk2=rk2)
        exact = 1.0 + 0.2 * np.sin(2 * np.pi * (x - vel * steps * dt))
        errs.append(np.max(np.abs(q[:N] - exact)))
    assert errs[2] < 0.02
    assert 1.5 < errs[0] / errs[1] < 4.5 and 1.5 < errs[1] / errs[2] < 4.5


def test_spectral_radius_pressure_jump_special_case():
    """rho_L = rho_R, u = 0, isolated pressure jump between cells k and k+1.  On the initial data the limiter
    is off on both sides of the jump (pressure ratios are 0 or inf), so the interface flux is
    0.5 (F_L + F_R + r_sp (Q_L - Q_R)) with first-order states and the energy flux is 0.5 r_sp (E_L - E_R).
    With equal densities reading X3 reduces to the closed form r_sp^2 = (c_L^2 + c_R^2) / 2.

    The first-stage flux divergence f(q0) is recovered exactly from two full steps that share the same
    predictor q* = q0 + (dt/2) f(q0):  midpoint(dt) = q0 + dt f(q*),  Heun(dt/2) = q0 + (dt/4)(f(q0) + f(q*))."""
    N, k = 16, 7
    rho = np.ones(N)
    p = np.where(np.arange(N) <= k, 1.0, 0.4)
    E = p / (G - 1)
    q0 = np.concatenate([rho, np.zeros(N), E])
    dx, dt = 1.0, 2.0 ** -10
    mid = oracle.run(oracle.EULER, q0, N, 1, dx, dt, gamma=G, rk2=oracle.RK2_MIDPOINT)
    heun = oracle.run(oracle.EULER, q0, N, 1, dx, dt / 2, gamma=G, rk2=oracle.RK2_HEUN)
    f0 = 4.0 * (heun - q0) / dt - (mid - q0) / dt
    dE = f0[2 * N + k]                          # = -(Flux_E(k+1/2) - Flux_E(k-1/2)) / dx,  Flux_E(k-1/2) = 0
    rsp = -dE * 2.0 / (E[k] - E[k + 1])
    cl2, cr2 = G * 1.0 / 1.0, G * 0.4 / 1.0
    assert abs(rsp - np.sqrt(0.5 * (cl2 + cr2))) < 1e-9
    # mass: 0.5 r_sp (rho_L - rho_R) = 0; momentum: 0.5 (P_L + P_R) - P_L
    assert abs(f0[k]) < 1e-9 and abs(f0[N + k] - 0.3) < 1e-9


def mp_step(q0, N, dx, dt, rk2, g):
    """(D.4)-(D.12) as printed, 50 digits, periodic."""
    mp.mp.dps = 50
    g = mp.mpf(g)
    Q = [[mp.mpf(float(q0[c * N + j])) for j in range(N)] for c in range(3)]

    def stage(V, base, hs):
        P = [(g - 1) * (V[2][j] - V[1][j] ** 2 / V[0][j] / 2) for j in range(N)]          # (D.4)

        def lim(num, den):
            if den == 0:
                return mp.mpf(0)  # ratio is inf or 0/0: "otherwise" branch of (D.7)/(D.8)
            r = num / den
            return min(r, 1) / 2 if r > 0 else mp.mpf(0)

        F = [[None] * N for _ in range(3)]
        for k in range(N):
            kp, km, kpp = (k + 1) % N, (k - 1) % N, (k + 2) % N
            phiL = lim(P[kp] - P[k], P[k] - P[km])            # P_r at k           (D.6), (D.7)
            phiR = lim(P[kp] - P[k], P[kpp] - P[kp])          # 1/P_r at k+1       (D.8)
            QL = [V[c][k] + phiL * (V[c][kp] - V[c][k]) for c in range(3)]
            QR = [V[c][kp] + phiR * (V[c][k] - V[c][kp]) for c in range(3)]

            def flux(S):
                u = S[1] / S[0]
                Pp = (g - 1) * (S[2] - S[0] * u * u / 2)
                return [S[1], S[0] * u * u + Pp, u * (S[2] + Pp)], u, S[2] / S[0]         # (D.3)

            FL, uL, eL = flux(QL)
            FR, uR, eR = flux(QR)
            sL, sR = mp.sqrt(QL[0]), mp.sqrt(QR[0])
            usp = (sL * uL + sR * uR) / (sL + sR)                                        # (D.10), X3
            esp = (sL * eL + sR * eR) / (sL + sR)
            rsp = mp.sqrt(g * (g - 1) * (esp - usp * usp / 2)) + abs(usp)                 # (D.11)
            for c in range(3):
                F[c][k] = (FR[c] + FL[c] + rsp * (QL[c] - QR[c])) / 2                     # (D.9)
        return [[base[c][j] - hs * (F[c][j] - F[c][(j - 1) % N]) for j in range(N)] for c in range(3)]

    lam = mp.mpf(dt) / mp.mpf(dx)
    if rk2 == oracle.RK2_MIDPOINT:
        Qs = stage(Q, Q, lam / 2)
        Qn = stage(Qs, Q, lam)
    else:
        Qs = stage(Q, Q, lam)
        Qt = stage(Qs, Qs, lam)
        Qn = [[(Q[c][j] + Qt[c][j]) / 2 for j in range(N)] for c in range(3)]
    return np.array([float(Qn[c][j]) for c in range(3) for j in range(N)])


@pytest.mark.parametrize("rk2", [oracle.RK2_MIDPOINT, oracle.RK2_HEUN])
def test_p9_mpmath_brute_force(rk2):
    N = 14
    q0 = si.random_smooth(si.EULER, N, 99)
    rho, M, E = q0[:N].copy(), q0[N:2 * N].copy(), q0[2 * N:].copy()
    # cells 3,4 identical -> P_4 - P_3 = 0 exactly: limiter-off (division by zero) paths are exercised
    rho[4], M[4], E[4] = rho[3], M[3], E[3]
    q0 = np.concatenate([rho, M, E])
    dx, dt = 0.1, 0.01
    got = oracle.run(oracle.EULER, q0, N, 1, dx, dt, gamma=G, rk2=rk2)
    ref = mp_step(q0, N, dx, dt, rk2, G)
    assert np.max(np.abs(got - ref) / np.maximum(1.0, np.abs(ref))) < 1e-14
    # the data set exercises both limiter regimes: some pressure ratios > 1, some in (0,1), some <= 0
    _, _, p = prim(q0, N)
    d = np.roll(p, -1) - p
    with np.errstate(divide="ignore", invalid="ignore"):
        r = d / np.roll(d, 1)
    assert (r > 1).any() and ((r > 0) & (r < 1)).any() and (r <= 0).any()


def test_fp32_instantiation_tracks_fp64():
    w = si.config(4, N=256, nsteps=100)
    q64 = oracle.run_workload(w)
    q32 = oracle.run_workload(w, dtype=np.float32)
    assert 0 < np.max(np.abs(q32 - q64)) < 2e-2  # the limiter switches make float rounding visible
