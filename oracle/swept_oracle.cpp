// swept_oracle.cpp — CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code, header, table or constant generator with the
// CUDA library under paper_1705_03162_b200/; neither side includes or imports the other.
//
// What it computes: plain timestep-by-timestep explicit time stepping of the paper's three 1-D
// test problems on a periodic grid, i.e. the *definition* of the result the swept rule must reach
// ("the swept rule performs the same operations in a different order and location",
// PAPER.md:37, §2).  No tiles, no phases, no blocking, no fusion: one full sweep over i per
// (sub-)timestep, ping-pong arrays.
//
//   heat  : FTCS, Eq. (B.4), PAPER.md:325 (App. B)                     — 3-point, 1 stage / step
//   KS    : central 2nd-order, Eq. (C.2), midpoint RK2
//           Eqs. (C.3)-(C.4) PAPER.md:348-354 (App. C)                 — 5-point, 2 stages / step
//   Euler : 2nd-order finite volume, Eqs. (D.3)-(D.12) PAPER.md:366-416,
//           RK2 "with the same procedure" as (C.3)-(C.4), PAPER.md:418 — 5-point, 2 stages / step
//   KS3   : Eq. (C.2) advanced by the three-stage Shu-Osher SSP-RK3 (row f3: "more than two
//           sub-timesteps per timestep")                  — 5-point, 3 stages / step
//
// Readings of garbled / silent / ambiguous passages (all listed in DESIGN.md §3):
//   X1  (D.12) update is Q - dt/dx (F_{i+1/2} - F_{i-1/2}) (conservation law D.1).
//   X2  (B.3, C.2) second difference is u_{i+1} - 2u_i + u_{i-1}.
//   X3  (D.10) Roe average: sqrt(rho)-weighted u and e = E/rho; P_sp by (D.4).
//       PARITY UNPINNED beyond its L=R reduction (c + |u|) and the Sod/convergence pins.
//   X4  (D.2/D.4) third conserved component is total energy per volume E;
//       P = (gamma-1)(E - M^2/(2 rho)).
//   X5  (D.8) "(P_r)^-1" is the swapped quotient (P_i - P_{i-1})/(P_{i+1} - P_i).
//       PARITY UNPINNED (any reading with the same 0/inf/NaN classes is the same scheme in exact
//       arithmetic away from those classes).
//   X6  RK2 flavour: midpoint (the paper's) and Heun (BASELINE.json config 4) both provided.
//   X10 periodic boundaries for all three problems (BASELINE.json configs); the paper's own heat
//       boundary condition, insulated ends (B.5) PAPER.md:328-331, is available as bc = 1:
//       T_{-1} = T_1 and T_N = T_{N-2} for points 0..N-1 (mirror about the end POINTS; the paper's
//       index "n+1" is read with points 0..n).  Euler: Dirichlet ends, bc = 1: ghost cells
//       -2, -1 / N, N+1 hold the initial state of the first / last cell at every stage.
//
// Floating point: every expression below is a fixed tree of IEEE-754 operations.  Build with
// -ffp-contract=off so the compiler never fuses a*b+c on its own; the fused operations that ARE
// part of the tree are written std::fma.  Constants are computed once, in double, from
// (dx, dt, params) and rounded once to REAL.  OpenMP splits the i-loops only (each i independent,
// so the result does not depend on the thread count).
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): closed-form FTCS amplification factor,
// exact binomial delta response, Nyquist/constant modes, conservation, KS linear growth factor and
// PDE-consistency of the nonlinear term, Euler conservation / mirror symmetry / uniform fixed
// point / exact-Riemann Sod star state / advected-wave convergence, brute-force rational stencils.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// below this size a parallel region costs more than the loop (thread count never changes results)
constexpr int64_t OMP_MIN_N = 16384;

inline int64_t wrap(int64_t i, int64_t N) {
    i %= N;
    return i < 0 ? i + N : i;
}

// ---------------------------------------------------------------- heat, Eq. (B.4)
// T_i^{m+1} = Fo (T_{i+1} + T_{i-1}) + (1 - 2 Fo) T_i
// bc = 0: periodic neighbours.  bc = 1: insulated ends, Eq. (B.5): T_{-1} = T_1, T_N = T_{N-2}.
inline int64_t heat_nb(int64_t i, int64_t N, int bc) {
    if (bc == 0) return wrap(i, N);
    if (i < 0) return -i;
    if (i >= N) return 2 * (N - 1) - i;
    return i;
}

template <class R>
void heat_run(R* u, int64_t N, int64_t nsteps, double dx, double dt, double alpha, int bc = 0) {
    const double Fo_d = alpha * dt / (dx * dx);  // Fourier number
    const R Fo = (R)Fo_d;
    const R c0 = (R)(1.0 - 2.0 * Fo_d);
    std::vector<R> buf((size_t)N);
    R* a = u;
    R* b = buf.data();
    for (int64_t s = 0; s < nsteps; ++s) {
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
        for (int64_t i = 0; i < N; ++i) {
            const R um = a[heat_nb(i - 1, N, bc)], u0 = a[i], up = a[heat_nb(i + 1, N, bc)];
            const R sum = um + up;
            const R t = c0 * u0;
            b[i] = std::fma(Fo, sum, t);
        }
        R* tmp = a; a = b; b = tmp;
    }
    if (a != u) std::memcpy(u, a, sizeof(R) * (size_t)N);
}

// ---------------------------------------------------------------- KS, Eq. (C.2)
// rhs = -f = (u_{+1}^2 - u_{-1}^2)/(4dx) + (u_{+1} - 2u_0 + u_{-1})/dx^2
//          + (u_{+2} - 4u_{+1} + 6u_0 - 4u_{-1} + u_{-2})/dx^4
template <class R>
struct KSConst {
    R cx, cxx, cxxxx, dt, half_dt;
};

template <class R>
inline R ks_rhs(const R* v, int64_t i, int64_t N, const KSConst<R>& k) {
    const R vm2 = v[wrap(i - 2, N)], vm1 = v[wrap(i - 1, N)], v0 = v[i];
    const R vp1 = v[wrap(i + 1, N)], vp2 = v[wrap(i + 2, N)];
    const R s1 = vp1 + vm1;
    const R s2 = vp2 + vm2;
    const R q = std::fma(-vm1, vm1, vp1 * vp1);
    const R lap = std::fma((R)-2, v0, s1);
    const R bih = std::fma((R)6, v0, std::fma((R)-4, s1, s2));
    return std::fma(k.cxxxx, bih, std::fma(k.cxx, lap, k.cx * q));
}

template <class R>
void ks_run(R* u, int64_t N, int64_t nsteps, double dx, double dt, int rk2) {
    KSConst<R> k;
    k.cx = (R)(1.0 / (4.0 * dx));
    k.cxx = (R)(1.0 / (dx * dx));
    k.cxxxx = (R)(1.0 / ((dx * dx) * (dx * dx)));
    k.dt = (R)dt;
    k.half_dt = (R)(0.5 * dt);
    std::vector<R> us((size_t)N), un((size_t)N);
    R* a = u;
    R* b = un.data();
    R* p = us.data();
    for (int64_t s = 0; s < nsteps; ++s) {
        if (rk2 == 0) {  // midpoint, Eqs. (C.3), (C.4) PAPER.md:348-354
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
            for (int64_t i = 0; i < N; ++i) p[i] = std::fma(-k.half_dt, ks_rhs(a, i, N, k), a[i]);
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
            for (int64_t i = 0; i < N; ++i) b[i] = std::fma(-k.dt, ks_rhs(p, i, N, k), a[i]);
        } else {  // Heun: u* = u + dt f(u);  u^{n+1} = (u + (u* + dt f(u*)))/2   (reading X6)
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
            for (int64_t i = 0; i < N; ++i) p[i] = std::fma(-k.dt, ks_rhs(a, i, N, k), a[i]);
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
            for (int64_t i = 0; i < N; ++i) {
                const R t = std::fma(-k.dt, ks_rhs(p, i, N, k), p[i]);
                b[i] = (R)0.5 * (a[i] + t);
            }
        }
        R* tmp = a; a = b; b = tmp;
    }
    if (a != u) std::memcpy(u, a, sizeof(R) * (size_t)N);
}

// ---------------------------------------------------------------- KS with THREE sub-timesteps per timestep
// SURVEY.md §8(f) row f3.  The paper stops at two sub-timesteps per timestep and says the decomposition "must be
// adjusted ... when there are more than two sub-timesteps per timestep" and "adjusted further" beyond four
// (PAPER.md:103-115 on sub-timesteps that all use the minimum stencil).  The scheme taken for that
// row: the same spatial discretisation (C.2) advanced by the three-stage strong-stability-preserving Runge-Kutta
// method of Shu and Osher (a textbook scheme, not in the paper), every stage on the same 5-point stencil:
//     u1      = u^n + dt f(u^n)
//     u2      = 3/4 u^n + 1/4 (u1 + dt f(u1))
//     u^{n+1} = 1/3 u^n + 2/3 (u2 + dt f(u2))
// Stage s reads the previous stage on the stencil and u^n at its own point (s-1 sub-timesteps back): with three
// sub-timesteps the paper's two-row working array would have overwritten it (the conflict of PAPER.md Fig. 3).
// Canonical trees:  e = fma(-dt, rhs(v), v) with rhs of F-KS;  stage 1: e;  stage 2: fma(1/4, e, (3/4) u^n);
// stage 3: fma(c23, e, c13 u^n) with c13 = REAL(1.0/3.0), c23 = REAL(2.0/3.0) (rounded once, like every constant).
// Pins: tests/test_oracle_ks3.py (growth polynomial 1 + z + z^2/2 + z^3/6, third-order convergence in dt,
// conservation of the mean, PDE consistency, exact-rational hand expansion).
template <class R>
void ks3_run(R* u, int64_t N, int64_t nsteps, double dx, double dt) {
    KSConst<R> k;
    k.cx = (R)(1.0 / (4.0 * dx));
    k.cxx = (R)(1.0 / (dx * dx));
    k.cxxxx = (R)(1.0 / ((dx * dx) * (dx * dx)));
    k.dt = (R)dt;
    k.half_dt = (R)(0.5 * dt);
    const R c14 = (R)0.25, c34 = (R)0.75, c13 = (R)(1.0 / 3.0), c23 = (R)(2.0 / 3.0);
    std::vector<R> s1((size_t)N), s2((size_t)N), un((size_t)N);
    R* a = u;
    R* b = un.data();
    R* p = s1.data();
    R* q = s2.data();
    for (int64_t s = 0; s < nsteps; ++s) {
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
        for (int64_t i = 0; i < N; ++i) p[i] = std::fma(-k.dt, ks_rhs(a, i, N, k), a[i]);
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
        for (int64_t i = 0; i < N; ++i) {
            const R e = std::fma(-k.dt, ks_rhs(p, i, N, k), p[i]);
            q[i] = std::fma(c14, e, c34 * a[i]);
        }
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
        for (int64_t i = 0; i < N; ++i) {
            const R e = std::fma(-k.dt, ks_rhs(q, i, N, k), q[i]);
            b[i] = std::fma(c23, e, c13 * a[i]);
        }
        R* tmp = a; a = b; b = tmp;
    }
    if (a != u) std::memcpy(u, a, sizeof(R) * (size_t)N);
}

// ---------------------------------------------------------------- Euler, Eqs. (D.3)-(D.12)
template <class R>
struct EulerConst {
    R gm1, ggm1;
};

// Eq. (D.4) PAPER.md:372 with reading X4:  P = (gamma-1)(E - M^2/(2 rho)),  u = M/rho
template <class R>
inline R pressure(R rho, R M, R E, const EulerConst<R>& c) {
    const R u = M / rho;
    return c.gm1 * std::fma(-((R)0.5 * M), u, E);
}

// limiter factor min(r,1)/2 if 0 < r < inf else 0 — Eqs. (D.7)/(D.8) PAPER.md:386-390
template <class R>
inline R half_minmod(R r) {
    const R inf = std::numeric_limits<R>::infinity();
    return (r > (R)0 && r < inf) ? (R)0.5 * std::fmin(r, (R)1) : (R)0;
}

// One stage: out = acc_base - hs * (Flux_{j+1/2} - Flux_{j-1/2}), flux evaluated on state V.
//   V, base, out: component-major arrays rho[N], M[N], E[N].
template <class R>
void euler_stage(const R* V, const R* base, R* out, int64_t N, R hs, const EulerConst<R>& c,
                 std::vector<R>& P, std::vector<R>& F) {
    const R* rho = V;
    const R* mom = V + N;
    const R* ene = V + 2 * N;
    // pressure in every cell, Eq. (D.4)
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
    for (int64_t j = 0; j < N; ++j) P[(size_t)j] = pressure(rho[j], mom[j], ene[j], c);
    // flux at every interface k+1/2 (between cells k and k+1), Eqs. (D.6)-(D.11)
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
    for (int64_t k = 0; k < N; ++k) {
        const int64_t km = wrap(k - 1, N), kp = wrap(k + 1, N), kpp = wrap(k + 2, N);
        const R dm = P[(size_t)k] - P[(size_t)km];     // P_k     - P_{k-1}
        const R d0 = P[(size_t)kp] - P[(size_t)k];     // P_{k+1} - P_k
        const R dp = P[(size_t)kpp] - P[(size_t)kp];   // P_{k+2} - P_{k+1}
        const R rL = d0 / dm;                          // P_r at cell k,     Eq. (D.6)
        const R rRinv = d0 / dp;                       // 1/P_r at cell k+1, reading X5
        const R phiL = half_minmod(rL);
        const R phiR = half_minmod(rRinv);
        R QL[3], QR[3];
        for (int cpt = 0; cpt < 3; ++cpt) {
            const R vl = V[cpt * N + k], vr = V[cpt * N + kp];
            const R dq = vr - vl;
            QL[cpt] = std::fma(phiL, dq, vl);          // Eq. (D.7)
            QR[cpt] = std::fma(-phiR, dq, vr);         // Eq. (D.8)
        }
        // physical fluxes, Eq. (D.3)
        const R uL = QL[1] / QL[0];
        const R PL = c.gm1 * std::fma(-((R)0.5 * QL[1]), uL, QL[2]);
        const R eL = QL[2] / QL[0];
        const R uR = QR[1] / QR[0];
        const R PR = c.gm1 * std::fma(-((R)0.5 * QR[1]), uR, QR[2]);
        const R eR = QR[2] / QR[0];
        const R FL[3] = {QL[1], std::fma(QL[1], uL, PL), uL * (QL[2] + PL)};
        const R FR[3] = {QR[1], std::fma(QR[1], uR, PR), uR * (QR[2] + PR)};
        // Roe-averaged spectral radius, Eqs. (D.10)-(D.11) PAPER.md:404-411, reading X3
        const R sL = std::sqrt(QL[0]), sR = std::sqrt(QR[0]);
        const R den = sL + sR;
        const R usp = (sL * uL + sR * uR) / den;      // two products then one add: L<->R symmetric
        const R esp = (sL * eL + sR * eR) / den;
        const R c2 = c.ggm1 * std::fma(-((R)0.5 * usp), usp, esp);
        const R rsp = std::sqrt(c2) + std::fabs(usp);
        // Eq. (D.9)
        for (int cpt = 0; cpt < 3; ++cpt)
            F[(size_t)(cpt * N + k)] = (R)0.5 * std::fma(rsp, QL[cpt] - QR[cpt], FR[cpt] + FL[cpt]);
    }
    // Eq. (D.12) PAPER.md:415 with reading X1 (minus sign)
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
    for (int64_t j = 0; j < N; ++j) {
        const int64_t jm = wrap(j - 1, N);
        for (int cpt = 0; cpt < 3; ++cpt) {
            const R dF = F[(size_t)(cpt * N + j)] - F[(size_t)(cpt * N + jm)];
            out[cpt * N + j] = std::fma(-hs, dF, base[cpt * N + j]);
        }
    }
}

// Dirichlet ends ("The spatial boundary conditions are these values at their respective ends of
// the tube"): cells -2, -1 hold the initial state of cell 0 and cells N, N+1 that of cell N-1, at every stage.
// Implemented by running the very same euler_stage on arrays padded with those four ghost cells and made
// "periodic" over N+4 cells: the wrap-around then only ever couples ghost cells with each other (a ghost's
// update is discarded and the ghosts are re-imposed before every stage), and every interior cell j reads exactly
// cells j-2..j+2 of the padded array.
template <class R>
void euler_run_dirichlet(R* q, int64_t N, int64_t nsteps, double dx, double dt, double gamma, int rk2) {
    EulerConst<R> c;
    c.gm1 = (R)(gamma - 1.0);
    c.ggm1 = (R)(gamma * (gamma - 1.0));
    const double lam_d = dt / dx;
    const R lam = (R)lam_d, half_lam = (R)(0.5 * lam_d);
    const int64_t M = N + 4;
    const size_t m3 = (size_t)(3 * M);
    std::vector<R> qa(m3), qs(m3), qn(m3), P((size_t)M), F(m3);
    R left[3], right[3];
    for (int cpt = 0; cpt < 3; ++cpt) {
        left[cpt] = q[cpt * N];
        right[cpt] = q[cpt * N + N - 1];
        for (int64_t j = 0; j < N; ++j) qa[(size_t)(cpt * M + 2 + j)] = q[cpt * N + j];
    }
    auto impose = [&](R* v) {
        for (int cpt = 0; cpt < 3; ++cpt) {
            v[cpt * M + 0] = v[cpt * M + 1] = left[cpt];
            v[cpt * M + M - 2] = v[cpt * M + M - 1] = right[cpt];
        }
    };
    R* a = qa.data();
    R* b = qn.data();
    R* p = qs.data();
    for (int64_t s = 0; s < nsteps; ++s) {
        impose(a);
        if (rk2 == 0) {
            euler_stage(a, a, p, M, half_lam, c, P, F);
            impose(p);
            euler_stage(p, a, b, M, lam, c, P, F);
        } else {
            euler_stage(a, a, p, M, lam, c, P, F);
            impose(p);
            euler_stage(p, p, b, M, lam, c, P, F);
            for (int64_t j = 0; j < (int64_t)m3; ++j) b[j] = (R)0.5 * (a[j] + b[j]);
        }
        R* tmp = a; a = b; b = tmp;
    }
    for (int cpt = 0; cpt < 3; ++cpt)
        for (int64_t j = 0; j < N; ++j) q[cpt * N + j] = a[(size_t)(cpt * M + 2 + j)];
}

template <class R>
void euler_run(R* q, int64_t N, int64_t nsteps, double dx, double dt, double gamma, int rk2) {
    EulerConst<R> c;
    c.gm1 = (R)(gamma - 1.0);
    c.ggm1 = (R)(gamma * (gamma - 1.0));
    const double lam_d = dt / dx;
    const R lam = (R)lam_d, half_lam = (R)(0.5 * lam_d);
    const size_t n3 = (size_t)(3 * N);
    std::vector<R> qs(n3), qn(n3), P((size_t)N), F(n3);
    R* a = q;
    R* b = qn.data();
    R* p = qs.data();
    for (int64_t s = 0; s < nsteps; ++s) {
        if (rk2 == 0) {  // midpoint (PAPER.md:418 -> Eqs. C.3, C.4)
            euler_stage(a, a, p, N, half_lam, c, P, F);
            euler_stage(p, a, b, N, lam, c, P, F);
        } else {  // Heun (BASELINE.json config 4, reading X6)
            euler_stage(a, a, p, N, lam, c, P, F);
            euler_stage(p, p, b, N, lam, c, P, F);  // b = u* + dt f(u*)
#pragma omp parallel for schedule(static) if (N >= OMP_MIN_N)
            for (int64_t j = 0; j < (int64_t)n3; ++j) b[j] = (R)0.5 * (a[j] + b[j]);
        }
        R* tmp = a; a = b; b = tmp;
    }
    if (a != q) std::memcpy(q, a, sizeof(R) * n3);
}

}  // namespace

extern "C" {

// All entry points: in-place on a caller-owned host array; return 0, or -1 on bad arguments.
int oracle_heat_f64(double* u, int64_t N, int64_t nsteps, double dx, double dt, double alpha) {
    if (!u || N < 3 || nsteps < 0) return -1;
    heat_run<double>(u, N, nsteps, dx, dt, alpha);
    return 0;
}
int oracle_heat_f32(float* u, int64_t N, int64_t nsteps, double dx, double dt, double alpha) {
    if (!u || N < 3 || nsteps < 0) return -1;
    heat_run<float>(u, N, nsteps, dx, dt, alpha);
    return 0;
}
// heat with an explicit boundary condition: bc = 0 periodic, 1 insulated (B.5)
int oracle_heat_bc_f64(double* u, int64_t N, int64_t nsteps, double dx, double dt, double alpha, int bc) {
    if (!u || N < 3 || nsteps < 0 || bc < 0 || bc > 1) return -1;
    heat_run<double>(u, N, nsteps, dx, dt, alpha, bc);
    return 0;
}
int oracle_heat_bc_f32(float* u, int64_t N, int64_t nsteps, double dx, double dt, double alpha, int bc) {
    if (!u || N < 3 || nsteps < 0 || bc < 0 || bc > 1) return -1;
    heat_run<float>(u, N, nsteps, dx, dt, alpha, bc);
    return 0;
}
int oracle_ks_f64(double* u, int64_t N, int64_t nsteps, double dx, double dt, int rk2) {
    if (!u || N < 5 || nsteps < 0) return -1;
    ks_run<double>(u, N, nsteps, dx, dt, rk2);
    return 0;
}
int oracle_ks_f32(float* u, int64_t N, int64_t nsteps, double dx, double dt, int rk2) {
    if (!u || N < 5 || nsteps < 0) return -1;
    ks_run<float>(u, N, nsteps, dx, dt, rk2);
    return 0;
}
// KS, three sub-timesteps per timestep (SSP-RK3)
int oracle_ks3_f64(double* u, int64_t N, int64_t nsteps, double dx, double dt) {
    if (!u || N < 5 || nsteps < 0) return -1;
    ks3_run<double>(u, N, nsteps, dx, dt);
    return 0;
}
int oracle_euler_f64(double* q, int64_t N, int64_t nsteps, double dx, double dt, double gamma,
                     int rk2) {
    if (!q || N < 5 || nsteps < 0) return -1;
    euler_run<double>(q, N, nsteps, dx, dt, gamma, rk2);
    return 0;
}
int oracle_euler_f32(float* q, int64_t N, int64_t nsteps, double dx, double dt, double gamma,
                     int rk2) {
    if (!q || N < 5 || nsteps < 0) return -1;
    euler_run<float>(q, N, nsteps, dx, dt, gamma, rk2);
    return 0;
}
// Euler with Dirichlet ends = the initial states of the first and last cell
int oracle_euler_bc_f64(double* q, int64_t N, int64_t nsteps, double dx, double dt, double gamma, int rk2) {
    if (!q || N < 5 || nsteps < 0) return -1;
    euler_run_dirichlet<double>(q, N, nsteps, dx, dt, gamma, rk2);
    return 0;
}
int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

}  // extern "C"
