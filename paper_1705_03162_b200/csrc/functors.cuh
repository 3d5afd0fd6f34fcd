// functors.cuh — stencil functors for the three test problems of PAPER.md §5.2.
//
// Each functor advances P contiguous points by ONE sub-timestep ("tier") from a window of the previous
// tier.  The same functor is used by the per-step kernels and by every swept kernel, so all variants
// evaluate identical IEEE-754 expression trees (compiled with -fmad=false; every fused multiply-add
// below is explicit) and are bit-identical to one another ("the same operations in a different order and
// location").
//
//   win [c][k], k = 0 .. P+2H-1 : stage input (tier t-1) at points x0-H .. x0+P-1+H, component c
//   base[c][j], j = 0 .. P-1    : value at tier t-2 (= u^n) for the final stage; for the predictor
//                                 stage the caller passes the window centre (tier t-1 = u^n)
//   odd                         : global tier index modulo SIGMA.  Two-stage schemes: 1 = predictor sub-timestep
//                                 (odd tier), 0 = final sub-timestep (odd tiers hold predictor
//                                 values, even tiers final values).  Three-stage scheme (KS3): 1, 2 = first and
//                                 second stage, 0 = final stage.  base is u^n whenever odd != 1.
//   ROWS                        : rows of the inter-launch state (tier modulo ROWS); u^n lives in row 0
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace swept {

__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
// x = fma(a, b, c) where rel <= span (unsigned), x unchanged elsewhere: the same fma.rn, issued under a predicate, so that a
// register-resident tier (swept_cluster.cuh) needs no select between its arithmetic and the next tier's shuffle
__device__ __forceinline__ void fma_if_(double& x, double a, double b, double c, unsigned rel, unsigned span) {
  asm("{\n\t.reg .pred p;\n\tsetp.le.u32 p, %4, %5;\n\t@p fma.rn.f64 %0, %1, %2, %3;\n\t}"
      : "+d"(x) : "d"(a), "d"(b), "d"(c), "r"(rel), "r"(span));
}
__device__ __forceinline__ void fma_if_(float& x, float a, float b, float c, unsigned rel, unsigned span) {
  asm("{\n\t.reg .pred p;\n\tsetp.le.u32 p, %4, %5;\n\t@p fma.rn.f32 %0, %1, %2, %3;\n\t}"
      : "+f"(x) : "f"(a), "f"(b), "f"(c), "r"(rel), "r"(span));
}
__device__ __forceinline__ double sqrt_(double a) { return sqrt(a); }
__device__ __forceinline__ float sqrt_(float a) { return sqrtf(a); }
__device__ __forceinline__ double fabs_(double a) { return fabs(a); }
__device__ __forceinline__ float fabs_(float a) { return fabsf(a); }
__device__ __forceinline__ double fmin_(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float fmin_(float a, float b) { return fminf(a, b); }
template <class R> __device__ __forceinline__ R inf_();
template <> __device__ __forceinline__ double inf_<double>() { return __longlong_as_double(0x7ff0000000000000LL); }
template <> __device__ __forceinline__ float inf_<float>() { return __int_as_float(0x7f800000); }

// a / b, bit for bit the IEEE round-to-nearest quotient, arranged so that the common special operand does not leave
// the fast path of the division.  nvcc expands an FP64 division into a reciprocal refinement (about 10 FP64
// instructions) followed by a range check that sends a ZERO or tiny numerator, a zero / infinite / NaN operand or a
// subnormal quotient to a subroutine of several dozen instructions.  A gas at rest has zero momentum in every cell, so
// in the undisturbed part of the Sod tube (most of the domain for most of a run) every velocity M / rho went through
// that subroutine.  The quotient of a zero by a finite non-zero number is a signed zero with the sign of the product:
// a * b yields exactly that.  Every other case still runs the division itself.
template <class R>
__device__ __forceinline__ R div_(R a, R b) {
  const bool zero = a == (R)0 && fabs_(b) > (R)0 && fabs_(b) < inf_<R>();
  const R q = (zero ? (R)1 : a) / b;
  return zero ? a * b : q;
}

// Scheme constants, computed once on the host in double and rounded once to REAL (host side: api).
template <class R>
struct Consts {
  R a0, a1, a2, a3, a4;  // meaning per problem, see each functor
};

// Boundary treatment handed to the kernels (include/swept.h SWEPT_BC_*): 0 periodic; 1 mirror about the end points
// (insulated heat ends, Eq. (B.5)); 2 Dirichlet: ghost cells hold the end states l / r at every
// stage (Euler tube).
enum { BC_WRAP = 0, BC_MIRROR = 1, BC_FIXED = 2 };
template <class R>
struct BcVals {
  R l[3], r[3];
};

// ---------------------------------------------------------------------------------------------
// Heat, FTCS, Eq. (B.4):  T_i^{m+1} = Fo (T_{i+1} + T_{i-1}) + (1 - 2 Fo) T_i
//   a0 = Fo = alpha dt / dx^2,  a1 = 1 - 2 Fo
template <class R_>
struct Heat {
  using R = R_;
  static constexpr int H = 1, C = 1, SIGMA = 1, ROWS = 2;
  static constexpr int MAX_THREADS = 1024;  // per CTA, for __launch_bounds__ (register budget)
  static constexpr int TIER_MAX_THREADS = 1024;
  __device__ __forceinline__ static R point(R um, R u0, R up, const Consts<R>& k) {
    const R s = um + up;
    const R t = k.a1 * u0;
    return fma_(k.a0, s, t);
  }
  template <int P>
  __device__ __forceinline__ static void stage(const R (&win)[C][P + 2 * H], const R (&base)[C][P],
                                               R (&out)[C][P], int /*odd*/, const Consts<R>& k) {
#pragma unroll
    for (int j = 0; j < P; ++j) out[0][j] = point(win[0][j], win[0][j + 1], win[0][j + 2], k);
  }
  // the same stage written into dst where point j's relative tier lies in its window (rel[j] <= span[j]); the other
  // points of dst keep their values.  Same expression tree as point(): the last operation alone carries the predicate.
  static constexpr bool HAS_STAGE_IF = true;
  template <int P>
  __device__ __forceinline__ static void stage_if(const R (&win)[C][P + 2 * H], const R (&/*base*/)[C][P],
                                                  R (&dst)[C][P], int /*odd*/, const Consts<R>& k,
                                                  const unsigned (&rel)[P], const unsigned (&span)[P]) {
#pragma unroll
    for (int j = 0; j < P; ++j) {
      const R s = win[0][j] + win[0][j + 2];
      const R t = k.a1 * win[0][j + 1];
      fma_if_(dst[0][j], k.a0, s, t, rel[j], span[j]);
    }
  }
};

// ---------------------------------------------------------------------------------------------
// Kuramoto-Sivashinsky, Eq. (C.2) PAPER.md:342 (sign of 2u_i per reading X2), RK2 (C.3)/(C.4)
// PAPER.md:348-354.   a0 = 1/(4dx), a1 = 1/dx^2, a2 = 1/dx^4, a3 = dt, a4 = dt/2;  heun = template flag
template <class R_, int HEUN>
struct KS {
  using R = R_;
  static constexpr int H = 2, C = 1, SIGMA = 2, ROWS = 2;
  static constexpr int MAX_THREADS = 1024;
  static constexpr int TIER_MAX_THREADS = 1024;
  __device__ __forceinline__ static R rhs(R vm2, R vm1, R v0, R vp1, R vp2, const Consts<R>& k) {
    const R s1 = vp1 + vm1;
    const R s2 = vp2 + vm2;
    const R q = fma_(-vm1, vm1, vp1 * vp1);
    const R lap = fma_((R)-2, v0, s1);
    const R bih = fma_((R)6, v0, fma_((R)-4, s1, s2));
    return fma_(k.a2, bih, fma_(k.a1, lap, k.a0 * q));
  }
  // one point; base = u^n_i (tier t-2) for the final stage, = v0 for the predictor
  __device__ __forceinline__ static R point(R vm2, R vm1, R v0, R vp1, R vp2, R base, int odd,
                                            const Consts<R>& k) {
    const R f = rhs(vm2, vm1, v0, vp1, vp2, k);
    if (HEUN) {
      const R t = fma_(-k.a3, f, v0);            // v + dt f(v)
      return odd ? t : (R)0.5 * (base + t);      // predictor: u* ; final: (u^n + u* + dt f(u*))/2
    } else {
      const R hs = odd ? k.a4 : k.a3;            // (C.3) dt/2 ; (C.4) dt
      const R b = odd ? v0 : base;
      return fma_(-hs, f, b);
    }
  }
  template <int P>
  __device__ __forceinline__ static void stage(const R (&win)[C][P + 2 * H], const R (&base)[C][P],
                                               R (&out)[C][P], int odd, const Consts<R>& k) {
#pragma unroll
    for (int j = 0; j < P; ++j)
      out[0][j] = point(win[0][j], win[0][j + 1], win[0][j + 2], win[0][j + 3], win[0][j + 4],
                        base[0][j], odd, k);
  }
};

// ---------------------------------------------------------------------------------------------
// KS3 — a scheme with THREE sub-timesteps per timestep (the decomposition
// "must be adjusted ... when there are more than two sub-timesteps per timestep"): Eq. (C.2) advanced by the
// three-stage Shu-Osher SSP Runge-Kutta method, every stage on the same 5-point stencil,
//     u1 = u^n + dt f(u^n);   u2 = 3/4 u^n + 1/4 (u1 + dt f(u1));   u^{n+1} = 1/3 u^n + 2/3 (u2 + dt f(u2)).
// The final stage reads u^n three tiers back, which the paper's two-row working array has overwritten by then
// (Fig. 3): the state has ROWS = 3 rows (tier modulo 3), u^n in row 0.   Constants as KS (a3 = dt).
template <class R_>
struct KS3 {
  using R = R_;
  static constexpr int H = 2, C = 1, SIGMA = 3, ROWS = 3;
  static constexpr int MAX_THREADS = 1024;
  static constexpr int TIER_MAX_THREADS = 1024;
  __device__ __forceinline__ static R point(R vm2, R vm1, R v0, R vp1, R vp2, R base, int st, const Consts<R>& k) {
    const R f = KS<R, 0>::rhs(vm2, vm1, v0, vp1, vp2, k);
    const R e = fma_(-k.a3, f, v0);                                   // v + dt f(v)
    if (st == 1) return e;
    if (st == 2) return fma_((R)0.25, e, (R)0.75 * base);
    return fma_((R)(2.0 / 3.0), e, (R)(1.0 / 3.0) * base);
  }
  template <int P>
  __device__ __forceinline__ static void stage(const R (&win)[C][P + 2 * H], const R (&base)[C][P],
                                               R (&out)[C][P], int st, const Consts<R>& k) {
#pragma unroll
    for (int j = 0; j < P; ++j)
      out[0][j] = point(win[0][j], win[0][j + 1], win[0][j + 2], win[0][j + 3], win[0][j + 4], base[0][j], st, k);
  }
};

// ---------------------------------------------------------------------------------------------
// Euler, second-order finite volume, Eqs. (D.3)-(D.12) PAPER.md:366-416 (readings X1, X3, X4, X5).
//   a0 = gamma - 1, a1 = gamma (gamma - 1), a2 = dt/dx, a3 = dt/(2dx)
template <class R_, int HEUN>
struct Euler {
  using R = R_;
  static constexpr int H = 2, C = 3, SIGMA = 2, ROWS = 2;
  static constexpr int MAX_THREADS = 256;  // ~250 live registers per thread (P:270 'greater low-level memory usage')
  static constexpr int TIER_MAX_THREADS = 1024;  // the TIER kernel shares pressures and fluxes: 64 registers

  __device__ __forceinline__ static R pressure(R rho, R M, R E, const Consts<R>& k) {  // (D.4), X4
    const R u = div_(M, rho);
    return k.a0 * fma_(-((R)0.5 * M), u, E);
  }
  // min(r,1)/2 if 0 < r < inf else 0 (D.7)/(D.8), written with comparisons only: 0.5 * fmin(r, 1) is 0.5 r below 1 and
  // 0.5 from 1 on; NaN fails every comparison and gives 0
  __device__ __forceinline__ static R half_minmod(R r) {
    const R half_r = (R)0.5 * r;
    const R v = r < (R)1 ? half_r : (R)0.5;
    return (r > (R)0 && r < inf_<R>()) ? v : (R)0;
  }
  // half_minmod(num / den).  Where the pressure is flat num or den is exactly zero and the quotient is 0, NaN or
  // +-inf, each of which the limiter maps to 0: decided here, and the division runs on harmless operands instead of
  // falling into its special-case subroutine (see div_).  NaN operands still reach the division.
  __device__ __forceinline__ static R limiter(R num, R den) {
    const bool flat = num == (R)0 || den == (R)0;
    const R r = (flat ? (R)1 : num) / (flat ? (R)1 : den);
    return flat ? (R)0 : half_minmod(r);
  }
  // flux at the interface between cells k (state vl) and k+1 (state vr);
  // dm = P_k - P_{k-1}, d0 = P_{k+1} - P_k, dp = P_{k+2} - P_{k+1}
  __device__ __forceinline__ static void flux(const R (&vl)[3], const R (&vr)[3], R dm, R d0, R dp,
                                              R (&F)[3], const Consts<R>& k) {
    const R phiL = limiter(d0, dm);  // P_r at cell k (D.6)
    const R phiR = limiter(d0, dp);  // 1/P_r at cell k+1 as the swapped quotient (X5)
    R QL[3], QR[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const R dq = vr[c] - vl[c];
      QL[c] = fma_(phiL, dq, vl[c]);   // (D.7)
      QR[c] = fma_(-phiR, dq, vr[c]);  // (D.8)
    }
    const R uL = div_(QL[1], QL[0]);
    const R PL = k.a0 * fma_(-((R)0.5 * QL[1]), uL, QL[2]);
    const R eL = QL[2] / QL[0];
    const R uR = div_(QR[1], QR[0]);
    const R PR = k.a0 * fma_(-((R)0.5 * QR[1]), uR, QR[2]);
    const R eR = QR[2] / QR[0];
    const R FL0 = QL[1], FL1 = fma_(QL[1], uL, PL), FL2 = uL * (QL[2] + PL);  // (D.3)
    const R FR0 = QR[1], FR1 = fma_(QR[1], uR, PR), FR2 = uR * (QR[2] + PR);
    const R sL = sqrt_(QL[0]), sR = sqrt_(QR[0]);
    const R den = sL + sR;
    const R usp = div_(sL * uL + sR * uR, den);  // (D.10), X3; products then one add: L<->R symmetric
    const R esp = (sL * eL + sR * eR) / den;
    const R c2 = k.a1 * fma_(-((R)0.5 * usp), usp, esp);
    const R rsp = sqrt_(c2) + fabs_(usp);     // (D.11)
    F[0] = (R)0.5 * fma_(rsp, QL[0] - QR[0], FR0 + FL0);  // (D.9)
    F[1] = (R)0.5 * fma_(rsp, QL[1] - QR[1], FR1 + FL1);
    F[2] = (R)0.5 * fma_(rsp, QL[2] - QR[2], FR2 + FL2);
  }
  // one component of one cell: v = stage input, base = u^n, dF = Flux_{j+1/2} - Flux_{j-1/2}
  __device__ __forceinline__ static R update(R v, R base, R dF, int odd, const Consts<R>& k) {
    if (HEUN) {
      const R t = fma_(-k.a2, dF, v);                   // v + dt f(v)
      return odd ? t : (R)0.5 * (base + t);
    } else {
      const R hs = odd ? k.a3 : k.a2;                    // (D.12) with X1 (minus)
      const R b = odd ? v : base;
      return fma_(-hs, dF, b);
    }
  }
  template <int P>
  __device__ __forceinline__ static void stage(const R (&win)[C][P + 2 * H], const R (&base)[C][P],
                                               R (&out)[C][P], int odd, const Consts<R>& k) {
    R pr[P + 4];
#pragma unroll
    for (int j = 0; j < P + 4; ++j) pr[j] = pressure(win[0][j], win[1][j], win[2][j], k);
    R d[P + 3];
#pragma unroll
    for (int j = 0; j < P + 3; ++j) d[j] = pr[j + 1] - pr[j];
    // interface i (i = 0..P) lies between window cells i+1 and i+2  (cell j of the output = window j+2)
    R Fprev[3];
#pragma unroll
    for (int i = 0; i <= P; ++i) {
      const R vl[3] = {win[0][i + 1], win[1][i + 1], win[2][i + 1]};
      const R vr[3] = {win[0][i + 2], win[1][i + 2], win[2][i + 2]};
      R F[3];
      flux(vl, vr, d[i], d[i + 1], d[i + 2], F, k);
      if (i > 0) {
        const int j = i - 1;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          out[c][j] = update(win[c][j + 2], base[c][j], F[c] - Fprev[c], odd, k);
        }
      }
#pragma unroll
      for (int c = 0; c < 3; ++c) Fprev[c] = F[c];
    }
  }
};

}  // namespace swept
