// per_step.cuh — the per-step ("Classic") kernel: one launch per sub-timestep, working array in global
// memory (Fig. 6).  SURVEY.md §8(a) row a0.
//
// B200 layout: each thread advances P contiguous points; the P-point body of the window is one (or two)
// 16-byte vector loads, the 2h halo values are scalar loads that hit L1 (they are the neighbours' bodies);
// the periodic wrap (PAPER.md:196-201 uses `& lastidx`, which needs N = 2^k) is a compare-and-add so any
// N divisible by P works.  Algorithmic traffic per point and sub-timestep: C*sizeof(R) read + the same
// written (+ the same again for the final stage's base read).
#pragma once
#include "functors.cuh"

namespace swept {

template <class R, int P>
__device__ __forceinline__ void load_vec(const R* __restrict__ p, R (&v)[P]) {
  if constexpr (sizeof(R) * P >= 16 && (sizeof(R) * P) % 16 == 0) {
    constexpr int NV = (int)(sizeof(R) * P / 16);
    const int4* q = reinterpret_cast<const int4*>(p);
    int4 t[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) t[i] = __ldg(q + i);
#pragma unroll
    for (int i = 0; i < NV; ++i) reinterpret_cast<int4*>(v)[i] = t[i];
  } else {
#pragma unroll
    for (int i = 0; i < P; ++i) v[i] = __ldg(p + i);
  }
}
template <class R, int P>
__device__ __forceinline__ void store_vec(R* __restrict__ p, const R (&v)[P]) {
  if constexpr (sizeof(R) * P >= 16 && (sizeof(R) * P) % 16 == 0) {
    constexpr int NV = (int)(sizeof(R) * P / 16);
#pragma unroll
    for (int i = 0; i < NV; ++i) reinterpret_cast<int4*>(p)[i] = reinterpret_cast<const int4*>(v)[i];
  } else {
#pragma unroll
    for (int i = 0; i < P; ++i) p[i] = v[i];
  }
}

// in: stage input (tier t-1), base: u^n (only read by the stages after the first: SIGMA >= 2 and odd != 1), out: tier t.
// odd = tier modulo SIGMA (functors.cuh).
template <class Prob, int P>
__global__ void __launch_bounds__(Prob::MAX_THREADS)
per_step_kernel(const typename Prob::R* __restrict__ in, const typename Prob::R* __restrict__ base,
                typename Prob::R* __restrict__ out, int64_t N, int odd, Consts<typename Prob::R> k, int bc, BcVals<typename Prob::R> bv) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C;
  const int64_t i0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * P;
  if (i0 >= N) return;
  alignas(16) R win[C][P + 2 * H];
  alignas(16) R bs[C][P];
  alignas(16) R o[C][P];
#pragma unroll
  for (int c = 0; c < C; ++c) {
    const R* src = in + (int64_t)c * N;
    alignas(16) R body[P];
    load_vec<R, P>(src + i0, body);
#pragma unroll
    for (int j = 0; j < P; ++j) win[c][H + j] = body[j];
#pragma unroll
    for (int j = 0; j < H; ++j) {
      int64_t il = i0 - H + j;
      const bool fix_l = bc == BC_FIXED && il < 0;       // Dirichlet ghost cells
      if (il < 0) il = bc ? -il : il + N;                // mirror: T_{-k} = T_k, T_{N-1+k} = T_{N-1-k} (B.5)
      int64_t ir = i0 + P + j;
      const bool fix_r = bc == BC_FIXED && ir >= N;
      if (ir >= N) ir = bc ? 2 * (N - 1) - ir : ir - N;
      win[c][j] = fix_l ? bv.l[c] : __ldg(src + il);
      win[c][H + P + j] = fix_r ? bv.r[c] : __ldg(src + ir);
    }
  }
  if (Prob::SIGMA >= 2 && odd != 1) {
#pragma unroll
    for (int c = 0; c < C; ++c) load_vec<R, P>(base + (int64_t)c * N + i0, bs[c]);
  } else {
#pragma unroll
    for (int c = 0; c < C; ++c)
#pragma unroll
      for (int j = 0; j < P; ++j) bs[c][j] = win[c][H + j];
  }
  Prob::template stage<P>(win, bs, o, odd, k);
#pragma unroll
  for (int c = 0; c < C; ++c) store_vec<R, P>(out + (int64_t)c * N + i0, o[c]);
}

// ---------------------------------------------------------------------------------------------------------
// Per-step kernel for a two-stage scalar scheme (KS), one launch per TIMESTEP (north_star allows "one launch per
// timestep or RK stage"): a thread reads the window of its P points widened by 2h on either side, evaluates the
// predictor stage on its P points and their h neighbours on either side (recomputed, not communicated), then
// the final stage on its P points.  Same Prob::stage trees as the two-launch form, so the same bits; half the
// launches and no predictor array in global memory (16 B instead of 40 B per point and timestep).
// SHFL = true takes the halo from the neighbouring lanes (large N: the kernel is then bound by memory, not by the L1
// tag stage); SHFL = false loads it (small N: one load latency instead of load + shuffle on the critical path of a
// launch that is over in two microseconds).
template <class Prob, int P, bool SHFL>
__global__ void __launch_bounds__(Prob::MAX_THREADS)
per_step_fused_kernel(const typename Prob::R* __restrict__ in, typename Prob::R* __restrict__ out, int64_t N,
                      Consts<typename Prob::R> k) {
  using R = typename Prob::R;
  constexpr int H = Prob::H;
  static_assert(Prob::C == 1 && Prob::SIGMA == 2, "fused two-stage kernel: scalar RK2 schemes");
  const int64_t i0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * P;
  constexpr int Q = P + 2 * H;  // points whose predictor value this thread needs
  alignas(16) R win[1][Q + 2 * H];
  alignas(16) R body[P];
  if constexpr (SHFL && P >= 2 * H && P % (2 * H) == 0) {
    // The 2h values either side are the neighbouring lanes' bodies: warp shuffles, not loads.  (With eight scalar
    // halo loads per thread this kernel was bound by the L1 tag stage — l1tex throughput 98 %, DRAM 44 % at N = 2^24,
    // profiles/r2_ks_per_step.md — although every one of them hit L1.)  Only the two end lanes of a warp, and a lane
    // whose neighbour lies beyond N, load their halo, as one vector; the whole warp stays for the shuffles.
    const bool valid = i0 < N;
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int j = 0; j < P; ++j) body[j] = (R)0;
    const bool edge_l = valid && lane == 0, edge_r = valid && (lane == 31 || i0 + P >= N);
    alignas(16) R left[2 * H], right[2 * H];
#pragma unroll
    for (int j = 0; j < 2 * H; ++j) left[j] = right[j] = (R)0;
    // all loads first, so that the end lanes' halo loads travel with the body loads instead of after the shuffles
    if (valid) load_vec<R, P>(in + i0, body);
    if (edge_l) load_vec<R, 2 * H>(in + (i0 >= 2 * H ? i0 - 2 * H : N - 2 * H), left);
    if (edge_r) load_vec<R, 2 * H>(in + (i0 + P < N ? i0 + P : 0), right);
#pragma unroll
    for (int j = 0; j < 2 * H; ++j) {
      const R fromL = __shfl_up_sync(0xffffffffu, body[P - 2 * H + j], 1);
      const R fromR = __shfl_down_sync(0xffffffffu, body[j], 1);
      win[0][j] = edge_l ? left[j] : fromL;
      win[0][2 * H + P + j] = edge_r ? right[j] : fromR;
    }
    if (!valid) return;
  } else {
    if (i0 >= N) return;
    load_vec<R, P>(in + i0, body);
#pragma unroll
    for (int j = 0; j < 2 * H; ++j) {
      int64_t il = i0 - 2 * H + j;
      if (il < 0) il += N;
      int64_t ir = i0 + P + j;
      if (ir >= N) ir -= N;
      win[0][j] = __ldg(in + il);
      win[0][2 * H + P + j] = __ldg(in + ir);
    }
  }
#pragma unroll
  for (int j = 0; j < P; ++j) win[0][2 * H + j] = body[j];
  R ctr[1][Q], pred[1][Q];
#pragma unroll
  for (int j = 0; j < Q; ++j) ctr[0][j] = win[0][H + j];
  Prob::template stage<Q>(win, ctr, pred, 1, k);  // predictor u* at i0-h .. i0+P+h-1 (odd tier)
  R bs[1][P], o[1][P];
#pragma unroll
  for (int j = 0; j < P; ++j) bs[0][j] = body[j];
  Prob::template stage<P>(pred, bs, o, 0, k);      // final stage: window = u*, base = u^n
  store_vec<R, P>(out + i0, o[0]);
}

// ---------------------------------------------------------------------------------------------------------
// Per-step kernel for the finite-volume Euler scheme, one INTERFACE per lane.  The generic kernel above lets every
// thread rebuild the P+4 pressures and P+1 interface fluxes of its P cells (P = 2: three pressures and 1.5 fluxes
// per cell, each flux with 8 divisions and 3 square roots).  Here lane l of a warp holds cell j = 28 w + l - 2,
// computes that cell's pressure and the flux at its right interface j+1/2 once, and receives the neighbours'
// pressures, the right neighbour's state and the left interface's flux by warp shuffles; lanes 2..29 then update
// their cell (28 cells per warp: 1.14 pressures and 1.14 fluxes per cell).  Same pressure(), flux() and update
// expressions as Euler::stage, so the result is bit-identical.
template <class Prob>
__global__ void __launch_bounds__(256)
per_step_lane_kernel(const typename Prob::R* __restrict__ in, const typename Prob::R* __restrict__ base,
                     typename Prob::R* __restrict__ out, int64_t N, int odd, Consts<typename Prob::R> k, int bc,
                     BcVals<typename Prob::R> bv) {
  using R = typename Prob::R;
  static_assert(Prob::C == 3 && Prob::H == 2, "interface-per-lane kernel is written for the Euler scheme");
  constexpr int USE = 28;  // cells updated per warp
  const int lane = threadIdx.x & 31;
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w * USE >= N) return;  // whole warp
  const int64_t j = w * USE + lane - 2;
  // state of cell j: periodic wrap, or the fixed end states of the tube in the ghost cells
  int64_t g = j;
  const bool ghost = bc == BC_FIXED && (j < 0 || j >= N);
  if (g < 0) g += N;
  while (g >= N) g -= N;  // the tail warp may reach a few cells past N + 1: any valid cell will do, nothing is stored
  R V[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) V[c] = ghost ? (j < 0 ? bv.l[c] : bv.r[c]) : __ldg(in + (int64_t)c * N + g);
  const R pr = Prob::pressure(V[0], V[1], V[2], k);
  const R pm1 = __shfl_up_sync(0xffffffffu, pr, 1);
  const R pp1 = __shfl_down_sync(0xffffffffu, pr, 1);
  const R pp2 = __shfl_down_sync(0xffffffffu, pr, 2);
  R Vr[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) Vr[c] = __shfl_down_sync(0xffffffffu, V[c], 1);
  R F[3], Fl[3];
  Prob::flux(V, Vr, pr - pm1, pp1 - pr, pp2 - pp1, F, k);  // interface j + 1/2 (meaningless in lanes 0, 30, 31)
#pragma unroll
  for (int c = 0; c < 3; ++c) Fl[c] = __shfl_up_sync(0xffffffffu, F[c], 1);  // interface j - 1/2
  if (lane >= 2 && lane < 2 + USE && j < N) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const R b0 = (!odd) ? __ldg(base + (int64_t)c * N + j) : V[c];
      out[(int64_t)c * N + j] = Prob::update(V[c], b0, F[c] - Fl[c], odd, k);
    }
  }
}

}  // namespace swept
