// per_step_resident.cuh — the per-step scheme WITHOUT a launch per sub-timestep (per-step
// half; PAPER.md:297-303 names a device-side synchronisation instead of kernel relaunch as future work).
//
// Same arithmetic and the same order of sub-timesteps as per_step.cuh (one sub-timestep of every point before the
// next one starts: the "Classic" decomposition), but ONE persistent launch runs all of them:
//   * the field lives in registers: thread g owns the P contiguous points [gP, gP+P) for the whole run;
//   * inside a CTA the h halo values of each neighbour go through a double-buffered shared-memory edge array, one
//     __syncthreads() per sub-timestep;
//   * between CTAs only the two neighbours are synchronised (not the whole grid): each CTA publishes its outermost
//     h values per side to a double-buffered global exchange array and release-stores its sub-step counter; the
//     neighbour's edge thread polls that counter (relaxed, then an acquire fence) and reads the values.
// Global traffic per sub-timestep: 2 h C values per CTA instead of the whole field.  The launch is cooperative
// (cudaLaunchCooperativeKernel) only to be certain that all CTAs are co-resident; no grid-wide barrier is used.
//
// Exchange-slot reuse: slot s&1 written at sub-step s is overwritten at s+2; a CTA cannot start s+2 before it has
// the neighbour's edges of s+1, which the neighbour publishes only after it has read the slot of s.
#pragma once
#include "functors.cuh"
#include "per_step.cuh"

namespace swept {

template <class R>
struct ResidentArgs {
  const R* in;     // field at entry (C components, stride N)
  R* out;          // field at exit
  int64_t N;
  int64_t nsteps;  // full timesteps
  R* xch;          // [2 parities][G CTAs][2 sides] slots of RS_LINE bytes, each holding [C][H] edge values
  int* flags;      // sub-steps published by CTA i at flags[i * RS_LINE / 4]; zero on entry
  int* err;        // error word: set if a neighbour wait timed out
  int bc;          // BC_WRAP, BC_MIRROR (insulated heat ends) or BC_FIXED (Euler tube): applied by the two end threads
  BcVals<R> bv;
  Consts<R> k;
};

// the neighbour's counter is polled with an acquire load (2 polling threads per CTA: the per-poll L1 invalidation
// is cheap here), so that no separate fence sits on the critical path of a sub-timestep
__device__ __forceinline__ int rs_ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// every flag and every exchange slot has its own 128-byte line: polled lines are not shared between CTAs
constexpr int RS_LINE = 128;

template <class Prob, int P>
__global__ void __launch_bounds__(Prob::MAX_THREADS < 512 ? Prob::MAX_THREADS : 512) per_step_resident_kernel(const ResidentArgs<typename Prob::R> a) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C, SIGMA = Prob::SIGMA;
  static_assert(P >= H, "a thread's halo must come from its immediate neighbours");
  extern __shared__ __align__(16) unsigned char rs_smem[];
  // edge[parity][side][c][e][tid]: side 0 = the thread's first H points, side 1 = its last H points
  R* edge = reinterpret_cast<R*>(rs_smem);
  const int T = blockDim.x, tid = threadIdx.x, G = gridDim.x, cta = blockIdx.x;
  const int64_t N = a.N, nthr = N / P;                   // active threads over the whole grid
  const int64_t g = (int64_t)cta * T + tid;
  const bool on = g < nthr;
  const int t_last = (int)(((int64_t)(cta + 1) * T <= nthr ? T : nthr - (int64_t)cta * T) - 1);  // last active thread
  const int left_cta = cta == 0 ? G - 1 : cta - 1, right_cta = cta + 1 == G ? 0 : cta + 1;
  auto eslot = [&](int par, int side, int c, int e, int t) -> R& {
    return edge[((((par * 2 + side) * C + c) * H + e) * T) + t];
  };
  auto xslot = [&](int par, int who, int side, int c, int e) -> R* {
    return a.xch + (((int64_t)par * G + who) * 2 + side) * (RS_LINE / (int)sizeof(R)) + c * H + e;
  };

  alignas(16) R cur[C][P], stg[C][P];
  if (on) {
#pragma unroll
    for (int c = 0; c < C; ++c) load_vec<R, P>(a.in + (int64_t)c * N + g * P, cur[c]);
  }
  int sub = 0;  // sub-timesteps completed = index of the exchange about to happen
  for (int64_t step = 0; step < a.nsteps; ++step) {
#pragma unroll
    for (int st = 0; st < SIGMA; ++st) {
      const int odd = (SIGMA == 2 && st == 0) ? 1 : 0;     // predictor sub-timestep
      R(&src)[C][P] = (SIGMA == 2 && st == 1) ? stg : cur;  // stage input
      const int par = sub & 1;
      if (on) {
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int e = 0; e < H; ++e) {
            eslot(par, 0, c, e, tid) = src[c][e];
            eslot(par, 1, c, e, tid) = src[c][P - H + e];
          }
        if (G > 1) {
          if (tid == 0)
#pragma unroll
            for (int c = 0; c < C; ++c)
#pragma unroll
              for (int e = 0; e < H; ++e) *xslot(par, cta, 0, c, e) = src[c][e];
          if (tid == t_last)
#pragma unroll
            for (int c = 0; c < C; ++c)
#pragma unroll
              for (int e = 0; e < H; ++e) *xslot(par, cta, 1, c, e) = src[c][P - H + e];
        }
      }
      __syncthreads();
      if (G > 1 && tid == 0) {  // release is cumulative over the edge writes ordered before it by the barrier
        asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(a.flags + cta * (RS_LINE / 4)), "r"(sub + 1) : "memory");
      }
      if (on) {
        R win[C][P + 2 * H];
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int j = 0; j < P; ++j) win[c][H + j] = src[c][j];
        // left halo = last H points of the thread before, right halo = first H points of the thread after
        // the two ends of the domain under a non-periodic boundary condition: no neighbour, the halo is the mirror
        // image of the thread's own points (B.5) or the fixed end state
        const bool wall_l = a.bc != BC_WRAP && g == 0, wall_r = a.bc != BC_WRAP && g == nthr - 1;
        const bool gl_left = tid == 0 && G > 1 && !wall_l, gl_right = tid == t_last && G > 1 && !wall_r;
        if (gl_left || gl_right) {
          const int who = gl_left ? left_cta : right_cta;
          unsigned polls = 0;
          while (rs_ld_acquire(a.flags + who * (RS_LINE / 4)) < sub + 1) {
            __nanosleep(20);
            if (++polls > (1u << 22)) {  // never while the grid is co-resident: report instead of hanging
              atomicExch(a.err, 1);
              break;
            }
          }
        }
        const int tl = tid == 0 ? t_last : tid - 1, tr = tid == t_last ? 0 : tid + 1;  // G == 1: periodic inside the CTA
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int e = 0; e < H; ++e) {
            win[c][e] = gl_left ? __ldcg(xslot(par, left_cta, 1, c, e)) : eslot(par, 1, c, e, tl);
            win[c][H + P + e] = gl_right ? __ldcg(xslot(par, right_cta, 0, c, e)) : eslot(par, 0, c, e, tr);
          }
        if (wall_l) {
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int e = 0; e < H; ++e) win[c][e] = a.bc == BC_FIXED ? a.bv.l[c] : src[c][H - e];
        }
        if (wall_r) {
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int e = 0; e < H; ++e) win[c][H + P + e] = a.bc == BC_FIXED ? a.bv.r[c] : src[c][P - 2 - e];
        }
        if (gl_left && gl_right) {  // one active thread in this CTA: it needs both neighbours
          unsigned polls = 0;
          while (rs_ld_acquire(a.flags + right_cta * (RS_LINE / 4)) < sub + 1 && ++polls < (1u << 22)) {}
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int e = 0; e < H; ++e) win[c][H + P + e] = __ldcg(xslot(par, right_cta, 0, c, e));
        }
        R o[C][P];
        Prob::template stage<P>(win, cur, o, odd, a.k);  // base = u^n for the final stage (cur is untouched by stage 1)
        if (SIGMA == 2 && st == 0) {
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int j = 0; j < P; ++j) stg[c][j] = o[c][j];
        } else {
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int j = 0; j < P; ++j) cur[c][j] = o[c][j];
        }
      }
      ++sub;
    }
  }
  if (on) {
#pragma unroll
    for (int c = 0; c < C; ++c) store_vec<R, P>(a.out + (int64_t)c * N + g * P, cur[c]);
  }
}

template <class Prob>
inline size_t resident_smem_bytes(int threads) {
  return (size_t)2 * 2 * Prob::C * Prob::H * threads * sizeof(typename Prob::R);
}

}  // namespace swept
