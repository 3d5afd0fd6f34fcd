// kernels_impl.cuh — templated host launchers shared by kernels_{heat,ks,euler}.cu.
#pragma once
#include "internal.h"
#include "per_step.cuh"
#include "swept_tier.cuh"
#include "swept_char.cuh"
#include "../../include/swept.h"

namespace swept {

template <class R>
inline Consts<R> round_consts(const double* c) {
  Consts<R> k;
  k.a0 = (R)c[0]; k.a1 = (R)c[1]; k.a2 = (R)c[2]; k.a3 = (R)c[3]; k.a4 = (R)c[4];
  return k;
}

template <class R>
inline BcVals<R> round_bcvals(const double* v) {
  BcVals<R> b;
  for (int c = 0; c < 3; ++c) {
    b.l[c] = v ? (R)v[c] : (R)0;
    b.r[c] = v ? (R)v[3 + c] : (R)0;
  }
  return b;
}

template <class Prob, int P>
inline int per_step_go(const PerStepLaunch& a) {
  using R = typename Prob::R;
  const int64_t nthreads = a.N / P;
  const int threads = a.threads < Prob::MAX_THREADS ? a.threads : Prob::MAX_THREADS;
  const unsigned grid = (unsigned)((nthreads + threads - 1) / threads);
  per_step_kernel<Prob, P><<<grid, threads, 0, a.stream>>>((const R*)a.in, (const R*)a.base, (R*)a.out,
                                                             a.N, a.odd, round_consts<R>(a.consts), a.bc,
                                                             round_bcvals<R>(a.bcv));
  return (int)cudaGetLastError();
}

// scalar RK2 schemes: both stages of a timestep in one launch (per_step.cuh)
template <class Prob, int P>
inline int per_step_fused_go(const PerStepLaunch& a) {
  using R = typename Prob::R;
  if (a.N % P || a.bc) return NO_KERNEL;
  const int64_t nthreads = a.N / P;
  const int threads = a.threads < Prob::MAX_THREADS ? a.threads : Prob::MAX_THREADS;
  const unsigned grid = (unsigned)((nthreads + threads - 1) / threads);
  // halo by warp shuffles where the launch is throughput-bound (measured cross-over between N = 2^17 and 2^20)
  if (a.N >= ((int64_t)1 << 19))
    per_step_fused_kernel<Prob, P, true><<<grid, threads, 0, a.stream>>>((const R*)a.in, (R*)a.out, a.N,
                                                                           round_consts<R>(a.consts));
  else
    per_step_fused_kernel<Prob, P, false><<<grid, threads, 0, a.stream>>>((const R*)a.in, (R*)a.out, a.N,
                                                                            round_consts<R>(a.consts));
  return (int)cudaGetLastError();
}

// Euler: one interface per lane, 28 cells per warp (per_step.cuh)
template <class Prob>
inline int per_step_lane_go(const PerStepLaunch& a) {
  using R = typename Prob::R;
  const int threads = 256;
  const int64_t warps = (a.N + 27) / 28;
  const unsigned grid = (unsigned)((warps * 32 + threads - 1) / threads);
  per_step_lane_kernel<Prob><<<grid, threads, 0, a.stream>>>((const R*)a.in, (const R*)a.base, (R*)a.out, a.N, a.odd,
                                                             round_consts<R>(a.consts), a.bc, round_bcvals<R>(a.bcv));
  return (int)cudaGetLastError();
}

template <class Prob, int PMAX>
inline int per_step_T(const PerStepLaunch& a) {
  if (a.N % a.P != 0) return NO_KERNEL;
  switch (a.P) {
    case 1: return per_step_go<Prob, 1>(a);
    case 2: return per_step_go<Prob, 2>(a);
    case 4: if (PMAX >= 4) return per_step_go<Prob, (PMAX >= 4 ? 4 : 1)>(a); break;
  }
  return NO_KERNEL;
}

template <class Prob, int P, int KIND>
inline int tier_go(const TileLaunch& a) {
  using R = typename Prob::R;
  TierArgs<R> t;
  t.in0 = (const R*)a.in0; t.in1 = (const R*)a.in1; t.out0 = (R*)a.out0; t.out1 = (R*)a.out1;
  t.N = a.N; t.n = a.n; t.shift = a.shift; t.ntiers = a.ntiers; t.k = round_consts<R>(a.consts);
  t.bc = a.bc;
  t.bv = round_bcvals<R>(a.bcv);
  t.tile_base = a.tile_base; t.tile_step = a.tile_step; t.skip_first = 0; t.skip_last = 0;
  t.in2 = (const R*)a.in2; t.out2 = (R*)a.out2; t.tmod = a.tmod;
  const size_t smem = tier_smem_bytes<Prob>(a.n);
  auto kern = swept_tier_kernel<Prob, P, KIND>;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
  }
  kern<<<(unsigned)(a.tile_count > 0 ? a.tile_count : a.N / a.n), a.n / P, smem, a.stream>>>(t);
  return (int)cudaGetLastError();
}

template <class Prob, int P>
inline int tier_kind(const TileLaunch& a) {
  switch (a.kind) {
    case KIND_UP: return tier_go<Prob, P, KIND_UP>(a);
    case KIND_SPLIT: return tier_go<Prob, P, KIND_SPLIT>(a);
    case KIND_WHOLE: return tier_go<Prob, P, KIND_WHOLE>(a);
    case KIND_DOWN: return tier_go<Prob, P, KIND_DOWN>(a);
  }
  return NO_KERNEL;
}

template <class Prob>
inline bool tier_ok(int n, int P, int pmax) {
  if (n < 32 || n > 4096 || (n & (n - 1))) return false;
  if (P != 1 && P != 2 && P != 4) return false;
  if (P > pmax) return false;
  const int threads = n / P;
  if (threads < 8 || threads > Prob::TIER_MAX_THREADS) return false;
  return tier_smem_bytes<Prob>(n) <= 227 * 1024;
}

template <class Prob, int PMAX>
int tier_T(const TileLaunch& a) {
  if (!tier_ok<Prob>(a.n, a.P, PMAX)) return NO_KERNEL;
  switch (a.P) {
    case 1: return tier_kind<Prob, 1>(a);
    case 2: return tier_kind<Prob, 2>(a);
    case 4: if (PMAX >= 4) return tier_kind<Prob, (PMAX >= 4 ? 4 : 1)>(a); break;
  }
  return NO_KERNEL;
}


// ---- CHAR flavour: a.P = L (lanes per tile), B = n / L lines per lane ---------------------------------
inline int char_threads(int64_t N, int B) {
  for (int T : {64, 32})
    if (N % ((int64_t)T * B) == 0) return T;
  return 0;
}

template <class Prob, int B, int L, int KIND>
inline int char_go(const TileLaunch& a) {
  using R = typename Prob::R;
  const int T = char_threads(a.N, B);
  if (T == 0 || T < L) return NO_KERNEL;
  TierArgs<R> t;
  t.in0 = (const R*)a.in0; t.in1 = (const R*)a.in1; t.out0 = (R*)a.out0; t.out1 = (R*)a.out1;
  t.N = a.N; t.n = a.n; t.shift = a.shift; t.ntiers = a.ntiers; t.k = round_consts<R>(a.consts);
  t.bc = 0;
  t.bv = round_bcvals<R>(nullptr);
  t.tile_base = 0; t.tile_step = 1; t.skip_first = a.skip_first; t.skip_last = a.skip_last;
  const size_t smem = char_smem_bytes<Prob>(T, B);
  auto kern = swept_char_kernel<Prob, B, L, KIND>;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
  }
  kern<<<(unsigned)(a.N / ((int64_t)T * B)), T, smem, a.stream>>>(t);
  return (int)cudaGetLastError();
}

template <class Prob, int B, int L>
inline int char_kind(const TileLaunch& a) {
  switch (a.kind) {
    case KIND_UP: return char_go<Prob, B, L, KIND_UP>(a);
    case KIND_SPLIT: return char_go<Prob, B, L, KIND_SPLIT>(a);
    case KIND_WHOLE: return char_go<Prob, B, L, KIND_WHOLE>(a);
    case KIND_DOWN: return char_go<Prob, B, L, KIND_DOWN>(a);
  }
  return NO_KERNEL;
}

template <class Prob, int BMAX>
inline bool char_ok(int64_t N, int n, int L) {
  if (L != 8 && L != 16 && L != 32) return false;
  if (n % L) return false;
  const int B = n / L;
  // B = 4 (3-point stencil only: the chain length B/2h must stay even for the 5-point RK2 schemes) serves the
  // narrow tiles of the remainder cycles: n = 32 with L = 8
  if (B != 8 && B != 16 && B != 32 && !(B == 4 && Prob::H == 1)) return false;
  if (B > BMAX || B % (2 * Prob::H)) return false;
  const int T = char_threads(N, B);
  return T >= L && N % n == 0;
}

template <class Prob, int B>
int char_L(const TileLaunch& a) {
  switch (a.P) {
    case 8: return char_kind<Prob, B, 8>(a);
    case 16: return char_kind<Prob, B, 16>(a);
    case 32: return char_kind<Prob, B, 32>(a);
  }
  return NO_KERNEL;
}

template <class Prob, int BMAX>
int char_T(const TileLaunch& a) {
  if (!char_ok<Prob, BMAX>(a.N, a.n, a.P)) return NO_KERNEL;
  switch (a.n / a.P) {
    case 4: if (Prob::H == 1) return char_L<Prob, (Prob::H == 1 ? 4 : 8)>(a); break;
    case 8: return char_L<Prob, 8>(a);
    case 16: if (BMAX >= 16) return char_L<Prob, (BMAX >= 16 ? 16 : 8)>(a); break;
    case 32: if (BMAX >= 32) return char_L<Prob, (BMAX >= 32 ? 32 : 8)>(a); break;
  }
  return NO_KERNEL;
}

}  // namespace swept
