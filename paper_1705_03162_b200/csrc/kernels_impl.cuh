// kernels_impl.cuh — templated host launchers shared by kernels_{heat,ks,euler}.cu.
#pragma once
#include "internal.h"
#include "per_step.cuh"
#include "swept_tier.cuh"
#include "../../include/swept.h"

namespace swept {

template <class R>
inline Consts<R> round_consts(const double* c) {
  Consts<R> k;
  k.a0 = (R)c[0]; k.a1 = (R)c[1]; k.a2 = (R)c[2]; k.a3 = (R)c[3]; k.a4 = (R)c[4];
  return k;
}

template <class Prob, int P>
inline int per_step_go(const PerStepLaunch& a) {
  using R = typename Prob::R;
  const int64_t nthreads = a.N / P;
  const unsigned grid = (unsigned)((nthreads + a.threads - 1) / a.threads);
  per_step_kernel<Prob, P><<<grid, a.threads, 0, a.stream>>>((const R*)a.in, (const R*)a.base, (R*)a.out,
                                                             a.N, a.odd, round_consts<R>(a.consts));
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
  const size_t smem = tier_smem_bytes<Prob>(a.n);
  auto kern = swept_tier_kernel<Prob, P, KIND>;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
  }
  kern<<<(unsigned)(a.N / a.n), a.n / P, smem, a.stream>>>(t);
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
  if (threads < 8 || threads > 1024) return false;
  return tier_smem_bytes<Prob>(n) <= 227 * 1024;
}

template <class Prob, int PMAX>
inline int tier_T(const TileLaunch& a) {
  if (!tier_ok<Prob>(a.n, a.P, PMAX)) return NO_KERNEL;
  switch (a.P) {
    case 1: return tier_kind<Prob, 1>(a);
    case 2: return tier_kind<Prob, 2>(a);
    case 4: if (PMAX >= 4) return tier_kind<Prob, (PMAX >= 4 ? 4 : 1)>(a); break;
  }
  return NO_KERNEL;
}

}  // namespace swept
