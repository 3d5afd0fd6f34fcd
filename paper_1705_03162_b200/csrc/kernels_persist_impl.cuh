// kernels_persist_impl.cuh — host launchers of the two persistent flavours (PS_RESIDENT, FLOW), kept apart from
// kernels_impl.cuh so that the slow Euler swept-kernel slices (kernels_euler_inst.cu) do not depend on them.
#pragma once
#include "kernels_impl.cuh"
#include "per_step_resident.cuh"
#include "swept_flow.cuh"
#include "swept_cluster.cuh"

namespace swept {

// ---- resident per-step: one cooperative launch, the field in registers ---------------------------------
template <class Prob, int P>
inline int resident_try(const ResidentLaunch& a, int threads, int pass) {
  using R = typename Prob::R;
  if (a.N % P) return NO_KERNEL;
  const int64_t nthr = a.N / P;
  if (nthr < threads) threads = (int)((nthr + 31) / 32 * 32);
  const int64_t G = (nthr + threads - 1) / threads;
  auto kern = per_step_resident_kernel<Prob, P>;
  const size_t smem = resident_smem_bytes<Prob>(threads);
  int dev = 0, sms = 0, occ = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem) != cudaSuccess || occ < 1) {
    cudaGetLastError();
    return NO_KERNEL;
  }
  // pass 0: a single CTA (no global exchange at all); 1: one CTA per SM; 2: any co-resident grid
  if (G > RESIDENT_MAX_CTAS || G > (pass == 0 ? 1 : (int64_t)sms * (pass == 1 ? 1 : occ))) return NO_KERNEL;
  ResidentArgs<R> r;
  r.in = (const R*)a.in; r.out = (R*)a.out; r.N = a.N; r.nsteps = a.nsteps;
  r.flags = (int*)a.xch;
  r.err = r.flags + RESIDENT_MAX_CTAS * 32;
  r.bc = a.bc;
  r.bv = round_bcvals<R>(a.bcv);
  r.xch = (R*)((char*)a.xch + resident_flag_bytes(RESIDENT_MAX_CTAS));
  r.k = round_consts<R>(a.consts);
  void* args[] = {&r};
  return (int)cudaLaunchCooperativeKernel((const void*)kern, dim3((unsigned)G), dim3((unsigned)threads), args, smem,
                                          a.stream);
}

// smallest P (most lanes busy per point) whose grid fits one CTA per SM, else any co-resident grid
template <class Prob, int PMAX>
int resident_T(const ResidentLaunch& a) {
  constexpr int TMAX = Prob::MAX_THREADS < 512 ? Prob::MAX_THREADS : 512;
  for (int pass = 0; pass < 3; ++pass) {
    int rc = NO_KERNEL;
    if (rc == NO_KERNEL && Prob::H <= 2 && PMAX >= 2) rc = resident_try<Prob, 2>(a, TMAX, pass);
    if (rc == NO_KERNEL && PMAX >= 4) rc = resident_try<Prob, (PMAX >= 4 ? 4 : 2)>(a, TMAX, pass);
    if (rc == NO_KERNEL && PMAX >= 8) rc = resident_try<Prob, (PMAX >= 8 ? 8 : 2)>(a, TMAX, pass);
    if (rc == NO_KERNEL && PMAX >= 16) rc = resident_try<Prob, (PMAX >= 16 ? 16 : 2)>(a, TMAX, pass);
    if (rc != NO_KERNEL) return rc;
  }
  return NO_KERNEL;
}

// ---- CLUSTER flavour: the whole domain in one thread-block cluster, a warp per tile of n = 32 P points -------
// warps per CTA for K tiles: the caller's choice, else as few as still fit a cluster of 16 CTAs (one warp per scheduler
// is the shortest tier latency); 0 if K tiles cannot be laid out
template <class Prob>
inline int cluster_warps_per_cta(int64_t K, int n, int want) {
  const int P = n / 32;
  const int max_wpc = ClusterMaxThreads<16>::value / 32 * (P >= 8 ? 1 : 2);  // = ClusterMaxThreads<P> / 32
  for (int wpc : {1, 2, 4, 8, 16, 32}) {
    if (want ? wpc != want : (wpc < 4 && K > wpc)) continue;
    if (wpc > max_wpc || K % wpc || K / wpc > 16) continue;
    if (cluster_smem_bytes<Prob>(wpc * n) > (size_t)200 * 1024) continue;  // (the two-row kernel's buffers: + 2h per row)
    return wpc;
  }
  return 0;
}

template <class Prob>
inline bool cluster_ok(int64_t N, int n, int want_wpc) {
  if (n != 64 && n != 128 && n != 256 && n != 512 && !(n == 32 && Prob::H == 1 && Prob::ROWS == 2)) return false;
  if (Prob::ROWS == 3 && n > 256) return false;  // three register rows per lane: at most 8 points each
  if (N % n || n / 32 < Prob::H || (n / (2 * Prob::H)) % 2) return false;
  return cluster_warps_per_cta<Prob>(N / n, n, want_wpc) != 0;
}

template <class Prob, int P>
inline int cluster_go(const ClusterLaunch& a) {
  using R = typename Prob::R;
  const int64_t K = a.N / a.n;
  const int wpc = cluster_warps_per_cta<Prob>(K, a.n, a.warps_per_cta);
  if (!wpc) return NO_KERNEL;
  const int cs = (int)(K / wpc);
  ClusterArgs<R> c;
  c.init = (const R*)a.init; c.out = (R*)a.out; c.N = a.N; c.n = a.n; c.rows = a.rows;
  c.k = round_consts<R>(a.consts);
  c.bc = a.bc;
  if (a.bc && !(Prob::H == 1 && Prob::ROWS == 2 && a.bc == BC_MIRROR)) return NO_KERNEL;  // walls: the heat problem
  const size_t smem = cluster_push_smem_bytes<Prob>(wpc, a.n);
  void (*kern)(const ClusterArgs<R>) = nullptr;
  if constexpr (Prob::ROWS == 3) kern = swept_cluster3_kernel<Prob, P>;
  else if constexpr (Prob::H == 1) kern = a.bc ? swept_cluster_kernel<Prob, P, true> : swept_cluster_kernel<Prob, P, false>;
  else kern = swept_cluster_kernel<Prob, P, false>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess && cs > 8) e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e != cudaSuccess) return (int)e;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)cs);
  cfg.blockDim = dim3((unsigned)(wpc * 32));
  cfg.dynamicSmemBytes = smem;
  cfg.stream = a.stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cs;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int nclusters = 0;
  e = cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg);
  if (e != cudaSuccess || nclusters < 1) {
    cudaGetLastError();
    return NO_KERNEL;  // this cluster shape cannot be scheduled on this device
  }
  return (int)cudaLaunchKernelEx(&cfg, kern, c);
}

template <class Prob>
int cluster_T(const ClusterLaunch& a) {
  if (!cluster_ok<Prob>(a.N, a.n, a.warps_per_cta)) return NO_KERNEL;
  switch (a.n / 32) {
    case 1: if constexpr (Prob::H == 1 && Prob::ROWS == 2) return cluster_go<Prob, 1>(a); break;
    case 2: return cluster_go<Prob, 2>(a);
    case 4: return cluster_go<Prob, 4>(a);
    case 8: return cluster_go<Prob, 8>(a);
    case 16: if constexpr (Prob::ROWS == 2) return cluster_go<Prob, 16>(a); break;
  }
  return NO_KERNEL;
}

// ---- FLOW flavour: persistent launch, L = 32 lanes per tile, B = n / 32 lines per lane -----------------
template <class Prob, int BMAX>
inline bool flow_ok(int64_t N, int n) {
  if (n % 32 || N % n) return false;
  const int B = n / 32;
  if (B != 8 && B != 16 && B != 32) return false;
  return B <= BMAX && B % (2 * Prob::H) == 0 && n / (2 * Prob::H) >= 32;
}

template <class Prob, int B, bool TMA, bool PROF = false, bool WALLS = false>
inline int flow_go(const FlowLaunch& a) {
  using R = typename Prob::R;
  constexpr int warps = 4;  // one per scheduler
  constexpr int threads = warps * 32;
  FlowArgs<R> f;
  f.init = (const R*)a.init;
  for (int i = 0; i < 2; ++i)
    for (int j = 0; j < 2; ++j) f.buf[i][j] = (R*)a.buf[i][j];
  f.N = a.N; f.K = (int)(a.N / a.n); f.rows = a.rows; f.flags = a.flags; f.ticket = a.ticket;
  f.k = round_consts<R>(a.consts);
  f.prof = a.prof;
  f.bc = a.bc;
  const size_t smem = flow_smem_bytes<Prob>(warps, a.n);
  auto kern = swept_flow_kernel<Prob, B, TMA, PROF, WALLS>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return (int)e;
  // never launch more CTAs than can be co-resident: waiting tasks must not keep their parents off the machine
  int dev = 0, sms = 0, occ = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem);
  if (e != cudaSuccess) return (int)e;
  if (occ < 1) return (int)cudaErrorLaunchOutOfResources;
  const int64_t ntasks = (int64_t)f.rows * f.K;
  // Resident warps.  All warps run at the same pace, so the tile a warp takes next has its parents still in
  // flight when the resident warps span a whole row (K tiles): waiting warps then only poll.  Default: about
  // 7/8 K warps for the 3-point problem, K/2 for the 5-point ones (their tiles have more parallelism inside a
  // warp and more registers); `ctas_per_sm` (autotuned) overrides.
  int64_t per_sm = a.ctas_per_sm & 15;
  if (per_sm <= 0) {
    const int64_t want = (Prob::H == 1 ? (int64_t)f.K * 7 / 8 : (int64_t)f.K / 2) / warps;  // CTAs
    per_sm = (want + sms / 2) / sms;
  }
  if (per_sm < 1) per_sm = 1;
  if (per_sm > occ) per_sm = occ;
  int64_t grid = per_sm * sms;
  if (grid > (ntasks + warps - 1) / warps) grid = (ntasks + warps - 1) / warps;
  kern<<<(unsigned)grid, threads, smem, a.stream>>>(f);
  return (int)cudaGetLastError();
}

template <class Prob, int BMAX>
int flow_T(const FlowLaunch& a) {
  if (!flow_ok<Prob, BMAX>(a.N, a.n)) return NO_KERNEL;
  // group bit 4: stage the tiles with TMA bulk copies; group 0 (library defaults) does too — measured faster at every
  // size once the kernel around them compiled as tightly as the 16-byte-copy one (profiles/r2_flow_phases.md)
  const bool tma = (a.ctas_per_sm & 16) != 0 || a.ctas_per_sm == 0;
  if (a.bc) {  // insulated ends (heat): the TMA-staged kernel with the wall-tile path
    if constexpr (Prob::H == 1 && Prob::C == 1 && Prob::SIGMA == 1) {
      if (a.bc != BC_MIRROR || a.prof) return NO_KERNEL;
      switch (a.n / 32) {
        case 8: return flow_go<Prob, 8, true, false, true>(a);
        case 16: return flow_go<Prob, 16, true, false, true>(a);
        case 32: return flow_go<Prob, 32, true, false, true>(a);
      }
    }
    return NO_KERNEL;
  }
  if (a.prof) {  // instrumented kernels (swept_flow_profile): the 3-point FP64 problem, the headline's kernel family
    if constexpr (Prob::H == 1 && sizeof(typename Prob::R) == 8) {
      switch (a.n / 32) {
        case 8: return tma ? flow_go<Prob, 8, true, true>(a) : flow_go<Prob, 8, false, true>(a);
        case 16: return tma ? flow_go<Prob, 16, true, true>(a) : flow_go<Prob, 16, false, true>(a);
        case 32: return tma ? flow_go<Prob, 32, true, true>(a) : flow_go<Prob, 32, false, true>(a);
      }
    }
    return NO_KERNEL;
  }
  switch (a.n / 32) {
    case 8: return tma ? flow_go<Prob, 8, true>(a) : flow_go<Prob, 8, false>(a);
    case 16: if (BMAX >= 16) return tma ? flow_go<Prob, (BMAX >= 16 ? 16 : 8), true>(a) : flow_go<Prob, (BMAX >= 16 ? 16 : 8), false>(a); break;
    case 32: if (BMAX >= 32) return tma ? flow_go<Prob, (BMAX >= 32 ? 32 : 8), true>(a) : flow_go<Prob, (BMAX >= 32 ? 32 : 8), false>(a); break;
  }
  return NO_KERNEL;
}

}  // namespace swept
