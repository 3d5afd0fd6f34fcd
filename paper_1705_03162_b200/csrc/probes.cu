// probes.cu — measurement helpers behind swept_probe_fp64 / swept_probe_launch (include/swept.h).
// They provide the roofline denominators that MEASURED_PEAKS.json does not carry (FP64 pipe rate) and the
// B200 counterpart of the paper's 4 us empty-kernel launch cost.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/swept.h"
#include "swept_char.cuh"

namespace {

constexpr int CHAINS = 8;

__global__ void __launch_bounds__(256) dfma_chain_kernel(double* sink, int iters, double a, double b) {
  double x[CHAINS];
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) x[c] = (double)(threadIdx.x + c) * 1e-3;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) x[c] = fma(x[c], a, b);
  }
  double s = 0;
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) s += x[c];
  if (s == 123.456) sink[0] = s;  // never true in practice; keeps the chains alive
}

__global__ void empty_kernel() {}

// ---- one dependent FP64 chain per thread, one warp: the latency of DADD -> DFMA, the pair a heat update puts on
// the critical path of a tier (s = um + up; out = fma(Fo, s, t))
__global__ void __launch_bounds__(32) dep_chain_kernel(double* sink, int iters, double a, double b, long long* cycles) {
  double x = (double)threadIdx.x * 1e-3;
  const long long t0 = clock64();
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      x = x + b;           // DADD
      x = fma(a, x, b);    // DFMA
    }
  }
  const long long t1 = clock64();
  if (threadIdx.x == 0) cycles[0] = t1 - t0;
  if (x == 123.456) sink[0] = x;
}

// ---- the dependent chain of a REGISTER-RESIDENT tier (swept_cluster.cuh), one warp, one point per lane:
// MODE 0: shuffle -> shuffle; 1: both neighbours by 64-bit shuffles -> DADD -> DFMA; 2: the same -> select on the tier
// window (a whole heat tier); 3: DFMA -> select
template <int MODE>
__global__ void __launch_bounds__(32) tier_chain_kernel(double* sink, int iters, double a0, double a1, int span,
                                                        long long* cycles) {
  const int lane = threadIdx.x & 31;
  double u = (double)lane * 1e-3;
  int w = lane;
  const int sl = (lane + 31) & 31, sr = (lane + 1) & 31;
  const long long t0 = clock64();
  for (int i = 0; i < iters; ++i) {
    if (MODE == 0) w = __shfl_sync(0xffffffffu, w, sr);
    if (MODE == 1) u = fma(a0, __shfl_sync(0xffffffffu, u, sl) + __shfl_sync(0xffffffffu, u, sr), a1 * u);
    if (MODE == 2) {
      const double o = fma(a0, __shfl_sync(0xffffffffu, u, sl) + __shfl_sync(0xffffffffu, u, sr), a1 * u);
      u = (unsigned)(i - lane) <= (unsigned)span ? o : u;
    }
    if (MODE == 3) {
      const double o = fma(a0, u, a1);
      u = (unsigned)(i - lane) <= (unsigned)span ? o : u;
    }
  }
  const long long t1 = clock64();
  if (threadIdx.x == 0) cycles[0] = t1 - t0;
  if (u + w == 123.456) sink[0] = u;
}

// ---- shared-memory bandwidth: every thread streams conflict-free 16-byte loads from its CTA's shared memory
// (integer XORs keep the loaded values alive without touching the FP64 pipe)
__global__ void __launch_bounds__(1024) smem_read_int_kernel(unsigned* sink, int iters) {
  extern __shared__ __align__(16) unsigned char sm_raw[];
  uint4* sm = reinterpret_cast<uint4*>(sm_raw);
  const int nvec = 2048;  // 32 KiB
  for (int i = threadIdx.x; i < nvec; i += blockDim.x) sm[i] = make_uint4(i, i + 1, i + 2, i + 3);
  __syncthreads();
  uint4 acc = make_uint4(0, 0, 0, 0);
  int idx = threadIdx.x;
  const uint32_t base = swept::smem_u32(sm);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      uint4 v;  // volatile: one LDS.128 per lane and iteration, never hoisted or merged
      asm volatile("ld.volatile.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                   : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                   : "r"(base + 16u * (uint32_t)((idx + u * 256) & (nvec - 1))));
      acc.x ^= v.x; acc.y ^= v.y; acc.z ^= v.z; acc.w ^= v.w;
    }
    idx = (idx + 32) & (nvec - 1);
  }
  if ((acc.x ^ acc.y ^ acc.z ^ acc.w) == 0x12345678u) sink[0] = acc.x;
}

// ---- the characteristic sweep of the CHAR / FLOW flavours on ONE SM, no global traffic: `warps` warps (4 x the
// warps per scheduler) each sweep their own staged WholeDiamond tile `reps` times; cycles from clock64.  This is the
// micro-benchmark behind DESIGN.md §5.6 (issue-rate model of the sweep).
template <class Prob, int B>
__global__ void __launch_bounds__(B == 32 ? 384 : (B == 16 ? 768 : 1024))
sweep_probe_kernel(swept::Consts<typename Prob::R> k, int reps, long long* cycles) {
  using R = typename Prob::R;
  constexpr int PAD = swept::Pad16<R>::value, L = 32, n = B * L, RS = n + 2 * PAD;
  extern __shared__ __align__(128) unsigned char sm_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  R* rows = reinterpret_cast<R*>(sm_raw) + (size_t)warp * 2 * Prob::C * RS;
  for (int i = lane; i < 2 * Prob::C * RS; i += 32) rows[i] = (R)(1.0 + 1e-3 * (i % 17));
  __syncthreads();
  const long long t0 = clock64();
  for (int r = 0; r < reps; ++r) {
    swept::char_sweep_tile<Prob, B, L, swept::KIND_WHOLE, RS>(rows, RS, PAD + n / 2, lane, k);
    __syncwarp();
  }
  __syncthreads();
  const long long t1 = clock64();
  if (threadIdx.x == 0) cycles[0] = t1 - t0;
}

template <class Prob, int B>
int sweep_probe_go(int warps, int reps, cudaStream_t stream, long long* dcycles) {
  using R = typename Prob::R;
  constexpr int PAD = swept::Pad16<R>::value, n = B * 32, RS = n + 2 * PAD;
  const size_t smem = (size_t)warps * 2 * Prob::C * RS * sizeof(R);
  if (smem > 227 * 1024 || warps * 32 > (B == 32 ? 384 : (B == 16 ? 768 : 1024))) return SWEPT_EUNSUPPORTED;
  auto kern = sweep_probe_kernel<Prob, B>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SWEPT_ECUDA;
  swept::Consts<R> k;
  if (Prob::H == 1) { k.a0 = (R)0.25; k.a1 = (R)0.5; k.a2 = k.a3 = k.a4 = (R)0; }
  else { k.a0 = (R)0.5; k.a1 = (R)4; k.a2 = (R)16; k.a3 = (R)0.005; k.a4 = (R)0.0025; }
  kern<<<1, warps * 32, smem, stream>>>(k, reps, dcycles);
  return cudaGetLastError() == cudaSuccess ? SWEPT_OK : SWEPT_ECUDA;
}

}  // namespace

extern "C" {

int swept_probe_fp64(int device, void* stream_, double* out) {
  if (!out) return SWEPT_EINVAL;
  cudaStream_t stream = (cudaStream_t)stream_;
  if (device >= 0 && cudaSetDevice(device) != cudaSuccess) return SWEPT_ECUDA;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return SWEPT_ECUDA;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double* sink = nullptr;
  if (cudaMalloc(&sink, 8) != cudaSuccess) return SWEPT_ENOMEM;
  const int iters = 20000, blocks = sms * 8, threads = 256;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, stream);
    dfma_chain_kernel<<<blocks, threads, 0, stream>>>(sink, iters, 0.999999, 1e-9);
    cudaEventRecord(e1, stream);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(sink); return SWEPT_ECUDA; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double ops = (double)blocks * threads * (double)iters * CHAINS;
    if (rep > 0 && ops / (ms * 1e-3) > best) best = ops / (ms * 1e-3);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  *out = best;
  return SWEPT_OK;
}

int swept_probe_launch(int device, void* stream_, int count, double* us_per_launch) {
  if (!us_per_launch || count <= 0) return SWEPT_EINVAL;
  cudaStream_t stream = (cudaStream_t)stream_;
  if (device >= 0 && cudaSetDevice(device) != cudaSuccess) return SWEPT_ECUDA;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  for (int i = 0; i < 16; ++i) empty_kernel<<<1, 32, 0, stream>>>();
  cudaEventRecord(e0, stream);
  for (int i = 0; i < count; ++i) empty_kernel<<<1, 32, 0, stream>>>();
  cudaEventRecord(e1, stream);
  if (cudaEventSynchronize(e1) != cudaSuccess) return SWEPT_ECUDA;
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *us_per_launch = (double)ms * 1e3 / count;
  return SWEPT_OK;
}

}  // extern "C"

extern "C" {

int swept_probe_chain(int device, void* stream_, double* cycles_per_dadd_dfma) {
  if (!cycles_per_dadd_dfma) return SWEPT_EINVAL;
  cudaStream_t stream = (cudaStream_t)stream_;
  if (device >= 0 && cudaSetDevice(device) != cudaSuccess) return SWEPT_ECUDA;
  double* sink = nullptr;
  long long* dc = nullptr;
  if (cudaMalloc(&sink, 8) != cudaSuccess || cudaMalloc(&dc, 8) != cudaSuccess) { cudaFree(sink); return SWEPT_ENOMEM; }
  const int iters = 4096;
  long long c = 0;
  for (int rep = 0; rep < 2; ++rep) dep_chain_kernel<<<1, 32, 0, stream>>>(sink, iters, 0.999999, 1e-9, dc);
  const cudaError_t e = cudaMemcpyAsync(&c, dc, 8, cudaMemcpyDeviceToHost, stream);
  const cudaError_t e2 = cudaStreamSynchronize(stream);
  cudaFree(sink);
  cudaFree(dc);
  if (e != cudaSuccess || e2 != cudaSuccess) return SWEPT_ECUDA;
  *cycles_per_dadd_dfma = (double)c / ((double)iters * 8);
  return SWEPT_OK;
}

int swept_probe_tier(int device, void* stream_, double* cycles4) {
  if (!cycles4) return SWEPT_EINVAL;
  cudaStream_t stream = (cudaStream_t)stream_;
  if (device >= 0 && cudaSetDevice(device) != cudaSuccess) return SWEPT_ECUDA;
  double* sink = nullptr;
  long long* dc = nullptr;
  if (cudaMalloc(&sink, 8) != cudaSuccess || cudaMalloc(&dc, 4 * 8) != cudaSuccess) { cudaFree(sink); return SWEPT_ENOMEM; }
  const int iters = 20000, span = 1 << 30;
  long long c[4] = {0, 0, 0, 0};
  for (int rep = 0; rep < 2; ++rep) {
    tier_chain_kernel<0><<<1, 32, 0, stream>>>(sink, iters, 0.25, 0.5, span, dc + 0);
    tier_chain_kernel<1><<<1, 32, 0, stream>>>(sink, iters, 0.25, 0.5, span, dc + 1);
    tier_chain_kernel<2><<<1, 32, 0, stream>>>(sink, iters, 0.25, 0.5, span, dc + 2);
    tier_chain_kernel<3><<<1, 32, 0, stream>>>(sink, iters, 0.25, 0.5, span, dc + 3);
  }
  const cudaError_t e = cudaMemcpyAsync(c, dc, 4 * 8, cudaMemcpyDeviceToHost, stream);
  const cudaError_t e2 = cudaStreamSynchronize(stream);
  cudaFree(sink);
  cudaFree(dc);
  if (e != cudaSuccess || e2 != cudaSuccess) return SWEPT_ECUDA;
  for (int i = 0; i < 4; ++i) cycles4[i] = (double)c[i] / (double)iters;
  return SWEPT_OK;
}

int swept_probe_smem(int device, void* stream_, double* bytes_per_s, double* bytes_per_clk_per_sm) {
  if (!bytes_per_s) return SWEPT_EINVAL;
  cudaStream_t stream = (cudaStream_t)stream_;
  if (device >= 0 && cudaSetDevice(device) != cudaSuccess) return SWEPT_ECUDA;
  int dev = 0, sms = 0, khz = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return SWEPT_ECUDA;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
  unsigned* sink = nullptr;
  if (cudaMalloc(&sink, 8) != cudaSuccess) return SWEPT_ENOMEM;
  const int iters = 4000, threads = 1024, smem = 32 * 1024;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, stream);
    smem_read_int_kernel<<<sms * 2, threads, smem, stream>>>(sink, iters);
    cudaEventRecord(e1, stream);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(sink); return SWEPT_ECUDA; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double bytes = (double)sms * 2 * threads * (double)iters * 8 * 16;
    if (rep > 0 && bytes / (ms * 1e-3) > best) best = bytes / (ms * 1e-3);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  *bytes_per_s = best;
  if (bytes_per_clk_per_sm) *bytes_per_clk_per_sm = best / ((double)khz * 1e3) / sms;
  return SWEPT_OK;
}

int swept_probe_sweep(int device, void* stream_, int problem, int lines_per_lane, int warps_per_scheduler,
                      double* cycles_per_step, double* fp64_busy) {
  if (!cycles_per_step) return SWEPT_EINVAL;
  if (warps_per_scheduler < 1 || warps_per_scheduler > 8) return SWEPT_EINVAL;
  cudaStream_t stream = (cudaStream_t)stream_;
  if (device >= 0 && cudaSetDevice(device) != cudaSuccess) return SWEPT_ECUDA;
  long long* dc = nullptr;
  if (cudaMalloc(&dc, 8) != cudaSuccess) return SWEPT_ENOMEM;
  const int warps = 4 * warps_per_scheduler, reps = 8, B = lines_per_lane;
  int rc = SWEPT_EUNSUPPORTED, h = 1, fp64_per_point = 3;
  for (int pass = 0; pass < 2; ++pass) {  // pass 0 warms up
    if (problem == SWEPT_HEAT) {
      if (B == 8) rc = sweep_probe_go<swept::Heat<double>, 8>(warps, reps, stream, dc);
      else if (B == 16) rc = sweep_probe_go<swept::Heat<double>, 16>(warps, reps, stream, dc);
      else if (B == 32) rc = sweep_probe_go<swept::Heat<double>, 32>(warps, reps, stream, dc);
    } else if (problem == SWEPT_KS) {
      h = 2;
      fp64_per_point = 11;
      if (B == 8) rc = sweep_probe_go<swept::KS<double, 0>, 8>(warps, reps, stream, dc);
      else if (B == 16) rc = sweep_probe_go<swept::KS<double, 0>, 16>(warps, reps, stream, dc);
      else if (B == 32) rc = sweep_probe_go<swept::KS<double, 0>, 32>(warps, reps, stream, dc);
    }
    if (rc != SWEPT_OK) break;
  }
  long long c = 0;
  if (rc == SWEPT_OK && (cudaMemcpyAsync(&c, dc, 8, cudaMemcpyDeviceToHost, stream) != cudaSuccess ||
                         cudaStreamSynchronize(stream) != cudaSuccess))
    rc = SWEPT_ECUDA;
  cudaFree(dc);
  if (rc != SWEPT_OK) return rc;
  const int n = 32 * B, m = n / (2 * h);
  const double steps = (double)reps * (m + 32);  // super-steps per warp, skew ramp included
  *cycles_per_step = (double)c / steps;
  // FP64 warp-instructions of a super-step (B points) x 2 issue cycles on the 16-lane pipe of a scheduler
  if (fp64_busy) *fp64_busy = warps_per_scheduler * (double)(fp64_per_point * B) * 2.0 / *cycles_per_step;
  return SWEPT_OK;
}

}  // extern "C"
