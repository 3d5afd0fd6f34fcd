// probes.cu — measurement helpers behind swept_probe_fp64 / swept_probe_launch (include/swept.h).
// They provide the roofline denominators that MEASURED_PEAKS.json does not carry (FP64 pipe rate) and the
// B200 counterpart of the paper's 4 us empty-kernel launch cost.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/swept.h"

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
