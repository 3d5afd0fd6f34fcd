// flow_static.cu — swept_heat_flow_static (include/swept.h): one swept cycle of the heat problem by the persistent
// FLOW kernel (swept_flow.cuh) for callers that must not allocate — code under CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc.  Everything the existing path gets from swept_create's allocations lives
// in ONE file-scope device array here: the kernel's ticket / leave counters and per-tile flags, and three of the four
// row slabs of the two-row inter-launch state (the fourth is the caller's output buffer).  The entry point calls no
// cudaMalloc, cudaFree or allocating library routine; the array is held by every GPU that loads the library until the
// process exits.
//
// In HOST code the array's name is a host-side stand-in, not a device address: its device address is taken once per
// device with cudaGetSymbolAddress (same translation unit, that device current) and only that pointer reaches a kernel.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/swept.h"
#include "kernels_persist_impl.cuh"

namespace {

constexpr int64_t MAX_N = SWEPT_STATIC_MAX_N;  // points
constexpr size_t HEAD_BYTES = 4096;            // 4 counter words + 2 * MAX_N / 256 flags (516 ints), padded
constexpr size_t SLAB_BYTES = (size_t)MAX_N * sizeof(double);
constexpr size_t SCRATCH_BYTES = HEAD_BYTES + 3 * SLAB_BYTES;  // 1 576 960 bytes
static_assert((4 + 2 * (MAX_N / 256)) * sizeof(int) <= HEAD_BYTES, "counters and flags must fit the head of the scratch");
static_assert(SCRATCH_BYTES == SWEPT_STATIC_SCRATCH_BYTES, "include/swept.h states the size of the static scratch");

static __device__ __align__(256) unsigned char g_flow_static_scratch[SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_mutex;
unsigned char* g_scratch_dev[MAX_DEVICES] = {};  // device address of the array, per device ordinal

int fail(int code, const char* msg) {
  swept::set_last_error(msg);
  return code;
}

// device address of the scratch on the CURRENT device (looked up once per device)
int scratch_address(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(SWEPT_ECUDA, "swept_heat_flow_static: cudaGetDevice failed (no CPU fallback exists)");
  if (dev < 0 || dev >= MAX_DEVICES) return fail(SWEPT_EUNSUPPORTED, "swept_heat_flow_static: device ordinal out of range");
  std::lock_guard<std::mutex> lock(g_mutex);
  if (!g_scratch_dev[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_flow_static_scratch);
    if (e != cudaSuccess || !p) {
      char buf[256];
      snprintf(buf, sizeof buf, "swept_heat_flow_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
      return fail(SWEPT_ECUDA, buf);
    }
    g_scratch_dev[dev] = (unsigned char*)p;
  }
  *out = g_scratch_dev[dev];
  return 0;
}

}  // namespace

extern "C" int swept_heat_flow_static(const double* in_dev, double* out_dev, int64_t N, int64_t nsteps,
                                      int32_t tile_width, double dx, double dt, double alpha, void* stream_) {
  char msg[320];
  if (!in_dev || !out_dev) return fail(SWEPT_EINVAL, "swept_heat_flow_static: null buffer");
  if (N <= 0 || N > MAX_N) {
    snprintf(msg, sizeof msg, "swept_heat_flow_static: N = %lld exceeds the static scratch (maximum N = %lld points); "
             "use swept_create / swept_run for larger problems", (long long)N, (long long)MAX_N);
    return fail(SWEPT_EINVAL, msg);
  }
  const int n = tile_width;
  if (n != 256 && n != 512 && n != 1024) return fail(SWEPT_EINVAL, "swept_heat_flow_static: tile_width must be 256, 512 or 1024");
  if (N % n) return fail(SWEPT_EINVAL, "swept_heat_flow_static: N must be a multiple of tile_width");
  const int64_t m = n / 2;  // sub-timesteps per row of tiles (h = 1)
  if (nsteps < m || nsteps % m) {
    snprintf(msg, sizeof msg, "swept_heat_flow_static: nsteps = %lld must be a positive multiple of tile_width / 2 = %lld "
             "(one Up .. Down cycle, no remainder)", (long long)nsteps, (long long)m);
    return fail(SWEPT_EINVAL, msg);
  }
  if (nsteps / m + 1 > (1 << 20)) return fail(SWEPT_EINVAL, "swept_heat_flow_static: too many rows of tiles in one cycle");
  if (!(dx > 0) || !(dt > 0)) return fail(SWEPT_EINVAL, "swept_heat_flow_static: dx and dt must be positive");
  const char* a0 = (const char*)in_dev;
  const char* b0 = (const char*)out_dev;
  const size_t bytes = (size_t)N * sizeof(double);
  if (a0 < b0 + bytes && b0 < a0 + bytes) return fail(SWEPT_EINVAL, "swept_heat_flow_static: in and out must not overlap");
  if (((uintptr_t)in_dev | (uintptr_t)out_dev) & 15) return fail(SWEPT_EINVAL, "swept_heat_flow_static: buffers must be 16-byte aligned");

  unsigned char* scratch = nullptr;
  if (int rc = scratch_address(&scratch)) return rc;
  cudaStream_t stream = (cudaStream_t)stream_;
  // The array keeps the last call's contents.  The counters and flags must start at zero (a launch leaves them zero
  // again, but a failed or aborted one may not): cleared here, on the caller's stream.  The row slabs need no clearing:
  // every slot a tile reads was written by its parents in this launch (swept_flow.cuh, hazards).
  cudaError_t e = cudaMemsetAsync(scratch, 0, HEAD_BYTES, stream);
  if (e != cudaSuccess) {
    snprintf(msg, sizeof msg, "swept_heat_flow_static: clearing the counters: %s", cudaGetErrorString(e));
    return fail(SWEPT_ECUDA, msg);
  }
  double* slab[3];
  for (int i = 0; i < 3; ++i) slab[i] = (double*)(scratch + HEAD_BYTES + (size_t)i * SLAB_BYTES);

  // scheme constants as swept_create computes them (Eq. (B.4))
  const double Fo = alpha * dt / (dx * dx);
  const double consts[5] = {Fo, 1.0 - 2.0 * Fo, 0, 0, 0};

  swept::FlowLaunch f{};
  f.init = in_dev;
  f.N = N;
  f.n = n;
  f.rows = (int)(nsteps / m) + 1;  // Up + D diamond rows + Down = D + 2, T = (D + 1) m
  // row r writes buffer r & 1; the Down row (r = rows - 1) leaves the full time level in row 0 of its buffer: that
  // slab is the caller's output, the other three are in the static scratch
  const int last = (f.rows - 1) & 1;
  f.buf[last][0] = out_dev;
  f.buf[last][1] = slab[0];
  f.buf[1 - last][0] = slab[1];
  f.buf[1 - last][1] = slab[2];
  f.ticket = (unsigned*)scratch;
  f.flags = (int*)scratch + 4;
  f.ctas_per_sm = 0;  // library default: resident CTAs from the tiles per row
  f.consts = consts;
  f.stream = stream;
  int rc;
  switch (n / 32) {
    case 8: rc = swept::flow_go<swept::Heat<double>, 8, true>(f); break;
    case 16: rc = swept::flow_go<swept::Heat<double>, 16, true>(f); break;
    default: rc = swept::flow_go<swept::Heat<double>, 32, true>(f); break;
  }
  if (rc == swept::NO_KERNEL) return fail(SWEPT_EUNSUPPORTED, "swept_heat_flow_static: no kernel for this configuration");
  if (rc != 0) {
    snprintf(msg, sizeof msg, "swept_heat_flow_static: launch: %s", cudaGetErrorString((cudaError_t)rc));
    return fail(SWEPT_ECUDA, msg);
  }
  return SWEPT_OK;
}

// did the last launches on this device give up waiting for a dependency?  (sticky word 1 of the counters)
extern "C" int swept_heat_flow_static_check(void* stream_) {
  unsigned char* scratch = nullptr;
  if (int rc = scratch_address(&scratch)) return rc;
  cudaStream_t stream = (cudaStream_t)stream_;
  int err = 0;
  cudaError_t e = cudaMemcpyAsync(&err, (int*)scratch + 1, sizeof(int), cudaMemcpyDeviceToHost, stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
  if (e != cudaSuccess) {
    char msg[256];
    snprintf(msg, sizeof msg, "swept_heat_flow_static_check: %s", cudaGetErrorString(e));
    return fail(SWEPT_ECUDA, msg);
  }
  if (err) return fail(SWEPT_ECUDA, "swept_heat_flow_static: a tile waited too long for its parents; the output is invalid");
  return SWEPT_OK;
}
