// internal.h — host-side launcher interface between swept_api.cu and the per-problem kernel files.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace swept {

struct PerStepLaunch {
  const void* in;
  const void* base;
  void* out;
  int64_t N;
  int odd;
  int threads;  // threads per block
  int P;        // points per thread (N % P == 0)
  const double* consts;  // 5 doubles, rounded once to REAL by the launcher
  cudaStream_t stream;
  int bc = 0;   // kernel boundary mode: 0 wrap, 1 mirror (heat B.5), 2 fixed end states (Euler tube)
  const double* bcv = nullptr;  // bc == 2: left[3], right[3] end states
};

struct TileLaunch {
  int kind;  // KIND_*
  const void* in0;
  const void* in1;
  void* out0;
  void* out1;
  int64_t N;
  int n, shift, ntiers;
  int P;       // TIER: points per thread.  CHAR: lanes per tile (L)
  int flavor;  // SWEPT_FLAVOR_TIER / SWEPT_FLAVOR_CHAR
  const double* consts;
  cudaStream_t stream;
  int bc = 0;  // kernel boundary mode (TIER flavour only): 0 wrap, 1 mirror, 2 fixed end states
  const double* bcv = nullptr;
  // hybrid wall handling: TIER launches only the tiles tile_base + b * tile_step, b < tile_count (0 = all tiles);
  // CHAR leaves the first / last tile of the row unwritten
  int tile_base = 0, tile_step = 1, tile_count = 0;
  int skip_first = 0, skip_last = 0;
  // three-row schemes (KS3: three sub-timesteps per timestep): the third row, and the global tier of the phase's
  // relative tier 0 modulo 3 (which stage its first tier is)
  const void* in2 = nullptr;
  void* out2 = nullptr;
  int tmod = 0;
};

// FLOW flavour: one whole Up / diamonds / Down cycle of tile width n in a single persistent launch
struct FlowLaunch {
  const void* init;  // full time level at the start of the cycle
  void* buf[2][2];   // [buffer][row]; row r of the cycle writes buffer r & 1
  int64_t N;
  int n, rows;       // tile width; rows = D + 2
  int* flags;        // 2 * N/n words, zero (the kernel leaves them zero again; swept_flow.cuh)
  unsigned* ticket;  // 4 words: task counter, sticky error word, leave counter, unused; counters zero
  int ctas_per_sm;   // bits 0..3: resident CTAs (of 4 warps) per SM, 0 = default policy; bit 4: TMA staging
  unsigned long long* prof = nullptr;  // 8 device counters: run the instrumented kernel (swept_flow_profile)
  int bc = 0;        // kernel boundary mode: 0 wrap, 1 mirror (insulated heat ends: wall tiles advance tier by tier)
  const double* consts;
  cudaStream_t stream;
};

// CLUSTER flavour: one whole Up / diamonds / Down cycle of tile width n in a single launch of one thread-block cluster
struct ClusterLaunch {
  const void* init;  // full time level at the start of the cycle
  void* out;         // full time level at its end (another slab)
  int64_t N;
  int n, rows;       // tile width; rows = D + 2
  int warps_per_cta; // 0 = as few as fit a cluster of 16 CTAs
  int bc = 0;        // kernel boundary mode: 0 wrap, 1 mirror (insulated heat ends)
  const double* consts;
  cudaStream_t stream;
};

// resident per-step: all sub-timesteps in one persistent cooperative launch (per_step_resident.cuh)
struct ResidentLaunch {
  const void* in;
  void* out;
  int64_t N, nsteps;
  void* xch;       // device scratch, resident_scratch_bytes() bytes, 16-byte aligned; first the flags
  const double* consts;
  cudaStream_t stream;
  int bc = 0;      // kernel boundary mode (0 wrap, 1 mirror, 2 fixed end states)
  const double* bcv = nullptr;
};
// scratch needed for at most `max_ctas` CTAs (flags + error word, then the exchange slots of the widest problem)
// layout: one 128-byte line per CTA flag, one line for the error word, then 2 x max_ctas x 2 exchange lines
inline size_t resident_flag_bytes(int max_ctas) { return (size_t)(max_ctas + 1) * 128; }
inline size_t resident_scratch_bytes(int max_ctas) {
  return resident_flag_bytes(max_ctas) + (size_t)2 * max_ctas * 2 * 128;
}
constexpr int RESIDENT_MAX_CTAS = 4096;

// edge of a shard <-> contiguous message buffer (shard_kernels.cu)
struct ShardCopy {
  void* rows[3];   // row slabs (nrows of them used), component c at rows[r] + c * Next elements
  int nrows, C;
  int64_t Next;    // points of the shard's extended (own + ghost) array
  int64_t off;     // first local point of the edge (periodic in Next; may be negative)
  int count;       // points
  void* buf;       // device buffer of nrows * C * count elements, [row][component][point]
  int elem;        // bytes per element (8 or 4)
  cudaStream_t stream;
  bool pack;       // true: rows -> buf; false: buf -> rows
};
int launch_shard_copy(const ShardCopy& a);

// dtype: 0 f64, 1 f32.  rk2: 0 midpoint, 1 Heun.  Return cudaError_t as int, or -1000 if the
// combination has no kernel.
int launch_per_step_heat(int dtype, const PerStepLaunch& a);
int launch_per_step_ks(int dtype, int rk2, const PerStepLaunch& a);
int launch_per_step_ks_fused(int dtype, int rk2, const PerStepLaunch& a);  // both stages of a timestep in one launch
int launch_per_step_euler(int dtype, int rk2, const PerStepLaunch& a);
int launch_tile_heat(int dtype, const TileLaunch& a);
int launch_tile_ks(int dtype, int rk2, const TileLaunch& a);
int launch_tile_euler(int dtype, int rk2, const TileLaunch& a);
int launch_per_step_ks3(int dtype, const PerStepLaunch& a);  // a.odd = stage (1, 2, 0)
int launch_tile_ks3(int dtype, const TileLaunch& a);
bool tile_config_ok_ks3(int dtype, int flavor, int64_t N, int n, int P);
// does a kernel exist for (flavor, n, P)?  (host-only query used by the autotuner and argument checks)
int launch_resident_heat(int dtype, const ResidentLaunch& a);
int launch_resident_ks(int dtype, int rk2, const ResidentLaunch& a);
int launch_resident_euler(int dtype, int rk2, const ResidentLaunch& a);
int launch_flow_heat(int dtype, const FlowLaunch& a);
int launch_flow_ks(int dtype, int rk2, const FlowLaunch& a);
int launch_cluster_heat(int dtype, const ClusterLaunch& a);
int launch_cluster_ks(int dtype, int rk2, const ClusterLaunch& a);
int launch_cluster_ks3(int dtype, const ClusterLaunch& a);
bool tile_config_ok_heat(int dtype, int flavor, int64_t N, int n, int P);
bool tile_config_ok_ks(int dtype, int flavor, int64_t N, int n, int P);
bool tile_config_ok_euler(int dtype, int flavor, int64_t N, int n, int P);

constexpr int NO_KERNEL = -1000;

// sets the thread-local text swept_last_error() returns (for entry points that live outside swept_api.cu)
void set_last_error(const char* msg);

}  // namespace swept
