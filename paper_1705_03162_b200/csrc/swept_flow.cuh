// swept_flow.cuh — swept kernels, flavour FLOW: one whole swept cycle (UpTriangle, D Split/WholeDiamond rows,
// DownTriangle; §4.2-4.3) in ONE persistent launch, the rows chained by per-tile dependencies.
//
// The paper synchronises the rows of tiles by returning to the host between launches ("kernel calls are
// implicitly synchronized by returning control to the queue") and names a cheaper device-side
// synchronisation as future work.  What a tile of row r really needs is only the two tiles of
// row r-1 it overlaps (the edges it receives), not the whole row.  So here every tile of the
// cycle is a task (row-major ticket order, one atomic ticket counter); a WARP takes a ticket, waits until the
// two parent tiles have published their edges (one flag per tile, release/acquire at GPU scope), stages the
// tile's two rows from global memory into a private shared-memory slice with TMA 1-D bulk copies
// (cp.async.bulk, mbarrier completion), sweeps the tile exactly as the CHAR flavour does (swept_char.cuh:
// registers + shuffles, L = 32 lanes, B = n/32 lines per lane), writes the rows back with bulk stores and raises
// its flag.  (Staging the NEXT tile behind the sweep — two slices per warp — was built and measured: no gain at
// any size, because at the sizes where the next tile is ready early the load is 0.1 % of the tile time, and
// claiming a ticket ahead of time costs the dynamic balance.)  This removes the launch gaps, the load / compute / store serialisation of a
// whole row, and the load imbalance of 2^k equal tiles on 148 SMs (a fast SM simply takes the next ticket).
//
// Global state: the same two-row layout as the other flavours.  Row r of the cycle
// reads buffer (r-1)&1 and writes buffer r&1 (two rows each; the Up row reads the initial time level `init`,
// the Down row writes only row 0 = the full time level).  Tiling of row r is shifted by n/2 when r is odd
// (Up = row 0 aligned; the paper's half-tile shift).
//
// Hazards.  RAW: tile (r,k) reads [S-h, S+n+h) of buffer (r-1)&1, which lies inside the ranges of the two tiles
// of row r-1 that overlap [S, S+n) — its parents — and both have published (flag) before it loads.  WAR: tile
// (r,k) overwrites [S, S+n) of buffer r&1, last written by row r-2 and read by row r-1; the only tiles of row r-1
// whose reads (range plus h-wide halo) touch [S, S+n) are again the two parents, which finished reading before
// they published.  The Up row's input `init` may be one of the slabs of buffer 1: row 1 overwrites a range of it
// only after both Up tiles that read that range have published.  Deadlock freedom: tickets are taken in
// row-major order and a task only waits for tasks with smaller tickets, which are held by warps that are
// already running — the launch never exceeds the number of co-resident CTAs (host side: occupancy query).
#pragma once
#include "common.cuh"
#include "functors.cuh"
#include "swept_char.cuh"
#include "swept_cluster.cuh"

namespace swept {

template <class R>
struct FlowArgs {
  const R* init;  // full time level at the start of the cycle (C components, stride N)
  R* buf[2][2];   // [buffer][row]
  int64_t N;
  int K;          // tiles per row = N / n
  int rows;       // D + 2
  int* flags;     // 2 * K words, zero on entry: flags[(r & 1) * K + k] = r + 1 once tile (r, k) is in global memory.
                  // Reusing the slot two rows later is safe: tile (r+2, k) cannot finish before both children of
                  // tile (r, k) — the only readers of its flag — have finished.
  unsigned* ticket;  // ticket[0] = task counter, ticket[2] = warps that have left; both zero on entry.  The last
                     // warp to leave clears them and the flags again, so a launch needs no host-side reset and a
                     // captured launch can be replayed.  ticket[1] = sticky error word (a dependency wait timed
                     // out), read and cleared by the host.
  Consts<R> k;
  // PROF kernels only: 8 counters, summed over all warps — SM cycles spent [0] taking a ticket, [1] waiting for the
  // parents' flags, [2] staging the tile, [3] sweeping, [4] storing and publishing; [5] tiles done
  unsigned long long* prof;
  int bc;  // WALLS kernels: BC_MIRROR = insulated ends (heat, Eq. (B.5)); else 0
};

// polling load: relaxed at GPU scope (no L1 invalidation per poll); the acquire fence follows once the flag is seen
__device__ __forceinline__ int ld_relaxed_gpu(const int* p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// 16-byte copies global <-> shared of `count` elements starting at global element g0 (periodic in N; g0 and the
// wrap point are multiples of the vector width), by the 32 lanes of a warp.  Loads bypass L1 (ld.global.cg):
// the data was written by other SMs during this launch.
template <class R>
__device__ __forceinline__ void warp_load_row(R* dst, const R* __restrict__ src, int64_t g0, int count, int64_t N,
                                              int lane) {
  constexpr int V = 16 / (int)sizeof(R);
  for (int i = lane * V; i < count; i += 32 * V) {
    int64_t g = g0 + i;
    if (g >= N) g -= N;
    const int4 t = __ldcg(reinterpret_cast<const int4*>(src + g));
    *reinterpret_cast<int4*>(dst + i) = t;
  }
}
template <class R>
__device__ __forceinline__ void warp_store_row(R* __restrict__ dst, const R* src, int64_t g0, int count, int64_t N,
                                               int lane) {
  constexpr int V = 16 / (int)sizeof(R);
  for (int i = lane * V; i < count; i += 32 * V) {
    int64_t g = g0 + i;
    if (g >= N) g -= N;
    *reinterpret_cast<int4*>(dst + g) = *reinterpret_cast<const int4*>(src + i);
  }
}

// Predicated forms of the bulk-copy primitives (common.cuh): the FLOW kernel issues them from lane 0 WITHOUT a C++
// branch.  With `if (lane == 0) { ... }` around them the compiler could no longer prove the warp converged at the sweep's
// shuffles and guarded each with a divergence test (BRA.DIV + out-of-line WARPSYNC.COLLECTIVE): 134 instead of 118
// instructions per pair of steps and 78 registers.
__device__ __forceinline__ void bulk_g2s_if(bool p, void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
  asm volatile(
      "{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %4, 0;\n\t"
      "@q cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n\t}" ::"r"(
          smem_u32(dst_smem)),
      "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "r"((uint32_t)p)
      : "memory");
}
__device__ __forceinline__ void bulk_s2g_if(bool p, void* dst_gmem, const void* src_smem, uint32_t bytes) {
  asm volatile(
      "{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %3, 0;\n\t"
      "@q cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n\t}" ::"l"(dst_gmem),
      "r"(smem_u32(src_smem)), "r"(bytes), "r"((uint32_t)p)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx_if(bool p, uint64_t* bar, uint32_t bytes) {
  asm volatile(
      "{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %2, 0;\n\t"
      "@q mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n\t}" ::"r"(smem_u32(bar)),
      "r"(bytes), "r"((uint32_t)p)
      : "memory");
}
__device__ __forceinline__ void st_release_gpu_if(bool p, int* ptr, int v) {
  asm volatile(
      "{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %2, 0;\n\t"
      "@q st.release.gpu.global.s32 [%0], %1;\n\t}" ::"l"(ptr),
      "r"(v), "r"((uint32_t)p)
      : "memory");
}

// TMA 1-D bulk copies of `len` elements starting at global element g0 of a periodic row of N elements (g0 may be
// negative by less than N); g0, len and N are multiples of the 16-byte granule, so every piece is aligned.
template <class R>
__device__ __forceinline__ void bulk_load_wrapped(bool p, R* dst, const R* __restrict__ src, int64_t g0, int len, int64_t N,
                                                  uint64_t* bar) {
  // at most three pieces (len <= N + 2 pads; a single tile, n = N, wraps at both ends): up to the end of the row, a
  // whole row or the rest from its start, and what is still left from the start again
  const int64_t g = g0 < 0 ? g0 + N : g0;
  const int first = (int)((N - g) < (int64_t)len ? (N - g) : (int64_t)len);
  const int second = (int)((int64_t)(len - first) < N ? (int64_t)(len - first) : N);
  const int third = len - first - second;
  bulk_g2s_if(p, dst, src + g, (uint32_t)(first * sizeof(R)), bar);
  bulk_g2s_if(p && second > 0, dst + first, src, (uint32_t)(second * sizeof(R)), bar);
  bulk_g2s_if(p && third > 0, dst + first + second, src, (uint32_t)(third * sizeof(R)), bar);
}
template <class R>
__device__ __forceinline__ void bulk_store_wrapped(bool p, R* __restrict__ dst, const R* src, int64_t g0, int len, int64_t N) {
  const int first = (int)((N - g0) < (int64_t)len ? (N - g0) : (int64_t)len);
  bulk_s2g_if(p, dst + g0, src, (uint32_t)(first * sizeof(R)));
  bulk_s2g_if(p && len > first, dst, src + first, (uint32_t)((len - first) * sizeof(R)));
}
// orders this thread's generic-proxy view against the async (TMA) proxy, all state spaces: after a flag has been
// acquired and before a bulk load of what it guards; after bulk stores have completed and before the flag is raised
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

// A tile that touches a wall (non-periodic ends, row f1): "node 0 is split across the spatial boundary and must apply the
// boundary conditions at its center".  The characteristic sweep cannot run through a wall (its lines
// reflect there), so the warp that draws such a tile advances it tier by tier in its shared-memory slice, as the TIER
// flavour does for a whole CTA: lane l owns the P = n/32 points l P .. l P + P - 1, a tier reads the other row, and the
// insulated ends T_{-1} = T_1, T_N = T_{N-2} (Eq. (B.5)) are applied where the stencil would cross the wall:
//   wl / wr : the tile's first / last point is the domain's (aligned rows: the first / last tile of the row);
//   split   : the tile wraps, point N-1 sits at slot n/2 - 1 and point 0 at slot n/2 (shifted rows: the last tile).
// One __syncwarp() per tier; the same tier ranges and the same Heat::point as every other flavour, so the same bits.
// Points are dealt to the lanes in quads, round-robin (lane l owns points 4 l .. 4 l + 3, 128 + 4 l .., ...: consecutive
// lanes touch consecutive 16-byte words — with a block of n/32 points per lane every access was a 32-way bank conflict and
// a wall tile took 5.5 tile times); all loads of a tier are issued before its first store (a skip of the groups outside
// the tier's range was tried: the branches serialise the loads and cost more than they save).
// The wall tiles of successive rows depend on one another, so rows x (time of a wall tile) bounds the launch from
// below.  Through shared memory a wall tile computes every point at every tier (1.8 x the arithmetic of a swept tile) on
// a scheduler it shares with two sweeping warps: 1.6 (n = 256) to 2 (n = 512) tile times.  For n = 256 the tile is
// therefore kept in the warp's REGISTERS (the B == 8 branch below: the CLUSTER flavour's tier): 0.9 tile times, and walls
// cost nothing any more (insulated heat N = 2^20, n = 256: 3.54e12, the periodic run's figure; N = 2^17: 8.3e11 against
// 4.5e11 through shared memory).
template <class Prob, int B, int KIND>
__device__ __forceinline__ void flow_wall_tile(typename Prob::R* rows, const int RS, const int pad, const int lane,
                                               const bool wl, const bool wr, const bool split,
                                               const Consts<typename Prob::R>& k) {
  using R = typename Prob::R;
  static_assert(Prob::H == 1 && Prob::C == 1 && Prob::SIGMA == 1, "walls in the FLOW flavour: the heat problem");
  constexpr int n = 32 * B, m = n / 2;
  const int ntiers = KIND == KIND_UP ? m - 1 : (KIND == KIND_DOWN ? m : 2 * m - 1);
  if constexpr (B == 8) {
    // n = 256: the tile fits the warp's registers (8 points of both rows per lane): the tiers run as in the CLUSTER
    // flavour (swept_cluster.cuh: one shuffle exchange per tier, no shared-memory round trip, no warp barrier), the
    // walls are its lane selects.  The wall tiles of successive rows form the critical path at N <= 2^19, so their
    // latency is what counts.
    constexpr int P = B;
    R v0[1][P], v1[1][P], hl0[1][1], hr0[1][1], hl1[1][1], hr1[1][1];
    R* r0 = rows + pad;
    R* r1 = rows + RS + pad;
#pragma unroll
    for (int j = 0; j < P; ++j) {
      v0[0][j] = r0[lane * P + j];
      v1[0][j] = r1[lane * P + j];
    }
    hl0[0][0] = r0[-1]; hr0[0][0] = r0[n];
    hl1[0][0] = r1[-1]; hr1[0][0] = r1[n];
    int ta[P];
    unsigned span[P];
#pragma unroll
    for (int j = 0; j < P; ++j) {  // tier window of each point (as swept_cluster_kernel)
      const int x = lane * P + j;
      const int d = x < n / 2 ? n / 2 - x : x - n / 2 + 1;
      const int edge = x < n - 1 - x ? x : n - 1 - x;
      const int t0 = KIND == KIND_UP ? 1 : d;
      const int tb = KIND == KIND_UP ? edge : (KIND == KIND_DOWN ? m : 2 * m - d);
      const bool never = tb < t0;
      span[j] = never ? 0u : (unsigned)(tb - t0);
      ta[j] = never ? (1 << 30) : t0;
    }
    const bool wall_l = split ? lane == 16 : (wl && lane == 0);
    const bool wall_r = split ? lane == 15 : (wr && lane == 31);
    const TierLanes TL = tier_lanes(lane);
    for (int t = 1; t <= ntiers; t += 2) {
      cluster_tier<Prob, P, true>(v0, v1, v0, hl0, hr0, 1, t, ta, span, TL, k, wall_l, wall_r);
      if (t + 1 <= ntiers) cluster_tier<Prob, P, true>(v1, v0, v0, hl1, hr1, 0, t + 1, ta, span, TL, k, wall_l, wall_r);
    }
#pragma unroll
    for (int j = 0; j < P; ++j) {
      r0[lane * P + j] = v0[0][j];
      r1[lane * P + j] = v1[0][j];
    }
    __syncwarp();
    return;
  }
  for (int t = 1; t <= ntiers; ++t) {
    // (source and destination are different rows: all loads of a tier are issued before its first store)
    const R* __restrict__ src = rows + ((t - 1) & 1) * RS + pad;  // phases start on even tiers: odd tiers read row 0
    R* __restrict__ dst = rows + (t & 1) * RS + pad;
    int lo, hi;
    tier_range<KIND>(t, n, 1, m, lo, hi);
    // lane l owns the quads of consecutive points 4 (32 g + l) .. + 3, g < B/4: one 16-byte-vector load of the quad (two
    // for FP64) and its two outer neighbours instead of three loads per point; every quad, in range or not (no branch,
    // so that the loads of a tier overlap)
    R o[B];
#pragma unroll
    for (int g = 0; g < B / 4; ++g) {
      const int q0 = 4 * (g * 32 + lane);
      alignas(16) R body[4];
      constexpr int NV = (int)(4 * sizeof(R) / 16);
#pragma unroll
      for (int v = 0; v < NV; ++v)
        reinterpret_cast<int4*>(body)[v] = reinterpret_cast<const int4*>(src + q0)[v];
      R left = src[q0 - 1], right = src[q0 + 4];
      if ((wl && q0 == 0) || (split && q0 == n / 2)) left = body[1];                   // T_{-1} = T_1
      if ((wr && q0 + 4 == n) || (split && q0 + 4 == n / 2)) right = body[2];          // T_N = T_{N-2}
      o[4 * g + 0] = Prob::point(left, body[0], body[1], k);
      o[4 * g + 1] = Prob::point(body[0], body[1], body[2], k);
      o[4 * g + 2] = Prob::point(body[1], body[2], body[3], k);
      o[4 * g + 3] = Prob::point(body[2], body[3], right, k);
    }
#pragma unroll
    for (int g = 0; g < B / 4; ++g)
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int j = 4 * (g * 32 + lane) + e;
        if (j >= lo && j < hi) dst[j] = o[4 * g + e];
      }
    __syncwarp();
  }
}

#ifndef FLOW_MAX_SLEEP
#define FLOW_MAX_SLEEP 256
#endif

// TMA = true : the tile's rows are staged by cp.async.bulk loads completing on an mbarrier and written back by bulk
//              stores, issued by one lane;
// TMA = false: by 16-byte ld.global.cg / st.global of all 32 lanes.
// Same task loop, same sweep, same protocol.  Both are kept because the compiler's code for the sweep loop depends on
// which one surrounds it (profiles/r2_flow_phases.md); swept_autotune measures both.
// PROF = true: the same kernel with clock64() stamps between the parts of a task (swept_flow_profile; the timings
// in profiles/r2_flow_phases.md).
// WALLS = true: non-periodic ends (a.bc): the one or two tiles of a row that touch a wall go to flow_wall_tile.
template <class Prob, int B, bool TMA, bool PROF = false, bool WALLS = false>
__global__ void __launch_bounds__(128) swept_flow_kernel(const FlowArgs<typename Prob::R> a) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C, PAD = Pad16<R>::value, L = 32;
  constexpr int n = B * L;
  constexpr int RS = n + 2 * PAD;
  static_assert(H <= PAD, "the halo must fit the 16-byte pad of a staged row");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  R* rows = reinterpret_cast<R*>(smem_raw) + (size_t)warp * 2 * C * RS;
  uint64_t* mbar = reinterpret_cast<uint64_t*>(smem_raw + (size_t)(blockDim.x >> 5) * 2 * C * RS * sizeof(R)) + warp;
  const int64_t N = a.N;
  const unsigned ntasks = (unsigned)a.rows * (unsigned)a.K;
  unsigned phase = 0;  // parity the mbarrier completes next
  long long pc[5] = {0, 0, 0, 0, 0}, ptiles = 0, t0 = 0, t1 = 0;
  (void)pc; (void)ptiles; (void)t0; (void)t1;
  if constexpr (TMA) {
    if (lane == 0) {
      mbar_init(mbar, 1);
      fence_mbar_init();
    }
    __syncwarp();
  }

  for (;;) {
    if constexpr (PROF) t0 = clock64();
    unsigned t = 0;
    if (lane == 0) t = atomicAdd(a.ticket, 1u);
    t = __shfl_sync(0xffffffffu, t, 0);
    if (t >= ntasks) break;
    if constexpr (PROF) { t1 = clock64(); pc[0] += t1 - t0; t0 = t1; }
    const int r = (int)(t / (unsigned)a.K);
    int k = (int)(t % (unsigned)a.K);
    if constexpr (WALLS) {
      // The wall tiles of successive rows depend on one another and each costs about two tile times: their chain is the
      // critical path of the launch.  Hand them out FIRST in every row (aligned rows: tiles 0 and K-1; shifted rows: the
      // split tile K-1), so that the chain runs beside the bulk of the row instead of after it.  Any order inside a row
      // keeps the protocol (a tile waits only for tiles of the previous row, which hold smaller tickets).
      if (a.K >= 2) {
        const int j = k;
        if (r & 1) k = j == 0 ? a.K - 1 : j - 1;
        else k = j == 0 ? 0 : (j == 1 ? a.K - 1 : j - 1);
      }
    }
    const int64_t S = (int64_t)k * n + ((r & 1) ? n / 2 : 0);  // < N; copies wrap
    if (r > 0) {
      // parents: the tiles of row r-1 overlapping [S, S+n); row r-1 publishes (r-1) + 1
      const int p0 = (r & 1) ? k : (k == 0 ? a.K - 1 : k - 1);
      const int p1 = (r & 1) ? (k + 1 == a.K ? 0 : k + 1) : k;
      const int* f = a.flags + (size_t)((r - 1) & 1) * a.K;
      unsigned ns = 32, polls = 0;
      bool dead = false;
      while (ld_relaxed_gpu(f + p0) < r || ld_relaxed_gpu(f + p1) < r) {
        __nanosleep(ns);
        if (ns < FLOW_MAX_SLEEP) ns *= 2;
        // cannot happen while the grid is co-resident; bounded so that a scheduling surprise yields an error
        // code (the next synchronising call reports it) instead of a hung device: 2^22 polls x >= 0.25 us.
        // A warp that gives up raises the sticky error word; every other waiting warp sees it and leaves too,
        // and nobody stores a tile computed from unready inputs.
        ++polls;
        if (polls > (1u << 22) || ((polls & 255u) == 0 && ld_relaxed_gpu((const int*)a.ticket + 1) != 0)) {
          if (lane == 0) atomicExch(a.ticket + 1, 1u);
          dead = true;
          break;
        }
      }
      if (dead) break;
      fence_acq_rel_gpu();
    }
    if constexpr (PROF) { t1 = clock64(); pc[1] += t1 - t0; t0 = t1; }
    // ---- stage the tile: both rows with their halo [S-h, S+n+h) (Up: row 0 of the initial level; the other row
    // is zero: tier -1 does not exist)
    const R* in0 = r == 0 ? a.init : ((r & 1) ? a.buf[0][0] : a.buf[1][0]);
    const R* in1 = (r & 1) ? a.buf[0][1] : a.buf[1][1];
    if constexpr (TMA) {
      // bulk loads over [S-PAD, S+n+PAD): the 16-byte pad holds the halo (what lies beyond it is never used)
      const bool issuer = lane == 0;  // the copies are issued by one lane, by predication, not by a branch
      fence_proxy_async_all();        // what the flags guard is read through the async proxy
      mbar_arrive_expect_tx_if(issuer, mbar, (uint32_t)((r == 0 ? 1 : 2) * C * RS * sizeof(R)));
#pragma unroll
      for (int c = 0; c < C; ++c) {
        bulk_load_wrapped<R>(issuer, rows + c * RS, in0 + (int64_t)c * N, S - PAD, RS, N, mbar);
        bulk_load_wrapped<R>(issuer && r != 0, rows + (C + c) * RS, in1 + (int64_t)c * N, S - PAD, RS, N, mbar);
      }
      if (r == 0)
        for (int i = lane; i < C * RS; i += 32) rows[C * RS + i] = (R)0;
      mbar_wait_warp(mbar, phase);
      phase ^= 1u;
    } else {
      if (r == 0) {
#pragma unroll
        for (int c = 0; c < C; ++c) warp_load_row<R>(rows + c * RS + PAD, in0 + (int64_t)c * N, S, n, N, lane);
        for (int i = lane; i < C * RS; i += 32) rows[C * RS + i] = (R)0;
      } else {
#pragma unroll
        for (int c = 0; c < C; ++c) {
          warp_load_row<R>(rows + c * RS + PAD, in0 + (int64_t)c * N, S, n, N, lane);
          warp_load_row<R>(rows + (C + c) * RS + PAD, in1 + (int64_t)c * N, S, n, N, lane);
        }
        if (lane < 2 * C * 2 * H) {
          const int rr = lane / (C * 2 * H), c = (lane / (2 * H)) % C, j = lane % (2 * H);
          int64_t g = (j < H) ? (S - H + j) : (S + n + (j - H));  // S < N, so one wrap suffices
          if (g < 0) g += N;
          if (g >= N) g -= N;
          const int sl = (j < H) ? (PAD - H + j) : (PAD + n + (j - H));
          rows[(rr * C + c) * RS + sl] = __ldcg((rr ? in1 : in0) + (int64_t)c * N + g);
        }
      }
    }
    __syncwarp();
    if constexpr (PROF) { t1 = clock64(); pc[2] += t1 - t0; t0 = t1; }
    // ---- sweep (identical arithmetic and order to the CHAR flavour)
    bool walled = false;
    if constexpr (WALLS) {
      const bool wl = !(r & 1) && k == 0, wr = !(r & 1) && k == a.K - 1, split = (r & 1) && k == a.K - 1;
      walled = wl || wr || split;
      if (walled) {
        if (r == 0) flow_wall_tile<Prob, B, KIND_UP>(rows, RS, PAD, lane, wl, wr, split, a.k);
        else if (r == a.rows - 1) flow_wall_tile<Prob, B, KIND_DOWN>(rows, RS, PAD, lane, wl, wr, split, a.k);
        else flow_wall_tile<Prob, B, KIND_WHOLE>(rows, RS, PAD, lane, wl, wr, split, a.k);
      }
    }
    if (walled) {
    } else if (r == 0) char_sweep_tile<Prob, B, L, KIND_UP, RS>(rows, RS, PAD + n / 2, lane, a.k);
    else if (r == a.rows - 1) char_sweep_tile<Prob, B, L, KIND_DOWN, RS>(rows, RS, PAD + n / 2, lane, a.k);
    else char_sweep_tile<Prob, B, L, KIND_WHOLE, RS>(rows, RS, PAD + n / 2, lane, a.k);
    if constexpr (PROF) { __syncwarp(); t1 = clock64(); pc[3] += t1 - t0; t0 = t1; }
    // ---- publish: the rows over [S, S+n), then the flag
    R* out0 = (r & 1) ? a.buf[1][0] : a.buf[0][0];
    R* out1 = (r & 1) ? a.buf[1][1] : a.buf[0][1];
    if constexpr (TMA) {
      fence_proxy_async_smem();
      __syncwarp();
      const bool issuer = lane == 0;
#pragma unroll
      for (int c = 0; c < C; ++c) {
        bulk_store_wrapped<R>(issuer, out0 + (int64_t)c * N, rows + c * RS + PAD, S, n, N);
        // Down leaves only row 0: the full time level
        bulk_store_wrapped<R>(issuer && r != a.rows - 1, out1 + (int64_t)c * N, rows + (C + c) * RS + PAD, S, n, N);
      }
      bulk_commit();    // (a lane without copies commits and waits for an empty group)
      bulk_wait_all();  // the writes are complete (not just the shared-memory reads)
      fence_proxy_async_all();
      st_release_gpu_if(issuer, a.flags + (size_t)(r & 1) * a.K + k, r + 1);
    } else {
      __syncwarp();
#pragma unroll
      for (int c = 0; c < C; ++c) {
        warp_store_row<R>(out0 + (int64_t)c * N, rows + c * RS + PAD, S, n, N, lane);
        if (r != a.rows - 1) warp_store_row<R>(out1 + (int64_t)c * N, rows + (C + c) * RS + PAD, S, n, N, lane);
      }
      __syncwarp();
      if (lane == 0) {
        __threadfence();
        st_release_gpu(a.flags + (size_t)(r & 1) * a.K + k, r + 1);
      }
    }
    __syncwarp();  // the slice is restaged by the next task of this warp
    if constexpr (PROF) { t1 = clock64(); pc[4] += t1 - t0; ++ptiles; }
  }
  if constexpr (PROF) {
    if (lane == 0 && a.prof) {
#pragma unroll
      for (int i = 0; i < 5; ++i) atomicAdd(a.prof + i, (unsigned long long)pc[i]);
      atomicAdd(a.prof + 5, (unsigned long long)ptiles);
    }
  }
  // Leave the scratch as it was found.  A warp arrives here after its last task is in global memory; the warp that
  // arrives last therefore knows that every task of the launch is done.
  unsigned gone = 0;
  if (lane == 0) gone = atomicAdd(a.ticket + 2, 1u);
  gone = __shfl_sync(0xffffffffu, gone, 0);
  if (gone == gridDim.x * (blockDim.x >> 5) - 1) {
    for (int i = lane; i < 2 * a.K; i += 32) a.flags[i] = 0;
    if (lane == 0) {
      a.ticket[2] = 0;
      a.ticket[0] = 0;
    }
  }
}

template <class Prob>
inline size_t flow_smem_bytes(int warps, int n) {
  using R = typename Prob::R;
  return (size_t)warps * (2 * Prob::C * ((size_t)n + 2 * Pad16<R>::value) * sizeof(R) + 8);
}

}  // namespace swept
