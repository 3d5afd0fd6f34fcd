// swept_cluster.cuh — swept kernels, flavour CLUSTER: the WHOLE domain inside one thread-block cluster, for the
// small problems where every other flavour is bound by latency, not by arithmetic (BASELINE.json config 1: N = 2048).
//
// The paper names a device-side synchronisation between the rows of tiles as future work and its
// "Register" variant keeps a 32-point tile in the registers of one warp.  Here:
//   * one WARP per tile ("node") of n = 32 P points; lane l holds the P contiguous points l P .. l P + P - 1 of both
//     rows of the two-row working array in registers;
//   * a tier is one shuffle exchange of the h values either side of a lane's block and P stencil evaluations — no
//     block barrier, no shared-memory traffic inside a phase; the tile's outermost h halo values are read once per
//     phase (they do not change during it);
//   * the whole cycle — UpTriangle, D Split/WholeDiamond rows, DownTriangle (§4.2) — runs in ONE launch: a
//     tile that finishes a row PUSHES the left half of its two rows into a receive buffer in the shared memory of the
//     warp that continues them (half a tile to the left), the right half to the warp half a tile to the right
//     (the edges a node passes on) — st.async through the cluster's distributed shared memory, possibly
//     into a neighbouring SM, each store counting its bytes on the receiver's mbarrier.  The receiver waits on its own
//     barrier for its two producers only and reads its own shared memory: no cluster-wide barrier, no fence, no remote
//     load between rows (the first version had all three: 1.3 k cycles per row).
//     Global memory is touched twice: the Up row reads the time level, the Down row writes it.
//   * receive buffers ping-pong with the row's parity; a buffer is rewritten only by tiles that consumed this warp's
//     output of the row that read it (see the hand-off comment below).
// What it buys: a tier costs a shuffle round trip plus one dependent DADD -> DFMA -> select (64 cycles measured for one
// point per lane) instead of the 130 cycles per tier the characteristic sweep needs at N = 2048 (its skew and chain
// latency), and no launch gap or L2 round trip between rows.  Lane efficiency is the paper's ~50 %;
// irrelevant here, because the bound at these sizes is the dependent chain, not the FP64 pipe.  Same
// functors, so the same bits.
#pragma once
#include <cooperative_groups.h>
#include <type_traits>

#include "common.cuh"
#include "functors.cuh"
#include "swept_tier.cuh"

namespace swept {

template <class R>
struct ClusterArgs {
  const R* init;  // full time level at the start of the cycle (C components, stride N)
  R* out;         // full time level at its end
  int64_t N;
  int n;          // tile width = 32 P
  int rows;       // D + 2
  Consts<R> k;
  int bc = 0;  // BC_MIRROR: insulated ends (heat, Eq. (B.5)), applied by the lanes next to a wall
};

__device__ __forceinline__ double shfl_idx_(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ float shfl_idx_(float v, int src) { return __shfl_sync(0xffffffffu, v, src); }

// One tier of a warp's tile: source row vs (tier t-1), destination row vd (tier t; holds tier t-2 before), halo values
// of the source row beyond the tile's ends in hl / hr.  Point j of the lane is updated when relative tier t lies in
// its window [ta[j], ta[j] + span[j]] (the tier ranges of swept_tier.cuh turned round: per point instead of per tier,
// so that the test is one subtraction and one compare on plain registers).
// which lanes a lane exchanges with, and whether it takes the tile's outer halo instead (lanes 0 / 31 by default)
struct TierLanes {
  int srcL, srcR;      // source lanes of the left / right neighbour values
  bool use_hl, use_hr; // this lane's left / right neighbour lies beyond the tile
};
__device__ __forceinline__ TierLanes tier_lanes(int lane) {
  return TierLanes{(lane + 31) & 31, (lane + 1) & 31, lane == 0, lane == 31};
}

template <class Prob, class = void> struct HasStageIf { static constexpr bool value = false; };
template <class Prob> struct HasStageIf<Prob, std::enable_if_t<Prob::HAS_STAGE_IF>> { static constexpr bool value = true; };

// HALO = false: a tier on which no active point reads beyond the tile's ends (every tier of a triangle or diamond but
// the full-width one, tier m): lanes 0 and 31 take the shuffle's wrapped-round value, which only inactive points read.
template <class Prob, int P, bool WALLS = false, bool HALO = true>
__device__ __forceinline__ void cluster_tier(const typename Prob::R (&vs)[Prob::C][P], typename Prob::R (&vd)[Prob::C][P],
                                             const typename Prob::R (&v0)[Prob::C][P],
                                             const typename Prob::R (&hl)[Prob::C][Prob::H],
                                             const typename Prob::R (&hr)[Prob::C][Prob::H], const int par, const int t,
                                             const int (&ta)[P], const unsigned (&span)[P], const TierLanes& L,
                                             const Consts<typename Prob::R>& k, const bool wall_l = false,
                                             const bool wall_r = false) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C;
  R win[C][P + 2 * H], bs[C][P], o[C][P];
#pragma unroll
  for (int c = 0; c < C; ++c) {
#pragma unroll
    for (int e = 0; e < H; ++e) {
      // left neighbours: the top H values of lane - 1; right neighbours: the bottom H values of lane + 1
      const R fromL = shfl_idx_(vs[c][P - H + e], L.srcL);
      const R fromR = shfl_idx_(vs[c][e], L.srcR);
      win[c][e] = (HALO && L.use_hl) ? hl[c][e] : fromL;
      win[c][H + P + e] = (HALO && L.use_hr) ? hr[c][e] : fromR;
    }
#pragma unroll
    for (int j = 0; j < P; ++j) {
      win[c][H + j] = vs[c][j];
      bs[c][j] = (Prob::SIGMA >= 2 && par != 1) ? v0[c][j] : vs[c][j];  // u^n: row 0
    }
    if constexpr (WALLS && H == 1 && P > 2) {
      // (P <= 2: the mirror point is what a shuffle from another SOURCE LANE delivers — the caller sets L.srcL / L.srcR
      // of the wall lanes and nothing is selected per tier)
      // (compiled only into the kernels that run with walls: the selects cost the periodic run 5-12 % at N <= 2^14)
      // a lane whose first / last point is an END POINT of the domain: the stencil's outer value is the mirror image
      // of its own second / second-to-last point, T_{-1} = T_1 and T_N = T_{N-2} (Eq. (B.5), reading X17)
      // (written on the window, so that P = 1 — the neighbour point lives in the next lane — needs no other case)
      win[c][0] = wall_l ? win[c][2] : win[c][0];
      win[c][P + 1] = wall_r ? win[c][P - 1] : win[c][P + 1];
    }
  }
  if constexpr (HasStageIf<Prob>::value) {
    unsigned rel[P];
#pragma unroll
    for (int j = 0; j < P; ++j) rel[j] = (unsigned)(t - ta[j]);
    Prob::template stage_if<P>(win, bs, vd, par, k, rel, span);
  } else {
    Prob::template stage<P>(win, bs, o, par, k);
#pragma unroll
    for (int j = 0; j < P; ++j) {
      const bool act = (unsigned)(t - ta[j]) <= span[j];
#pragma unroll
      for (int c = 0; c < C; ++c) vd[c][j] = act ? o[c][j] : vd[c][j];
    }
  }
}

// threads per CTA (register budget: two rows of P points, the window and the tier windows per lane)
template <int P> struct ClusterMaxThreads { static constexpr int value = P >= 8 ? 256 : 512; };

// ---- hand-off between the rows of tiles: PUSHED, not fetched.  Every warp owns, in its CTA's shared memory, two
// receive buffers (rows ping-pong) of [2 rows][C][n + 2h] values, each with an mbarrier.  A tile that finishes a row
// stores the left half of its points (both rows of the working array) straight into the buffer of the tile that
// continues them — half a tile to the left — and the right half into the buffer of the tile half a tile to the right
// ("the edges a node passes on"), with st.async: each 8-byte store lands in the consumer's shared memory
// and counts its bytes on the consumer's mbarrier in one operation.  The consumer waits for (n + 2h) values per row and
// component on its OWN barrier and reads its OWN shared memory.  No cluster-wide barrier, no fence, no remote load: a
// row costs one store latency across the cluster (about 215 cycles) instead of release fence + cluster barrier (380) +
// remote load (215), and a warp waits for its two producers only.
//   Slots of a buffer row: point i of the consumer's tile at (i % P) * 32 + i / P (lane-major: conflict-free reads);
//   the h values left of the tile at n + e, the h values right of it at n + h + e.
//   Reuse: buffer b of a warp is written for row r + 1 by the row-r tiles and next for row r + 3 by row-(r + 2) tiles,
//   each of which consumed the output of this warp's row-(r + 1) tile — which read buffer b before it computed.
__device__ __forceinline__ uint32_t mapa_u32(uint32_t local_addr, uint32_t cta_rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(cta_rank));
  return r;
}
__device__ __forceinline__ void st_async_(uint32_t addr, double v, uint32_t bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(addr), "d"(v), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void st_async_(uint32_t addr, float v, uint32_t bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f32 [%0], %1, [%2];" ::"r"(addr), "f"(v), "r"(bar)
               : "memory");
}
// all lanes wait for the phase; a phase that does not complete within ~1 s is a bug: trap instead of hanging the GPU
__device__ __forceinline__ void mbar_wait_warp_bounded(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  int spins = 0;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"  // the producers sit in other CTAs
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    if (++spins > (1 << 22)) __trap();
  } while (!__all_sync(0xffffffffu, done));
}
__host__ __device__ constexpr int cluster_bar_bytes(int wpc) { return (wpc * 16 + 127) / 128 * 128; }

template <class Prob, int P, bool WALLS = false>
__global__ void __launch_bounds__(ClusterMaxThreads<P>::value) swept_cluster_kernel(const ClusterArgs<typename Prob::R> a) {
  namespace cg = cooperative_groups;
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C;
  static_assert(Prob::ROWS == 2, "two-row schemes");
  static_assert(P >= H, "a lane's block must hold its neighbour's halo");
  constexpr int n = 32 * P, m = n / (2 * H);
  constexpr int W = n + 2 * H;                              // slots per (row, component)
  constexpr int BUF = 2 * C * W;                            // values per receive buffer
  constexpr uint32_t TX = (uint32_t)(BUF * sizeof(R));      // bytes a tile receives per row of tiles
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cg::cluster_group cluster = cg::this_cluster();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int wpc = blockDim.x >> 5;
  const unsigned rank = cluster.block_rank();
  const int64_t N = a.N;
  const int K = (int)(N / n);
  const int k_tile = (int)rank * wpc + warp;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);                      // [warp][buffer]
  R* recv = reinterpret_cast<R*>(smem_raw + cluster_bar_bytes(wpc));          // [warp][buffer][row][C][W]
  const uint32_t smem_base = smem_u32(smem_raw);
  // shared-memory offsets (bytes from smem_raw) of warp w's barrier / receive buffer b: the same in every CTA
  auto bar_off = [&](int w, int b) -> uint32_t { return (uint32_t)((w * 2 + b) * 8); };
  auto buf_off = [&](int w, int b) -> uint32_t {
    return (uint32_t)cluster_bar_bytes(wpc) + (uint32_t)((w * 2 + b) * BUF * (int)sizeof(R));
  };
  if (lane == 0) {
    mbar_init(&bars[warp * 2 + 0], 1);
    mbar_init(&bars[warp * 2 + 1], 1);
  }
  fence_mbar_init();
  cluster.sync();  // every barrier of the cluster exists before the first store can reach it
  if (lane == 0) {  // row 1 reads buffer 0, row 2 buffer 1
    if (a.rows > 1) mbar_arrive_expect_tx(&bars[warp * 2 + 0], TX);
    if (a.rows > 2) mbar_arrive_expect_tx(&bars[warp * 2 + 1], TX);
  }
  auto wrap = [&](int64_t g) -> int64_t { return g < 0 ? g + N : (g >= N ? g - N : g); };
  // Where this lane's values go, for an aligned (0) and a shifted (1) row of tiles; a row's parity is also its buffer.
  // Aligned tile k: its left half continues in shifted tile k - 1, its right half in shifted tile k; shifted tile k:
  // aligned tiles k and k + 1.  Lanes 0..15 hold the left half; lane 15's last h points are also the LEFT halo of the
  // right-hand consumer, lane 16's first h points the RIGHT halo of the left-hand one.  (wpc is a power of two.)
  uint32_t main_dst[2], main_bar[2], halo_dst[2], halo_bar[2];
  const int wshift = 31 - __clz(wpc);
#pragma unroll
  for (int p = 0; p < 2; ++p) {
    const int kL = p ? k_tile : (k_tile == 0 ? K - 1 : k_tile - 1);
    const int kR = p ? (k_tile == K - 1 ? 0 : k_tile + 1) : k_tile;
    const int mine = lane < 16 ? kL : kR, other = lane < 16 ? kR : kL;
    main_bar[p] = mapa_u32(smem_base + bar_off(mine & (wpc - 1), p), (uint32_t)(mine >> wshift));
    main_dst[p] = mapa_u32(smem_base + buf_off(mine & (wpc - 1), p), (uint32_t)(mine >> wshift)) +
                  (uint32_t)((lane ^ 16) * sizeof(R));
    halo_bar[p] = mapa_u32(smem_base + bar_off(other & (wpc - 1), p), (uint32_t)(other >> wshift));
    halo_dst[p] = mapa_u32(smem_base + buf_off(other & (wpc - 1), p), (uint32_t)(other >> wshift)) +
                  (uint32_t)((n + (lane == 16 ? H : 0)) * sizeof(R));
  }
  const R* recv_mine = recv + (size_t)(warp * 2) * BUF;
  uint64_t* bars_mine = bars + warp * 2;
  const int rows = a.rows;

  R v0[C][P], v1[C][P];  // row 0 (even tiers) and row 1 (odd tiers) of this lane's P points
  R hl0[C][H], hr0[C][H], hl1[C][H], hr1[C][H];
  int ta[P];           // tier window of each point of the lane (below), kept across the rows of one kind
  unsigned span[P];
  int window_kind = -1;
  for (int r = 0; r < rows; ++r) {
    const int kind = r == 0 ? KIND_UP : (r == rows - 1 ? KIND_DOWN : KIND_WHOLE);
    const int inb = (r + 1) & 1, outb = r & 1;
    // ---- the tile's rows (Up: the time level from global memory; tier -1 does not exist)
    if (kind == KIND_UP) {
      const int64_t g0 = (int64_t)k_tile * n + lane * P;  // row 0 is an aligned row
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int j = 0; j < P; ++j) {
          v0[c][j] = __ldg(a.init + (int64_t)c * N + g0 + j);
          v1[c][j] = (R)0;
        }
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int e = 0; e < H; ++e) hl0[c][e] = hr0[c][e] = hl1[c][e] = hr1[c][e] = (R)0;  // never used by a triangle
    } else {
      mbar_wait_warp_bounded(bars_mine + inb, (uint32_t)(((r - 1) >> 1) & 1));
      if (lane == 0 && r + 2 < rows) mbar_arrive_expect_tx(bars_mine + inb, TX);  // the buffer's next use
      const R* b0 = recv_mine + (size_t)inb * BUF;
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const R* q0 = b0 + (size_t)c * W;
        const R* q1 = b0 + (size_t)(C + c) * W;
#pragma unroll
        for (int j = 0; j < P; ++j) {
          v0[c][j] = q0[j * 32 + lane];
          v1[c][j] = q1[j * 32 + lane];
        }
#pragma unroll
        for (int e = 0; e < H; ++e) {  // the h-wide halo beyond either end of the tile, both rows (broadcast reads)
          hl0[c][e] = q0[n + e];
          hl1[c][e] = q1[n + e];
          hr0[c][e] = q0[n + H + e];
          hr1[c][e] = q1[n + H + e];
        }
      }
    }
    // ---- tiers (phases start on even global tiers, so odd relative tiers are predictor / odd-row tiers).
    // Tier window of every point x of the tile: Up (tier t covers [ht, n-ht)): 1 .. min(x, n-1-x)/h;
    // diamond (tier t covers the centre +- ht, then +- h(2m-t)): ceil(d/h) .. 2m - ceil(d/h) with d the
    // distance from the centre; Down: ceil(d/h) .. m.
    const int ntiers = kind == KIND_UP ? m - 1 : (kind == KIND_DOWN ? m : 2 * m - 1);
    if (kind != window_kind) {  // the windows change with the kind of row only: three times per cycle
      window_kind = kind;
#pragma unroll
      for (int j = 0; j < P; ++j) {
        const int x = lane * P + j;
        const int d = x < n / 2 ? n / 2 - x : x - n / 2 + 1;
        const int first = (d + H - 1) / H;
        const int edge = (x < n - 1 - x ? x : n - 1 - x) / H;
        const int t0 = kind == KIND_UP ? 1 : first;
        const int tb = kind == KIND_UP ? edge : (kind == KIND_DOWN ? m : 2 * m - first);
        const bool never = tb < t0;  // the end points of an UpTriangle's base row
        span[j] = never ? 0u : (unsigned)(tb - t0);
        ta[j] = never ? (1 << 30) : t0;
      }
    }
    // (Two tiers behind one shuffle exchange — 2h redundant evaluations per lane instead of a second exchange — was
    // built and measured: no faster for the 3-point scheme, 3 % for the 5-point one; not kept.)
    // walls ("node 0 is split across the spatial boundary and must apply the boundary conditions at its center",
    // PAPER.md:79-81): aligned rows: point 0 is lane 0 of the first tile, point N-1 lane 31 of the last; shifted rows:
    // the last tile wraps, point N-1 is the last point of its lane 15 and point 0 the first of its lane 16
    const bool shifted = (r & 1) != 0;
    const bool wall_l = WALLS && a.bc != 0 && (shifted ? (k_tile == K - 1 && lane == 16) : (k_tile == 0 && lane == 0));
    const bool wall_r = WALLS && a.bc != 0 && (shifted ? (k_tile == K - 1 && lane == 15) : (k_tile == K - 1 && lane == 31));
    TierLanes L = tier_lanes(lane);
    if constexpr (WALLS && H == 1 && P <= 2) {
      // the mirror image by the shuffle's source lane: T_{-1} = T_1 is this lane's own second point (P = 2: the register
      // the left-going shuffle reads) or the next lane's point (P = 1); the same on the right.  A wall lane never takes
      // the tile's outer halo.
      if (wall_l) { L.srcL = P == 2 ? lane : (lane + 1) & 31; L.use_hl = false; }
      if (wall_r) { L.srcR = P == 2 ? lane : (lane + 31) & 31; L.use_hr = false; }
    }
    // The values beyond the tile's ends are read by active points on ONE tier only, the full-width tier m (an even one):
    // the loop is split round it so that every other tier runs without the two halo selects in its dependent chain.
    int t = 1;
#pragma unroll 1
    for (; t + 1 < m; t += 2) {  // tiers 1 .. m-2
      cluster_tier<Prob, P, WALLS, false>(v0, v1, v0, hl0, hr0, 1, t, ta, span, L, a.k, wall_l, wall_r);  // odd: 0 -> 1
      cluster_tier<Prob, P, WALLS, false>(v1, v0, v0, hl1, hr1, 0, t + 1, ta, span, L, a.k, wall_l, wall_r);  // even
    }
    cluster_tier<Prob, P, WALLS, false>(v0, v1, v0, hl0, hr0, 1, t, ta, span, L, a.k, wall_l, wall_r);  // tier m-1
    if (t + 1 <= ntiers)
      cluster_tier<Prob, P, WALLS, true>(v1, v0, v0, hl1, hr1, 0, t + 1, ta, span, L, a.k, wall_l, wall_r);  // tier m
#pragma unroll 1
    for (t += 2; t <= ntiers; t += 2) {  // tiers m+1 .. 2m-1 (diamonds)
      cluster_tier<Prob, P, WALLS, false>(v0, v1, v0, hl0, hr0, 1, t, ta, span, L, a.k, wall_l, wall_r);
      if (t + 1 <= ntiers)
        cluster_tier<Prob, P, WALLS, false>(v1, v0, v0, hl1, hr1, 0, t + 1, ta, span, L, a.k, wall_l, wall_r);
    }
    // ---- hand the rows on: Down leaves the full time level (row 0) in global memory
    if (kind == KIND_DOWN) {
      const int64_t S = wrap((int64_t)k_tile * n + (shifted ? n / 2 : 0));
      const int64_t g0 = wrap(S + lane * P);  // this lane's first point; its P points do not straddle the wrap
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int j = 0; j < P; ++j) a.out[(int64_t)c * N + g0 + j] = v0[c][j];
    } else {
      {
        const uint32_t bar = outb ? main_bar[1] : main_bar[0];
        const uint32_t dst = outb ? main_dst[1] : main_dst[0];
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int j = 0; j < P; ++j) {
            st_async_(dst + (uint32_t)((c * W + j * 32) * sizeof(R)), v0[c][j], bar);
            st_async_(dst + (uint32_t)(((C + c) * W + j * 32) * sizeof(R)), v1[c][j], bar);
          }
      }
      if (lane == 15 || lane == 16) {
        // lane 15: the last h points of the left half are the LEFT halo of the right-hand consumer;
        // lane 16: the first h points of the right half are the RIGHT halo of the left-hand consumer
        const uint32_t bar = outb ? halo_bar[1] : halo_bar[0];
        const uint32_t dst = outb ? halo_dst[1] : halo_dst[0];
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int e = 0; e < H; ++e) {
            const R x0 = lane == 15 ? v0[c][P - H + e] : v0[c][e];
            const R x1 = lane == 15 ? v1[c][P - H + e] : v1[c][e];
            st_async_(dst + (uint32_t)((c * W + e) * sizeof(R)), x0, bar);
            st_async_(dst + (uint32_t)(((C + c) * W + e) * sizeof(R)), x1, bar);
          }
      }
    }
  }
  cluster.sync();  // nobody leaves while a store into its shared memory may still be in flight
}

// ---------------------------------------------------------------------------------------------------------------
// The same for a scheme with THREE sub-timesteps per timestep on a three-row state (Prob::ROWS == 3: KS3, SURVEY.md
// §8(f) row f3).  Row p of a lane's registers holds the latest value with tier = p (mod 3); the tier with
// global index g reads row (g - 1) % 3, writes row g % 3, is stage g % 3 of its timestep (1, 2, 0) and takes u^n from
// row 0.  A cycle starts on a full time level, so row r >= 1 of tiles starts at global tier (r - 1) m (the Up row at 0),
// whose residue differs from row to row (m is a power of two): the tier loop is instantiated for the three residues and
// rotates the register rows statically.
template <class Prob, int P, int G>
__device__ __forceinline__ void cluster3_tier(typename Prob::R (&v)[3][Prob::C][P],
                                              const typename Prob::R (&hl)[3][Prob::C][Prob::H],
                                              const typename Prob::R (&hr)[3][Prob::C][Prob::H], const int t,
                                              const int (&ta)[P], const unsigned (&span)[P], const int lane,
                                              const Consts<typename Prob::R>& k) {
  constexpr int SRC = (G + 2) % 3;
  cluster_tier<Prob, P>(v[SRC], v[G], v[0], hl[SRC], hr[SRC], G, t, ta, span, tier_lanes(lane), k);
}

template <class Prob, int P, int Q0>
__device__ __forceinline__ void cluster3_tiers(typename Prob::R (&v)[3][Prob::C][P],
                                               const typename Prob::R (&hl)[3][Prob::C][Prob::H],
                                               const typename Prob::R (&hr)[3][Prob::C][Prob::H], const int ntiers,
                                               const int (&ta)[P], const unsigned (&span)[P], const int lane,
                                               const Consts<typename Prob::R>& k) {
  int t = 1;  // relative tier t has global residue (Q0 + t) % 3
  for (; t + 2 <= ntiers; t += 3) {
    cluster3_tier<Prob, P, (Q0 + 1) % 3>(v, hl, hr, t, ta, span, lane, k);
    cluster3_tier<Prob, P, (Q0 + 2) % 3>(v, hl, hr, t + 1, ta, span, lane, k);
    cluster3_tier<Prob, P, Q0 % 3>(v, hl, hr, t + 2, ta, span, lane, k);
  }
  if (t <= ntiers) cluster3_tier<Prob, P, (Q0 + 1) % 3>(v, hl, hr, t, ta, span, lane, k);
  if (t + 1 <= ntiers) cluster3_tier<Prob, P, (Q0 + 2) % 3>(v, hl, hr, t + 1, ta, span, lane, k);
}

template <class Prob, int P>
__global__ void __launch_bounds__(ClusterMaxThreads<P>::value) swept_cluster3_kernel(const ClusterArgs<typename Prob::R> a) {
  namespace cg = cooperative_groups;
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C;
  static_assert(Prob::ROWS == 3 && Prob::SIGMA == 3, "three sub-timesteps per timestep on three rows");
  static_assert(P >= H, "a lane's block must hold its neighbour's halo");
  constexpr int n = 32 * P, m = n / (2 * H);
  constexpr int W = n + 2 * H;                          // slots per (row, component)
  constexpr int BUF = 3 * C * W;                        // values per receive buffer: three rows
  constexpr uint32_t TX = (uint32_t)(BUF * sizeof(R));  // bytes a tile receives per row of tiles
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cg::cluster_group cluster = cg::this_cluster();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int wpc = blockDim.x >> 5;
  const unsigned rank = cluster.block_rank();
  const int64_t N = a.N;
  const int K = (int)(N / n);
  const int k_tile = (int)rank * wpc + warp;
  // the pushed hand-off of swept_cluster_kernel (see there), with three rows per buffer
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);              // [warp][buffer]
  R* recv = reinterpret_cast<R*>(smem_raw + cluster_bar_bytes(wpc));  // [warp][buffer][row 3][C][W]
  const uint32_t smem_base = smem_u32(smem_raw);
  auto bar_off = [&](int w, int b) -> uint32_t { return (uint32_t)((w * 2 + b) * 8); };
  auto buf_off = [&](int w, int b) -> uint32_t {
    return (uint32_t)cluster_bar_bytes(wpc) + (uint32_t)((w * 2 + b) * BUF * (int)sizeof(R));
  };
  if (lane == 0) {
    mbar_init(&bars[warp * 2 + 0], 1);
    mbar_init(&bars[warp * 2 + 1], 1);
  }
  fence_mbar_init();
  cluster.sync();
  const int rows = a.rows;
  if (lane == 0) {
    if (rows > 1) mbar_arrive_expect_tx(&bars[warp * 2 + 0], TX);
    if (rows > 2) mbar_arrive_expect_tx(&bars[warp * 2 + 1], TX);
  }
  auto wrap = [&](int64_t g) -> int64_t { return g < 0 ? g + N : (g >= N ? g - N : g); };
  uint32_t main_dst[2], main_bar[2], halo_dst[2], halo_bar[2];
  const int wshift = 31 - __clz(wpc);
#pragma unroll
  for (int p = 0; p < 2; ++p) {
    const int kL = p ? k_tile : (k_tile == 0 ? K - 1 : k_tile - 1);
    const int kR = p ? (k_tile == K - 1 ? 0 : k_tile + 1) : k_tile;
    const int mine = lane < 16 ? kL : kR, other = lane < 16 ? kR : kL;
    main_bar[p] = mapa_u32(smem_base + bar_off(mine & (wpc - 1), p), (uint32_t)(mine >> wshift));
    main_dst[p] = mapa_u32(smem_base + buf_off(mine & (wpc - 1), p), (uint32_t)(mine >> wshift)) +
                  (uint32_t)((lane ^ 16) * sizeof(R));
    halo_bar[p] = mapa_u32(smem_base + bar_off(other & (wpc - 1), p), (uint32_t)(other >> wshift));
    halo_dst[p] = mapa_u32(smem_base + buf_off(other & (wpc - 1), p), (uint32_t)(other >> wshift)) +
                  (uint32_t)((n + (lane == 16 ? H : 0)) * sizeof(R));
  }
  const R* recv_mine = recv + (size_t)(warp * 2) * BUF;
  uint64_t* bars_mine = bars + warp * 2;

  R v[3][C][P], hl[3][C][H], hr[3][C][H];
  int ta[P];
  unsigned span[P];
  int window_kind = -1;
  for (int r = 0; r < rows; ++r) {
    const int kind = r == 0 ? KIND_UP : (r == rows - 1 ? KIND_DOWN : KIND_WHOLE);
    const int inb = (r + 1) & 1, outb = r & 1;
    if (kind == KIND_UP) {
      const int64_t g0 = (int64_t)k_tile * n + lane * P;  // row 0 is an aligned row
#pragma unroll
      for (int c = 0; c < C; ++c) {
#pragma unroll
        for (int j = 0; j < P; ++j) {
          v[0][c][j] = __ldg(a.init + (int64_t)c * N + g0 + j);
          v[1][c][j] = v[2][c][j] = (R)0;  // tiers before the cycle's first do not exist
        }
#pragma unroll
        for (int e = 0; e < H; ++e)
#pragma unroll
          for (int row = 0; row < 3; ++row) hl[row][c][e] = hr[row][c][e] = (R)0;  // never used by a triangle
      }
    } else {
      mbar_wait_warp_bounded(bars_mine + inb, (uint32_t)(((r - 1) >> 1) & 1));
      if (lane == 0 && r + 2 < rows) mbar_arrive_expect_tx(bars_mine + inb, TX);  // the buffer's next use
      const R* b0 = recv_mine + (size_t)inb * BUF;
#pragma unroll
      for (int row = 0; row < 3; ++row)
#pragma unroll
        for (int c = 0; c < C; ++c) {
          const R* q = b0 + (size_t)(row * C + c) * W;
#pragma unroll
          for (int j = 0; j < P; ++j) v[row][c][j] = q[j * 32 + lane];
#pragma unroll
          for (int e = 0; e < H; ++e) {
            hl[row][c][e] = q[n + e];
            hr[row][c][e] = q[n + H + e];
          }
        }
    }
    const int ntiers = kind == KIND_UP ? m - 1 : (kind == KIND_DOWN ? m : 2 * m - 1);
    if (kind != window_kind) {
      window_kind = kind;
#pragma unroll
      for (int j = 0; j < P; ++j) {  // tier window of each point: as in swept_cluster_kernel
        const int x = lane * P + j;
        const int d = x < n / 2 ? n / 2 - x : x - n / 2 + 1;
        const int first = (d + H - 1) / H;
        const int edge = (x < n - 1 - x ? x : n - 1 - x) / H;
        const int t0 = kind == KIND_UP ? 1 : first;
        const int tb = kind == KIND_UP ? edge : (kind == KIND_DOWN ? m : 2 * m - first);
        const bool never = tb < t0;
        span[j] = never ? 0u : (unsigned)(tb - t0);
        ta[j] = never ? (1 << 30) : t0;
      }
    }
    // residue of the global tier this row of tiles starts at: the Up row at tier 0, diamond / Down row r at (r - 1) m
    const int q0 = r == 0 ? 0 : (int)(((int64_t)(r - 1) * m) % 3);
    if (q0 == 0) cluster3_tiers<Prob, P, 0>(v, hl, hr, ntiers, ta, span, lane, a.k);
    else if (q0 == 1) cluster3_tiers<Prob, P, 1>(v, hl, hr, ntiers, ta, span, lane, a.k);
    else cluster3_tiers<Prob, P, 2>(v, hl, hr, ntiers, ta, span, lane, a.k);
    if (kind == KIND_DOWN) {  // the cycle ends on a full timestep: row 0 is the time level
      const int64_t S = wrap((int64_t)k_tile * n + ((r & 1) ? n / 2 : 0));
      const int64_t g0 = wrap(S + lane * P);
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int j = 0; j < P; ++j) a.out[(int64_t)c * N + g0 + j] = v[0][c][j];
    } else {
      {
        const uint32_t bar = outb ? main_bar[1] : main_bar[0];
        const uint32_t dst = outb ? main_dst[1] : main_dst[0];
#pragma unroll
        for (int row = 0; row < 3; ++row)
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int j = 0; j < P; ++j)
              st_async_(dst + (uint32_t)(((row * C + c) * W + j * 32) * sizeof(R)), v[row][c][j], bar);
      }
      if (lane == 15 || lane == 16) {  // the h points next to the tile's centre are a neighbour consumer's halo
        const uint32_t bar = outb ? halo_bar[1] : halo_bar[0];
        const uint32_t dst = outb ? halo_dst[1] : halo_dst[0];
#pragma unroll
        for (int row = 0; row < 3; ++row)
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int e = 0; e < H; ++e) {
              const R x = lane == 15 ? v[row][c][P - H + e] : v[row][c][e];
              st_async_(dst + (uint32_t)(((row * C + c) * W + e) * sizeof(R)), x, bar);
            }
      }
    }
  }
  cluster.sync();  // nobody leaves while a store into its shared memory may still be in flight
}

// per warp two barriers and two receive buffers of [ROWS][C][n + 2h] values
template <class Prob>
inline size_t cluster_push_smem_bytes(int wpc, int n) {
  return (size_t)cluster_bar_bytes(wpc) +
         (size_t)wpc * 2 * Prob::ROWS * Prob::C * (size_t)(n + 2 * Prob::H) * sizeof(typename Prob::R);
}

// (admission test of cluster_warps_per_cta: the buffers without their halo slots)
template <class Prob>
inline size_t cluster_smem_bytes(int chunk) {
  return (size_t)2 * Prob::ROWS * Prob::C * (size_t)chunk * sizeof(typename Prob::R);
}

}  // namespace swept
