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
//   * the whole cycle — UpTriangle, D Split/WholeDiamond rows, DownTriangle (§4.2) — runs in ONE launch: between
//     two rows every warp writes its tile's rows to the cluster's DISTRIBUTED SHARED MEMORY (point x of the domain
//     lives in CTA x / chunk), one cluster barrier, and every warp reads the rows of its next tile, half a tile
//     further on (the edges a node passes on), from there — possibly from a neighbouring SM.  Inside
//     an aligned block of n points the slots are lane-major (point lane * P + j sits at j * 32 + lane), so that the 32
//     lanes of one load or store touch consecutive addresses: a remote shared-memory access is one request per lane
//     unless the lanes are contiguous (measured: 1200 cycles per strided warp access).
//     Global memory is touched twice: the Up row reads the time level, the Down row writes it.
//   * rows ping-pong between two shared-memory buffers, so one barrier per row suffices (a tile reads an h-wide halo
//     that its neighbour rewrites in the same row: SURVEY.md §8(d) note).
// What it buys: a tier costs a shuffle round trip plus one dependent DADD -> DFMA (about 50 cycles for P = 4) instead of
// the 130 cycles per tier the characteristic sweep needs at N = 2048 (its skew and chain latency), and no launch gap or
// L2 round trip between rows.  Lane efficiency is the paper's ~50 %; irrelevant here, because the bound
// at these sizes is the dependent chain, not the FP64 pipe.  Same functors, so the same bits.
#pragma once
#include <cooperative_groups.h>

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
  int chunk;      // points per CTA = warps per CTA * n (a power of two)
  int chunk_log2;
  Consts<R> k;
  int bc = 0;  // BC_MIRROR: insulated ends (heat, Eq. (B.5)), applied by the lanes next to a wall
};

__device__ __forceinline__ double shfl_idx_(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ float shfl_idx_(float v, int src) { return __shfl_sync(0xffffffffu, v, src); }

// One tier of a warp's tile: source row vs (tier t-1), destination row vd (tier t; holds tier t-2 before), halo values
// of the source row beyond the tile's ends in hl / hr.  Point j of the lane is updated when relative tier t lies in
// its window [ta[j], ta[j] + span[j]] (the tier ranges of swept_tier.cuh turned round: per point instead of per tier,
// so that the test is one subtraction and one compare on plain registers).
template <class Prob, int P>
__device__ __forceinline__ void cluster_tier(const typename Prob::R (&vs)[Prob::C][P], typename Prob::R (&vd)[Prob::C][P],
                                             const typename Prob::R (&v0)[Prob::C][P],
                                             const typename Prob::R (&hl)[Prob::C][Prob::H],
                                             const typename Prob::R (&hr)[Prob::C][Prob::H], const int par, const int t,
                                             const int (&ta)[P], const unsigned (&span)[P], const int lane,
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
      const R fromL = shfl_idx_(vs[c][P - H + e], (lane + 31) & 31);
      const R fromR = shfl_idx_(vs[c][e], (lane + 1) & 31);
      win[c][e] = lane == 0 ? hl[c][e] : fromL;
      win[c][H + P + e] = lane == 31 ? hr[c][e] : fromR;
    }
#pragma unroll
    for (int j = 0; j < P; ++j) {
      win[c][H + j] = vs[c][j];
      bs[c][j] = (Prob::SIGMA >= 2 && par != 1) ? v0[c][j] : vs[c][j];  // u^n: row 0
    }
    if constexpr (H == 1 && P >= 2) {
      // a lane whose first / last point is an END POINT of the domain: the stencil's outer value is the mirror image
      // of its own second / second-to-last point, T_{-1} = T_1 and T_N = T_{N-2} (Eq. (B.5), reading X17)
      win[c][0] = wall_l ? vs[c][1] : win[c][0];
      win[c][P + 1] = wall_r ? vs[c][P - 2] : win[c][P + 1];
    }
  }
  Prob::template stage<P>(win, bs, o, par, k);
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const bool act = (unsigned)(t - ta[j]) <= span[j];
#pragma unroll
    for (int c = 0; c < C; ++c) vd[c][j] = act ? o[c][j] : vd[c][j];
  }
}

// threads per CTA (register budget: two rows of P points, the window and the tier windows per lane)
template <int P> struct ClusterMaxThreads { static constexpr int value = P >= 8 ? 256 : 512; };

template <class Prob, int P>
__global__ void __launch_bounds__(ClusterMaxThreads<P>::value) swept_cluster_kernel(const ClusterArgs<typename Prob::R> a) {
  namespace cg = cooperative_groups;
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C;
  static_assert(Prob::ROWS == 2, "two-row schemes");
  static_assert(P >= H, "a lane's block must hold its neighbour's halo");
  constexpr int n = 32 * P, m = n / (2 * H);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  R* sm = reinterpret_cast<R*>(smem_raw);  // [buffer 2][row 2][component C][chunk]
  cg::cluster_group cluster = cg::this_cluster();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int wpc = blockDim.x >> 5;
  const unsigned rank = cluster.block_rank();
  const int64_t N = a.N;
  const int64_t k_tile = (int64_t)rank * wpc + warp;
  const int chunk = a.chunk;
  // address of point g (0 <= g < N) of (buffer, row, component) in the cluster's distributed shared memory
  auto dsm = [&](int buf, int row, int c, int64_t g) -> R* {
    const int i = (int)(g & (n - 1));                              // position inside the aligned block of n points
    const int off = (int)(g & (chunk - 1)) - i + (i % P) * 32 + i / P;  // lane-major inside the block
    R* local = sm + (size_t)((buf * 2 + row) * C + c) * chunk + off;
    return cluster.map_shared_rank(local, (unsigned)(g >> a.chunk_log2));
  };
  auto wrap = [&](int64_t g) -> int64_t { return g < 0 ? g + N : (g >= N ? g - N : g); };

  R v0[C][P], v1[C][P];  // row 0 (even tiers) and row 1 (odd tiers) of this lane's P points
  R hl0[C][H], hr0[C][H], hl1[C][H], hr1[C][H];
  for (int r = 0; r < a.rows; ++r) {
    const int kind = r == 0 ? KIND_UP : (r == a.rows - 1 ? KIND_DOWN : KIND_WHOLE);
    const int64_t S = wrap(k_tile * n + ((r & 1) ? n / 2 : 0));
    const int64_t g0 = wrap(S + lane * P);  // this lane's first point; its P points do not straddle the wrap
    const int inb = (r + 1) & 1, outb = r & 1;
    // ---- load the tile's rows (Up: the time level from global memory; tier -1 does not exist)
    if (kind == KIND_UP) {
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
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const R* p0 = dsm(inb, 0, c, g0);
        const R* p1 = dsm(inb, 1, c, g0);
#pragma unroll
        for (int j = 0; j < P; ++j) {  // g0 is a multiple of P: its slot is the lane's column, the points are 32 apart
          v0[c][j] = p0[j * 32];
          v1[c][j] = p1[j * 32];
        }
#pragma unroll
        for (int e = 0; e < H; ++e) {  // the h-wide halo beyond either end of the tile, both rows (all lanes: broadcast)
          const int64_t gl = wrap(S - H + e), gr = wrap(S + n + e);
          hl0[c][e] = *dsm(inb, 0, c, gl);
          hl1[c][e] = *dsm(inb, 1, c, gl);
          hr0[c][e] = *dsm(inb, 0, c, gr);
          hr1[c][e] = *dsm(inb, 1, c, gr);
        }
      }
    }
    // ---- tiers (phases start on even global tiers, so odd relative tiers are predictor / odd-row tiers).
    // Tier window of every point x of the tile: Up (tier t covers [ht, n-ht)): 1 .. min(x, n-1-x)/h;
    // diamond (tier t covers the centre +- ht, then +- h(2m-t)): ceil(d/h) .. 2m - ceil(d/h) with d the
    // distance from the centre; Down: ceil(d/h) .. m.
    const int ntiers = kind == KIND_UP ? m - 1 : (kind == KIND_DOWN ? m : 2 * m - 1);
    int ta[P];
    unsigned span[P];
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
    // (Two tiers behind one shuffle exchange — 2h redundant evaluations per lane instead of a second exchange — was
    // built and measured: no faster for the 3-point scheme, 3 % for the 5-point one; not kept.)
    // walls ("node 0 is split across the spatial boundary and must apply the boundary conditions at its center",
    // PAPER.md:79-81): aligned rows: point 0 is lane 0 of the first tile, point N-1 lane 31 of the last; shifted rows:
    // the last tile wraps, point N-1 is the last point of its lane 15 and point 0 the first of its lane 16
    const int64_t K = N / n;
    const bool shifted = (r & 1) != 0;
    const bool wall_l = a.bc != 0 && (shifted ? (k_tile == K - 1 && lane == 16) : (k_tile == 0 && lane == 0));
    const bool wall_r = a.bc != 0 && (shifted ? (k_tile == K - 1 && lane == 15) : (k_tile == K - 1 && lane == 31));
    for (int t = 1; t <= ntiers; t += 2) {
      cluster_tier<Prob, P>(v0, v1, v0, hl0, hr0, 1, t, ta, span, lane, a.k, wall_l, wall_r);  // odd tier: row 0 -> row 1
      if (t + 1 <= ntiers)
        cluster_tier<Prob, P>(v1, v0, v0, hl1, hr1, 0, t + 1, ta, span, lane, a.k, wall_l, wall_r);  // even: row 1 -> row 0
    }
    // ---- hand the rows on: Down leaves the full time level (row 0) in global memory
    if (kind == KIND_DOWN) {
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int j = 0; j < P; ++j) a.out[(int64_t)c * N + g0 + j] = v0[c][j];
    } else {
#pragma unroll
      for (int c = 0; c < C; ++c) {
        R* p0 = dsm(outb, 0, c, g0);
        R* p1 = dsm(outb, 1, c, g0);
#pragma unroll
        for (int j = 0; j < P; ++j) {
          p0[j * 32] = v0[c][j];
          p1[j * 32] = v1[c][j];
        }
      }
      cluster.sync();  // release / acquire at cluster scope: every tile of row r is in shared memory
    }
  }
  cluster.sync();  // nobody leaves while a slower CTA may still be reading its shared memory
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
  cluster_tier<Prob, P>(v[SRC], v[G], v[0], hl[SRC], hr[SRC], G, t, ta, span, lane, k);
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
  extern __shared__ __align__(128) unsigned char smem_raw[];
  R* sm = reinterpret_cast<R*>(smem_raw);  // [buffer 2][row 3][component C][chunk]
  cg::cluster_group cluster = cg::this_cluster();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int wpc = blockDim.x >> 5;
  const unsigned rank = cluster.block_rank();
  const int64_t N = a.N;
  const int64_t k_tile = (int64_t)rank * wpc + warp;
  const int chunk = a.chunk;
  auto dsm = [&](int buf, int row, int c, int64_t g) -> R* {
    const int i = (int)(g & (n - 1));
    const int off = (int)(g & (chunk - 1)) - i + (i % P) * 32 + i / P;  // lane-major inside the aligned block
    R* local = sm + (size_t)((buf * 3 + row) * C + c) * chunk + off;
    return cluster.map_shared_rank(local, (unsigned)(g >> a.chunk_log2));
  };
  auto wrap = [&](int64_t g) -> int64_t { return g < 0 ? g + N : (g >= N ? g - N : g); };

  R v[3][C][P], hl[3][C][H], hr[3][C][H];
  for (int r = 0; r < a.rows; ++r) {
    const int kind = r == 0 ? KIND_UP : (r == a.rows - 1 ? KIND_DOWN : KIND_WHOLE);
    const int64_t S = wrap(k_tile * n + ((r & 1) ? n / 2 : 0));
    const int64_t g0 = wrap(S + lane * P);
    const int inb = (r + 1) & 1, outb = r & 1;
    if (kind == KIND_UP) {
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
#pragma unroll
      for (int row = 0; row < 3; ++row)
#pragma unroll
        for (int c = 0; c < C; ++c) {
          const R* p = dsm(inb, row, c, g0);
#pragma unroll
          for (int j = 0; j < P; ++j) v[row][c][j] = p[j * 32];
#pragma unroll
          for (int e = 0; e < H; ++e) {
            hl[row][c][e] = *dsm(inb, row, c, wrap(S - H + e));
            hr[row][c][e] = *dsm(inb, row, c, wrap(S + n + e));
          }
        }
    }
    const int ntiers = kind == KIND_UP ? m - 1 : (kind == KIND_DOWN ? m : 2 * m - 1);
    int ta[P];
    unsigned span[P];
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
    // residue of the global tier this row of tiles starts at: the Up row at tier 0, diamond / Down row r at (r - 1) m
    const int q0 = r == 0 ? 0 : (int)(((int64_t)(r - 1) * m) % 3);
    if (q0 == 0) cluster3_tiers<Prob, P, 0>(v, hl, hr, ntiers, ta, span, lane, a.k);
    else if (q0 == 1) cluster3_tiers<Prob, P, 1>(v, hl, hr, ntiers, ta, span, lane, a.k);
    else cluster3_tiers<Prob, P, 2>(v, hl, hr, ntiers, ta, span, lane, a.k);
    if (kind == KIND_DOWN) {  // the cycle ends on a full timestep: row 0 is the time level
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int j = 0; j < P; ++j) a.out[(int64_t)c * N + g0 + j] = v[0][c][j];
    } else {
#pragma unroll
      for (int row = 0; row < 3; ++row)
#pragma unroll
        for (int c = 0; c < C; ++c) {
          R* p = dsm(outb, row, c, g0);
#pragma unroll
          for (int j = 0; j < P; ++j) p[j * 32] = v[row][c][j];
        }
      cluster.sync();
    }
  }
  cluster.sync();
}

template <class Prob>
inline size_t cluster_smem_bytes(int chunk) {
  return (size_t)2 * Prob::ROWS * Prob::C * (size_t)chunk * sizeof(typename Prob::R);
}

}  // namespace swept
