// swept_tier.cuh — swept kernels, flavour TIER: one CTA per tile ("node"), the two-row
// working array of PAPER.md:97-99 staged in shared memory, one block barrier per tier.
//
// SURVEY.md §8(a) rows a1 (UpTriangle), a3 (SplitDiamond), a4 (WholeDiamond), a5 (DownTriangle); the
// inter-launch state is row a2: two global rows, row0[x] / row1[x] = latest even- / odd-tier value at x
// (the paper's L/R edge arrays, re-expressed with the same bytes).
//
// A tile starting at S = shift + blockIdx.x * n (periodic; the last shifted tile wraps across the
// boundary = the paper's boundary-split node) does:
//   1. TMA 1-D bulk copies (cp.async.bulk, mbarrier completion) of row0/row1[S, S+n) into shared memory,
//      plus 2h halo values per row with plain loads (the widest tier reads [S-h, S+n+h));
//   2. tiers t = 1..ntiers: each thread owns P contiguous points, reads its (P+2h)-wide window of the other
//      row, applies the stencil functor, overwrites its own row where the tier is active (interior values
//      are overwritten once used, edges survive: PAPER.md:97); __syncthreads() per tier;
//        Up:       tier t covers [S + h t, S + n - h t),           t = 1 .. m-1
//        Diamond:  tier t covers [c - h t, c + h t) for t <= m and
//                  [c - h(2m-t), c + h(2m-t)) for t > m,            t = 1 .. 2m-1
//        Down:     tier t covers [c - h t, c + h t),                t = 1 .. m
//      with c = S + n/2 and m = n/(2h);
//   3. TMA bulk stores of both rows (Down: row0 only = the full time level) to the OTHER global buffer
//      (phases ping-pong between two 2 x N buffers, SURVEY.md §8(d) note).
#pragma once
#include "common.cuh"
#include "functors.cuh"

namespace swept {

enum { KIND_UP = 0, KIND_SPLIT = 1, KIND_WHOLE = 2, KIND_DOWN = 3 };

template <class R>
struct TierArgs {
  const R* in0;  // row0 of the input buffer (C components, stride N)
  const R* in1;  // row1 of the input buffer (unused by Up)
  R* out0;
  R* out1;  // unused by Down
  const R* in2 = nullptr;  // third row, schemes with three sub-timesteps per timestep (Prob::ROWS == 3)
  R* out2 = nullptr;
  int tmod = 0;  // global tier of the phase's relative tier 0, modulo Prob::ROWS (0 for the two-row schemes, whose
                 // phases all start on even tiers)
  int64_t N;
  int n;       // tile width in points
  int shift;   // 0 or n/2
  int ntiers;  // tiers to compute
  int bc;      // BC_WRAP, BC_MIRROR (heat, Eq. (B.5): T_{-k} = T_k, T_{N-1+k} = T_{N-1-k}) or
               // BC_FIXED (Euler tube: ghost cells hold the end states bv.l / bv.r)
  BcVals<R> bv;
  // tile selection.  TIER: block b computes tile tile_base + b * tile_step (default 0, 1: every tile).  CHAR: the
  // first / last tile of the row is left to a TIER launch that applies the walls (hybrid mode)
  int tile_base, tile_step;
  int skip_first, skip_last;
  Consts<R> k;
};

template <int KIND>
__device__ __forceinline__ void tier_range(int t, int n, int h, int m, int& lo, int& hi) {
  if (KIND == KIND_UP) {
    lo = h * t;
    hi = n - h * t;
  } else {
    const int w = (KIND == KIND_DOWN || t <= m) ? h * t : h * (2 * m - t);
    lo = n / 2 - w;
    hi = n / 2 + w;
  }
}

template <class Prob, int P, int KIND>
__global__ void __launch_bounds__(Prob::TIER_MAX_THREADS) swept_tier_kernel(const TierArgs<typename Prob::R> a) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C, PAD = Pad16<R>::value, ROWS = Prob::ROWS;
  static_assert(ROWS == 2 || (ROWS == Prob::SIGMA && C == 1), "rows = tier modulo ROWS; u^n in row 0");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = a.n;
  const int RS = n + 4 * PAD;  // padded row stride: body starts 16 bytes in; room for the wall gap (see below)
  R* rows = reinterpret_cast<R*>(smem_raw);
  uint64_t* mbar = reinterpret_cast<uint64_t*>(smem_raw + (size_t)ROWS * C * RS * sizeof(R));
  R* xtr = reinterpret_cast<R*>(smem_raw + (size_t)ROWS * C * RS * sizeof(R) + 16);  // Euler: pressures, fluxes
  (void)xtr;
  const int64_t N = a.N;
  const int tid = threadIdx.x;
  int64_t S = (int64_t)a.shift + ((int64_t)a.tile_base + (int64_t)blockIdx.x * a.tile_step) * n;
  if (S >= N) S -= N;
  const int len1 = (int)((N - S) < (int64_t)n ? (N - S) : (int64_t)n);  // part before the periodic wrap
  const int len2 = n - len1;
  constexpr int NROWS_IN = (KIND == KIND_UP) ? 1 : ROWS;
  // Non-periodic ends ("node 0 is split across the spatial boundary and must apply the boundary conditions at its
  // center"): the tile that wraps holds the last n/2 and the first n/2 points of the domain with the
  // two walls between them.  Its halves are staged 2*PAD slots apart and the gap holds each wall's h ghost values;
  // tiles that end at a wall keep the ghosts in their halo slots.  A ghost is the mirror image of a point the tile
  // itself updates (mirror), so whoever writes a point within h of a wall also writes its image (no extra barrier);
  // Dirichlet ghosts are constants written once.
  const bool bcm = a.bc != 0;
  const int GAP = (bcm && len2 > 0) ? 2 * PAD : 0;
  const int jl = !bcm ? -100000 : (len2 > 0 ? len1 : (S == 0 ? 0 : -100000));              // local index of point 0
  const int jr = !bcm ? -100000 : (len2 > 0 ? len1 - 1 : (S + n == N ? n - 1 : -100000));  // ... of point N-1
  auto slot_of = [&](int j) -> int { return PAD + j + (j >= len1 ? GAP : 0); };

  if (tid == 0) {
    mbar_init(mbar, 1);
    fence_mbar_init();
  }
  __syncthreads();
  if (tid == 0) {
    mbar_arrive_expect_tx(mbar, (uint32_t)(NROWS_IN * C * n * sizeof(R)));
#pragma unroll
    for (int r = 0; r < NROWS_IN; ++r) {
      const R* src = r == 0 ? a.in0 : (r == 1 ? a.in1 : a.in2);
#pragma unroll
      for (int c = 0; c < C; ++c) {
        R* dst = rows + (r * C + c) * RS + PAD;
        bulk_g2s(dst, src + (int64_t)c * N + S, (uint32_t)(len1 * sizeof(R)), mbar);
        if (len2 > 0) bulk_g2s(dst + len1 + GAP, src + (int64_t)c * N, (uint32_t)(len2 * sizeof(R)), mbar);
      }
    }
  }
  if (KIND == KIND_UP) {
    // tiers before the cycle's first do not exist: give the other rows a defined value (their edge slots are
    // stored but never used)
    for (int i = tid; i < (ROWS - 1) * C * RS; i += blockDim.x) rows[C * RS + i] = (R)0;
  } else {
    // halo: H points either side of the tile, every row, plain loads (periodic, or mirrored at a wall)
    for (int i = tid; i < ROWS * C * 2 * H; i += blockDim.x) {
      const int r = i / (C * 2 * H), c = (i / (2 * H)) % C, j = i % (2 * H);
      const R* src = (r == 0 ? a.in0 : (r == 1 ? a.in1 : a.in2)) + (int64_t)c * N;
      int64_t g = (j < H) ? (S - H + j) : (S + n + (j - H));
      if (len2 > 0 && j >= H) g = len2 + (j - H);  // the wrapping tile continues at point n/2 (no wall there)
      const bool fixed = a.bc == BC_FIXED && (g < 0 || g >= N);
      const R fv = g < 0 ? a.bv.l[c] : a.bv.r[c];
      if (g < 0) g = bcm ? -g : g + N;
      if (g >= N) g = bcm ? 2 * (N - 1) - g : g - N;
      const int s = (j < H) ? (PAD - H + j) : (PAD + n + GAP + (j - H));
      rows[(r * C + c) * RS + s] = fixed ? fv : src[g];
    }
    if (GAP > 0) {  // ghosts of the two walls inside the wrapping tile: T_{N-1+k} = T_{N-1-k}, T_{-k} = T_k
      for (int i = tid; i < 2 * C * 2 * H; i += blockDim.x) {
        const int r = i / (C * 2 * H), c = (i / (2 * H)) % C, j = i % (2 * H);
        const R* src = (r == 0 ? a.in0 : a.in1) + (int64_t)c * N;
        const int k = (j < H) ? j + 1 : j - H + 1;
        const int s = (j < H) ? slot_of(jr) + k : slot_of(jl) - k;
        if (a.bc == BC_FIXED) rows[(r * C + c) * RS + s] = (j < H) ? a.bv.r[c] : a.bv.l[c];
        else rows[(r * C + c) * RS + s] = (j < H) ? src[N - 1 - k] : src[k];
      }
    }
  }
  mbar_wait(mbar, 0);
  __syncthreads();

  const int m = n / (2 * H);
  const int j0 = tid * P;
  const int sb = slot_of(j0);  // a thread's P points lie on one side of the wrap (n/2 is a multiple of P)
  for (int t = 1; t <= a.ntiers; ++t) {
    // global tier g = tmod + t (mod ROWS): reads row (g-1) % ROWS, writes row g % ROWS; the stage is g % SIGMA
    // (two-row schemes: phases start on even global tiers, m is even, so par = t & 1: odd = predictor)
    const int gm = (a.tmod + t) % ROWS;
    const int par = ROWS == 2 ? (t & 1) : gm;
    const R* src = rows + (ROWS == 2 ? 1 - par : (gm + ROWS - 1) % ROWS) * C * RS;
    R* dst = rows + par * C * RS;
    int lo, hi;
    tier_range<KIND>(t, n, H, m, lo, hi);
    if constexpr (Prob::C == 3) {
      // Euler: every pressure and every interface flux of the tier is computed ONCE and shared through shared
      // memory (Prob::stage would rebuild P+4 pressures and P+1 fluxes per thread: 8 divisions and 3 square roots
      // per flux).  Three steps per tier, all threads of the CTA share the slots of the active range evenly:
      //   A  pressure (D.4) of the slots [lo-2, hi+2);  B  flux (D.6)-(D.11) at the right interface of the slots
      //   [lo-1, hi);  C  update (D.12) of the points [lo, hi).  Same pressure()/flux()/update() as Prob::stage.
      R* prs = xtr;
      R* flx = xtr + RS;
      const int s_lo = slot_of(lo), s_hi = slot_of(hi - 1) + 1;  // slot range of the active points (gap included)
      for (int q = s_lo - 2 + tid; q < s_hi + 2; q += blockDim.x)
        prs[q] = Prob::pressure(src[q], src[RS + q], src[2 * RS + q], a.k);
      __syncthreads();
      for (int q = s_lo - 1 + tid; q < s_hi; q += blockDim.x) {
        const R vl[3] = {src[q], src[RS + q], src[2 * RS + q]};
        const R vr[3] = {src[q + 1], src[RS + q + 1], src[2 * RS + q + 1]};
        R F[3];
        Prob::flux(vl, vr, prs[q] - prs[q - 1], prs[q + 1] - prs[q], prs[q + 2] - prs[q + 1], F, a.k);
        flx[q] = F[0];
        flx[RS + q] = F[1];
        flx[2 * RS + q] = F[2];
      }
      __syncthreads();
#pragma unroll
      for (int j = 0; j < P; ++j)
        if (j0 + j >= lo && j0 + j < hi) {
#pragma unroll
          for (int c = 0; c < C; ++c) {
            const R v = src[c * RS + sb + j];
            const R b = !par ? dst[c * RS + sb + j] : v;
            dst[c * RS + sb + j] = Prob::update(v, b, flx[c * RS + sb + j] - flx[c * RS + sb + j - 1], par, a.k);
          }
        }
    } else if (j0 < hi && j0 + P > lo) {
      R win[C][P + 2 * H], bs[C][P], o[C][P];
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int q = 0; q < P + 2 * H; ++q) win[c][q] = src[c * RS + sb - H + q];
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int j = 0; j < P; ++j)
          bs[c][j] = (Prob::SIGMA >= 2 && par != 1) ? rows[c * RS + sb + j] : win[c][H + j];  // u^n: row 0
      Prob::template stage<P>(win, bs, o, par, a.k);
#pragma unroll
      for (int j = 0; j < P; ++j)
        if (j0 + j >= lo && j0 + j < hi) {
#pragma unroll
          for (int c = 0; c < C; ++c) dst[c * RS + sb + j] = o[c][j];
          if (a.bc == BC_MIRROR) {
            const int dl = j0 + j - jl, dr = jr - (j0 + j);
            if (dl > 0 && dl <= H) {
#pragma unroll
              for (int c = 0; c < C; ++c) dst[c * RS + slot_of(jl) - dl] = o[c][j];
            }
            if (dr > 0 && dr <= H) {
#pragma unroll
              for (int c = 0; c < C; ++c) dst[c * RS + slot_of(jr) + dr] = o[c][j];
            }
          }
        }
    }
    __syncthreads();
  }

  fence_proxy_async_smem();
  __syncthreads();
  if (tid == 0) {
    constexpr int NROWS_OUT = (KIND == KIND_DOWN) ? 1 : ROWS;
#pragma unroll
    for (int r = 0; r < NROWS_OUT; ++r) {
      R* dstg = r == 0 ? a.out0 : (r == 1 ? a.out1 : a.out2);
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const R* s = rows + (r * C + c) * RS + PAD;
        bulk_s2g(dstg + (int64_t)c * N + S, s, (uint32_t)(len1 * sizeof(R)));
        if (len2 > 0) bulk_s2g(dstg + (int64_t)c * N, s + len1 + GAP, (uint32_t)(len2 * sizeof(R)));
      }
    }
    bulk_commit();
    bulk_wait_all();
  }
}

template <class Prob>
inline size_t tier_smem_bytes(int n) {
  using R = typename Prob::R;
  const size_t row = ((size_t)n + 4 * Pad16<R>::value) * sizeof(R);
  return (size_t)Prob::ROWS * Prob::C * row + 16 + (Prob::C == 3 ? 4 * row : 0);  // Euler: + one pressure and three flux rows
}

}  // namespace swept
