// swept_char.cuh — swept kernels, flavour CHAR: register-resident sweep of a tile along its characteristics.
//
// Same space-time regions as swept_tier.cuh (UpTriangle / Split-, WholeDiamond / DownTriangle of PAPER.md
// §4.2-4.3, edges through the two global rows, half-tile shift) — only the ORDER in which the points of one
// tile are evaluated on chip differs, which the swept rule leaves free.
//
// Geometry.  In a diamond of width n centred at c, relative tier t, x' = x - c, use the characteristic
// coordinates  p = x' + h t,  q = h t - x' - 1.  The diamond is exactly the square 0 <= p, q < n (lattice
// points: p + q + 1 = 2 h t).  Point (p, q) depends on (p-2h+k, q-k), k = 0..2h (its 2h+1 stencil inputs at
// tier t-1) and, for a final stage, on (p-2h, q-2h) (its own value at tier t-2).  So any order with p
// ascending and, inside a column, q ascending is valid, and a "line" q = const needs only ONE live value:
// its latest point.  A tile is owned by a group of L lanes; lane gl keeps the B = n/L lines
// q in [gl B, gl B + B) in registers (v[.]), sweeps p upwards 2h columns ("super-column") per step, and lags
// its lower neighbour by one step, so the only communication is: per step, the 2h top lines of lane gl-1
// by __shfl_up.  Lane 0 takes them from the staged input rows instead (the diamond's lower-right edge),
// lane L-1 streams its top lines out (the upper-left edge), and the last values of all lines form the
// upper-right edge.  Every lane is busy m = n/(2h) of the m + L - 1 steps: lane utilisation m/(m+L-1)
// instead of the ~50 % of a tier-by-tier diamond (PAPER.md:211 names idle threads as the first drawback).
// No block barrier and no shared-memory traffic inside the sweep.
//
// Up / Down are the upper / lower half of the same square (tiers t > m, resp. t <= m, with m the tier of the
// anti-diagonal p + q + 1 = n); the other half is masked.
//
// Shared memory holds the CTA's chunk of both rows (T*B contiguous points, all tiles of the CTA), loaded and
// stored with TMA 1-D bulk copies, and is updated in place: stream / final writes only touch slots whose
// input value has already been consumed (see DESIGN.md §5.4 for the hazard argument).
#pragma once
#include "common.cuh"
#include "functors.cuh"
#include "swept_tier.cuh"

namespace swept {

template <class R>
__device__ __forceinline__ R shfl_up_(R v, int width);
template <>
__device__ __forceinline__ double shfl_up_<double>(double v, int width) {
  return __shfl_up_sync(0xffffffffu, v, 1, width);
}
template <>
__device__ __forceinline__ float shfl_up_<float>(float v, int width) {
  return __shfl_up_sync(0xffffffffu, v, 1, width);
}

// Predicated shared-memory access of the two I/O lanes of a group with an immediate byte offset from one running
// 32-bit shared address.  Written in PTX so that the load lands in the very register the shuffle filled (the
// tied "+" operand: no select, no move) and the address arithmetic stays out of the loop.
template <int OFF> __device__ __forceinline__ void lds_tied(double& x, uint32_t addr) {
  asm volatile("ld.volatile.shared.f64 %0, [%1+%2];" : "+d"(x) : "r"(addr), "n"(OFF) : "memory");
}
template <int OFF> __device__ __forceinline__ void lds_tied(float& x, uint32_t addr) {
  asm volatile("ld.volatile.shared.f32 %0, [%1+%2];" : "+f"(x) : "r"(addr), "n"(OFF) : "memory");
}
template <int OFF> __device__ __forceinline__ void sts_imm(uint32_t addr, double x) {
  asm volatile("st.volatile.shared.f64 [%0+%1], %2;" ::"r"(addr), "n"(OFF), "d"(x) : "memory");
}
template <int OFF> __device__ __forceinline__ void sts_imm(uint32_t addr, float x) {
  asm volatile("st.volatile.shared.f32 [%0+%1], %2;" ::"r"(addr), "n"(OFF), "f"(x) : "memory");
}
// scheme constants pinned in registers: the compiler otherwise reloads them from the constant bank inside the
// sweep loop (two LDC per pair of steps)
__device__ __forceinline__ void pin_reg(double& x) { asm volatile("" : "+d"(x)); }
__device__ __forceinline__ void pin_reg(float& x) { asm volatile("" : "+f"(x)); }
template <class R>
__device__ __forceinline__ Consts<R> pinned_consts(const Consts<R>& k) {
  Consts<R> r = k;
  pin_reg(r.a0); pin_reg(r.a1); pin_reg(r.a2); pin_reg(r.a3); pin_reg(r.a4);
  return r;
}

// Advance the B lines of one lane by one super-column `sc` (0 <= sc < m): 2h sub-columns (p mod 2h fixed), each a
// dependent chain of B/2h points.  hal = the 2h lines below the lane's block after the neighbour's super-column
// sc, halp = the same one super-column earlier (own-point-two-tiers-back operand of the first chain links).
template <class Prob, int B, int L, int KIND>
__device__ __forceinline__ void char_update_lines(typename Prob::R (&v)[Prob::C][B],
                                                  const typename Prob::R (&hal)[Prob::C][2 * Prob::H],
                                                  const typename Prob::R (&halp)[Prob::C][2 * Prob::H], const int sc,
                                                  const int gl, const Consts<typename Prob::R>& kc) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C;
  constexpr int n = B * L, m = n / (2 * H), BP = B / (2 * H);
#pragma unroll
  for (int rho = 0; rho < 2 * H; ++rho) {
    R carry[C];  // previous value of line i-2h (tier t-2 of the point being computed)
#pragma unroll
    for (int c = 0; c < C; ++c) carry[c] = halp[c][rho];
#pragma unroll
    for (int aa = 0; aa < BP; ++aa) {
      const int i = 2 * H - 1 - rho + 2 * H * aa;  // line updated in this sub-column
      const int t = sc + gl * BP + aa + 1;         // its relative tier
      const int odd = t & 1;
      const bool act = KIND == KIND_UP ? (t > m) : (KIND == KIND_DOWN ? (t <= m) : true);
      R win[C][2 * H + 1], bs[C][1], o[C][1];
#pragma unroll
      for (int c = 0; c < C; ++c) {
#pragma unroll
        for (int k = 0; k <= 2 * H; ++k)
          win[c][k] = (i - k >= 0) ? v[c][(i - k >= 0) ? i - k : 0] : hal[c][(i - k >= 0) ? 0 : k - i - 1];
        bs[c][0] = (Prob::SIGMA == 2 && !odd) ? carry[c] : win[c][H];
      }
      Prob::template stage<1>(win, bs, o, odd, kc);
#pragma unroll
      for (int c = 0; c < C; ++c) {
        carry[c] = v[c][i];
        if (act) v[c][i] = o[c][0];
      }
    }
  }
}

// One super-step of a lane: fetch the 2h-line halo (shuffle, or the staged edge for group lane 0), update the
// B lines of this lane (2h sub-columns, each a dependent chain of B/2h points), stream the top lines out
// (group lane L-1).  GUARD = some lanes of the warp are outside their m super-columns (ramp up / down).
// Steps come in pairs (PH = 0: s even, PH = 1: s odd) and L is even, so the rows the two I/O lanes touch are fixed
// per PH and every address is `base` plus a compile-time offset, with base = rows + ctr + h * (s - PH) advanced
// by 2h per pair by the caller (no per-lane pointer, no row toggling in the loop):
//   reader (group lane 0):    line -1-e at super-column s is (x' = h s + e, tier s): row PH
//   writer (group lane L-1):  at its super-column sc = s - (L-1) its top line e leaves at
//                             (x' = -n/2 + h sc + e, tier m + sc): row (sc & 1) = 1 - PH
template <class Prob, int B, int L, int KIND, bool GUARD, int PH, int RSC>
__device__ __forceinline__ void char_step(typename Prob::R (&v)[Prob::C][B],
                                          typename Prob::R (&hal)[Prob::C][2 * Prob::H],
                                          const typename Prob::R (&halp)[Prob::C][2 * Prob::H],
                                          typename Prob::R* base, const uint32_t sbase, const int s, const int gl,
                                          const int RS, const Consts<typename Prob::R>& kc) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C;
  constexpr int n = B * L, m = n / (2 * H);
  const int sc = s - gl;  // this lane's super-column
#pragma unroll
  for (int c = 0; c < C; ++c)
#pragma unroll
    for (int e = 0; e < 2 * H; ++e) hal[c][e] = shfl_up_<R>(v[c][B - 1 - e], L);
  if (gl == 0 && (!GUARD || s < m)) {
    if constexpr (RSC > 0) {  // row stride known at compile time: immediate offsets from the running shared address
      if constexpr (C >= 1) { lds_tied<(int)sizeof(R) * ((PH * C + 0) * RSC + PH * H + 0)>(hal[0][0], sbase);
                              lds_tied<(int)sizeof(R) * ((PH * C + 0) * RSC + PH * H + 1)>(hal[0][1], sbase); }
      if constexpr (H == 2) { lds_tied<(int)sizeof(R) * ((PH * C + 0) * RSC + PH * H + 2)>(hal[0][2], sbase);
                              lds_tied<(int)sizeof(R) * ((PH * C + 0) * RSC + PH * H + 3)>(hal[0][3], sbase); }
      static_assert(C == 1, "the compile-time-stride path is instantiated for the scalar problems");
    } else {
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int e = 0; e < 2 * H; ++e) hal[c][e] = base[(PH * C + c) * RS + PH * H + e];
    }
  }
  if (!GUARD || (sc >= 0 && sc < m)) {
    char_update_lines<Prob, B, L, KIND>(v, hal, halp, sc, gl, kc);
    // upper-left edge: the top 2h lines of the last lane leave the tile
    if (KIND != KIND_DOWN && gl == L - 1) {
      if constexpr (RSC > 0) {
        constexpr int W0 = ((1 - PH) * C + 0) * RSC + PH * H - n / 2 - H * (L - 1);
        sts_imm<(int)sizeof(R) * (W0 + 0)>(sbase, v[0][B - 1]);
        sts_imm<(int)sizeof(R) * (W0 + 1)>(sbase, v[0][B - 2]);
        if constexpr (H == 2) {
          sts_imm<(int)sizeof(R) * (W0 + 2)>(sbase, v[0][B - 3]);
          sts_imm<(int)sizeof(R) * (W0 + 3)>(sbase, v[0][B - 4]);
        }
      } else {
#pragma unroll
        for (int c = 0; c < C; ++c)
#pragma unroll
          for (int e = 0; e < 2 * H; ++e)
            base[((1 - PH) * C + c) * RS + PH * H - n / 2 - H * (L - 1) + e] = v[c][B - 1 - e];
      }
    }
  }
}

// Line values of one lane <-> the staged rows of its tile (rows, RS, ctr as in char_sweep_tile).
template <class Prob, int B, int L, int KIND>
__device__ __forceinline__ void char_load_lines(typename Prob::R (&v)[Prob::C][B], const typename Prob::R* rows, const int RS,
                                   const int ctr, const int gl) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C, n = B * L;
  auto slot = [&](int row, int c, int xp) -> const R& { return rows[(row * C + c) * RS + ctr + xp]; };
  // initial line values: the point of line q just below the square (super-column -1), which is the latest
  // (or second latest) tier stored at x' = -(h tq + r + 1); Up: the anti-diagonal = tier-0 data
#pragma unroll
  for (int i = 0; i < B; ++i) {
    const int q = gl * B + i;
    int xp, row;
    if (KIND == KIND_UP) {
      xp = n / 2 - 1 - q;
      row = 0;
    } else {
      const int tq = q / (2 * H), r = i % (2 * H);
      xp = -(H * tq + r + 1);
      row = tq & 1;
    }
#pragma unroll
    for (int c = 0; c < C; ++c) v[c][i] = slot(row, c, xp);
  }
}

template <class Prob, int B, int L, int KIND>
__device__ __forceinline__ void char_store_lines(const typename Prob::R (&v)[Prob::C][B], typename Prob::R* rows, const int RS,
                                   const int ctr, const int gl) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C, n = B * L;
  auto slot = [&](int row, int c, int xp) -> R& { return rows[(row * C + c) * RS + ctr + xp]; };
  // upper-right edge (Down: the full time level): last value of every line
#pragma unroll
  for (int i = 0; i < B; ++i) {
    const int q = gl * B + i;
    int xp, row;
    if (KIND == KIND_DOWN) {
      xp = n / 2 - 1 - q;
      row = 0;
    } else {
      const int tq = q / (2 * H), r = i % (2 * H);
      xp = n / 2 - 1 - H * tq - r;
      row = tq & 1;
    }
#pragma unroll
    for (int c = 0; c < C; ++c) slot(row, c, xp) = v[c][i];
  }
}

// The sweep of ONE tile by its group of L lanes (all of one warp): initial line values from the staged rows,
// m + L - 1 skewed super-steps, final line values back to the staged rows (in place).
//   rows : staged two-row state, component c of row r at rows[(r*C + c)*RS + slot]
//   ctr  : slot of x' = 0 (the tile centre);  gl : lane within the group
// RSC = the row stride RS when it is a compile-time constant (FLOW), else 0 (CHAR: it depends on the launch).
template <class Prob, int B, int L, int KIND, int RSC = 0>
__device__ __forceinline__ void char_sweep_tile(typename Prob::R* rows, const int RS, const int ctr, const int gl,
                                                const Consts<typename Prob::R>& kc) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C;
  constexpr int n = B * L;          // tile width
  constexpr int m = n / (2 * H);    // super-columns per tile = tiers per half diamond
  static_assert(B % (2 * H) == 0, "lines per lane must be a multiple of 2h");
  static_assert(L % 2 == 0 && m % 2 == 0 && m >= L, "step pairing needs even L, even m >= L");
  auto slot = [&](int row, int c, int xp) -> R& { return rows[(row * C + c) * RS + ctr + xp]; };

  R v[C][B], halA[C][2 * H], halB[C][2 * H];
  char_load_lines<Prob, B, L, KIND>(v, rows, RS, ctr, gl);
#pragma unroll
  for (int c = 0; c < C; ++c)
#pragma unroll
    for (int e = 0; e < 2 * H; ++e) halA[c][e] = halB[c][e] = (R)0;
  __syncwarp();

  // Loop I/O (group lanes 0 and L-1 only) goes through one pointer advanced by 2h per pair of steps (char_step)
  R* base = rows + ctr;
  uint32_t sbase = smem_u32(base);
  int s = 0;
  for (; s < L; s += 2, base += 2 * H, sbase += 2 * H * (int)sizeof(R)) {  // ramp up: lane gl starts at step gl
    char_step<Prob, B, L, KIND, true, 0, RSC>(v, halA, halB, base, sbase, s, gl, RS, kc);
    char_step<Prob, B, L, KIND, true, 1, RSC>(v, halB, halA, base, sbase, s + 1, gl, RS, kc);
  }
  for (; s < m; s += 2, base += 2 * H, sbase += 2 * H * (int)sizeof(R)) {  // steady state: every lane is inside its m super-columns
    char_step<Prob, B, L, KIND, false, 0, RSC>(v, halA, halB, base, sbase, s, gl, RS, kc);
    char_step<Prob, B, L, KIND, false, 1, RSC>(v, halB, halA, base, sbase, s + 1, gl, RS, kc);
  }
  for (; s < m + L; s += 2, base += 2 * H, sbase += 2 * H * (int)sizeof(R)) {  // ramp down (the last step, s = m+L-1, is empty and keeps the pairing)
    char_step<Prob, B, L, KIND, true, 0, RSC>(v, halA, halB, base, sbase, s, gl, RS, kc);
    char_step<Prob, B, L, KIND, true, 1, RSC>(v, halB, halA, base, sbase, s + 1, gl, RS, kc);
  }
  __syncwarp();
  char_store_lines<Prob, B, L, KIND>(v, rows, RS, ctr, gl);
}

template <class Prob, int B, int L, int KIND>
__global__ void __launch_bounds__(128) swept_char_kernel(const TierArgs<typename Prob::R> a) {
  using R = typename Prob::R;
  constexpr int H = Prob::H, C = Prob::C, PAD = Pad16<R>::value;
  constexpr int n = B * L;          // tile width
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int T = blockDim.x;
  const int chunk = T * B;  // points staged by this CTA (T/L adjacent tiles)
  const int RS = chunk + 2 * PAD;
  R* rows = reinterpret_cast<R*>(smem_raw);
  uint64_t* mbar = reinterpret_cast<uint64_t*>(smem_raw + (size_t)2 * C * RS * sizeof(R));
  const int64_t N = a.N;
  const int tid = threadIdx.x;
  int64_t S = ((int64_t)a.shift + (int64_t)blockIdx.x * chunk) % N;
  const int len1 = (int)((N - S) < (int64_t)chunk ? (N - S) : (int64_t)chunk);
  const int len2 = chunk - len1;
  constexpr int NROWS_IN = (KIND == KIND_UP) ? 1 : 2;

  if (tid == 0) {
    mbar_init(mbar, 1);
    fence_mbar_init();
  }
  __syncthreads();
  if (tid == 0) {
    mbar_arrive_expect_tx(mbar, (uint32_t)(NROWS_IN * C * chunk * sizeof(R)));
#pragma unroll
    for (int r = 0; r < NROWS_IN; ++r) {
      const R* src = r == 0 ? a.in0 : a.in1;
#pragma unroll
      for (int c = 0; c < C; ++c) {
        R* dst = rows + (r * C + c) * RS + PAD;
        bulk_g2s(dst, src + (int64_t)c * N + S, (uint32_t)(len1 * sizeof(R)), mbar);
        if (len2 > 0) bulk_g2s(dst + len1, src + (int64_t)c * N, (uint32_t)(len2 * sizeof(R)), mbar);
      }
    }
  }
  if (KIND == KIND_UP) {
    for (int i = tid; i < C * RS; i += T) rows[C * RS + i] = (R)0;  // tier -1 does not exist
  } else {
    for (int i = tid; i < 2 * C * 2 * H; i += T) {  // halo of the chunk, both rows (periodic)
      const int r = i / (C * 2 * H), c = (i / (2 * H)) % C, j = i % (2 * H);
      const R* src = (r == 0 ? a.in0 : a.in1) + (int64_t)c * N;
      int64_t g = (j < H) ? (S - H + j) : (S + chunk + (j - H));
      if (g < 0) g += N;
      if (g >= N) g -= N;
      const int s = (j < H) ? (PAD - H + j) : (PAD + chunk + (j - H));
      rows[(r * C + c) * RS + s] = src[g];
    }
  }
  mbar_wait(mbar, 0);
  __syncthreads();

  char_sweep_tile<Prob, B, L, KIND>(rows, RS, PAD + (tid / L) * n + n / 2, tid % L, a.k);

  fence_proxy_async_smem();
  __syncthreads();
  if (tid == 0) {
    constexpr int NROWS_OUT = (KIND == KIND_DOWN) ? 1 : 2;
#pragma unroll
    for (int r = 0; r < NROWS_OUT; ++r) {
      R* dstg = r == 0 ? a.out0 : a.out1;
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const R* sm = rows + (r * C + c) * RS + PAD;
        // [lo, hi) of the chunk is written; a wall tile at either end of the row belongs to the TIER launch
        const int lo = (a.skip_first && blockIdx.x == 0) ? n : 0;
        const int hi = chunk - ((a.skip_last && blockIdx.x == gridDim.x - 1) ? n : 0);
        const int e1 = hi < len1 ? hi : len1;  // end of the part before the periodic wrap
        if (e1 > lo) bulk_s2g(dstg + (int64_t)c * N + S + lo, sm + lo, (uint32_t)((e1 - lo) * sizeof(R)));
        const int b2 = lo > len1 ? lo : len1;
        if (hi > b2) bulk_s2g(dstg + (int64_t)c * N + (b2 - len1), sm + b2, (uint32_t)((hi - b2) * sizeof(R)));
      }
    }
    bulk_commit();
    bulk_wait_all();
  }
}

template <class Prob>
inline size_t char_smem_bytes(int threads, int B) {
  using R = typename Prob::R;
  return (size_t)2 * Prob::C * ((size_t)threads * B + 2 * Pad16<R>::value) * sizeof(R) + 16;
}

}  // namespace swept
