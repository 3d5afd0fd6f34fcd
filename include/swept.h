/* swept.h — C ABI of the B200 swept time-space decomposition library (libswept_b200.so).
 *
 * The hot path of "Accelerating solutions of one-dimensional unsteady PDEs with GPU-based swept
 * time-space decomposition" (arXiv 1705.03162; citations below are PAPER.md line numbers):
 * explicit finite-difference / finite-volume time stepping of 1-D periodic PDEs, advanced either
 *   - per step   ("Classic", Fig. 6): one kernel launch per sub-timestep,
 *                working array in global memory; or
 *   - swept      (§4.2, §4.3): UpTriangle, then alternating
 *                SplitDiamond / WholeDiamond, then DownTriangle; each thread block advances one tile of
 *                `tile_width` points through its whole domain of dependence on chip; only the two-row
 *                edge state goes through HBM between launches; the tiling
 *                shifts by half a tile each phase.
 * Both variants evaluate the same IEEE expression trees, so their results are bit-identical
 * ("the swept rule performs the same operations in a different order and location").
 *
 * Conventions
 *   - Every function is extern "C"; no exception crosses the boundary; no torch type appears.
 *   - "host" pointers are ordinary host memory (pageable or pinned), caller-owned.
 *     "device" pointers are CUDA device memory.
 *   - Field layout: component-major C arrays of N REALs.  heat/KS: u[N].  Euler: rho[N], rho*u[N], E[N]
 *     (E = total energy per volume; Eq. D.2 PAPER.md:366 with reading X4 of DESIGN.md).
 *     REAL is double (SWEPT_F64) or float (SWEPT_F32).
 *   - All work is enqueued on the state's stream (swept_set_stream); swept_run never synchronises.
 *   - Return codes: 0 ok; SWEPT_EINVAL bad argument; SWEPT_EUNSUPPORTED unsupported combination;
 *     SWEPT_ECUDA CUDA error (text in swept_last_error); SWEPT_ENOMEM allocation failed.
 *   - A swept_state is not thread-safe; distinct states are independent (multi-GPU = one state per
 *     device, "replicas only": the paper's method is single-GPU).
 *   - There is no CPU fallback: without a CUDA device every compute call fails with SWEPT_ECUDA.
 */
#ifndef SWEPT_H_
#define SWEPT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct swept_state swept_state; /* opaque; owns its device buffers */

enum { SWEPT_HEAT = 0, SWEPT_KS = 1, SWEPT_EULER = 2,       /* problem (App. B-D)  */
       SWEPT_KS3 = 3 };  /* the KS discretisation (C.2) with THREE sub-timesteps per timestep (Shu-Osher SSP-RK3):
                            the case PAPER.md:131 says the two-row decomposition "must be adjusted" for — the
                            inter-launch state has three rows (tier modulo 3).  FP64, periodic; per-step and the
                            swept TIER and CLUSTER flavours */
enum { SWEPT_PER_STEP = 0, SWEPT_SWEPT = 1 };               /* variant                           */
enum { SWEPT_F64 = 0, SWEPT_F32 = 1 };                      /* dtype                             */
enum { SWEPT_RK2_MIDPOINT = 0, SWEPT_RK2_HEUN = 1 };        /* KS/Euler integrator (
                                                               Heun is BASELINE.json config 4)   */
/* boundary conditions: periodic (all BASELINE.json configs) or the paper's own: insulated ends for heat,
 * Eq. (B.5), T_{-1} = T_1 and T_N = T_{N-2} for points 0..N-1; Dirichlet ends for the Euler
 * tube: cells -2, -1 and N, N+1 hold the states that swept_write found in the first and last
 * cell.  SWEPT_BC_PAPER is built for per-step (both flavours), the swept TIER flavour, where the
 * tile split across the boundary applies the condition at its centre, and for heat the CHAR
 * flavour in hybrid mode (wall tiles by the TIER kernels on a second stream), the FLOW flavour
 * (the one or two wall tiles of a row advance tier by tier inside the persistent launch) and the CLUSTER flavour (the
 * lanes next to a wall take the mirror image of their own neighbour point); KS (periodic in the paper)
 * and Euler with FLOW / CHAR / CLUSTER: SWEPT_EUNSUPPORTED. */
enum { SWEPT_BC_PERIODIC = 0, SWEPT_BC_PAPER = 1 };
enum { SWEPT_NKINDS = 6 };                                   /* phase kinds reported by swept_phase_times */
enum { SWEPT_OK = 0, SWEPT_EINVAL = -1, SWEPT_EUNSUPPORTED = -2, SWEPT_ECUDA = -3, SWEPT_ENOMEM = -4 };

/* swept kernel flavours (how a tile is evaluated on chip; results are identical) */
enum {
  SWEPT_FLAVOR_AUTO = 0,  /* library picks (autotuned value if swept_autotune was run)                 */
  SWEPT_FLAVOR_TIER = 1,  /* one CTA per tile, two-row working array in shared memory, one block barrier
                             per tier (the paper's "Shared" arrangement, re-sized)        */
  SWEPT_FLAVOR_CHAR = 2,  /* register-resident sweep along characteristics: a lane group per tile,
                             halo exchange by warp shuffles only, no block barrier       */
  SWEPT_FLAVOR_FLOW = 3,  /* the CHAR sweep inside ONE persistent launch per Up..Down cycle: tiles are
                             tasks, rows are chained by per-tile flags instead of kernel boundaries
                             (DESIGN.md §5.5).  heat and KS, n = 256, 512, 1024   */
  SWEPT_FLAVOR_CLUSTER = 4 /* small problems: the whole domain in ONE thread-block cluster, one launch per
                             Up..Down cycle; a warp per tile, its points in registers, one shuffle exchange per
                             tier; a tile stores its edges straight into the shared memory of the warps that
                             continue them (distributed shared memory, st.async + mbarrier) instead of global
                             memory and a launch.
                             Periodic heat (FP64, FP32), KS and KS3 (three register rows per lane, n <= 256);
                             n = 64, 128, 256, 512 (heat also 32: one point per lane); N / n <= 256 tiles (128 for
                             n >= 256); group = warps per CTA
                             (0 = as few as fit a cluster of 16 CTAs)                                      */
};

/* Optional device allocator hooks (so that PyTorch's caching allocator owns the memory).
 * alloc returns a device pointer or NULL; both are called on the thread that calls swept_create/destroy. */
typedef void* (*swept_alloc_fn)(void* ctx, uint64_t nbytes);
typedef void (*swept_free_fn)(void* ctx, void* device_ptr);

typedef struct {
  uint32_t struct_size; /* = sizeof(swept_params); ABI versioning                                    */
  int32_t dtype;        /* SWEPT_F64 (default) or SWEPT_F32                                          */
  int32_t rk2;          /* SWEPT_RK2_*; ignored for heat                                             */
  int32_t device;       /* CUDA ordinal, -1 = current device                                         */
  double alpha;         /* heat diffusivity (Eq. B.1)                                  */
  double gamma;         /* Euler heat-capacity ratio, 1.4                             */
  void* stream;         /* cudaStream_t used by all calls on this state (NULL = legacy default stream) */
  swept_alloc_fn alloc; /* NULL = cudaMalloc                                                         */
  swept_free_fn free;   /* NULL = cudaFree                                                           */
  void* alloc_ctx;      /* passed back to alloc/free                                                 */
  int32_t bc;           /* SWEPT_BC_PERIODIC (default) or SWEPT_BC_PAPER                                */
  int32_t reserved0;    /* 0                                                                           */
} swept_params;

/* swept_create — set up one problem: N periodic points, spacing dx, fixed timestep dt.
 * Scheme constants are computed once, in double, on the host (Fo = alpha dt/dx^2; etc.) and
 * rounded once to REAL.  p may be NULL (FP64, midpoint, alpha = 1, gamma = 1.4, current device).
 * Requires 8 <= N <= 2^31, dx > 0, dt > 0 (the swept variant additionally needs N to hold at least one tile:
 * N >= 32, see swept_run).  All device memory the state will ever use — four field slabs and the scratch of the
 * persistent flavours — is allocated here, through p->alloc when given; creation may synchronise p->stream.
 * p->stream = NULL means the CUDA legacy default stream (the Python binding passes torch's current stream and
 * re-sets it with swept_set_stream before every call).  Returns NULL on error.
 * Debugging aid: with the environment variable SWEPT_POISON set, every field slab is filled with 0xFF bytes (NaNs)
 * at creation, so that a kernel reading a value no kernel wrote yields a visibly wrong result. */
swept_state* swept_create(int problem, int64_t N, double dx, double dt, const swept_params* p);

/* swept_write — copy initial data from HOST memory (C*N REALs, layout above) to the device, asynchronously
 * on the state's stream (the host buffer must stay valid until the stream reaches the copy; pageable
 * memory makes the call synchronous).  Resets the step counter. */
int swept_write(swept_state* s, const void* host_buf);

/* swept_write_device — same, from DEVICE memory (device-to-device copy on the stream).  With SWEPT_BC_PAPER on
 * the Euler problem the six end-state scalars are read back on the state's stream and the call synchronises it.
 * (Both write calls: new Dirichlet end states discard the cached per-step CUDA graphs, which hold them.) */
int swept_write_device(swept_state* s, const void* device_buf);

/* swept_run — advance by nsteps full timesteps (PAPER.md:236 counts timesteps; KS/Euler timesteps have two
 * sub-timesteps).
 *   variant SWEPT_PER_STEP: tile_width = threads per block of the per-step kernel (32..1024, power of two;
 *                           0 = library default).  One launch per sub-timestep (heat, Euler) or per timestep
 *                           with both RK2 stages fused (KS), replayed from a CUDA graph in chunks.
 *   variant SWEPT_SWEPT   : tile_width = n = spatial points per tile ("node"), a power of two,
 *                           32 <= n <= 4096 (the paper sweeps 32..1024), n >= 16 h for the
 *                           5-point problems, N % n == 0; 0 = autotuned / default value.
 *                           The run is Up, D diamonds, Down, covering the largest T = (D+1) n/(2h)
 *                           sub-timesteps that fit; what is left runs further Up..Down cycles of width n/2,
 *                           n/4, ... >= 32 and finally per-step stages (readout granularity, PAPER.md:83;
 *                           reading G5).  If N has no admissible tile the call fails with
 *                           SWEPT_EUNSUPPORTED.
 * Asynchronous on the state's stream: the call enqueues kernels (and, the first time a 256-step per-step chunk is
 * needed, records a CUDA graph on a private stream); it neither allocates device memory nor synchronises, so it
 * may itself be captured into a CUDA graph.  Launch errors surface at the next synchronising call
 * (swept_read, swept_sync, swept_phase_times, swept_autotune). */
int swept_run(swept_state* s, int64_t nsteps, int32_t tile_width, int variant);

/* per-step flavours */
enum {
  SWEPT_PS_LAUNCH = 0,   /* one launch per sub-timestep (CUDA-graph replay): the paper's "Classic" */
  SWEPT_PS_RESIDENT = 1  /* the same sub-timesteps in ONE persistent cooperative launch: field in registers,
                            neighbour-only synchronisation through global flags (PAPER.md:297-303 future work;
                            DESIGN.md §5.7).  Needs N small enough for a co-resident grid (heat FP64: N <= 2^20
                            on B200), else SWEPT_EUNSUPPORTED; tile_width is ignored                            */
};

/* swept_run_flavor — swept_run with an explicit kernel flavour in bits 0..7 of `flavor` (SWEPT_FLAVOR_* for
 * variant SWEPT_SWEPT, SWEPT_PS_* for SWEPT_PER_STEP) and the flavour's group parameter in bits 8..15
 * (TIER: points per thread; CHAR: lanes per tile; CLUSTER: warps per CTA; FLOW: resident CTAs per SM in its bits 0..3,
 * 0 = default, and in its bit 4 (value 16) how a tile's rows travel between global and shared memory: 1 = TMA bulk
 * copies (cp.async.bulk + mbarrier) issued by one lane, 0 = 16-byte loads / stores of all lanes; group 0 = the
 * library's defaults: TMA copies, resident CTAs from the tiles per row). */
int swept_run_flavor(swept_state* s, int64_t nsteps, int32_t tile_width, int variant, int flavor);

/* swept_read — synchronise the stream and copy the current field to HOST memory (same layout as
 * swept_write).  Errors of the asynchronous launches since the last synchronising call surface here
 * (SWEPT_ECUDA), including a FLOW launch whose dependency wait timed out. */
int swept_read(swept_state* s, void* host_buf);

/* swept_sync — synchronise the state's stream and report what the asynchronous launches since the last
 * synchronising call left behind: SWEPT_ECUDA if a persistent launch (FLOW, PS_RESIDENT) gave up waiting for a
 * dependency — its tiles are then not stored and the field is invalid — else 0.  Callers that consume
 * swept_device_ptr directly (no swept_read) use this to learn about such a failure. */
int swept_sync(swept_state* s);

/* swept_device_ptr — DEVICE pointer to the current full time level (C*N REALs), valid until the next
 * swept_run/swept_write on this state; stream-ordered (no synchronisation). */
const void* swept_device_ptr(swept_state* s);

/* swept_autotune — time short runs over admissible tile widths (and flavours) for `variant`
 * (the paper also keeps the best block size per N), restore the field, remember and return
 * the best tile width.  Synchronises.  The result is also kept in a process-wide cache keyed by (device, problem,
 * dtype, rk2, bc, N): states created later for the same key start with it (tile_width = 0 uses it). */
int swept_autotune(swept_state* s, int variant, int32_t* best_tile_width);

/* swept_tuned — what swept_autotune remembered for `variant`: tile width, swept flavour and its group
 * parameter (TIER: points per thread; CHAR: lanes per tile; FLOW: resident CTAs per SM); zeros if autotune has not run. */
int swept_tuned(const swept_state* s, int variant, int32_t* tile_width, int32_t* flavor, int32_t* group);

/* swept_set_stream — change the stream used by subsequent calls (cudaStream_t). */
int swept_set_stream(swept_state* s, void* stream);

/* swept_steps_done — timesteps advanced since the last swept_write. */
int64_t swept_steps_done(const swept_state* s);

/* swept_last_launches — number of kernel launches (graph nodes included) issued by the last swept_run. */
int64_t swept_last_launches(const swept_state* s);

/* swept_set_phase_timing — on != 0: every later swept_run brackets each swept launch (and the per-step
 * remainder as a whole) with a pair of CUDA events recorded on the state's stream, so that the duration of
 * each kernel kind can be measured live, inside a timed region, without a profiler.  Off by default. */
int swept_set_phase_timing(swept_state* s, int on);

/* swept_phase_times — synchronise the stream (reporting failures like swept_sync) and return, per phase kind (index 0 Up, 1 SplitDiamond,
 * 2 WholeDiamond, 3 Down, 4 per-step remainder, 5 whole FLOW cycle), the summed device time in milliseconds
 * and the number of kernel launches recorded since timing was switched on or since the previous call; then
 * reset the record.  ms and launches are caller-owned HOST arrays of SWEPT_NKINDS (6) entries. */
int swept_phase_times(swept_state* s, double* ms, int64_t* launches);

void swept_destroy(swept_state* s);

/* swept_last_error — thread-local message of the last failing call on this thread. */
const char* swept_last_error(void);

/* ---- host-only helpers (no GPU needed) ------------------------------------------------------------ */

/* One phase of the swept schedule: kind 0 Up, 1 SplitDiamond, 2 WholeDiamond, 3 Down,
 * 4 per-step remainder.  `shift` = offset of the tiling in points (0 or n/2), `tier0` = global sub-timestep
 * index at which the phase's relative tier 0 sits, `ntiers` = tiers it computes at its tallest column,
 * `n` = tile width of the phase (0 for the per-step remainder). */
typedef struct {
  int32_t kind;
  int32_t shift;
  int64_t tier0;
  int64_t ntiers;
  int32_t n;
  int32_t reserved;
} swept_phase;

/* swept_plan — the phase list swept_run executes for nsub = sigma*nsteps sub-timesteps with tile width n and
 * stencil half-width h: one Up / D diamonds / Down cycle of width n covering the largest T = (D+1) n/(2h) <= nsub
 * (PAPER.md:83), then further cycles of width n/2, n/4, ... >= 32 for what is left (reading G5),
 * then a per-step remainder.  (swept_run additionally skips widths for which N has no kernel.)
 * Writes at most max_phases entries, returns the number of phases needed (or a negative error code). */
int64_t swept_plan(int64_t nsub, int32_t n, int32_t h, swept_phase* out, int64_t max_phases);

/* swept_plan_sigma — the same for a scheme with `sigma` sub-timesteps per timestep (1, 2 or 3; swept_plan is the
 * sigma <= 2 case).  A cycle must end on a full timestep, i.e. T = (D+1) n/(2h) must be a multiple of sigma: with
 * n/(2h) a power of two that is automatic for sigma = 1, 2 and means (D+1) % 3 == 0 for sigma = 3 (PAPER.md:131:
 * the decomposition "must be adjusted" for more than two sub-timesteps).  Phases of a sigma = 3 cycle may start on
 * any tier: tier0 % 3 tells the kernel which stage its first tier is. */
int64_t swept_plan_sigma(int64_t nsub, int32_t n, int32_t h, int32_t sigma, swept_phase* out, int64_t max_phases);

/* ---- sharding over several GPUs ------------------------------------------
 * The paper's motivation is distributed memory: a swept phase needs ONE exchange with the neighbour where a
 * per-step scheme needs one per sub-timestep.  Here the N points are cut into `nshards`
 * contiguous blocks of n_local = N / nshards points (a whole number of tiles), one swept_state per block, normally
 * one per GPU.  A shard keeps its own points 0 .. n_local-1 and a ghost zone of `tile_width` points behind them
 * (local points n_local .. n_local + tile_width - 1, which is also where its negative local points -1, -2, ... live:
 * the shard's array is periodic in n_local + tile_width).  On a shifted row of tiles the shard computes the tile that
 * straddles its right end, i.e. the first half tile of its right neighbour, and hands it over afterwards; before a
 * shifted row it receives the neighbour's first half tile (plus h halo points).  So there is exactly one message per
 * phase and neighbour pair, alternating in direction, of rows x C x (tile_width/2 + h) values — the paper's edge
 * hand-off across the GPU boundary.  The per-step remainder (fewer than 16 sub-timesteps) is done
 * with one exchange of ntiers*h points each way, after which the shards step independently.  Results are bit-identical
 * to the unsharded run (tests/test_gpu_shard.py).  The tiles a shard computes inside its ghost zone are redundant work
 * (one tile in n_local/tile_width + 1); whatever they write is overwritten by the next message before it is read.
 *
 * A shard state supports swept_write / swept_read / swept_sync / swept_device_ptr-free use as below; swept_run on it
 * fails (a shard cannot advance alone).  Only the phase-wise flavours (TIER, CHAR) exist for shards. */

/* One edge exchange of a sharded run.  Coordinates are LOCAL points of the sender / receiver (0 = first own point;
 * n_local .. = ghost zone; negative = left halo, stored at the end of the ghost zone). */
typedef struct {
  int32_t after_phase; /* happens after this entry of the phase list and before the next one (-1: before the first) */
  int32_t dir;         /* +1: every shard sends to its right neighbour (shard+1 mod nshards), -1: to its left one   */
  int64_t src_off;     /* first point sent, sender's local coordinates                                              */
  int64_t dst_off;     /* where it lands, receiver's local coordinates                                              */
  int32_t count;       /* points                                                                                    */
  int32_t rows;        /* rows of the inter-launch state sent (all of them, or 1 = the full time level)             */
} swept_exchange;

/* swept_shard_exchanges — host-only: the exchanges that go with a phase list from swept_plan / swept_plan_sigma for
 * shards of n_local points (rows_state = 2, or 3 for sigma = 3).  Writes at most max_out entries, returns the number
 * needed (or a negative error code).  The same list holds for every shard. */
int64_t swept_shard_exchanges(const swept_phase* plan, int64_t nphases, int32_t h, int32_t sigma, int64_t n_local,
                              swept_exchange* out, int64_t max_out);

/* swept_shard_create — one shard (index `shard` of `nshards`) of a problem of N periodic points advanced with swept
 * tile width `tile_width`; N % (nshards * tile_width) == 0.  Parameters as swept_create (periodic problems only).
 * swept_write / swept_read on the returned state move the shard's OWN n_local = N / nshards points per component
 * (host layout: C arrays of n_local REALs). */
swept_state* swept_shard_create(int problem, int64_t N, int32_t nshards, int32_t shard, int32_t tile_width, double dx,
                                double dt, const swept_params* p);

/* Phase-wise execution, for a caller that owns the transport (one process per GPU: torch.distributed / NCCL):
 *   swept_shard_begin(s, nsteps, flavor)  plan `nsteps` timesteps (flavor: SWEPT_FLAVOR_AUTO / _TIER / _CHAR with the
 *                                         group in bits 8..15); returns the number of phases, the same on every shard
 *   swept_shard_exchange_list(s, out, max) the exchanges of that plan (as swept_shard_exchanges)
 *   swept_shard_phase(s)                  enqueue the next phase on the state's stream
 *   swept_shard_pack(s, x, buf)           enqueue the gather of exchange x into the DEVICE buffer buf
 *                                         (swept_shard_message_bytes(s, x) bytes)
 *   swept_shard_unpack(s, x, buf)         enqueue the scatter of a received message
 *   swept_shard_end(s)                    close the run (step counter)
 * Order per phase i: phase; then for every exchange x with after_phase == i: pack, transport, unpack. */
int64_t swept_shard_begin(swept_state* s, int64_t nsteps, int flavor);
int64_t swept_shard_exchange_list(swept_state* s, swept_exchange* out, int64_t max_out);
int64_t swept_shard_message_bytes(swept_state* s, int64_t x);
int swept_shard_phase(swept_state* s);
int swept_shard_pack(swept_state* s, int64_t x, void* device_buf);
int swept_shard_unpack(swept_state* s, int64_t x, const void* device_buf);
int swept_shard_end(swept_state* s);

/* swept_shard_run — all shards in ONE process (shards[i] = shard i; on one device or on several with peer access):
 * runs the phases of every shard on its own stream and moves each message with one cudaMemcpyAsync between the
 * shards' staging buffers, ordered by events (no host synchronisation).  Asynchronous like swept_run. */
int swept_shard_run(swept_state* const* shards, int32_t nshards, int64_t nsteps, int flavor);

/* ---- an entry point that allocates nothing ---------------------------------------------------------------------
 * Some callers cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 * swept_heat_flow_static advances the periodic heat problem (FTCS, Eq. (B.4); FP64) by ONE swept cycle
 * — UpTriangle, D Split/WholeDiamond rows, DownTriangle in one persistent FLOW launch — with every
 * byte of scratch in a file-scope device array of the library: the kernel's ticket / leave counters and per-tile
 * flags, and three of the four row slabs of the two-row inter-launch state (the fourth is out_dev, which therefore
 * holds intermediate rows until the launch ends).  It calls no cudaMalloc, cudaFree or allocating library routine and
 * needs no swept_state.
 *   in_dev, out_dev : DEVICE buffers of N doubles, 16-byte aligned, not overlapping; caller-owned
 *   N               : points, a multiple of tile_width, N <= SWEPT_STATIC_MAX_N (65 536); larger -> SWEPT_EINVAL
 *   nsteps          : a positive multiple of tile_width / 2 (the cycle's (D + 1) n/(2h) sub-timesteps, no remainder)
 *   tile_width      : 256, 512 or 1024
 *   dx, dt, alpha   : as swept_create (Fo = alpha dt / dx^2 computed in double on the host)
 *   stream          : cudaStream_t; the call is asynchronous on it and runs on the CURRENT device
 * The result is bit-identical to swept_run(..., SWEPT_SWEPT) on a state of the same problem (same kernel, same
 * functor).  Limits: the array (SWEPT_STATIC_SCRATCH_BYTES = 1 576 960 bytes) is held by every GPU that loads the
 * library until the process exits; ALL calls on a device share it, and it keeps the last call's contents (the
 * counters and flags are cleared at the start of every call, on `stream`): calls that overlap on the GPU — two
 * streams, two host threads — race; serialise them.  swept_heat_flow_static_check(stream) synchronises the stream and
 * reports SWEPT_ECUDA if the last launch gave up waiting for a dependency (call it before the next launch clears the
 * word). */
enum { SWEPT_STATIC_MAX_N = 65536, SWEPT_STATIC_SCRATCH_BYTES = 4096 + 3 * 65536 * 8 };
int swept_heat_flow_static(const double* in_dev, double* out_dev, int64_t N, int64_t nsteps, int32_t tile_width,
                           double dx, double dt, double alpha, void* stream);
int swept_heat_flow_static_check(void* stream);

/* ---- measurement helpers --------------------------------------------------------------------------- */

/* swept_probe_fp64 — run a register-only DFMA chain on every SM of `device` and return FP64 pipe
 * instructions per second (warp-instructions * 32 lanes), i.e. the measured ALU roofline denominator. */
int swept_probe_fp64(int device, void* stream, double* fp64_lane_ops_per_s);

/* swept_probe_launch — average cost in microseconds of launching an empty kernel `count` times
 * back to back on `stream` (PAPER.md:253 measures the same on the K40c: about 4 us). */
int swept_probe_launch(int device, void* stream, int count, double* us_per_launch);

/* swept_flow_profile — where the warps of the FLOW flavour spend their time.  on != 0: later FLOW launches of this
 * state (heat FP64) run an instrumented copy of the kernel that stamps clock64() between the parts of every tile task;
 * on == 0: back to the plain kernel.  Either way the call synchronises, copies the 8 counters accumulated so far to
 * the caller's HOST array if it is not NULL — SM cycles summed over all warps spent [0] taking a ticket, [1] waiting
 * for the two parent tiles, [2] staging the rows, [3] sweeping, [4] storing and publishing; [5] = tiles done — and
 * clears them. */
int swept_flow_profile(swept_state* s, int on, uint64_t* counters);

/* swept_probe_chain — cycles per dependent DADD -> DFMA pair (one warp, one chain per lane): the latency a heat
 * update puts on the critical path of every tier, i.e. the denominator of the latency bound that governs small N
 * (a tile of n points cannot advance faster than one tier per chain link). */
int swept_probe_chain(int device, void* stream, double* cycles_per_dadd_dfma);

/* swept_probe_tier — cycles per link of the dependent chain of a register-resident tier (the CLUSTER flavour, one warp,
 * one point per lane), written to the caller's HOST array of 4 doubles: [0] shuffle -> shuffle; [1] both neighbours by
 * 64-bit shuffles -> DADD -> DFMA; [2] the same -> select on the tier window, i.e. one whole heat tier; [3] DFMA ->
 * select.  [2] is the floor of that flavour's time per tier. */
int swept_probe_tier(int device, void* stream, double* cycles4);

/* swept_probe_smem — shared-memory read bandwidth of the whole device (conflict-free 16-byte loads from 32 KiB per
 * CTA, 2 CTAs of 1024 threads per SM), in bytes per second and, if the pointer is given, bytes per clock and SM at
 * the device's maximum SM clock: the measured counterpart of the nominal 128 B/clk/SM. */
int swept_probe_smem(int device, void* stream, double* bytes_per_s, double* bytes_per_clk_per_sm);

/* swept_probe_sweep — the characteristic sweep of the CHAR / FLOW flavours (swept_char.cuh, L = 32 lanes per tile) on
 * ONE SM with no global traffic: 4 * warps_per_scheduler warps each sweep a staged WholeDiamond tile of
 * 32 * lines_per_lane points (lines_per_lane = 8, 16, 32; problem = SWEPT_HEAT or SWEPT_KS, FP64) several times.
 * Returns the SM cycles per super-step (all warps) and, if the pointer is given, the fraction of the FP64 pipe's
 * issue cycles that is busy.  The issue-rate model of DESIGN.md §5.6 is read off this probe. */
int swept_probe_sweep(int device, void* stream, int problem, int lines_per_lane, int warps_per_scheduler,
                      double* cycles_per_step, double* fp64_busy);

#ifdef __cplusplus
}
#endif
#endif /* SWEPT_H_ */
