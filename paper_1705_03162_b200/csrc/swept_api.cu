// swept_api.cu — the C ABI declared in include/swept.h: state, phase driver,
// per-step driver with CUDA-graph replay, autotuner (row a8) and measurement probes.
//
// Nothing here touches the field values on the host except the explicit copies of swept_write/read;
// there is no CPU fallback: every compute path is a kernel launch.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <tuple>
#include <vector>

#include "../../include/swept.h"
#include "internal.h"

namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}
#define CUDA_TRY(expr)                                                                      \
  do {                                                                                      \
    cudaError_t e_ = (expr);                                                                \
    if (e_ != cudaSuccess)                                                                  \
      return fail(e_ == cudaErrorMemoryAllocation ? SWEPT_ENOMEM : SWEPT_ECUDA, "%s: %s", #expr, \
                  cudaGetErrorString(e_));                                                  \
  } while (0)

constexpr int KIND_UP = 0, KIND_SPLIT = 1, KIND_WHOLE = 2, KIND_DOWN = 3, KIND_REMAINDER = 4, KIND_FLOW = 5;

struct ProblemShape {
  int h, sigma, C;
};
const ProblemShape kShape[4] = {{1, 1, 1}, {2, 2, 1}, {2, 2, 3}, {2, 3, 1}};
constexpr int MAX_SLABS = 6;

struct GraphKey {
  int threads, P, cur, steps;
  bool operator<(const GraphKey& o) const {
    return std::tie(threads, P, cur, steps) < std::tie(o.threads, o.P, o.cur, o.steps);
  }
};

// autotune results of this process, keyed by (device, problem, dtype, rk2, bc, N) — PAPER.md:236 keeps the best
// launch configuration per problem size; a state created later for the same key starts with it
struct TunedEntry {
  int width[2] = {0, 0};
  int flavor = 0, P = 0;
};
using TunedKey = std::tuple<int, int, int, int, int, int64_t>;
std::mutex g_tuned_mutex;
std::map<TunedKey, TunedEntry> g_tuned;

}  // namespace

namespace swept {
void set_last_error(const char* msg) { g_err = msg ? msg : ""; }
}  // namespace swept

struct swept_state {
  int problem = 0, dtype = 0, rk2 = 0, device = 0, bc = 0;
  int64_t N = 0;
  double dx = 0, dt = 0, alpha = 1, gamma = 1.4;
  double consts[5] = {0, 0, 0, 0, 0};
  double bcvals[6] = {0, 0, 0, 0, 0, 0};  // Dirichlet end states (Euler tube): left[3], right[3], set by swept_write
  int kernel_bc() const { return bc == 0 ? 0 : (problem == SWEPT_HEAT ? 1 : 2); }
  cudaStream_t stream = nullptr;
  cudaStream_t capture_stream = nullptr;  // graphs are recorded here (the legacy default stream cannot capture)
  swept_alloc_fn alloc = nullptr;
  swept_free_fn free_ = nullptr;
  void* alloc_ctx = nullptr;
  size_t slab_bytes = 0;
  // field slabs: twice the rows of the inter-launch state (phases ping-pong between two buffers): 4 for the two-row
  // schemes, 6 for the three-row one (KS3)
  void* slab[MAX_SLABS] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  int nslabs = 4;
  int rows() const { return nslabs / 2; }
  int cur = 0;  // slab holding the current full time level
  int64_t steps_done = 0, last_launches = 0;
  // autotune results: [variant] -> tile width, flavour, P
  int tuned_width[2] = {0, 0};
  int tuned_flavor = 0, tuned_P = 0;
  std::map<GraphKey, cudaGraphExec_t> graphs;
  // live per-kind timing (swept_set_phase_timing): event pairs recorded around launches
  struct Timed { int kind; int64_t launches; cudaEvent_t e0, e1; };
  bool timing = false;
  std::vector<Timed> timed;
  std::vector<cudaEvent_t> event_pool;
  // FLOW flavour scratch (allocated and zeroed by swept_create): word 0 = ticket counter, word 1 = sticky error
  // word, word 2 = leave counter, words 4.. = 2 * N/256 flags (swept_flow.cuh).  Every launch leaves the counters
  // and flags zero again, so nothing is cleared between launches.
  int* flow_scratch = nullptr;
  size_t flow_scratch_ints = 0;
  bool flow_pending_check = false;
  unsigned long long* flow_prof = nullptr;  // 8 counters of the instrumented FLOW kernel (swept_flow_profile)
  bool flow_prof_on = false;
  cudaStream_t wall_stream = nullptr;  // hybrid wall handling: the wall tiles run here, beside the CHAR launch
  cudaEvent_t wall_fork = nullptr, wall_join = nullptr;
  // the phase list of the swept run being executed (swept_run plans and runs it in one go; the shard driver,
  // swept_phase_begin / swept_phase_run, one phase at a time with edge exchanges in between)
  struct Planned {
    std::vector<swept_phase> plan;
    std::map<int, std::pair<int, int>> cfg;  // tile width -> (flavour, group)
    int rin[3] = {-1, -1, -1};               // slabs holding the rows written by the last phase
    int nrows_valid = 0;                     // rows of `rin` that hold data (1 after Down: the full time level)
    size_t next = 0;
    int64_t nsteps = 0;
  } pr;
  // shard mode (swept_shard_create): this state holds n_local own points and a ghost zone of shard_n points behind
  // them; N = shard_nloc + shard_n is the extent of its (periodic) arrays
  int64_t shard_nloc = 0;
  int shard_n = 0, nshards = 0, shard_index = 0;
  void* shard_send = nullptr;  // staging buffers of swept_shard_run: one message each
  void* shard_recv = nullptr;
  size_t shard_buf_bytes = 0;
  std::vector<swept_exchange> xch;  // exchanges of the planned run
  cudaEvent_t shard_packed = nullptr, shard_send_free = nullptr;
  bool shard_send_busy = false;
  bool is_shard() const { return nshards > 0; }
  void* resident_scratch = nullptr;  // flags + exchange slots of the resident per-step kernel
  bool resident_pending_check = false;  // a FLOW launch has run since the error word was last read
  size_t elem() const { return dtype == SWEPT_F64 ? 8 : 4; }
};

namespace {

using swept::NO_KERNEL;

int set_device(const swept_state* s) {
  CUDA_TRY(cudaSetDevice(s->device));
  return 0;
}

int launch_per_step(swept_state* s, const void* in, const void* base, void* out, int odd, int threads, int P) {
  swept::PerStepLaunch a{in, base, out, s->N, odd, threads, P, s->consts, s->stream, s->kernel_bc(), s->bcvals};
  int rc;
  switch (s->problem) {
    case SWEPT_HEAT: rc = swept::launch_per_step_heat(s->dtype, a); break;
    case SWEPT_KS: rc = swept::launch_per_step_ks(s->dtype, s->rk2, a); break;
    case SWEPT_KS3: rc = swept::launch_per_step_ks3(s->dtype, a); break;
    default: rc = swept::launch_per_step_euler(s->dtype, s->rk2, a); break;
  }
  if (rc == NO_KERNEL) return fail(SWEPT_EUNSUPPORTED, "no per-step kernel for this problem/dtype/P=%d", P);
  if (rc != 0) return fail(SWEPT_ECUDA, "per-step launch: %s", cudaGetErrorString((cudaError_t)rc));
  return 0;
}

int launch_tile(swept_state* s, swept::TileLaunch& a, cudaStream_t stream = nullptr) {
  a.N = s->N;
  a.consts = s->consts;
  a.stream = stream ? stream : s->stream;
  a.bc = s->kernel_bc();
  a.bcv = s->bcvals;
  int rc;
  switch (s->problem) {
    case SWEPT_HEAT: rc = swept::launch_tile_heat(s->dtype, a); break;
    case SWEPT_KS: rc = swept::launch_tile_ks(s->dtype, s->rk2, a); break;
    case SWEPT_KS3: rc = swept::launch_tile_ks3(s->dtype, a); break;
    default: rc = swept::launch_tile_euler(s->dtype, s->rk2, a); break;
  }
  if (rc == NO_KERNEL)
    return fail(SWEPT_EUNSUPPORTED, "no swept kernel for flavor=%d n=%d P=%d", a.flavor, a.n, a.P);
  if (rc != 0) return fail(SWEPT_ECUDA, "swept launch: %s", cudaGetErrorString((cudaError_t)rc));
  return 0;
}

// device memory through the caller's allocator hooks (swept_params.alloc / free), else cudaMalloc / cudaFree
void* dev_alloc(swept_state* s, size_t bytes) {
  void* ptr = nullptr;
  if (s->alloc) return s->alloc(s->alloc_ctx, bytes);
  if (cudaMalloc(&ptr, bytes) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  return ptr;
}
void dev_free(swept_state* s, void* ptr) {
  if (!ptr) return;
  if (s->free_) s->free_(s->alloc_ctx, ptr);
  else cudaFree(ptr);
}

constexpr int FLOW_MIN_WIDTH = 256;  // narrowest tile of the FLOW flavour: sizes the flag array

int launch_flow(swept_state* s, swept::FlowLaunch& a) {
  a.N = s->N;
  a.consts = s->consts;
  a.stream = s->stream;
  const size_t need = 4 + 2 * (size_t)(s->N / a.n);
  if (!s->flow_scratch || need > s->flow_scratch_ints)
    return fail(SWEPT_EUNSUPPORTED, "no FLOW kernel for this problem / n=%d", a.n);
  a.ticket = (unsigned*)s->flow_scratch;
  a.flags = s->flow_scratch + 4;
  a.prof = s->flow_prof_on ? s->flow_prof : nullptr;
  a.bc = s->kernel_bc();
  int rc;
  switch (s->problem) {
    case SWEPT_HEAT: rc = swept::launch_flow_heat(s->dtype, a); break;
    case SWEPT_KS: rc = swept::launch_flow_ks(s->dtype, s->rk2, a); break;
    default: rc = NO_KERNEL; break;
  }
  if (rc == NO_KERNEL) return fail(SWEPT_EUNSUPPORTED, "no FLOW kernel for this problem / n=%d", a.n);
  if (rc != 0) return fail(SWEPT_ECUDA, "flow launch: %s", cudaGetErrorString((cudaError_t)rc));
  s->flow_pending_check = true;
  return 0;
}

// after a stream synchronisation: did any FLOW launch give up waiting for a dependency?
int check_flow_error(swept_state* s) {
  if (s->resident_pending_check && s->resident_scratch) {
    s->resident_pending_check = false;
    int err = 0;
    int* word = (int*)s->resident_scratch + swept::RESIDENT_MAX_CTAS * 32;
    CUDA_TRY(cudaMemcpy(&err, word, sizeof(int), cudaMemcpyDeviceToHost));
    if (err) CUDA_TRY(cudaMemset(word, 0, sizeof(int)));
    if (err) return fail(SWEPT_ECUDA, "resident per-step kernel: a CTA waited too long for its neighbour");
  }
  if (!s->flow_pending_check || !s->flow_scratch) return 0;
  s->flow_pending_check = false;
  int err = 0;
  CUDA_TRY(cudaMemcpy(&err, s->flow_scratch + 1, sizeof(int), cudaMemcpyDeviceToHost));
  if (err) {
    CUDA_TRY(cudaMemset(s->flow_scratch + 1, 0, sizeof(int)));
    return fail(SWEPT_ECUDA, "FLOW kernel: a tile waited too long for its parents (grid not co-resident?); "
                             "the field is invalid, write it again");
  }
  return 0;
}

cudaEvent_t take_event(swept_state* s) {
  cudaEvent_t e = nullptr;
  if (!s->event_pool.empty()) {
    e = s->event_pool.back();
    s->event_pool.pop_back();
  } else {
    cudaEventCreate(&e);
  }
  return e;
}

// RAII bracket: records e0 now and e1 at scope exit when phase timing is on
struct TimedScope {
  swept_state* s;
  size_t idx = 0;
  bool on;
  TimedScope(swept_state* s_, int kind, int64_t launches) : s(s_), on(s_->timing) {
    if (!on) return;
    swept_state::Timed t{kind, launches, take_event(s), take_event(s)};
    cudaEventRecord(t.e0, s->stream);
    idx = s->timed.size();
    s->timed.push_back(t);
  }
  ~TimedScope() {
    if (on) cudaEventRecord(s->timed[idx].e1, s->stream);
  }
};

bool tile_ok(const swept_state* s, int flavor, int n, int P) {
  if (n <= 0 || s->N % n != 0) return false;
  // walls are applied by the TIER kernels; for heat also by the CHAR flavour in hybrid mode (wall tiles by TIER launches
  // beside it) and by the FLOW flavour (wall tiles tier by tier inside the persistent launch)
  if (s->bc && flavor != SWEPT_FLAVOR_TIER &&
      !((flavor == SWEPT_FLAVOR_CHAR || flavor == SWEPT_FLAVOR_FLOW || flavor == SWEPT_FLAVOR_CLUSTER) &&
        s->problem == SWEPT_HEAT))
    return false;
  if (s->bc && flavor == SWEPT_FLAVOR_CHAR && !swept::tile_config_ok_heat(s->dtype, SWEPT_FLAVOR_TIER, s->N, n, 1))
    return false;
  if (flavor == SWEPT_FLAVOR_CLUSTER && s->problem == SWEPT_EULER) return false;
  if (flavor == SWEPT_FLAVOR_FLOW && (s->problem == SWEPT_EULER || s->problem == SWEPT_KS3 || P < 0 || (P & 15) > 12 || P > 31 || !s->flow_scratch)) return false;
  switch (s->problem) {
    case SWEPT_HEAT: return swept::tile_config_ok_heat(s->dtype, flavor, s->N, n, P);
    case SWEPT_KS: return swept::tile_config_ok_ks(s->dtype, flavor, s->N, n, P);
    case SWEPT_KS3: return swept::tile_config_ok_ks3(s->dtype, flavor, s->N, n, P);
    default: return swept::tile_config_ok_euler(s->dtype, flavor, s->N, n, P);
  }
}

int per_step_P(const swept_state* s) {
  const int pmax = s->problem == SWEPT_EULER ? 2 : 4;
  for (int P = pmax; P > 1; P /= 2)
    if (s->N % P == 0 && (s->N / P) >= 32) return P;
  return 1;
}

// ---- per-step driver --------------------------------------------------------------------------------
// One timestep = sigma launches.  Buffers: cur -> (pred) -> nxt, then cur and nxt swap, so an even number
// of steps returns to the same buffer assignment and a captured chunk can be replayed.
int enqueue_steps(swept_state* s, int64_t steps, int threads, int P, int* cur_io) {
  const int sigma = kShape[s->problem].sigma;
  int cur = *cur_io;
  const int ns = s->nslabs;
  int nxt = (cur + 1) % ns, pred = (cur + 2) % ns, pred2 = (cur + 3) % ns;
  for (int64_t i = 0; i < steps; ++i) {
    if (sigma == 3) {
      // three stages: u1 from u^n; u2 from u1 and u^n; u^{n+1} from u2 and u^n (stage index = tier modulo 3)
      if (int rc = launch_per_step(s, s->slab[cur], s->slab[cur], s->slab[pred], 1, threads, P)) return rc;
      if (int rc = launch_per_step(s, s->slab[pred], s->slab[cur], s->slab[pred2], 2, threads, P)) return rc;
      if (int rc = launch_per_step(s, s->slab[pred2], s->slab[cur], s->slab[nxt], 0, threads, P)) return rc;
    } else if (sigma == 1) {
      if (int rc = launch_per_step(s, s->slab[cur], s->slab[cur], s->slab[nxt], 0, threads, P)) return rc;
    } else if (s->problem == SWEPT_KS && P >= 2) {
      // both RK2 stages in one launch (north_star: "one launch per timestep or RK stage")
      swept::PerStepLaunch a{s->slab[cur], s->slab[cur], s->slab[nxt], s->N, 0, threads, P, s->consts, s->stream, 0,
                             nullptr};
      const int rc = swept::launch_per_step_ks_fused(s->dtype, s->rk2, a);
      if (rc == NO_KERNEL) return fail(SWEPT_EUNSUPPORTED, "no fused per-step kernel for P=%d", P);
      if (rc != 0) return fail(SWEPT_ECUDA, "per-step launch: %s", cudaGetErrorString((cudaError_t)rc));
    } else {
      if (int rc = launch_per_step(s, s->slab[cur], s->slab[cur], s->slab[pred], 1, threads, P)) return rc;
      if (int rc = launch_per_step(s, s->slab[pred], s->slab[cur], s->slab[nxt], 0, threads, P)) return rc;
    }
    std::swap(cur, nxt);
  }
  *cur_io = cur;
  return 0;
}

int run_per_step(swept_state* s, int64_t steps, int threads) {
  if (steps <= 0) return 0;
  const int sigma = kShape[s->problem].sigma;
  const int P = per_step_P(s);
  const int lps = (s->problem == SWEPT_KS && P >= 2) ? 1 : sigma;  // launches per timestep (KS: fused stages)
  if (threads == 0) threads = 256;
  if (threads < 32 || threads > 1024 || (threads & (threads - 1)))
    return fail(SWEPT_EINVAL, "per-step tile_width (threads per block) must be a power of two in 32..1024");
  // replay chunks of CH steps from a captured graph (CH even so the buffer assignment is periodic)
  const int64_t CH = 256;
  int64_t left = steps;
  while (left >= CH) {
    GraphKey key{threads, P, s->cur, (int)CH};
    auto it = s->graphs.find(key);
    if (it == s->graphs.end()) {
      cudaGraph_t g = nullptr;
      if (!s->capture_stream) CUDA_TRY(cudaStreamCreateWithFlags(&s->capture_stream, cudaStreamNonBlocking));
      CUDA_TRY(cudaStreamBeginCapture(s->capture_stream, cudaStreamCaptureModeThreadLocal));
      int cur = s->cur;
      cudaStream_t user_stream = s->stream;
      s->stream = s->capture_stream;
      int rc = enqueue_steps(s, CH, threads, P, &cur);
      s->stream = user_stream;
      cudaError_t e = cudaStreamEndCapture(s->capture_stream, &g);
      if (rc) {
        if (g) cudaGraphDestroy(g);
        return rc;
      }
      if (e != cudaSuccess) return fail(SWEPT_ECUDA, "graph capture: %s", cudaGetErrorString(e));
      cudaGraphExec_t ge = nullptr;
      e = cudaGraphInstantiate(&ge, g, 0);
      cudaGraphDestroy(g);
      if (e != cudaSuccess) return fail(SWEPT_ECUDA, "graph instantiate: %s", cudaGetErrorString(e));
      it = s->graphs.emplace(key, ge).first;
    }
    CUDA_TRY(cudaGraphLaunch(it->second, s->stream));
    left -= CH;  // CH even: s->cur unchanged
    s->last_launches += CH * lps;
  }
  if (left > 0) {
    int cur = s->cur;
    if (int rc = enqueue_steps(s, left, threads, P, &cur)) return rc;
    s->cur = cur;
    s->last_launches += left * lps;
  }
  return 0;
}

// ---- resident per-step: every sub-timestep in one persistent launch (per_step_resident.cuh) -----------
int run_resident(swept_state* s, int64_t steps) {
  if (steps <= 0) return 0;
  if (!s->resident_scratch) return fail(SWEPT_EUNSUPPORTED, "no resident scratch (state creation failed to allocate it)");
  // flags restart from zero every launch; the error word behind them is sticky until swept_read looks at it
  CUDA_TRY(cudaMemsetAsync(s->resident_scratch, 0, (size_t)swept::RESIDENT_MAX_CTAS * 128, s->stream));
  if (s->problem == SWEPT_KS3)
    return fail(SWEPT_EUNSUPPORTED, "PS_RESIDENT is built for the paper's three problems, not for KS3");
  const int nxt = (s->cur + 1) & 3;
  swept::ResidentLaunch a{s->slab[s->cur], s->slab[nxt], s->N, steps, s->resident_scratch, s->consts, s->stream,
                          s->kernel_bc(), s->bcvals};
  int rc;
  switch (s->problem) {
    case SWEPT_HEAT: rc = swept::launch_resident_heat(s->dtype, a); break;
    case SWEPT_KS: rc = swept::launch_resident_ks(s->dtype, s->rk2, a); break;
    default: rc = swept::launch_resident_euler(s->dtype, s->rk2, a); break;
  }
  if (rc == NO_KERNEL)
    return fail(SWEPT_EUNSUPPORTED, "N=%lld does not fit a co-resident register-resident grid for this problem",
                (long long)s->N);
  if (rc != 0) return fail(SWEPT_ECUDA, "resident per-step launch: %s", cudaGetErrorString((cudaError_t)rc));
  s->cur = nxt;
  s->last_launches += 1;
  s->resident_pending_check = true;
  return 0;
}

// ---- swept phase plan -------------------------------------------------------------------------------
// One Up / D diamonds / Down cycle per admissible tile width, widest first (reading G5 of DESIGN.md §3): the
// sub-timesteps a cycle of width w cannot cover (fewer than m_w = w/(2h)) go to the next narrower width, and
// what is left below the narrowest one is finished with per-step launches.  Between cycles the state is a
// plain time level, so every cycle starts with an UpTriangle from row 0.
// A cycle must end on a full timestep: T = (D+1) m a multiple of sigma.  m is a power of two, so that is automatic
// for sigma = 1, 2 (m even) and means (D+1) % 3 == 0 for sigma = 3 (more than two sub-timesteps).
int64_t make_plan(int64_t nsub, const std::vector<int>& widths, int h, int sigma, std::vector<swept_phase>* out) {
  if (nsub < 0 || widths.empty() || nsub % sigma) return SWEPT_EINVAL;
  int64_t done = 0;
  for (int n : widths) {
    if (n < 4 * h || (n & (n - 1))) return SWEPT_EINVAL;
    const int64_t m = n / (2 * h);
    const int64_t left = nsub - done;
    int64_t q = left / m;  // rows of tiles after the Up row, Down included: D + 1
    if (sigma == 3) q -= q % 3;
    else if (m % sigma) return SWEPT_EINVAL;
    if (q < 1) continue;
    const int64_t D = q - 1;
    out->push_back({KIND_UP, 0, done, m - 1, n, 0});
    for (int64_t k = 1; k <= D; ++k) {
      const bool split = (k & 1) != 0;
      out->push_back({split ? KIND_SPLIT : KIND_WHOLE, split ? n / 2 : 0, done + (k - 1) * m, 2 * m - 1, n, 0});
    }
    out->push_back({KIND_DOWN, (D & 1) ? 0 : n / 2, done + D * m, m, n, 0});
    done += (D + 1) * m;
  }
  if (nsub > done) out->push_back({KIND_REMAINDER, 0, done, nsub - done, 0, 0});
  return (int64_t)out->size();
}

constexpr int MIN_LEVEL_WIDTH = 32;  // narrowest tile of the remainder cycles

int tier_default_P(const swept_state* s, int n) {
  // Euler's TIER tiers spread their pressure / flux work over all threads of the CTA: one thread per point
  // (measured: 256 threads per tile are best, more only add barrier cost)
  if (s->problem == SWEPT_EULER) return n <= 256 ? 1 : (n <= 2048 ? 2 : 4);
  if (s->problem == SWEPT_KS3) return n <= 1024 ? 1 : (n <= 2048 ? 2 : 4);
  const int pmax = 4, tmax = 1024;
  int P = std::min(pmax, std::max(1, n / 256));
  while (P < pmax && n / P > tmax) P *= 2;
  if (P == 3) P = 2;
  return P;
}

void default_tile(const swept_state* s, int* n_io, int* flavor_io, int* P_io) {
  int n = *n_io, flavor = *flavor_io, P = *P_io;
  if (n == 0 && s->tuned_width[SWEPT_SWEPT]) {
    n = s->tuned_width[SWEPT_SWEPT];
    if (flavor == SWEPT_FLAVOR_AUTO) {
      flavor = s->tuned_flavor;
      P = s->tuned_P;
    }
  }
  // untuned defaults (measured on B200): heat and KS run fastest with the register-resident
  // CHAR flavour on wide tiles, Euler (about 250 live registers per point) with the TIER flavour
  // fully default call (no width, no flavour, nothing tuned) on a large periodic heat / KS problem: the persistent
  // FLOW launch at the width measured best on B200 (N >= 2^19)
  // (the heat problem also with the paper's insulated ends: the wall tiles run inside the persistent launch, §5.8; n = 256
  // keeps them in registers and wins up to N = 2^20, profiles/r2_sweep_bc_heat.csv)
  const bool flow_default = (s->problem == SWEPT_HEAT || s->problem == SWEPT_KS) && (!s->bc || s->problem == SWEPT_HEAT);
  if (n == 0 && flavor == SWEPT_FLAVOR_AUTO && flow_default && s->N >= (1 << 19)) {
    const int cand = s->problem == SWEPT_HEAT ? ((s->bc && s->N < (1 << 21)) ? 256 : 512) : 1024;
    if (tile_ok(s, SWEPT_FLAVOR_FLOW, cand, 0)) {
      *n_io = cand;
      *flavor_io = SWEPT_FLAVOR_FLOW;
      *P_io = 0;
      return;
    }
  }
  // ... on a medium one (2^15 <= N < 2^19, a multiple of 256) the same flavour at n = 256: with TMA staging the persistent
  // launch beats a launch per row of tiles from N = 2^14 up (profiles/r2_sweep_heat_f64.csv, r2_sweep_ks.csv)
  if (n == 0 && flavor == SWEPT_FLAVOR_AUTO && flow_default &&
      s->N >= (1 << 15) && s->N < (1 << 19) && tile_ok(s, SWEPT_FLAVOR_FLOW, 256, 0)) {
    *n_io = 256;
    *flavor_io = SWEPT_FLAVOR_FLOW;
    *P_io = 0;
    return;
  }
  // ... and on a small one (N <= 2^14: at most 256 warp-sized tiles), where every flavour is bound by the latency of
  // the dependent tiers, the CLUSTER flavour: one launch per cycle, a warp per tile in registers, the rows chained by
  // stores into the next tile's shared memory.  Widths as measured (profiles/r2_sweep_*.csv): one warp per scheduler
  // as long as the tiles fit a cluster that way.
  const bool small_two_row = (s->problem == SWEPT_HEAT || s->problem == SWEPT_KS) && s->N <= 16384;
  const bool small_three_row = s->problem == SWEPT_KS3 && s->N <= 16384;  // measured: 1.5-2.2 x the TIER flavour there
  if (n == 0 && flavor == SWEPT_FLAVOR_AUTO && (!s->bc || s->problem == SWEPT_HEAT) && (small_two_row || small_three_row)) {
    const int first = s->problem == SWEPT_HEAT  ? (s->N <= 8192 ? 64 : 256)
                      : s->problem == SWEPT_KS ? (s->N <= 8192 ? 64 : 256)
                                               : (s->N <= 4096 ? 64 : (s->N <= 8192 ? 128 : 256));
    for (int cand : {first, 128, 256, 64})
      if (tile_ok(s, SWEPT_FLAVOR_CLUSTER, cand, 0)) {
        *n_io = cand;
        *flavor_io = SWEPT_FLAVOR_CLUSTER;
        *P_io = 0;
        return;
      }
  }
  if (flavor == SWEPT_FLAVOR_CLUSTER) {  // explicit flavour, library's width
    if (n == 0)
      for (int cand : {128, 64, 256, 512})
        if (n == 0 && tile_ok(s, SWEPT_FLAVOR_CLUSTER, cand, P)) n = cand;
    *n_io = n;
    *flavor_io = flavor;
    *P_io = P;
    return;
  }
  const bool want_char = flavor == SWEPT_FLAVOR_CHAR ||
                         (flavor == SWEPT_FLAVOR_AUTO && (s->problem == SWEPT_HEAT || s->problem == SWEPT_KS) && !s->bc);
  if (n == 0) {
    if (want_char) {
      for (int cand : {1024, 512, 256, 128, 64})
        for (int L : {32, 16, 8})
          if (n == 0 && (P == 0 || P == L) && tile_ok(s, SWEPT_FLAVOR_CHAR, cand, L)) n = cand;
    }
    if (n == 0 && flavor == SWEPT_FLAVOR_FLOW)
      for (int cand : {512, 1024, 256})
        if (n == 0 && tile_ok(s, SWEPT_FLAVOR_FLOW, cand, 0)) n = cand;
    if (n == 0 && flavor != SWEPT_FLAVOR_CHAR)
      for (int cand : {512, 256, 128, 1024, 64, 32, 2048, 4096})
        if (n == 0 && s->N % cand == 0) n = cand;
  }
  if (flavor == SWEPT_FLAVOR_AUTO) {
    flavor = SWEPT_FLAVOR_TIER;
    P = 0;
    if (want_char)
      for (int L : {32, 16, 8})
        if (flavor == SWEPT_FLAVOR_TIER && tile_ok(s, SWEPT_FLAVOR_CHAR, n, L)) {
          flavor = SWEPT_FLAVOR_CHAR;
          P = L;
        }
  }
  if (P == 0) {
    if (flavor == SWEPT_FLAVOR_TIER) P = tier_default_P(s, n);
    else if (flavor == SWEPT_FLAVOR_CHAR)
      for (int L : {32, 16, 8})
        if (P == 0 && tile_ok(s, SWEPT_FLAVOR_CHAR, n, L)) P = L;
  }
  *n_io = n;
  *flavor_io = flavor;
  *P_io = P;
}

// kernel configuration of a remainder cycle of width n, as close as possible to the top-level (flavor, P)
bool level_config(const swept_state* s, int n_top, int flavor_top, int P_top, int n, int* flavor, int* P) {
  if (n == n_top) {
    *flavor = flavor_top;
    *P = P_top;
    return tile_ok(s, flavor_top, n, P_top);
  }
  if (flavor_top == SWEPT_FLAVOR_CLUSTER) {
    if (tile_ok(s, SWEPT_FLAVOR_CLUSTER, n, 0)) {
      *flavor = SWEPT_FLAVOR_CLUSTER;
      *P = 0;
      return true;
    }
    for (int L : {32, 16, 8})
      if (tile_ok(s, SWEPT_FLAVOR_CHAR, n, L)) {
        *flavor = SWEPT_FLAVOR_CHAR;
        *P = L;
        return true;
      }
  }
  if (flavor_top == SWEPT_FLAVOR_FLOW) {
    if (tile_ok(s, SWEPT_FLAVOR_FLOW, n, P_top)) {
      *flavor = SWEPT_FLAVOR_FLOW;
      *P = P_top;
      return true;
    }
    for (int L : {32, 16, 8})
      if (tile_ok(s, SWEPT_FLAVOR_CHAR, n, L)) {
        *flavor = SWEPT_FLAVOR_CHAR;
        *P = L;
        return true;
      }
  }
  if (flavor_top == SWEPT_FLAVOR_CHAR) {
    const int B_top = n_top / P_top;
    for (int B : {B_top, 16, 8, 32, 4}) {
      if (n % B) continue;
      if (tile_ok(s, SWEPT_FLAVOR_CHAR, n, n / B)) {
        *flavor = SWEPT_FLAVOR_CHAR;
        *P = n / B;
        return true;
      }
    }
  }
  for (int Pt : {tier_default_P(s, n), 1, 2, 4}) {
    if (tile_ok(s, SWEPT_FLAVOR_TIER, n, Pt)) {
      *flavor = SWEPT_FLAVOR_TIER;
      *P = Pt;
      return true;
    }
  }
  return false;
}

// Plan a swept run: the cycles (tile widths) and their kernel configurations, then the phase list.
int plan_swept(swept_state* s, int64_t nsteps, int n, int flavor, int P) {
  const ProblemShape sh = kShape[s->problem];
  default_tile(s, &n, &flavor, &P);
  if (n <= 0) return fail(SWEPT_EUNSUPPORTED, "N=%lld has no admissible tile width", (long long)s->N);
  if (!tile_ok(s, flavor, n, P))
    return fail(s->N % n ? SWEPT_EINVAL : SWEPT_EUNSUPPORTED,
                "tile_width=%d (flavor %d, P=%d) not admissible for N=%lld", n, flavor, P, (long long)s->N);
  // widths of the cycles: n, then every narrower power of two that has a kernel for this N
  std::vector<int> widths;
  swept_state::Planned& pr = s->pr;
  pr.cfg.clear();
  pr.plan.clear();
  for (int w = n; w >= MIN_LEVEL_WIDTH && w >= 8 * sh.h; w /= 2) {
    int fl = 0, Pl = 0;
    if (!level_config(s, n, flavor, P, w, &fl, &Pl)) continue;
    widths.push_back(w);
    pr.cfg[w] = {fl, Pl};
  }
  const int64_t np = make_plan(nsteps * sh.sigma, widths, sh.h, sh.sigma, &pr.plan);
  if (np < 0) return fail(SWEPT_EINVAL, "cannot plan tile_width=%d", n);
  pr.rin[0] = pr.rin[1] = pr.rin[2] = -1;
  pr.nrows_valid = 0;
  pr.next = 0;
  pr.nsteps = nsteps;
  return 0;
}

// Launch phase pr.next of the planned run (a FLOW cycle counts as one: it consumes its Up .. Down entries).
int run_next_phase(swept_state* s) {
  const ProblemShape sh = kShape[s->problem];
  swept_state::Planned& pr = s->pr;
  if (pr.next >= pr.plan.size()) return fail(SWEPT_EINVAL, "no phase left in the planned run");
  const size_t ip = pr.next;
  const swept_phase& ph = pr.plan[ip];
  const int ns = s->nslabs, R = s->rows();
  if (ph.kind == KIND_UP && pr.cfg[ph.n].first == SWEPT_FLAVOR_CLUSTER) {
    // the whole cycle Up .. Down of this width in one launch of one thread-block cluster (swept_cluster.cuh)
    size_t jp = ip;
    while (pr.plan[jp].kind != KIND_DOWN) ++jp;
    swept::ClusterLaunch c{};
    c.init = s->slab[s->cur];
    const int o = (s->cur + 1) % ns;
    c.out = s->slab[o];
    c.N = s->N;
    c.n = ph.n;
    c.rows = (int)(jp - ip + 1);
    c.warps_per_cta = pr.cfg[ph.n].second;
    c.bc = s->kernel_bc();
    c.consts = s->consts;
    c.stream = s->stream;
    int rc;
    {
      TimedScope ts(s, KIND_FLOW, 1);
      rc = s->problem == SWEPT_HEAT ? swept::launch_cluster_heat(s->dtype, c)
           : s->problem == SWEPT_KS ? swept::launch_cluster_ks(s->dtype, s->rk2, c)
                                    : swept::launch_cluster_ks3(s->dtype, c);
    }
    if (rc == NO_KERNEL) return fail(SWEPT_EUNSUPPORTED, "no CLUSTER kernel for N=%lld n=%d", (long long)s->N, ph.n);
    if (rc != 0) return fail(SWEPT_ECUDA, "cluster launch: %s", cudaGetErrorString((cudaError_t)rc));
    s->last_launches += 1;
    s->cur = o;
    pr.rin[0] = o;
    pr.nrows_valid = 1;
    pr.next = jp + 1;
    return 0;
  }
  if (ph.kind == KIND_UP && pr.cfg[ph.n].first == SWEPT_FLAVOR_FLOW) {
    // the whole cycle Up .. Down of this width in one persistent launch
    size_t jp = ip;
    while (pr.plan[jp].kind != KIND_DOWN) ++jp;
    swept::FlowLaunch f{};
    f.n = ph.n;
    f.rows = (int)(jp - ip + 1);
    f.ctas_per_sm = pr.cfg[ph.n].second;
    f.init = s->slab[s->cur];
    // buffer 0 = the two slabs after cur, buffer 1 = the third one and cur itself (swept_flow.cuh: hazards)
    const int a0 = (s->cur + 1) & 3, a1 = (s->cur + 2) & 3, b0 = (s->cur + 3) & 3, b1 = s->cur;
    f.buf[0][0] = s->slab[a0]; f.buf[0][1] = s->slab[a1];
    f.buf[1][0] = s->slab[b0]; f.buf[1][1] = s->slab[b1];
    {
      TimedScope ts(s, KIND_FLOW, 1);
      if (int rc = launch_flow(s, f)) return rc;
    }
    s->last_launches += 1;
    s->cur = ((f.rows - 1) & 1) ? b0 : a0;  // the Down row wrote row 0 of its buffer
    pr.rin[0] = s->cur;
    pr.nrows_valid = 1;
    pr.next = jp + 1;
    return 0;
  }
  pr.next = ip + 1;
  if (ph.kind == KIND_REMAINDER) {
    TimedScope ts(s, KIND_REMAINDER, ph.ntiers);
    if (int rc = run_per_step(s, ph.ntiers / sh.sigma, 0)) return rc;
    pr.rin[0] = s->cur;
    pr.nrows_valid = 1;
    return 0;
  }
  swept::TileLaunch a{};
  a.kind = ph.kind;
  a.n = ph.n;
  a.shift = ph.shift;
  a.ntiers = (int)ph.ntiers;
  a.flavor = pr.cfg[ph.n].first;
  a.P = pr.cfg[ph.n].second;
  int o[3] = {-1, -1, -1};
  if (ph.kind == KIND_UP) {
    for (int r = 0; r < R; ++r) o[r] = (s->cur + 1 + r) % ns;
    a.in0 = s->slab[s->cur];
    a.in1 = nullptr;
  } else {
    // the slabs that are not the input rows
    int k = 0;
    for (int i = 0; i < ns && k < R; ++i)
      if (i != pr.rin[0] && i != pr.rin[1] && i != pr.rin[2]) o[k++] = i;
    a.in0 = s->slab[pr.rin[0]];
    a.in1 = s->slab[pr.rin[1]];
    if (R == 3) a.in2 = s->slab[pr.rin[2]];
  }
  a.out0 = s->slab[o[0]];
  a.out1 = s->slab[o[1]];
  if (R == 3) {
    a.out2 = s->slab[o[2]];
    a.tmod = (int)(ph.tier0 % 3);  // which stage the phase's first tier is
  }
  const bool hybrid = s->bc && a.flavor == SWEPT_FLAVOR_CHAR && ph.kind != KIND_UP;  // Up reads no halo
  if (hybrid) {
    // The tiles that touch a wall (aligned rows: the first and the last tile; shifted rows: the tile split across
    // the boundary) go to the TIER kernels, which apply the boundary condition, on a second
    // stream beside the register-resident launch — the paper's Hybrid idea with a stream in
    // place of the CPU.  Both read the same input rows and write disjoint ranges of the output rows.
    if (!s->wall_stream) return fail(SWEPT_ECUDA, "no wall stream (swept_create makes it for SWEPT_BC_PAPER heat)");
    CUDA_TRY(cudaEventRecord(s->wall_fork, s->stream));
    CUDA_TRY(cudaStreamWaitEvent(s->wall_stream, s->wall_fork, 0));
    a.skip_first = ph.shift == 0 ? 1 : 0;
    a.skip_last = 1;
    // wall tiles first, so that they are resident before the big launch takes every slot
    const int K = (int)(s->N / ph.n);
    swept::TileLaunch w = a;
    w.flavor = SWEPT_FLAVOR_TIER;
    w.P = 1;  // one thread per point: the shortest tier latency (measured), and the wall tile is a latency chain
    w.skip_first = w.skip_last = 0;
    if (ph.shift == 0) { w.tile_base = 0; w.tile_step = K - 1; w.tile_count = K > 1 ? 2 : 1; }
    else { w.tile_base = K - 1; w.tile_step = 0; w.tile_count = 1; }
    if (int rc = launch_tile(s, w, s->wall_stream)) return rc;
    s->last_launches += 1;
    CUDA_TRY(cudaEventRecord(s->wall_join, s->wall_stream));
  }
  {
    TimedScope ts(s, ph.kind, 1);
    if (int rc = launch_tile(s, a)) return rc;
  }
  s->last_launches += 1;
  if (hybrid) CUDA_TRY(cudaStreamWaitEvent(s->stream, s->wall_join, 0));
  for (int r = 0; r < 3; ++r) pr.rin[r] = o[r];
  pr.nrows_valid = R;
  if (ph.kind == KIND_DOWN) {
    s->cur = o[0];  // row 0 holds the full time level (T is a multiple of sigma)
    pr.nrows_valid = 1;
  }
  return 0;
}

int run_swept(swept_state* s, int64_t nsteps, int n, int flavor, int P) {
  if (int rc = plan_swept(s, nsteps, n, flavor, P)) return rc;
  while (s->pr.next < s->pr.plan.size())
    if (int rc = run_next_phase(s)) return rc;
  return 0;
}

}  // namespace

// =======================================================================================================
extern "C" {

const char* swept_last_error(void) { return g_err.c_str(); }

swept_state* swept_create(int problem, int64_t N, double dx, double dt, const swept_params* p) {
  if (problem < 0 || problem > 3) { fail(SWEPT_EINVAL, "unknown problem %d", problem); return nullptr; }
  if (N < 8 || N > (int64_t)1 << 31) { fail(SWEPT_EINVAL, "N out of range"); return nullptr; }
  if (!(dx > 0) || !(dt > 0)) { fail(SWEPT_EINVAL, "dx and dt must be positive"); return nullptr; }
  swept_params q;
  std::memset(&q, 0, sizeof q);
  q.struct_size = sizeof q;
  q.dtype = SWEPT_F64;
  q.device = -1;
  q.alpha = 1.0;
  q.gamma = 1.4;
  if (p) {
    if (p->struct_size < 4 || p->struct_size > sizeof q) { fail(SWEPT_EINVAL, "bad params.struct_size"); return nullptr; }
    std::memcpy(&q, p, p->struct_size);
  }
  if (q.dtype != SWEPT_F64 && q.dtype != SWEPT_F32) { fail(SWEPT_EINVAL, "bad dtype"); return nullptr; }
  if (q.rk2 != SWEPT_RK2_MIDPOINT && q.rk2 != SWEPT_RK2_HEUN) { fail(SWEPT_EINVAL, "bad rk2"); return nullptr; }
  if (problem == SWEPT_KS3) q.rk2 = 0;  // its integrator is fixed (SSP-RK3)
  if (q.dtype == SWEPT_F32 && problem != SWEPT_HEAT) {
    fail(SWEPT_EUNSUPPORTED, "FP32 is provided for the heat problem only (BASELINE.json config 2)");
    return nullptr;
  }
  if (q.bc != SWEPT_BC_PERIODIC && q.bc != SWEPT_BC_PAPER) { fail(SWEPT_EINVAL, "bad bc"); return nullptr; }
  if (q.bc == SWEPT_BC_PAPER && (problem == SWEPT_KS || problem == SWEPT_KS3)) {
    fail(SWEPT_EUNSUPPORTED, "SWEPT_BC_PAPER: the paper's KS runs are periodic (PAPER.md:356); heat and Euler only");
    return nullptr;
  }
  if ((q.alloc == nullptr) != (q.free == nullptr)) { fail(SWEPT_EINVAL, "alloc and free must be given together"); return nullptr; }
  int dev = q.device;
  if (dev < 0) {
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { fail(SWEPT_ECUDA, "cudaGetDevice: %s (no CPU fallback exists)", cudaGetErrorString(e)); return nullptr; }
  }
  {
    cudaError_t e = cudaSetDevice(dev);
    if (e != cudaSuccess) { fail(SWEPT_ECUDA, "cudaSetDevice(%d): %s (no CPU fallback exists)", dev, cudaGetErrorString(e)); return nullptr; }
  }
  swept_state* s = new swept_state();
  s->problem = problem; s->dtype = q.dtype; s->rk2 = q.rk2; s->device = dev; s->bc = q.bc;
  s->N = N; s->dx = dx; s->dt = dt; s->alpha = q.alpha; s->gamma = q.gamma;
  s->stream = (cudaStream_t)q.stream;
  s->alloc = q.alloc; s->free_ = q.free; s->alloc_ctx = q.alloc_ctx;
  // scheme constants: double on the host, rounded once to REAL at launch
  if (problem == SWEPT_HEAT) {
    const double Fo = q.alpha * dt / (dx * dx);
    s->consts[0] = Fo;
    s->consts[1] = 1.0 - 2.0 * Fo;
  } else if (problem == SWEPT_KS || problem == SWEPT_KS3) {
    s->consts[0] = 1.0 / (4.0 * dx);
    s->consts[1] = 1.0 / (dx * dx);
    s->consts[2] = 1.0 / ((dx * dx) * (dx * dx));
    s->consts[3] = dt;
    s->consts[4] = 0.5 * dt;
  } else {
    const double lam = dt / dx;
    s->consts[0] = q.gamma - 1.0;
    s->consts[1] = q.gamma * (q.gamma - 1.0);
    s->consts[2] = lam;
    s->consts[3] = 0.5 * lam;
  }
  {
    std::lock_guard<std::mutex> lock(g_tuned_mutex);
    auto it = g_tuned.find(TunedKey{dev, problem, q.dtype, q.rk2, q.bc, N});
    if (it != g_tuned.end()) {
      s->tuned_width[0] = it->second.width[0];
      s->tuned_width[1] = it->second.width[1];
      s->tuned_flavor = it->second.flavor;
      s->tuned_P = it->second.P;
    }
  }
  s->slab_bytes = (size_t)kShape[problem].C * (size_t)N * s->elem();
  s->nslabs = problem == SWEPT_KS3 ? 6 : 4;
  for (int i = 0; i < s->nslabs; ++i) {
    void* ptr = dev_alloc(s, s->slab_bytes);
    if (!ptr) {
      fail(SWEPT_ENOMEM, "device allocation of %zu bytes failed", s->slab_bytes);
      swept_destroy(s);
      return nullptr;
    }
    s->slab[i] = ptr;
    if (((uintptr_t)ptr & 15) != 0) {
      fail(SWEPT_EINVAL, "allocator returned a pointer that is not 16-byte aligned");
      swept_destroy(s);
      return nullptr;
    }
    // debugging aid (include/swept.h): every field slab starts as NaNs, so that a kernel reading a value nobody
    // wrote produces a wrong result instead of a plausible one
    if (std::getenv("SWEPT_POISON")) cudaMemsetAsync(ptr, 0xFF, s->slab_bytes, s->stream);
  }
  // Scratch of the persistent flavours, sized here for the worst admissible plan so that swept_run never
  // allocates or synchronises: FLOW (periodic heat / KS, N a multiple of its narrowest tile) needs a ticket word,
  // a leave counter, an error word and 2 N/256 flags; PS_RESIDENT one flag line and two exchange lines per CTA.
  cudaError_t e = cudaSuccess;
  if (((problem == SWEPT_HEAT || problem == SWEPT_KS) && q.bc == SWEPT_BC_PERIODIC || (problem == SWEPT_HEAT && q.bc)) &&
      N % FLOW_MIN_WIDTH == 0) {
    s->flow_scratch_ints = 4 + 2 * (size_t)(N / FLOW_MIN_WIDTH);
    s->flow_scratch = (int*)dev_alloc(s, s->flow_scratch_ints * sizeof(int));
    if (s->flow_scratch) e = cudaMemsetAsync(s->flow_scratch, 0, s->flow_scratch_ints * sizeof(int), s->stream);
    s->flow_prof = (unsigned long long*)dev_alloc(s, 8 * sizeof(unsigned long long));
    if (s->flow_prof && e == cudaSuccess) e = cudaMemsetAsync(s->flow_prof, 0, 8 * sizeof(unsigned long long), s->stream);
  }
  s->resident_scratch = dev_alloc(s, swept::resident_scratch_bytes(swept::RESIDENT_MAX_CTAS));
  if (s->resident_scratch && e == cudaSuccess)
    e = cudaMemsetAsync(s->resident_scratch, 0, swept::resident_flag_bytes(swept::RESIDENT_MAX_CTAS), s->stream);
  if (e == cudaSuccess && q.bc == SWEPT_BC_PAPER && problem == SWEPT_HEAT) {
    // hybrid wall handling: the wall tiles run on a second, highest-priority stream — the wall
    // tile is one long latency chain and must not wait for a slot behind the register-resident launch
    int lo_prio = 0, hi_prio = 0;
    e = cudaDeviceGetStreamPriorityRange(&lo_prio, &hi_prio);
    if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&s->wall_stream, cudaStreamNonBlocking, hi_prio);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->wall_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->wall_join, cudaEventDisableTiming);
  }
  // the clears above must not race with a later swept_set_stream: finish them here (creation may synchronise)
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e != cudaSuccess || !s->resident_scratch || (s->flow_scratch_ints && !s->flow_scratch)) {
    if (e != cudaSuccess) fail(SWEPT_ECUDA, "swept_create: %s", cudaGetErrorString(e));
    else fail(SWEPT_ENOMEM, "device allocation of the scratch buffers failed");
    swept_destroy(s);
    return nullptr;
  }
  return s;
}

void swept_destroy(swept_state* s) {
  if (!s) return;
  cudaSetDevice(s->device);
  cudaStreamSynchronize(s->stream);
  for (auto& kv : s->graphs) cudaGraphExecDestroy(kv.second);
  if (s->capture_stream) cudaStreamDestroy(s->capture_stream);
  for (auto& t : s->timed) { cudaEventDestroy(t.e0); cudaEventDestroy(t.e1); }
  for (cudaEvent_t e : s->event_pool) cudaEventDestroy(e);
  dev_free(s, s->flow_scratch);
  dev_free(s, s->flow_prof);
  dev_free(s, s->resident_scratch);
  dev_free(s, s->shard_send);
  dev_free(s, s->shard_recv);
  if (s->shard_packed) cudaEventDestroy(s->shard_packed);
  if (s->shard_send_free) cudaEventDestroy(s->shard_send_free);
  if (s->wall_stream) {
    cudaStreamSynchronize(s->wall_stream);
    cudaStreamDestroy(s->wall_stream);
  }
  if (s->wall_fork) cudaEventDestroy(s->wall_fork);
  if (s->wall_join) cudaEventDestroy(s->wall_join);
  for (int i = 0; i < MAX_SLABS; ++i) dev_free(s, s->slab[i]);
  delete s;
}

int swept_set_stream(swept_state* s, void* stream) {
  if (!s) return fail(SWEPT_EINVAL, "null state");
  s->stream = (cudaStream_t)stream;
  return 0;
}

int swept_set_phase_timing(swept_state* s, int on) {
  if (!s) return fail(SWEPT_EINVAL, "null state");
  s->timing = on != 0;
  return 0;
}

int swept_phase_times(swept_state* s, double* ms, int64_t* launches) {
  if (!s || !ms || !launches) return fail(SWEPT_EINVAL, "null argument");
  if (int rc = set_device(s)) return rc;
  CUDA_TRY(cudaStreamSynchronize(s->stream));
  for (int k = 0; k < SWEPT_NKINDS; ++k) { ms[k] = 0; launches[k] = 0; }
  for (auto& t : s->timed) {
    float f = 0;
    if (cudaEventElapsedTime(&f, t.e0, t.e1) == cudaSuccess && t.kind >= 0 && t.kind < SWEPT_NKINDS) {
      ms[t.kind] += f;
      launches[t.kind] += t.launches;
    }
    s->event_pool.push_back(t.e0);
    s->event_pool.push_back(t.e1);
  }
  s->timed.clear();
  cudaGetLastError();
  return check_flow_error(s);
}

int swept_flow_profile(swept_state* s, int on, uint64_t* counters) {
  if (!s) return fail(SWEPT_EINVAL, "null state");
  if (!s->flow_prof) return fail(SWEPT_EUNSUPPORTED, "this state has no FLOW flavour");
  if (int rc = set_device(s)) return rc;
  CUDA_TRY(cudaStreamSynchronize(s->stream));
  if (counters) CUDA_TRY(cudaMemcpy(counters, s->flow_prof, 8 * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  CUDA_TRY(cudaMemset(s->flow_prof, 0, 8 * sizeof(uint64_t)));
  s->flow_prof_on = on != 0;
  return check_flow_error(s);
}

int swept_sync(swept_state* s) {
  if (!s) return fail(SWEPT_EINVAL, "null state");
  if (int rc = set_device(s)) return rc;
  CUDA_TRY(cudaStreamSynchronize(s->stream));
  return check_flow_error(s);
}

// The field between a slab and a caller's buffer.  A shard's slab has N = n_local + ghost points per component, the
// caller's buffer only the n_local own points (include/swept.h): a strided copy.
static int copy_field(swept_state* s, void* dst, const void* src, bool to_slab, cudaMemcpyKind kind) {
  if (!s->is_shard()) {
    CUDA_TRY(cudaMemcpyAsync(dst, src, s->slab_bytes, kind, s->stream));
    return 0;
  }
  const size_t own = (size_t)s->shard_nloc * s->elem(), ext = (size_t)s->N * s->elem();
  CUDA_TRY(cudaMemcpy2DAsync(dst, to_slab ? ext : own, src, to_slab ? own : ext, own, (size_t)kShape[s->problem].C, kind,
                             s->stream));
  return 0;
}

// Dirichlet end states of the Euler tube = the initial states of the first and last cell.  The
// captured per-step graphs hold them as kernel arguments: new values invalidate the cache.
static int set_end_states(swept_state* s, const double (&v)[6]) {
  if (std::memcmp(s->bcvals, v, sizeof v) == 0) return 0;
  std::memcpy(s->bcvals, v, sizeof v);
  if (!s->graphs.empty()) {
    CUDA_TRY(cudaStreamSynchronize(s->stream));  // a replay may still be in flight
    for (auto& kv : s->graphs) cudaGraphExecDestroy(kv.second);
    s->graphs.clear();
  }
  return 0;
}

int swept_write(swept_state* s, const void* host_buf) {
  if (!s || !host_buf) return fail(SWEPT_EINVAL, "null argument");
  if (int rc = set_device(s)) return rc;
  if (s->bc && s->problem == SWEPT_EULER) {
    double v[6];
    for (int c = 0; c < 3; ++c) {
      v[c] = ((const double*)host_buf)[(size_t)c * s->N];
      v[3 + c] = ((const double*)host_buf)[(size_t)c * s->N + s->N - 1];
    }
    if (int rc = set_end_states(s, v)) return rc;
  }
  if (int rc = copy_field(s, s->slab[s->cur], host_buf, true, cudaMemcpyHostToDevice)) return rc;
  s->steps_done = 0;
  return 0;
}

int swept_write_device(swept_state* s, const void* device_buf) {
  if (!s || !device_buf) return fail(SWEPT_EINVAL, "null argument");
  if (int rc = set_device(s)) return rc;
  if (s->bc && s->problem == SWEPT_EULER) {
    // end states: six scalars read back on the state's stream (ordered after whatever produced device_buf there)
    double v[6];
    for (int c = 0; c < 3; ++c) {
      const double* d = (const double*)device_buf + (size_t)c * s->N;
      CUDA_TRY(cudaMemcpyAsync(&v[c], d, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
      CUDA_TRY(cudaMemcpyAsync(&v[3 + c], d + s->N - 1, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    }
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    if (int rc = set_end_states(s, v)) return rc;
  }
  if (int rc = copy_field(s, s->slab[s->cur], device_buf, true, cudaMemcpyDeviceToDevice)) return rc;
  s->steps_done = 0;
  return 0;
}

int swept_read(swept_state* s, void* host_buf) {
  if (!s || !host_buf) return fail(SWEPT_EINVAL, "null argument");
  if (int rc = set_device(s)) return rc;
  if (int rc = copy_field(s, host_buf, s->slab[s->cur], false, cudaMemcpyDeviceToHost)) return rc;
  CUDA_TRY(cudaStreamSynchronize(s->stream));
  return check_flow_error(s);
}

const void* swept_device_ptr(swept_state* s) { return s ? s->slab[s->cur] : nullptr; }
int64_t swept_steps_done(const swept_state* s) { return s ? s->steps_done : -1; }
int64_t swept_last_launches(const swept_state* s) { return s ? s->last_launches : -1; }

int swept_run_flavor(swept_state* s, int64_t nsteps, int32_t tile_width, int variant, int flavor) {
  if (!s) return fail(SWEPT_EINVAL, "null state");
  if (nsteps < 0) return fail(SWEPT_EINVAL, "nsteps must be >= 0");
  if (tile_width < 0) return fail(SWEPT_EINVAL, "tile_width must be >= 0");
  if (s->is_shard())
    return fail(SWEPT_EINVAL, "a shard cannot advance alone: use swept_shard_run or the swept_shard_* phase calls");
  if (int rc = set_device(s)) return rc;
  s->last_launches = 0;
  int rc;
  if (variant == SWEPT_PER_STEP) {
    if ((flavor & 0xff) == SWEPT_PS_RESIDENT) {
      rc = run_resident(s, nsteps);
    } else if ((flavor & 0xff) != SWEPT_PS_LAUNCH) {
      return fail(SWEPT_EINVAL, "unknown per-step flavor %d", flavor & 0xff);
    } else {
      int tw = tile_width ? tile_width : s->tuned_width[SWEPT_PER_STEP];
      rc = run_per_step(s, nsteps, tw);
    }
  } else if (variant == SWEPT_SWEPT) {
    int fl = flavor & 0xff, P = (flavor >> 8) & 0xff;  // bits 8..15: explicit P / lane-group size (0 = default)
    if (fl != SWEPT_FLAVOR_AUTO && fl != SWEPT_FLAVOR_TIER && fl != SWEPT_FLAVOR_CHAR && fl != SWEPT_FLAVOR_FLOW &&
        fl != SWEPT_FLAVOR_CLUSTER)
      return fail(SWEPT_EINVAL, "unknown flavor %d", fl);
    rc = run_swept(s, nsteps, tile_width, fl, P);
  } else {
    return fail(SWEPT_EINVAL, "unknown variant %d", variant);
  }
  if (rc == 0) s->steps_done += nsteps;
  return rc;
}

int swept_run(swept_state* s, int64_t nsteps, int32_t tile_width, int variant) {
  return swept_run_flavor(s, nsteps, tile_width, variant, SWEPT_FLAVOR_AUTO);
}

int64_t swept_plan(int64_t nsub, int32_t n, int32_t h, swept_phase* out, int64_t max_phases) {
  return swept_plan_sigma(nsub, n, h, 1, out, max_phases);
}

int64_t swept_plan_sigma(int64_t nsub, int32_t n, int32_t h, int32_t sigma, swept_phase* out, int64_t max_phases) {
  if (h != 1 && h != 2) return fail(SWEPT_EINVAL, "h must be 1 or 2");
  if (sigma < 1 || sigma > 3) return fail(SWEPT_EINVAL, "sigma must be 1, 2 or 3");
  if (nsub % sigma) return fail(SWEPT_EINVAL, "nsub must be a whole number of timesteps (a multiple of sigma)");
  if (n < 8 * h || (n & (n - 1))) return fail(SWEPT_EINVAL, "tile width %d not plannable for h=%d", n, h);
  std::vector<int> widths;
  for (int w = n; w == n || (w >= MIN_LEVEL_WIDTH && w >= 8 * h); w /= 2) widths.push_back(w);
  std::vector<swept_phase> plan;
  const int64_t np = make_plan(nsub, widths, h, sigma, &plan);
  if (np < 0) return fail(SWEPT_EINVAL, "tile width %d not plannable for h=%d", n, h);
  if (out)
    for (int64_t i = 0; i < np && i < max_phases; ++i) out[i] = plan[(size_t)i];
  return np;
}

// ---- sharding (include/swept.h: "sharding over several GPUs") ---------------------------------------------------
int64_t swept_shard_exchanges(const swept_phase* plan, int64_t nphases, int32_t h, int32_t sigma, int64_t n_local,
                              swept_exchange* out, int64_t max_out) {
  if (!plan || nphases < 0 || (h != 1 && h != 2) || sigma < 1 || sigma > 3 || n_local <= 0)
    return fail(SWEPT_EINVAL, "bad argument");
  const int R = sigma == 3 ? 3 : 2;
  int64_t cnt = 0;
  auto emit = [&](int after, int dir, int64_t src, int64_t dst, int count, int rows) {
    if (out && cnt < max_out) out[cnt] = swept_exchange{after, dir, src, dst, count, rows};
    ++cnt;
  };
  for (int64_t i = 0; i < nphases; ++i) {
    const swept_phase& ph = plan[i];
    if (ph.kind == KIND_REMAINDER) {
      // per-step stages: one exchange of ntiers * h points each way, then every shard steps on its own (the valid
      // part of the ghost zone shrinks by h per sub-timestep and never reaches the own points)
      const int g = (int)ph.ntiers * h;
      emit((int)i - 1, +1, n_local - g, -g, g, 1);
      emit((int)i - 1, -1, 0, n_local, g, 1);
    } else if (ph.kind == KIND_DOWN) {
      // shifted Down: the tile straddling the right end left the neighbour's first half tile at the final level
      if (ph.shift != 0) emit((int)i, +1, n_local, 0, ph.n / 2, 1);
    } else if (ph.shift == 0) {
      // aligned row done, a shifted row follows: its straddling tile needs the right neighbour's first half tile + halo
      emit((int)i, -1, 0, n_local, ph.n / 2 + h, R);
    } else {
      // shifted row done, an aligned row follows: hand the neighbour its first half tile back, with its left halo
      emit((int)i, +1, n_local - h, -h, ph.n / 2 + h, R);
    }
  }
  return cnt;
}

swept_state* swept_shard_create(int problem, int64_t N, int32_t nshards, int32_t shard, int32_t tile_width, double dx,
                                double dt, const swept_params* p) {
  if (nshards < 1 || shard < 0 || shard >= nshards) { fail(SWEPT_EINVAL, "bad shard index %d of %d", shard, nshards); return nullptr; }
  if (tile_width < 32 || (tile_width & (tile_width - 1)) || tile_width > 4096) {
    fail(SWEPT_EINVAL, "tile_width must be a power of two in 32..4096");
    return nullptr;
  }
  if (N <= 0 || N % ((int64_t)nshards * tile_width)) {
    fail(SWEPT_EINVAL, "N must be a multiple of nshards * tile_width");
    return nullptr;
  }
  if (p && p->struct_size >= offsetof(swept_params, bc) + sizeof(int32_t) && p->bc != SWEPT_BC_PERIODIC) {
    fail(SWEPT_EUNSUPPORTED, "shards are built for the periodic problems");
    return nullptr;
  }
  const int64_t nloc = N / nshards;
  swept_state* s = swept_create(problem, nloc + tile_width, dx, dt, p);
  if (!s) return nullptr;
  s->shard_nloc = nloc;
  s->shard_n = tile_width;
  s->nshards = nshards;
  s->shard_index = shard;
  const ProblemShape sh = kShape[problem];
  s->shard_buf_bytes = (size_t)s->rows() * sh.C * (size_t)(tile_width / 2 + sh.h) * s->elem();
  s->shard_send = dev_alloc(s, s->shard_buf_bytes);
  s->shard_recv = dev_alloc(s, s->shard_buf_bytes);
  cudaError_t e = cudaEventCreateWithFlags(&s->shard_packed, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->shard_send_free, cudaEventDisableTiming);
  if (!s->shard_send || !s->shard_recv || e != cudaSuccess) {
    fail(e != cudaSuccess ? SWEPT_ECUDA : SWEPT_ENOMEM, "swept_shard_create: staging buffers / events");
    swept_destroy(s);
    return nullptr;
  }
  return s;
}

int64_t swept_shard_begin(swept_state* s, int64_t nsteps, int flavor) {
  if (!s || !s->is_shard()) return fail(SWEPT_EINVAL, "not a shard state");
  if (nsteps < 0) return fail(SWEPT_EINVAL, "nsteps must be >= 0");
  if (int rc = set_device(s)) return rc;
  const int fl = flavor & 0xff, P = (flavor >> 8) & 0xff;
  if (fl != SWEPT_FLAVOR_AUTO && fl != SWEPT_FLAVOR_TIER && fl != SWEPT_FLAVOR_CHAR)
    return fail(SWEPT_EUNSUPPORTED, "shards run the phase-wise flavours (TIER, CHAR); flavor %d is not one", fl);
  s->last_launches = 0;
  if (int rc = plan_swept(s, nsteps, s->shard_n, fl, P)) return rc;
  const ProblemShape sh = kShape[s->problem];
  const int64_t nx = swept_shard_exchanges(s->pr.plan.data(), (int64_t)s->pr.plan.size(), sh.h, sh.sigma, s->shard_nloc,
                                           nullptr, 0);
  if (nx < 0) return nx;
  s->xch.resize((size_t)nx);
  swept_shard_exchanges(s->pr.plan.data(), (int64_t)s->pr.plan.size(), sh.h, sh.sigma, s->shard_nloc, s->xch.data(), nx);
  for (const swept_exchange& x : s->xch)
    // both halves of the per-step remainder's exchange (dst_off != 0, one row) land in the ghost zone
    if ((size_t)x.rows * sh.C * (size_t)x.count * s->elem() > s->shard_buf_bytes ||
        (x.rows == 1 && x.dst_off != 0 && 2 * x.count > s->shard_n))
      return fail(SWEPT_EINVAL, "exchange of %d points does not fit the ghost zone of %d", x.count, s->shard_n);
  return (int64_t)s->pr.plan.size();
}

int64_t swept_shard_exchange_list(swept_state* s, swept_exchange* out, int64_t max_out) {
  if (!s || !s->is_shard()) return fail(SWEPT_EINVAL, "not a shard state");
  for (int64_t i = 0; out && i < (int64_t)s->xch.size() && i < max_out; ++i) out[i] = s->xch[(size_t)i];
  return (int64_t)s->xch.size();
}

int64_t swept_shard_message_bytes(swept_state* s, int64_t x) {
  if (!s || !s->is_shard() || x < 0 || x >= (int64_t)s->xch.size()) return fail(SWEPT_EINVAL, "bad exchange index");
  const swept_exchange& e = s->xch[(size_t)x];
  return (int64_t)e.rows * kShape[s->problem].C * (int64_t)e.count * (int64_t)s->elem();
}

int swept_shard_phase(swept_state* s) {
  if (!s || !s->is_shard()) return fail(SWEPT_EINVAL, "not a shard state");
  if (int rc = set_device(s)) return rc;
  return run_next_phase(s);
}

static int shard_copy(swept_state* s, int64_t x, void* buf, bool pack) {
  if (!s || !s->is_shard() || !buf) return fail(SWEPT_EINVAL, "bad argument");
  if (x < 0 || x >= (int64_t)s->xch.size()) return fail(SWEPT_EINVAL, "bad exchange index");
  if (int rc = set_device(s)) return rc;
  const swept_exchange& e = s->xch[(size_t)x];
  swept::ShardCopy c{};
  if (e.rows == 1) {
    c.rows[0] = s->slab[s->cur];  // the full time level (after Down, and before the per-step remainder)
  } else {
    for (int r = 0; r < e.rows; ++r) {
      if (s->pr.rin[r] < 0) return fail(SWEPT_EINVAL, "exchange %lld before its phase has run", (long long)x);
      c.rows[r] = s->slab[s->pr.rin[r]];
    }
  }
  c.nrows = e.rows;
  c.C = kShape[s->problem].C;
  c.Next = s->N;
  c.off = pack ? e.src_off : e.dst_off;
  c.count = e.count;
  c.buf = buf;
  c.elem = (int)s->elem();
  c.stream = s->stream;
  c.pack = pack;
  const int rc = swept::launch_shard_copy(c);
  if (rc != 0) return fail(SWEPT_ECUDA, "shard %s: %s", pack ? "pack" : "unpack", cudaGetErrorString((cudaError_t)rc));
  s->last_launches += 1;
  return 0;
}

int swept_shard_pack(swept_state* s, int64_t x, void* device_buf) { return shard_copy(s, x, device_buf, true); }
int swept_shard_unpack(swept_state* s, int64_t x, const void* device_buf) {
  return shard_copy(s, x, const_cast<void*>(device_buf), false);
}

int swept_shard_end(swept_state* s) {
  if (!s || !s->is_shard()) return fail(SWEPT_EINVAL, "not a shard state");
  if (s->pr.next != s->pr.plan.size()) return fail(SWEPT_EINVAL, "the planned run has phases left");
  s->steps_done += s->pr.nsteps;
  return 0;
}

int swept_shard_run(swept_state* const* shards, int32_t nshards, int64_t nsteps, int flavor) {
  if (!shards || nshards < 1) return fail(SWEPT_EINVAL, "bad argument");
  int64_t np = -1;
  for (int i = 0; i < nshards; ++i) {
    swept_state* s = shards[i];
    if (!s || !s->is_shard() || s->nshards != nshards || s->shard_index != i)
      return fail(SWEPT_EINVAL, "shards[%d] is not shard %d of %d", i, i, nshards);
    const int64_t n = swept_shard_begin(s, nsteps, flavor);
    if (n < 0) return (int)n;
    if (np >= 0 && (n != np || s->xch.size() != shards[0]->xch.size()))
      return fail(SWEPT_EINVAL, "the shards planned different runs (different problems or sizes?)");
    np = n;
  }
  const std::vector<swept_exchange>& xch = shards[0]->xch;
  size_t ix = 0;
  for (int64_t i = -1; i < np; ++i) {
    if (i >= 0)
      for (int k = 0; k < nshards; ++k)
        if (int rc = swept_shard_phase(shards[k])) return rc;
    for (; ix < xch.size() && xch[ix].after_phase == (int)i; ++ix) {
      const int64_t bytes = swept_shard_message_bytes(shards[0], (int64_t)ix);
      // gather on every sender (after whoever still reads its staging buffer has finished) ...
      for (int k = 0; k < nshards; ++k) {
        swept_state* s = shards[k];
        if (int rc = set_device(s)) return rc;
        if (s->shard_send_busy) CUDA_TRY(cudaStreamWaitEvent(s->stream, s->shard_send_free, 0));
        if (int rc = swept_shard_pack(s, (int64_t)ix, s->shard_send)) return rc;
        CUDA_TRY(cudaEventRecord(s->shard_packed, s->stream));
      }
      // ... then ONE copy per message on the receiver's stream (peer-to-peer when the shards sit on two devices),
      // and the scatter into the receiver's rows
      for (int k = 0; k < nshards; ++k) {
        swept_state* s = shards[k];
        swept_state* d = shards[((k + xch[ix].dir) % nshards + nshards) % nshards];
        if (int rc = set_device(d)) return rc;
        CUDA_TRY(cudaStreamWaitEvent(d->stream, s->shard_packed, 0));
        CUDA_TRY(cudaMemcpyAsync(d->shard_recv, s->shard_send, (size_t)bytes, cudaMemcpyDefault, d->stream));
        CUDA_TRY(cudaEventRecord(s->shard_send_free, d->stream));
        s->shard_send_busy = true;
        if (int rc = swept_shard_unpack(d, (int64_t)ix, d->shard_recv)) return rc;
      }
    }
  }
  for (int k = 0; k < nshards; ++k)
    if (int rc = swept_shard_end(shards[k])) return rc;
  return 0;
}

int swept_tuned(const swept_state* s, int variant, int32_t* tile_width, int32_t* flavor, int32_t* group) {
  if (!s || (variant != SWEPT_PER_STEP && variant != SWEPT_SWEPT)) return fail(SWEPT_EINVAL, "bad argument");
  if (tile_width) *tile_width = s->tuned_width[variant];
  if (flavor) *flavor = variant == SWEPT_SWEPT ? s->tuned_flavor : 0;
  if (group) *group = variant == SWEPT_SWEPT ? s->tuned_P : 0;
  return 0;
}

int swept_autotune(swept_state* s, int variant, int32_t* best_tile_width) {
  if (!s) return fail(SWEPT_EINVAL, "null state");
  if (s->is_shard()) return fail(SWEPT_EUNSUPPORTED, "autotune an unsharded state of the same size per GPU instead");
  if (variant != SWEPT_PER_STEP && variant != SWEPT_SWEPT) return fail(SWEPT_EINVAL, "unknown variant");
  if (int rc = set_device(s)) return rc;
  const ProblemShape sh = kShape[s->problem];
  // keep the field: the trial runs scribble over all four slabs
  void* backup = dev_alloc(s, s->slab_bytes);
  if (!backup) return fail(SWEPT_ENOMEM, "autotune: device allocation of %zu bytes failed", s->slab_bytes);
  const int64_t saved_steps = s->steps_done;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  int rc_final = 0;
  // every CUDA call below is checked; the first failure ends the search, and the clean-up still runs
  auto ok = [&](cudaError_t e, const char* what) {
    if (e != cudaSuccess && !rc_final) rc_final = fail(SWEPT_ECUDA, "autotune: %s: %s", what, cudaGetErrorString(e));
    return e == cudaSuccess;
  };
  ok(cudaMemcpyAsync(backup, s->slab[s->cur], s->slab_bytes, cudaMemcpyDeviceToDevice, s->stream), "backup copy");
  ok(cudaEventCreate(&e0), "event") && ok(cudaEventCreate(&e1), "event");
  double best = 1e300;
  int best_n = 0, best_fl = 0, best_P = 0;
  struct Cand { int n, fl, P; };
  std::vector<Cand> cands;
  if (variant == SWEPT_PER_STEP) {
    for (int t = 32; t <= 1024; t *= 2) cands.push_back({t, 0, 0});
  } else {
    for (int n = 32; n <= 4096; n *= 2)
      for (int fl : {SWEPT_FLAVOR_TIER, SWEPT_FLAVOR_CHAR})
        for (int P : {1, 2, 4, 8, 16, 32})
          if (tile_ok(s, fl, n, P)) cands.push_back({n, fl, P});
    for (int n : {32, 64, 128, 256, 512})
      for (int wpc : {0, 4, 8, 16, 32})  // warps per CTA of the CLUSTER flavour (0 = the fewest that fit)
        if (tile_ok(s, SWEPT_FLAVOR_CLUSTER, n, wpc)) cands.push_back({n, SWEPT_FLAVOR_CLUSTER, wpc});
    for (int n : {256, 512, 1024})
      for (int ctas : {1, 2, 3, 4, 6})  // resident CTAs per SM (clamped to the occupancy limit at launch)
        for (int tma : {0, 16})         // generic 16-byte copies, or TMA bulk copies (group bit 4)
          if (tile_ok(s, SWEPT_FLAVOR_FLOW, n, ctas | tma)) cands.push_back({n, SWEPT_FLAVOR_FLOW, ctas | tma});
  }
  for (const Cand& c : cands) {
    if (rc_final) break;
    // enough steps for Up + 14 diamonds + Down at this width, so that the Up/Down rows and the start-up of a
    // persistent FLOW launch weigh as little as in a long run (and a few graph chunks for per-step)
    int64_t steps;
    if (variant == SWEPT_PER_STEP) steps = 512;
    else steps = std::max<int64_t>(16 * (c.n / (2 * sh.h)) / sh.sigma, 64);
    double t_best = 1e300;
    for (int rep = 0; rep < 3 && !rc_final; ++rep) {  // rep 0 warms up (graph capture, attribute setting)
      if (!ok(cudaMemcpyAsync(s->slab[s->cur], backup, s->slab_bytes, cudaMemcpyDeviceToDevice, s->stream), "restore") ||
          !ok(cudaEventRecord(e0, s->stream), "event record"))
        break;
      int rc = variant == SWEPT_PER_STEP ? run_per_step(s, steps, c.n) : run_swept(s, steps, c.n, c.fl, c.P);
      if (rc) { rc_final = rc; break; }
      if (!ok(cudaEventRecord(e1, s->stream), "event record") || !ok(cudaEventSynchronize(e1), "trial run")) break;
      if (int rc2 = check_flow_error(s)) { rc_final = rc2; break; }
      float ms = 0;
      if (!ok(cudaEventElapsedTime(&ms, e0, e1), "event time")) break;
      if (rep > 0) t_best = std::min(t_best, (double)ms / (double)steps);
    }
    if (!rc_final && t_best < best) { best = t_best; best_n = c.n; best_fl = c.fl; best_P = c.P; }
  }
  // restore the field whatever happened (keep the first error)
  {
    cudaError_t e = cudaMemcpyAsync(s->slab[s->cur], backup, s->slab_bytes, cudaMemcpyDeviceToDevice, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    ok(e, "restoring the field");
  }
  dev_free(s, backup);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  s->steps_done = saved_steps;
  if (rc_final) return rc_final;
  if (best_n == 0) return fail(SWEPT_EUNSUPPORTED, "no admissible tile width for N=%lld", (long long)s->N);
  s->tuned_width[variant] = best_n;
  if (variant == SWEPT_SWEPT) { s->tuned_flavor = best_fl; s->tuned_P = best_P; }
  {
    std::lock_guard<std::mutex> lock(g_tuned_mutex);
    TunedEntry& e = g_tuned[TunedKey{s->device, s->problem, s->dtype, s->rk2, s->bc, s->N}];
    e.width[variant] = best_n;
    if (variant == SWEPT_SWEPT) { e.flavor = best_fl; e.P = best_P; }
  }
  if (best_tile_width) *best_tile_width = best_n;
  return 0;
}

}  // extern "C"
