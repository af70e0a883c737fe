// strat.cu — the C ABI of libstrat.so (include/strat.h): host side; the sm_100a kernels are in
// strat_io.cuh / strat_kernels.cuh / strat_fused.cuh / strat_search.cuh, the rules in strat_game.cuh.
//
// Execution model: a batch = 32 consecutive games.
//   * Logic is thread-per-game on 100-bit bitboards held in registers (strat_game.cuh),
//     reading/writing per-game rows of shared memory whose strides (144 B, 113 words, 139 words)
//     make the 32 lanes hit 32 different banks.
//   * I/O is warp-cooperative: mask rows (32 x 452 B contiguous) and observations (32 x 8800 B
//     contiguous) leave as coalesced 16-byte vector stores staged through shared memory.
//   * The observation is produced as a 4400-bit stream per game; byte q of the stream expands,
//     through a small shared-memory table, to the q-th 16-byte chunk of the bf16 planes.
//   * The fused step (k_rollout_step) is persistent and warp-specialised: per CTA one logic
//     warp and one store warp, decoupled by mbarriers; consecutive launches overlap through
//     programmatic dependent launch and are ordered batch by batch with version flags.
//   * The single-purpose kernels (k_legal_mask, k_step, k_encode_obs, ...) run one warp per CTA.
#include <cuda_runtime.h>
#include <stdint.h>
#include <memory>
#include <mutex>
#include <new>

#include "../../include/strat.h"
#include "strat_game.cuh"

#include "strat_io.cuh"
#include "strat_kernels.cuh"
#include "strat_fused.cuh"
#include "strat_search.cuh"

namespace {
using namespace strat;

// ------------------------------------------------------------------ host side
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline bool cfg_ok(const strat_config* c) {
  return c && c->num_games >= 1 && (c->variant == 0 || c->variant == 1) && c->max_plies >= 0 &&
         c->max_battleless >= 0 && (c->chase_rule == 0 || c->chase_rule == 1) &&
         c->game_base + (uint64_t)c->num_games <= (1ull << 32) &&  // RNG counters carry a 32-bit global game index
         (c->infostate == 0 || c->infostate == 1) && c->reserved == 0;
}
inline Params make_params(const strat_config& c) {
  Params P;
  P.key0 = (uint32_t)c.seed; P.key1 = (uint32_t)(c.seed >> 32);
  P.game_base = (uint32_t)c.game_base;
  P.num_games = c.num_games; P.variant = c.variant;
  P.ply_cap = (c.max_plies >= 1 && c.max_plies <= 65535) ? c.max_plies : 65535;
  P.max_battleless = c.max_battleless; P.auto_reset = c.auto_reset ? 1 : 0; P.two_square = c.two_square ? 1 : 0;
  P.chase_rule = c.chase_rule ? 1 : 0;
  P.movelog = nullptr;
  P.pool = nullptr; P.pool_size = 0;
  P.pin = nullptr; P.pin_log = nullptr;
  P.track = nullptr;
  return P;
}
inline int launch_status() { return cudaGetLastError() == cudaSuccess ? STRAT_OK : STRAT_CUDA_ERROR; }
inline int batches(int n) { return (n + kBatch - 1) / kBatch; }
// A launch cannot start before every CTA of the previous one has started, and each launch in
// flight holds at least one of the <= 32 x SMs resident CTA slots, so far fewer than kTicketRing
// launches are ever in flight and two launches never share a ticket counter.
constexpr int kTicketRing = 8192;
constexpr int kOtherTickets = 64;  // self-resetting work counters of the other persistent kernels: word 1 strat_probe_write,
                                   // words 2..63 strat_encode_infostate, one per call in rotation (calls on different streams
                                   // may be in flight together; 62 at once is more than the GPU holds resident)
inline size_t sync_words(int n) { return (size_t)kTicketRing + 2 * (size_t)batches(n) + kOtherTickets; }

template <typename T>
void copy_elems(const T* src, T* dst, size_t count, cudaStream_t s) {
  if (count == 0) return;
  // widen to 16-byte vectors when both ends and the size allow it
  size_t bytes = count * sizeof(T);
  if ((((uintptr_t)src | (uintptr_t)dst | bytes) & 15) == 0) {
    size_t n16 = bytes / 16;
    int blocks = (int)((n16 + 255) / 256 < 148 * 16 ? (n16 + 255) / 256 : 148 * 16);
    k_copy<uint4><<<blocks, 256, 0, s>>>(reinterpret_cast<const uint4*>(src), reinterpret_cast<uint4*>(dst), n16);
  } else {
    int blocks = (int)((count + 255) / 256 < 148 * 16 ? (count + 255) / 256 : 148 * 16);
    k_copy<T><<<blocks, 256, 0, s>>>(src, dst, count);
  }
}
// records [0,n) of the source go to rows (row+i) mod rows of the array: at most two runs (n <= rows).
template <typename T>
void push_array(const T* src, T* ring, size_t per_rec, int64_t row, int64_t rows, int64_t n, cudaStream_t s) {
  int64_t first = n < rows - row ? n : rows - row;
  copy_elems<T>(src, ring + (size_t)row * per_rec, (size_t)first * per_rec, s);
  copy_elems<T>(src + (size_t)first * per_rec, ring, (size_t)(n - first) * per_rec, s);
}

}  // namespace

// Which fused step was launched last on which stream, as far as the environments sharing this
// record know (one private record per environment; strat_share_chain merges two).  A fused step
// may skip griddepcontrol.wait only when it directly continues its own environment's chain.
struct ChainRecord {
  std::mutex m;
  const void* stream = nullptr;
  const strat_env* last = nullptr;
};

struct strat_env {
  std::shared_ptr<ChainRecord> chain;
  strat_config cfg;
  strat::Params P;
  uint32_t* lines;
  int* err;
  uint32_t* tickets;     // ring of kTicketRing self-resetting batch-ticket counters (slot = version % ring)
  uint32_t* f_state;     // [batches] version of the last fused step that finished the batch's state
  uint32_t* f_obs;       // [batches] ... that finished the batch's observation stores
  uint32_t version;      // fused-step launches so far
  int num_sms;
  strat_history* hist;   // attached board-history ring, or nullptr
  strat_replay* chained; // ring whose gathers run chained between this environment's fused steps, or nullptr
  mutable uint32_t info_calls;  // strat_encode_infostate calls so far: picks the call's work counter
};

// Circular buffer of `length` time steps: per step N device lines + N x
// (action i16, reward i8, done u8).
struct strat_history {
  int32_t num_games, length;
  int64_t cur;                 // CurrentStep: state updates recorded so far
  uint32_t* lines; int16_t* act; int8_t* rew; uint8_t* done;
  uint16_t* logs;              // scratch [N][64]: move logs rebuilt for a query about a past state (chasing rule)
  const strat_env* env;        // attached environment (live state = time step cur)
  strat::Params P;             // its rule parameters, kept for queries after a detach
  // a tracked ring (strat_history_create_tracked) also keeps, per time step, the 2 KB of S2 trackers of every game
  uint32_t* track;             // [length][N][kTrackWords], or nullptr for a plain ring
  uint32_t* tickets;           // kOtherTickets self-resetting work counters of the historical 487-channel encoder
  mutable uint32_t info_calls; // strat_history_encode_infostate calls so far: picks the call's counter
  int num_sms;
};

namespace {
inline HistSlot hist_slot(strat_history* h) {
  HistSlot s = {nullptr, nullptr, nullptr, nullptr};
  if (h) {
    size_t k = (size_t)(h->cur % h->length), n = (size_t)h->num_games;
    s.lines = h->lines + k * n * kLineWords; s.act = h->act + k * n; s.rew = h->rew + k * n; s.done = h->done + k * n;
  }
  return s;
}
// state lines of time step t, or nullptr if t is outside the ring / not the live state
inline const uint32_t* hist_lines_at(const strat_history* h, int64_t t) {
  if (!h) return nullptr;
  if (t == h->cur) return h->env ? h->env->lines : nullptr;
  if (t < 0 || t >= h->cur || t < h->cur - h->length) return nullptr;
  return h->lines + (size_t)(t % h->length) * (size_t)h->num_games * kLineWords;
}
// A tracked ring records the trackers of the state a step starts from: copied by one more kernel in front of
// the step (fused steps recorded this way are separated by it and do not overlap).  True if it was launched.
inline bool hist_record_trackers(const strat_env* env, cudaStream_t s) {
  strat_history* h = env->hist;
  if (!h || !h->track || !env->P.track) return false;
  const size_t words = (size_t)h->num_games * kTrackWords;
  copy_elems<uint32_t>(env->P.track, h->track + (size_t)(h->cur % h->length) * words, words, s);
  return true;
}
inline void hist_rebuild_logs(const strat_history* h, int64_t t, const uint16_t* pin_logs, uint16_t* logs, cudaStream_t s) {
  int64_t oldest = h->cur - h->length > 0 ? h->cur - h->length : 0;
  k_rebuild_logs<<<(h->num_games + 255) / 256, 256, 0, s>>>(h->num_games, hist_lines_at(h, t), h->act, h->done, h->length,
                                                            (long long)t, (long long)oldest, pin_logs, logs);
}
}  // namespace

// Record number s (0, 1, 2, ... in push order) lives in row s % rows of the four small arrays and
// in row s % obs_rows of the observation array; rows = obs_rows = capacity for a plain ring.  A
// ring made for in-place pushes has spare rows, so that the block a fused step is writing ahead
// (mask_t ... done_t of the records being completed, obs_{t+1} of the next ones) never aliases a
// live record.  `head` = total % capacity and the index p of strat_replay_sample are positions in
// the capacity-sized ring of SURVEY C6 (what the oracle's ring calls a physical record).
struct strat_replay {
  int64_t per_slot, slots, capacity, head, filled;
  int64_t total;           // records pushed so far
  int64_t rows, obs_rows;  // physical rows of mask/action/reward/done, of obs
  uint16_t* obs; uint32_t* mask; int16_t* action; int8_t* reward; uint8_t* done;
  uint32_t* sync;          // 3 device words: two CTA counters and the number of the last finished chained gather
  uint32_t gathers;        // chained gathers issued so far
  strat_env* env;          // environment whose fused steps the chained gathers sit between, or nullptr
  // the regular loop (fused step, commit, chained gather, fused step, ...): what the last chained gather saw
  bool have_last; uint32_t last_version; int64_t last_total;
  uint32_t vouch_version;  // every fused step up to this version had finished before some earlier gather started
};

namespace {
// Launch of the fused step.  Programmatic dependent launch: the launch may become resident while
// the previous launch in the stream is still running IF that one is also a fused step (the only
// kernel that executes griddepcontrol.launch_dependents); behind any other kernel the attribute
// changes nothing.  Ordering against the previous fused step is per batch (f_state / f_obs).
// A fused step skips griddepcontrol.wait only if the operation issued immediately before it for
// this environment (and for every environment sharing its chain record) was a fused step of the
// SAME environment on the SAME stream: the per-batch version flags then order the two.  Every
// other entry point that takes the environment breaks the chain (chain_break), and a step with
// caller-provided actions (kExternal) always waits: its input comes from a foreign kernel.
inline void chain_break(const strat_env* env) {
  if (!env || !env->chain) return;
  std::lock_guard<std::mutex> lock(env->chain->m);
  env->chain->last = nullptr; env->chain->stream = nullptr;
}

// (Re)start the S2 trackers of every game from its current line (no-op without infostate).
inline void track_restart(const strat_env* env, cudaStream_t s);

template <bool kExternal>
int launch_fused(strat_env* env, uint32_t* mask, int16_t* actions, int8_t* reward, uint8_t* done, uint16_t* obs,
                 void* stream) {
  // The launch carries a host-side launch counter (the version the batch flags are compared
  // with): replaying it from a captured CUDA graph would reuse a stale version and wait forever.
  cudaStreamCaptureStatus capture = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing((cudaStream_t)stream, &capture) != cudaSuccess) return STRAT_CUDA_ERROR;
  if (capture != cudaStreamCaptureStatusNone) return STRAT_BAD_STATE;
  const int nb = batches(env->P.num_games);
  // a launch that follows a policy kernel has the GPU to itself (kWsExternalCtasPerSm says how it uses it)
  const int per_sm = kExternal ? kWsExternalCtasPerSm : env->P.track ? kWsTrackCtasPerSm : kWsCtasPerSm;
  const int grid = nb < env->num_sms * per_sm ? nb : env->num_sms * per_sm;
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)grid); lc.blockDim = dim3(64); lc.dynamicSmemBytes = 0; lc.stream = (cudaStream_t)stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = 1;
  const uint32_t version = env->version + 1;
  if (hist_record_trackers(env, (cudaStream_t)stream)) chain_break(env);  // the copy kernel is not a fused step: wait for it
  int wait_prior;
  {
    ChainRecord& rec = *env->chain;
    std::lock_guard<std::mutex> lock(rec.m);
    // a step with caller-provided actions publishes nothing while it runs (flag_set<false>): whatever
    // follows it waits for its grid as a whole, so its own environment's chain restarts after it
    wait_prior = kExternal || !(rec.last == env && rec.stream == stream);
    rec.last = kExternal ? nullptr : env; rec.stream = kExternal ? nullptr : stream;
  }
  auto kernel = env->P.track ? (env->P.chase_rule ? k_rollout_step<kExternal, true, true> : k_rollout_step<kExternal, false, true>)
                             : (env->P.chase_rule ? k_rollout_step<kExternal, true, false> : k_rollout_step<kExternal, false, false>);
  // chained gathers: the first step after a gather may overlap it (the rows it writes are the ring's spare
  // rows) but not the gather before it; a further step without a gather in between (a block has been
  // committed since) would write rows the latest gather may still read, so it waits for that one
  const uint32_t* gflag = nullptr;
  uint32_t gnum = 0u;
  if (env->chained && env->chained->gathers >= 1u) {
    const strat_replay* r = env->chained;
    gnum = r->total > r->last_total ? r->gathers : r->gathers - 1u;
    if (gnum >= 1u) gflag = r->sync + 2;
  }
  if (cudaLaunchKernelEx(&lc, kernel, env->P, env->lines, mask, actions, reward, done, obs,
                         env->tickets + (version % kTicketRing), env->f_state, env->f_obs, version,
                         hist_slot(env->hist), env->err, wait_prior, gflag, gnum) != cudaSuccess)
    return STRAT_CUDA_ERROR;
  env->version = version;
  if (env->hist) env->hist->cur += 1;
  return STRAT_OK;
}
inline void track_restart(const strat_env* env, cudaStream_t s) {
  if (env->P.track) k_track_start<<<(env->P.num_games + 3) / 4, 128, 0, s>>>(env->P, env->lines);
}
}  // namespace

extern "C" {

const char* strat_error_string(int code) {
  switch (code) {
    case STRAT_OK: return "ok";
    case STRAT_BAD_ARG: return "bad argument";
    case STRAT_BAD_STATE: return "bad state";
    case STRAT_CUDA_ERROR: return "CUDA error";
    case STRAT_ILLEGAL_ACTION: return "illegal action for a live game";
    case STRAT_TOO_LARGE: return "more games than the built-in scratch holds (STRAT_STATIC_MAX_GAMES)";
    default: return "unknown error";
  }
}

size_t strat_workspace_bytes(const strat_config* cfg) {
  if (!cfg_ok(cfg)) return 0;
  return align_up((size_t)cfg->num_games * STRAT_LINE_BYTES, 256) + 256 + align_up(sync_words(cfg->num_games) * 4, 256) +
         (cfg->chase_rule ? align_up((size_t)cfg->num_games * kLogPlies * 2, 256) : 0) +  // move logs: the chasing rule's memory
         (cfg->infostate ? (size_t)cfg->num_games * kTrackWords * 4 : 0);                 // S2 trackers
}

int strat_create(const strat_config* cfg, void* workspace_dev, size_t bytes, void* stream, strat_env** out) {
  if (!cfg_ok(cfg) || !workspace_dev || !out || bytes < strat_workspace_bytes(cfg) ||
      ((uintptr_t)workspace_dev & 255) != 0)
    return STRAT_BAD_ARG;
  if (cudaSetDevice(cfg->device) != cudaSuccess) return STRAT_CUDA_ERROR;
  strat_env* e = new (std::nothrow) strat_env;
  if (!e) return STRAT_BAD_ARG;
  e->chain = std::make_shared<ChainRecord>();
  e->cfg = *cfg;
  e->P = make_params(*cfg);
  e->lines = reinterpret_cast<uint32_t*>(workspace_dev);
  e->err = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(workspace_dev) +
                                  align_up((size_t)cfg->num_games * STRAT_LINE_BYTES, 256));
  e->tickets = reinterpret_cast<uint32_t*>(e->err) + 64;
  e->f_state = e->tickets + kTicketRing;
  e->f_obs = e->f_state + batches(cfg->num_games);
  e->version = 0;
  e->hist = nullptr;
  e->chained = nullptr;
  e->info_calls = 0;
  uint8_t* extra = reinterpret_cast<uint8_t*>(e->tickets) + align_up(sync_words(cfg->num_games) * 4, 256);
  if (cfg->chase_rule) {
    e->P.movelog = reinterpret_cast<uint16_t*>(extra);
    extra += align_up((size_t)cfg->num_games * kLogPlies * 2, 256);
  }
  if (cfg->infostate) e->P.track = reinterpret_cast<uint32_t*>(extra);
  if (cudaMemsetAsync(e->tickets, 0, sync_words(cfg->num_games) * 4, (cudaStream_t)stream) != cudaSuccess) {
    delete e;
    return STRAT_CUDA_ERROR;
  }
  e->num_sms = 148;
  cudaDeviceGetAttribute(&e->num_sms, cudaDevAttrMultiProcessorCount, cfg->device);
  *out = e;
  return strat_reset(e, cfg->seed, stream);
}

int strat_destroy(strat_env* env) {
  if (env && env->hist) env->hist->env = nullptr;
  if (env && env->chained) env->chained->env = nullptr;
  chain_break(env);
  delete env;
  return STRAT_OK;
}

int strat_share_chain(strat_env* a, strat_env* b) {
  if (!a || !b) return STRAT_BAD_ARG;
  if (a->chain == b->chain) return STRAT_OK;
  // b joins a's group.  If b already shared its record with other environments, re-pointing b alone
  // would leave those unordered against a's group: groups grow one lone environment at a time.
  if (b->chain.use_count() > 1) return STRAT_BAD_STATE;
  chain_break(a); chain_break(b);
  b->chain = a->chain;
  return STRAT_OK;
}

int strat_reset(strat_env* env, uint64_t seed, void* stream) {
  if (!env) return STRAT_BAD_ARG;
  chain_break(env);
  cudaStream_t s = (cudaStream_t)stream;
  env->cfg.seed = seed;
  const uint32_t* pin = env->P.pin;
  const uint16_t* pin_log = env->P.pin_log;
  uint16_t* movelog = env->P.movelog;
  uint32_t* track = env->P.track;
  const uint8_t* pool = env->P.pool;
  int32_t pool_size = env->P.pool_size;
  env->P = make_params(env->cfg);
  env->P.pin = pin; env->P.pin_log = pin_log;
  env->P.movelog = movelog;
  env->P.track = track;
  env->P.pool = pool; env->P.pool_size = pool_size;
  k_set_int<<<1, 1, 0, s>>>(env->err, 0);
  k_reset<<<batches(env->P.num_games), 32, 0, s>>>(env->P, env->lines);
  track_restart(env, s);
  return launch_status();
}

int strat_reset_from(strat_env* env, const uint8_t* boards, void* stream) {
  if (!env || !boards) return STRAT_BAD_ARG;
  chain_break(env);
  int n = env->P.num_games;
  k_import<<<(n + 3) / 4, 128, 0, (cudaStream_t)stream>>>(n, boards, env->lines, env->err);
  track_restart(env, (cudaStream_t)stream);
  return launch_status();
}

int strat_reset_from_with_plies(strat_env* env, const uint8_t* boards, const uint8_t* plies, void* stream) {
  if (!env || !boards || !plies) return STRAT_BAD_ARG;
  chain_break(env);
  int n = env->P.num_games;
  k_import<<<(n + 3) / 4, 128, 0, (cudaStream_t)stream>>>(n, boards, env->lines, env->err);
  if (env->P.movelog)  // without the chasing rule nothing remembers plies
    k_load_plies<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>(n, plies, env->lines, env->P.movelog);
  track_restart(env, (cudaStream_t)stream);
  return launch_status();
}

int strat_set_setup_pool(strat_env* env, const uint8_t* pool_dev, int32_t K, void* stream) {
  if (!env) return STRAT_BAD_ARG;
  chain_break(env);
  if (!pool_dev || K <= 0) { env->P.pool = nullptr; env->P.pool_size = 0; return STRAT_OK; }
  k_check_pool<<<(2 * K + 127) / 128, 128, 0, (cudaStream_t)stream>>>(pool_dev, K, env->err);
  env->P.pool = pool_dev; env->P.pool_size = K;
  return launch_status();
}

int strat_pin_reset_state(strat_env* env, void* pin_lines_dev, const uint8_t* boards, void* stream) {
  if (!env) return STRAT_BAD_ARG;
  chain_break(env);
  if (!boards) { env->P.pin = nullptr; env->P.pin_log = nullptr; return STRAT_OK; }
  if (!pin_lines_dev || ((uintptr_t)pin_lines_dev & 15) != 0) return STRAT_BAD_ARG;
  int n = env->P.num_games;
  k_import<<<(n + 3) / 4, 128, 0, (cudaStream_t)stream>>>(n, boards, reinterpret_cast<uint32_t*>(pin_lines_dev), env->err);
  env->P.pin = reinterpret_cast<const uint32_t*>(pin_lines_dev);
  env->P.pin_log = nullptr;
  return launch_status();
}

int strat_pin_reset_state_with_plies(strat_env* env, void* pin_lines_dev, void* pin_logs_dev, const uint8_t* boards,
                                     const uint8_t* plies, void* stream) {
  if (!env || !boards || !plies || !pin_logs_dev || ((uintptr_t)pin_logs_dev & 15) != 0) return STRAT_BAD_ARG;
  int rc = strat_pin_reset_state(env, pin_lines_dev, boards, stream);
  if (rc != STRAT_OK || !env->P.movelog) return rc;
  int n = env->P.num_games;
  k_load_plies<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>(n, plies, reinterpret_cast<uint32_t*>(pin_lines_dev),
                                                                 reinterpret_cast<uint16_t*>(pin_logs_dev));
  env->P.pin_log = reinterpret_cast<const uint16_t*>(pin_logs_dev);
  return launch_status();
}

int strat_get_boards(const strat_env* env, uint8_t* boards, void* stream) {
  if (!env || !boards) return STRAT_BAD_ARG;
  chain_break(env);
  int n = env->P.num_games;
  k_export<<<(n + 3) / 4, 128, 0, (cudaStream_t)stream>>>(n, env->lines, boards);
  return launch_status();
}

int strat_legal_mask(const strat_env* env, uint32_t* mask, void* stream) {
  if (!env || !mask) return STRAT_BAD_ARG;
  chain_break(env);
  if (env->P.chase_rule) k_legal_mask<true><<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, mask);
  else k_legal_mask<false><<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, mask);
  return launch_status();
}

int strat_sample_uniform(const strat_env* env, const uint32_t* mask, int16_t* actions, void* stream) {
  if (!env || !mask || !actions) return STRAT_BAD_ARG;
  chain_break(env);
  int n = env->P.num_games;
  k_sample_uniform<<<(n + 3) / 4, 128, 0, (cudaStream_t)stream>>>(env->P, env->lines, mask, actions);
  return launch_status();
}

int strat_step(strat_env* env, const int16_t* actions, int8_t* reward, uint8_t* done, void* stream) {
  if (!env || !actions || !reward || !done) return STRAT_BAD_ARG;
  chain_break(env);
  auto kernel = env->P.track ? (env->P.chase_rule ? k_step<true, true> : k_step<false, true>)
                             : (env->P.chase_rule ? k_step<true, false> : k_step<false, false>);
  hist_record_trackers(env, (cudaStream_t)stream);
  kernel<<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, actions, reward, done, env->err,
                                                                     hist_slot(env->hist));
  if (env->hist) env->hist->cur += 1;
  return launch_status();
}

int strat_encode_obs(const strat_env* env, uint16_t* obs, void* stream) {
  if (!env || !obs) return STRAT_BAD_ARG;
  chain_break(env);
  k_encode_obs<<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, obs);
  return launch_status();
}

int strat_encode_infostate(const strat_env* env, uint16_t* out, void* stream) {
  if (!env || !out || ((uintptr_t)out & 7) != 0) return STRAT_BAD_ARG;
  if (!env->P.track) return STRAT_BAD_STATE;
  chain_break(env);
  int ctas = env->P.num_games < kInfoCtasPerSm * env->num_sms ? env->P.num_games : kInfoCtasPerSm * env->num_sms;
  uint32_t* ticket = env->f_obs + batches(env->P.num_games) + 2 + (env->info_calls++ % (uint32_t)(kOtherTickets - 2));
  k_encode_infostate<<<ctas, 64, 0, (cudaStream_t)stream>>>(env->P, env->lines, out, ticket);
  return launch_status();
}

int strat_probe_write(const strat_env* env, void* dst, size_t bytes, int32_t chunk_bytes, int32_t dynamic, void* stream) {
  if (!env || !dst || chunk_bytes < 16 || chunk_bytes % 16 != 0 || bytes % (size_t)chunk_bytes != 0 ||
      ((uintptr_t)dst & 15) != 0 || bytes / (size_t)chunk_bytes > 0x7FFFFFFFull)
    return STRAT_BAD_ARG;
  if (bytes == 0) return STRAT_OK;
  const uint32_t pieces = (uint32_t)(bytes / (size_t)chunk_bytes);
  const uint32_t grid = pieces < (uint32_t)(2 * env->num_sms) ? pieces : (uint32_t)(2 * env->num_sms);
  k_probe_write<<<grid, 128, 0, (cudaStream_t)stream>>>(reinterpret_cast<uint4*>(dst), pieces, (uint32_t)chunk_bytes / 16u,
                                                       env->f_obs + batches(env->P.num_games) + 1, dynamic ? 1 : 0);
  return launch_status();
}

int strat_rollout_step(strat_env* env, uint32_t* mask, int16_t* actions, int8_t* reward, uint8_t* done,
                       uint16_t* obs, void* stream) {
  if (!env || !obs) return STRAT_BAD_ARG;
  return launch_fused<false>(env, mask, actions, reward, done, obs, stream);
}

int strat_step_observe(strat_env* env, const int16_t* actions, int8_t* reward, uint8_t* done, uint32_t* mask,
                       uint16_t* obs, void* stream) {
  if (!env || !actions || !reward || !done || !obs) return STRAT_BAD_ARG;
  return launch_fused<true>(env, mask, const_cast<int16_t*>(actions), reward, done, obs, stream);
}

size_t strat_host_scratch_bytes(const strat_config* cfg) {
  if (!cfg_ok(cfg)) return 0;
  size_t n = (size_t)cfg->num_games;
  return align_up(n * STRAT_OBS_ELEMS * 2, 256) + align_up(n * STRAT_MASK_WORDS * 4, 256) + align_up(n * 2, 256) +
         align_up(n, 256) + align_up(n, 256);
}

int strat_rollout_step_host(strat_env* env, void* scratch_dev, uint32_t* mask_host, int16_t* actions_host,
                            int8_t* reward_host, uint8_t* done_host, uint16_t* obs_host, void* stream) {
  if (!env || !scratch_dev || !mask_host || !actions_host || !reward_host || !done_host || !obs_host)
    return STRAT_BAD_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  size_t n = (size_t)env->P.num_games;
  uint8_t* p = reinterpret_cast<uint8_t*>(scratch_dev);
  uint16_t* obs = reinterpret_cast<uint16_t*>(p); p += align_up(n * STRAT_OBS_ELEMS * 2, 256);
  uint32_t* mask = reinterpret_cast<uint32_t*>(p); p += align_up(n * STRAT_MASK_WORDS * 4, 256);
  int16_t* act = reinterpret_cast<int16_t*>(p); p += align_up(n * 2, 256);
  int8_t* rew = reinterpret_cast<int8_t*>(p); p += align_up(n, 256);
  uint8_t* done = p;
  int rc = strat_rollout_step(env, mask, act, rew, done, obs, stream);
  if (rc != STRAT_OK) return rc;
  bool ok = cudaMemcpyAsync(obs_host, obs, n * STRAT_OBS_ELEMS * 2, cudaMemcpyDeviceToHost, s) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(mask_host, mask, n * STRAT_MASK_WORDS * 4, cudaMemcpyDeviceToHost, s) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(actions_host, act, n * 2, cudaMemcpyDeviceToHost, s) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(reward_host, rew, n, cudaMemcpyDeviceToHost, s) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(done_host, done, n, cudaMemcpyDeviceToHost, s) == cudaSuccess;
  ok = ok && cudaStreamSynchronize(s) == cudaSuccess;
  return ok ? STRAT_OK : STRAT_CUDA_ERROR;
}

int strat_step_host(strat_env* env, void* scratch_dev, const int16_t* actions_host, int8_t* reward_host,
                    uint8_t* done_host, uint32_t* mask_host, uint16_t* obs_host, void* stream) {
  if (!env || !scratch_dev || !actions_host || !reward_host || !done_host || !mask_host || !obs_host)
    return STRAT_BAD_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  size_t n = (size_t)env->P.num_games;
  uint8_t* p = reinterpret_cast<uint8_t*>(scratch_dev);
  uint16_t* obs = reinterpret_cast<uint16_t*>(p); p += align_up(n * STRAT_OBS_ELEMS * 2, 256);
  uint32_t* mask = reinterpret_cast<uint32_t*>(p); p += align_up(n * STRAT_MASK_WORDS * 4, 256);
  int16_t* act = reinterpret_cast<int16_t*>(p); p += align_up(n * 2, 256);
  int8_t* rew = reinterpret_cast<int8_t*>(p); p += align_up(n, 256);
  uint8_t* done = p;
  if (cudaMemcpyAsync(act, actions_host, n * 2, cudaMemcpyHostToDevice, s) != cudaSuccess) return STRAT_CUDA_ERROR;
  int rc = strat_step_observe(env, act, rew, done, mask, obs, stream);
  if (rc != STRAT_OK) return rc;
  bool ok = cudaMemcpyAsync(reward_host, rew, n, cudaMemcpyDeviceToHost, s) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(done_host, done, n, cudaMemcpyDeviceToHost, s) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(mask_host, mask, n * STRAT_MASK_WORDS * 4, cudaMemcpyDeviceToHost, s) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(obs_host, obs, n * STRAT_OBS_ELEMS * 2, cudaMemcpyDeviceToHost, s) == cudaSuccess;
  ok = ok && cudaStreamSynchronize(s) == cudaSuccess;
  return ok ? STRAT_OK : STRAT_CUDA_ERROR;
}

int strat_rollout_uniform(strat_env* env, int32_t plies, void* stream) {
  if (!env || plies < 0) return STRAT_BAD_ARG;
  chain_break(env);
  if (env->hist || env->P.track) return STRAT_BAD_STATE;  // on-chip plies are neither recorded nor tracked
  if (env->P.chase_rule)
    k_rollout_uniform<true><<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, plies, env->err);
  else
    k_rollout_uniform<false><<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, plies, env->err);
  return launch_status();
}

int strat_check(strat_env* env) {
  if (!env) return STRAT_BAD_ARG;
  if (cudaDeviceSynchronize() != cudaSuccess) return STRAT_CUDA_ERROR;
  int v = 0;
  if (cudaMemcpy(&v, env->err, sizeof v, cudaMemcpyDeviceToHost) != cudaSuccess) return STRAT_CUDA_ERROR;
  return v;
}

int strat_clear_error(strat_env* env, void* stream) {
  if (!env) return STRAT_BAD_ARG;
  chain_break(env);
  k_set_int<<<1, 1, 0, (cudaStream_t)stream>>>(env->err, 0);
  return launch_status();
}

// ---- replay ring
namespace {
int replay_layout(int64_t rows, int64_t obs_rows, size_t off[6]) {
  size_t p = 0;
  off[0] = p; p += align_up((size_t)obs_rows * STRAT_OBS_ELEMS * 2, 256);
  off[1] = p; p += align_up((size_t)rows * STRAT_MASK_WORDS * 4, 256);
  off[2] = p; p += align_up((size_t)rows * 2, 256);
  off[3] = p; p += align_up((size_t)rows, 256);
  off[4] = p; p += align_up((size_t)rows, 256);
  off[5] = p;  // 256 bytes of synchronisation words follow
  return STRAT_OK;
}
inline bool ring_args_ok(int32_t per_slot, int32_t slots, int32_t block) {
  if (per_slot <= 0 || slots <= 0 || block < 0) return false;
  int64_t C = (int64_t)per_slot * slots;
  return C <= 0xFFFFFFFFll && (block == 0 || (block <= C && C % block == 0));
}
int replay_make(void* mem_dev, size_t bytes, int32_t per_slot, int32_t slots, int32_t block, strat_replay** out) {
  if (!mem_dev || !out || !ring_args_ok(per_slot, slots, block) || ((uintptr_t)mem_dev & 255) != 0) return STRAT_BAD_ARG;
  int64_t C = (int64_t)per_slot * slots, rows = C + block, obs_rows = C + 2 * (int64_t)block;
  size_t off[6];
  replay_layout(rows, obs_rows, off);
  if (bytes < off[5] + 256) return STRAT_BAD_ARG;
  strat_replay* r = new (std::nothrow) strat_replay;
  if (!r) return STRAT_BAD_ARG;
  uint8_t* b = reinterpret_cast<uint8_t*>(mem_dev);
  r->per_slot = per_slot; r->slots = slots; r->capacity = C; r->head = 0; r->filled = 0; r->total = 0;
  r->rows = rows; r->obs_rows = obs_rows;
  r->obs = reinterpret_cast<uint16_t*>(b + off[0]); r->mask = reinterpret_cast<uint32_t*>(b + off[1]);
  r->action = reinterpret_cast<int16_t*>(b + off[2]); r->reward = reinterpret_cast<int8_t*>(b + off[3]);
  r->done = b + off[4];
  r->sync = reinterpret_cast<uint32_t*>(b + off[5]); r->gathers = 0; r->env = nullptr; r->have_last = false; r->last_version = 0; r->last_total = 0; r->vouch_version = 0;
  *out = r;
  return STRAT_OK;
}
inline void replay_advance(strat_replay* r, int64_t n) {
  r->total += n;
  r->head = r->total % r->capacity;
  r->filled = r->filled + n > r->capacity ? r->capacity : r->filled + n;
}
// push-order number of the live record at ring position p (0 <= p < filled)
inline int64_t replay_seq(const strat_replay* r, int64_t p) {
  int64_t base = r->total - r->filled;
  return base + ((p - base % r->capacity) + r->capacity) % r->capacity;
}
}  // namespace

int strat_replay_layout(int32_t per_slot, int32_t slots, int32_t block, size_t off[5]) {
  if (!ring_args_ok(per_slot, slots, block) || !off) return STRAT_BAD_ARG;
  size_t o[6];
  int64_t C = (int64_t)per_slot * slots;
  replay_layout(C + block, C + 2 * (int64_t)block, o);
  for (int i = 0; i < 5; ++i) off[i] = o[i];
  return STRAT_OK;
}

size_t strat_replay_bytes(int32_t per_slot, int32_t slots) { return strat_replay_bytes_in_place(per_slot, slots, 0); }

size_t strat_replay_bytes_in_place(int32_t per_slot, int32_t slots, int32_t block) {
  if (!ring_args_ok(per_slot, slots, block)) return 0;
  size_t o[6];
  int64_t C = (int64_t)per_slot * slots;
  replay_layout(C + block, C + 2 * (int64_t)block, o);
  return o[5] + 256;
}

int strat_replay_create(void* mem_dev, size_t bytes, int32_t per_slot, int32_t slots, strat_replay** out) {
  return replay_make(mem_dev, bytes, per_slot, slots, 0, out);
}

int strat_replay_create_in_place(void* mem_dev, size_t bytes, int32_t per_slot, int32_t slots, int32_t block,
                                 strat_replay** out) {
  if (block <= 0) return STRAT_BAD_ARG;
  return replay_make(mem_dev, bytes, per_slot, slots, block, out);
}

int strat_replay_destroy(strat_replay* r) {
  if (r && r->env) r->env->chained = nullptr;
  delete r;
  return STRAT_OK;
}

int strat_replay_push(strat_replay* r, const uint16_t* obs, const uint32_t* mask, const int16_t* action,
                      const int8_t* reward, const uint8_t* done, int32_t n, void* stream) {
  if (!r || !obs || !mask || !action || !reward || !done || n < 0 || n > r->capacity) return STRAT_BAD_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  int64_t row = r->total % r->rows, orow = r->total % r->obs_rows;
  push_array<uint16_t>(obs, r->obs, STRAT_OBS_ELEMS, orow, r->obs_rows, n, s);
  push_array<uint32_t>(mask, r->mask, STRAT_MASK_WORDS, row, r->rows, n, s);
  push_array<int16_t>(action, r->action, 1, row, r->rows, n, s);
  push_array<int8_t>(reward, r->reward, 1, row, r->rows, n, s);
  push_array<uint8_t>(done, r->done, 1, row, r->rows, n, s);
  r->have_last = false;  // records copied in by other kernels: the next chained gather waits for the stream
  replay_advance(r, n);
  return launch_status();
}

// In-place pushes work in blocks of n records that never wrap inside a block, and need the spare
// rows of strat_replay_create_in_place: the block written `ahead` pushes ahead must not alias a
// record that is live when the push in between is sampled.
static bool in_place_ok(const strat_replay* r, int32_t n, int32_t ahead) {
  if (!r || n <= 0 || ahead < 0 || ahead > 1) return false;
  if (r->total % n || r->rows % n || r->obs_rows % n) return false;
  return r->rows >= r->capacity + n && r->obs_rows >= r->capacity + (int64_t)(ahead + 1) * n;
}

int strat_replay_reserve(strat_replay* r, int32_t n, int32_t ahead, uint16_t** obs, uint32_t** mask) {
  if (!obs || !mask || !in_place_ok(r, n, ahead)) return STRAT_BAD_ARG;
  int64_t first = r->total + (int64_t)ahead * n;
  *obs = r->obs + (size_t)(first % r->obs_rows) * STRAT_OBS_ELEMS;
  *mask = r->mask + (size_t)(first % r->rows) * STRAT_MASK_WORDS;
  return STRAT_OK;
}

int strat_replay_reserve_rows(strat_replay* r, int32_t n, int16_t** action, int8_t** reward, uint8_t** done) {
  if (!action || !reward || !done || !in_place_ok(r, n, 0)) return STRAT_BAD_ARG;
  int64_t row = r->total % r->rows;
  *action = r->action + row; *reward = r->reward + row; *done = r->done + row;
  return STRAT_OK;
}

int strat_replay_commit(strat_replay* r, const int16_t* action, const int8_t* reward, const uint8_t* done, int32_t n,
                        void* stream) {
  if (!in_place_ok(r, n, 0)) return STRAT_BAD_ARG;
  if ((action == nullptr) != (reward == nullptr) || (action == nullptr) != (done == nullptr)) return STRAT_BAD_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  if (action) {  // nullptr x 3: the rows were written in place (strat_replay_reserve_rows)
    int64_t row = r->total % r->rows;
    copy_elems<int16_t>(action, r->action + row, (size_t)n, s);
    copy_elems<int8_t>(reward, r->reward + row, (size_t)n, s);
    copy_elems<uint8_t>(done, r->done + row, (size_t)n, s);
    r->have_last = false;  // as in strat_replay_push
  }
  replay_advance(r, n);
  return launch_status();
}

int strat_replay_sample(const strat_replay* r, uint64_t seed, uint64_t draw_index, int32_t batch, uint16_t* obs,
                        uint32_t* mask, int16_t* action, int8_t* reward, uint8_t* done, void* stream) {
  if (!r || batch < 0) return STRAT_BAD_ARG;
  if (r->filled == 0) return STRAT_BAD_STATE;
  if (batch == 0) return STRAT_OK;
  RingMap map;
  map.filled = (uint32_t)r->filled; map.capacity = (uint64_t)r->capacity; map.base = (uint64_t)(r->total - r->filled);
  map.rows = (uint64_t)r->rows; map.obs_rows = (uint64_t)r->obs_rows;
  GatherChain none = {};
  k_replay_sample<false><<<(batch + 3) / 4, 128, 0, (cudaStream_t)stream>>>(
      (uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)draw_index, (uint32_t)(draw_index >> 32), batch, map,
      r->obs, r->mask, r->action, r->reward, r->done, obs, mask, action, reward, done, none);
  return launch_status();
}

int strat_replay_sample_chained(strat_replay* r, strat_env* env, uint64_t seed, uint64_t draw_index, int32_t batch,
                                uint16_t* obs, uint32_t* mask, int16_t* action, int8_t* reward, uint8_t* done, void* stream) {
  if (!r || !env || batch <= 0) return STRAT_BAD_ARG;
  if (r->filled == 0 || r->rows < r->capacity + 1) return STRAT_BAD_STATE;  // in-place rings only (spare rows)
  if (r->env && r->env != env) return STRAT_BAD_ARG;
  // the environment's fused steps wait for the gathers of ONE ring (env->chained): a second ring tied to it
  // would silently take that slot over and the first ring's rows would be rewritten while its gather reads them
  if (!r->env && env->chained && env->chained != r) return STRAT_BAD_STATE;
  cudaStream_t s = (cudaStream_t)stream;
  if (!r->env) {  // first chained gather: clear the synchronisation words, tie the ring to the environment
    if (cudaMemsetAsync(r->sync, 0, 256, s) != cudaSuccess) return STRAT_CUDA_ERROR;
    chain_break(env);  // the memset is not a fused step: the next one waits for it
    r->env = env; env->chained = r; r->gathers = 0; r->have_last = false; r->vouch_version = env->version;
  }
  RingMap map;
  map.filled = (uint32_t)r->filled; map.capacity = (uint64_t)r->capacity; map.base = (uint64_t)(r->total - r->filled);
  map.rows = (uint64_t)r->rows; map.obs_rows = (uint64_t)r->obs_rows;
  r->gathers += 1;
  // Regular loop: the operation before this gather was the environment's fused step on this stream, one
  // step and one block of num_games records after the previous chained gather.  Then every record's
  // producer is known by version and the gather orders itself by the per-batch flags; anything else
  // falls back to waiting for the whole stream before it (and vouches for every step so far).
  const int64_t n = env->P.num_games;
  bool step_before;
  {
    ChainRecord& rec = *env->chain;
    std::lock_guard<std::mutex> lock(rec.m);
    step_before = rec.last == env && rec.stream == stream;
  }
  const bool regular = step_before && r->have_last && env->version == r->last_version + 1u &&
                       r->total == r->last_total + n && r->total % n == 0;
  if (!regular) r->vouch_version = env->version;
  r->have_last = true; r->last_version = env->version; r->last_total = r->total;
  GatherChain chain = {};
  chain.counter = r->sync; chain.done_flag = r->sync + 2; chain.number = r->gathers;
  chain.use_flags = regular ? 1 : 0; chain.f_state = env->f_state; chain.f_obs = env->f_obs;
  chain.newest_version = env->version; chain.vouch = r->vouch_version; chain.block = (uint32_t)n;
  chain.newest_block = (uint64_t)(r->total / n) - 1u;
  cudaLaunchConfig_t lc = {};
  int ctas = (batch + 3) / 4 < env->num_sms ? (batch + 3) / 4 : env->num_sms;  // one small CTA per SM: it waits, resident, for the step before it
  lc.gridDim = dim3((unsigned)ctas); lc.blockDim = dim3(128); lc.dynamicSmemBytes = 0; lc.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = 1;
  if (cudaLaunchKernelEx(&lc, k_replay_sample<true>, (uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)draw_index,
                         (uint32_t)(draw_index >> 32), (int)batch, map, (const uint16_t*)r->obs, (const uint32_t*)r->mask,
                         (const int16_t*)r->action, (const int8_t*)r->reward, (const uint8_t*)r->done, obs, mask, action,
                         reward, done, chain) != cudaSuccess)
    return STRAT_CUDA_ERROR;
  return STRAT_OK;  // deliberately no chain_break: the environment's next fused step continues its chain
}

int strat_replay_state(const strat_replay* r, int64_t* head, int64_t* filled) {
  if (!r) return STRAT_BAD_ARG;
  if (head) *head = r->head;
  if (filled) *filled = r->filled;
  return STRAT_OK;
}

int strat_replay_locate(const strat_replay* r, int64_t p, int64_t* row, int64_t* obs_row) {
  if (!r || p < 0 || p >= r->filled) return STRAT_BAD_ARG;
  int64_t s = replay_seq(r, p);
  if (row) *row = s % r->rows;
  if (obs_row) *obs_row = s % r->obs_rows;
  return STRAT_OK;
}

// ---- board-history ring (Table S1)
size_t strat_history_bytes(int32_t num_games, int32_t length) {
  if (num_games <= 0 || length <= 0) return 0;
  size_t n = (size_t)num_games, T = (size_t)length;
  return align_up(T * n * STRAT_LINE_BYTES, 256) + align_up(T * n * 2, 256) + 2 * align_up(T * n, 256) +
         align_up(n * kLogPlies * 2, 256);
}

int strat_history_create(void* mem_dev, size_t bytes, int32_t num_games, int32_t length, strat_history** out) {
  size_t need = strat_history_bytes(num_games, length);
  if (!mem_dev || !out || need == 0 || bytes < need || ((uintptr_t)mem_dev & 255) != 0) return STRAT_BAD_ARG;
  strat_history* h = new (std::nothrow) strat_history;
  if (!h) return STRAT_BAD_ARG;
  size_t n = (size_t)num_games, T = (size_t)length;
  uint8_t* b = reinterpret_cast<uint8_t*>(mem_dev);
  h->num_games = num_games; h->length = length; h->cur = 0; h->env = nullptr;
  h->lines = reinterpret_cast<uint32_t*>(b); b += align_up(T * n * STRAT_LINE_BYTES, 256);
  h->act = reinterpret_cast<int16_t*>(b); b += align_up(T * n * 2, 256);
  h->rew = reinterpret_cast<int8_t*>(b); b += align_up(T * n, 256);
  h->done = b; b += align_up(T * n, 256);
  h->logs = reinterpret_cast<uint16_t*>(b);
  h->track = nullptr; h->tickets = nullptr; h->info_calls = 0; h->num_sms = 148;
  *out = h;
  return STRAT_OK;
}

size_t strat_history_bytes_tracked(int32_t num_games, int32_t length) {
  size_t plain = strat_history_bytes(num_games, length);
  if (plain == 0) return 0;
  return plain + (size_t)length * (size_t)num_games * kTrackWords * 4 + 256;
}

int strat_history_create_tracked(void* mem_dev, size_t bytes, int32_t num_games, int32_t length, void* stream,
                                 strat_history** out) {
  size_t need = strat_history_bytes_tracked(num_games, length);
  if (need == 0 || bytes < need) return STRAT_BAD_ARG;
  int rc = strat_history_create(mem_dev, bytes, num_games, length, out);
  if (rc != STRAT_OK) return rc;
  strat_history* h = *out;
  uint8_t* b = reinterpret_cast<uint8_t*>(mem_dev) + strat_history_bytes(num_games, length);
  h->tickets = reinterpret_cast<uint32_t*>(b);
  h->track = reinterpret_cast<uint32_t*>(b + 256);
  int dev = 0;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev);
  if (cudaMemsetAsync(h->tickets, 0, 256, (cudaStream_t)stream) != cudaSuccess) {
    delete h; *out = nullptr;
    return STRAT_CUDA_ERROR;
  }
  return STRAT_OK;
}

int strat_history_destroy(strat_history* h) {
  if (h && h->env) const_cast<strat_env*>(h->env)->hist = nullptr;
  delete h;
  return STRAT_OK;
}

int strat_history_attach(strat_env* env, strat_history* h) {
  if (!env) return STRAT_BAD_ARG;
  chain_break(env);
  if (h && (h->num_games != env->P.num_games || (h->env && h->env != env))) return STRAT_BAD_ARG;
  if (env->hist && env->hist != h) env->hist->env = nullptr;
  env->hist = h;
  if (h) { h->env = env; h->P = env->P; }
  return STRAT_OK;
}

int strat_history_current_step(const strat_history* h, int64_t* step) {
  if (!h || !step) return STRAT_BAD_ARG;
  *step = h->cur;
  return STRAT_OK;
}

int strat_history_legal_mask(const strat_history* h, int64_t t, uint32_t* mask, void* stream) {
  if (h) chain_break(h->env);
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !mask) return STRAT_BAD_ARG;
  Params P = h->env ? h->env->P : h->P;
  if (t != h->cur && P.chase_rule) {  // a past state is judged with the plies the ring still holds
    hist_rebuild_logs(h, t, P.pin_log, h->logs, (cudaStream_t)stream);
    P.movelog = h->logs;
  }
  if (P.chase_rule) k_legal_mask<true><<<batches(h->num_games), 32, 0, (cudaStream_t)stream>>>(P, L, mask);
  else k_legal_mask<false><<<batches(h->num_games), 32, 0, (cudaStream_t)stream>>>(P, L, mask);
  return launch_status();
}

int strat_history_encode_obs(const strat_history* h, int64_t t, uint16_t* obs, void* stream) {
  if (h) chain_break(h->env);
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !obs) return STRAT_BAD_ARG;
  const Params& P = h->env ? h->env->P : h->P;
  k_encode_obs<<<batches(h->num_games), 32, 0, (cudaStream_t)stream>>>(P, L, obs);
  return launch_status();
}

int strat_history_encode_infostate(const strat_history* h, int64_t t, uint16_t* out, void* stream) {
  if (h) chain_break(h->env);
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !out || ((uintptr_t)out & 7) != 0) return STRAT_BAD_ARG;
  Params P = h->env ? h->env->P : h->P;
  if (!h->track || !P.track) return STRAT_BAD_STATE;  // a plain ring, or an environment that keeps no trackers
  if (t != h->cur) P.track = h->track + (size_t)(t % h->length) * (size_t)h->num_games * kTrackWords;
  int ctas = h->num_games < kInfoCtasPerSm * h->num_sms ? h->num_games : kInfoCtasPerSm * h->num_sms;
  uint32_t* ticket = h->tickets + (h->info_calls++ % (uint32_t)kOtherTickets);
  k_encode_infostate<<<ctas, 64, 0, (cudaStream_t)stream>>>(P, L, out, ticket);
  return launch_status();
}

int strat_history_get_boards(const strat_history* h, int64_t t, uint8_t* boards, void* stream) {
  if (h) chain_break(h->env);
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !boards) return STRAT_BAD_ARG;
  k_export<<<(h->num_games + 3) / 4, 128, 0, (cudaStream_t)stream>>>(h->num_games, L, boards);
  return launch_status();
}

int strat_history_transition(const strat_history* h, int64_t t, const int16_t** actions, const int8_t** reward,
                             const uint8_t** done) {
  if (h) chain_break(h->env);  // the caller is about to read the rows
  if (!h || t < 0 || t >= h->cur || t < h->cur - h->length) return STRAT_BAD_ARG;
  size_t off = (size_t)(t % h->length) * (size_t)h->num_games;
  if (actions) *actions = h->act + off;
  if (reward) *reward = h->rew + off;
  if (done) *done = h->done + off;
  return STRAT_OK;
}

int strat_history_info(const strat_history* h, int64_t t, int32_t* info, void* stream) {
  if (h) chain_break(h->env);
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !info || ((uintptr_t)info & 15) != 0) return STRAT_BAD_ARG;
  k_line_info<<<(h->num_games + 255) / 256, 256, 0, (cudaStream_t)stream>>>(h->num_games, L, info);
  return launch_status();
}

int strat_history_flags(const strat_history* h, int64_t t, uint8_t* two_square_applies, uint8_t* unknown,
                        int32_t* terminated_since, void* stream) {
  if (h) chain_break(h->env);
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || ((uintptr_t)unknown & 3) != 0) return STRAT_BAD_ARG;
  Params P = h->env ? h->env->P : h->P;
  P.movelog = nullptr;
  int n = h->num_games;
  if (two_square_applies || unknown)
    k_line_flags<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(P, L, two_square_applies, unknown);
  if (terminated_since) {
    int64_t oldest = h->cur - h->length > 0 ? h->cur - h->length : 0;  // oldest recorded step still in the ring
    int depth = (int)(t - oldest);
    k_terminated_since<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>(n, L, h->done, h->length, t, depth,
                                                                         terminated_since);
  }
  return launch_status();
}

int strat_history_restore(const strat_history* h, int64_t t, strat_env* env, void* stream) {
  if (h) chain_break(h->env);
  chain_break(env);
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !env || env->P.num_games != h->num_games) return STRAT_BAD_ARG;
  if (L != env->lines) {
    copy_elems<uint32_t>(L, env->lines, (size_t)h->num_games * kLineWords, (cudaStream_t)stream);
    // the chasing rule's memory travels back too: rebuilt from the ring's actions
    const Params& Ph = h->env ? h->env->P : h->P;
    if (env->P.movelog && t == h->cur && Ph.movelog)  // the live state of another environment: its log as it is
      copy_elems<uint16_t>(Ph.movelog, env->P.movelog, (size_t)h->num_games * kLogPlies, (cudaStream_t)stream);
    else if (env->P.movelog && Ph.chase_rule)
      hist_rebuild_logs(h, t, Ph.pin_log, env->P.movelog, (cudaStream_t)stream);
    else
      k_clear_logn<<<(h->num_games + 255) / 256, 256, 0, (cudaStream_t)stream>>>(h->num_games, env->lines);
    // the trackers of the state at t: from a tracked ring they travel back with it, otherwise they restart
    const size_t words = (size_t)h->num_games * kTrackWords;
    if (env->P.track && Ph.track && h->track)
      copy_elems<uint32_t>(t == h->cur ? Ph.track : h->track + (size_t)(t % h->length) * words, env->P.track, words,
                           (cudaStream_t)stream);
    else
      track_restart(env, (cudaStream_t)stream);
  }
  return launch_status();
}

// ---- search-shaped batch
int strat_determinise(const strat_env* roots, int32_t samples_per_root, uint64_t seed, strat_env* out, void* stream) {
  if (!roots || !out || samples_per_root <= 0 ||
      (int64_t)roots->P.num_games * samples_per_root != (int64_t)out->P.num_games)
    return STRAT_BAD_ARG;
  chain_break(roots);
  chain_break(out);
  k_determinise<<<batches(out->P.num_games), 32, 0, (cudaStream_t)stream>>>(
      out->P.num_games, samples_per_root, (uint32_t)seed, (uint32_t)(seed >> 32), out->P.game_base, roots->lines,
      out->lines, roots->P.movelog, out->P.movelog, out->err);
  track_restart(out, (cudaStream_t)stream);
  return launch_status();
}

int strat_search_expand(const strat_env* roots, int32_t rollouts, uint64_t seed, strat_env* out, void* stream) {
  if (!roots || !out || rollouts <= 0 || (int64_t)roots->P.num_games * rollouts != (int64_t)out->P.num_games ||
      out->P.auto_reset || out->hist || out->P.track)
    return STRAT_BAD_ARG;
  chain_break(roots);
  chain_break(out);
  auto kernel = roots->P.chase_rule ? k_search_expand<true> : k_search_expand<false>;
  kernel<<<batches(out->P.num_games), 32, 0, (cudaStream_t)stream>>>(roots->P, out->P, rollouts, (uint32_t)seed,
                                                                     (uint32_t)(seed >> 32), roots->lines, out->lines, out->err);
  return launch_status();
}

int strat_search_policy(const strat_env* roots, const strat_env* games, int32_t rollouts, const float* pi_theta,
                        float alpha, float beta, float* qhat, float* rho, float* pi_search, void* stream) {
  return strat_search_policy_values(roots, games, rollouts, pi_theta, nullptr, alpha, beta, qhat, rho, pi_search, stream);
}

int strat_search_policy_values(const strat_env* roots, const strat_env* games, int32_t rollouts, const float* pi_theta,
                               const float* values, float alpha, float beta, float* qhat, float* rho, float* pi_search,
                               void* stream) {
  if (!roots || !games || rollouts <= 0 || (int64_t)roots->P.num_games * rollouts != (int64_t)games->P.num_games ||
      !qhat || !rho || !pi_search || !(alpha + beta > 0.f))
    return STRAT_BAD_ARG;
  chain_break(roots);
  chain_break(games);
  auto kernel = roots->P.chase_rule ? k_search_policy<true> : k_search_policy<false>;
  kernel<<<roots->P.num_games, kPolicyThreads, 0, (cudaStream_t)stream>>>(roots->P, rollouts, roots->lines, games->lines,
                                                                         pi_theta, values, alpha, beta, qhat, rho, pi_search);
  return launch_status();
}

int strat_reduce_returns(const strat_env* games, const uint8_t* root_side, int32_t samples_per_root, int32_t* out,
                         void* stream) {
  if (!games || !root_side || !out || samples_per_root <= 0 || games->P.num_games % samples_per_root != 0)
    return STRAT_BAD_ARG;
  chain_break(games);
  int R = games->P.num_games / samples_per_root;
  k_reduce_returns<<<R, 256, 0, (cudaStream_t)stream>>>(games->lines, root_side, samples_per_root, out);
  return launch_status();
}

}  // extern "C"

// ---- strat_legal_mask_static: the legal-mask query for callers that cannot allocate (strat.h) ----
// The scratch of this one entry point is part of the library's device image instead of a caller's
// workspace: kStaticLineBytes of device lines (what k_import writes and k_legal_mask reads), then a
// 256-byte block whose first word is the error word k_import raises.  Every GPU that loads the
// library holds these 512.25 KB until the process exits.
//
// In HOST code the name `g_static_scratch` is only a handle for the symbol, not a device address
// (handing it to a kernel would fault, or quietly hit host memory on a system where the GPU can
// reach it).  The address on a given device comes from cudaGetSymbolAddress with that device
// current; static_scratch() asks once per device and remembers the answer.
namespace {
constexpr size_t kStaticLineBytes = (size_t)STRAT_STATIC_MAX_GAMES * STRAT_LINE_BYTES;
constexpr int kStaticMaxDevices = 64;
}  // namespace
static __device__ __align__(256) unsigned char g_static_scratch[kStaticLineBytes + 256];
namespace {
std::mutex g_static_mutex;
unsigned char* g_static_addr[kStaticMaxDevices];  // device address of g_static_scratch per device ordinal, once known

// Device address of the built-in scratch on the current device.  Looks it up on the first call
// for that device (no allocation: the array already exists in the loaded module).
int static_scratch(unsigned char** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return STRAT_CUDA_ERROR;
  if (dev < 0 || dev >= kStaticMaxDevices) return STRAT_BAD_ARG;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_addr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) return STRAT_CUDA_ERROR;
    g_static_addr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_static_addr[dev];
  return STRAT_OK;
}
}  // namespace

extern "C" int strat_legal_mask_static(const uint8_t* boards, int32_t num_games, int32_t two_square, uint32_t* mask,
                                       int32_t* status, void* stream) {
  if (!boards || !mask || num_games < 1) return STRAT_BAD_ARG;
  if (num_games > STRAT_STATIC_MAX_GAMES) return STRAT_TOO_LARGE;
  unsigned char* base = nullptr;
  int rc = static_scratch(&base);
  if (rc != STRAT_OK) return rc;
  uint32_t* lines = reinterpret_cast<uint32_t*>(base);
  int* err = reinterpret_cast<int*>(base + kStaticLineBytes);
  cudaStream_t s = (cudaStream_t)stream;
  // the array still holds the previous call's lines and error word: the lines of games [0, num_games)
  // are overwritten below and no kernel looks beyond them; the error word has to start at zero
  k_set_int<<<1, 1, 0, s>>>(err, 0);
  k_import<<<(num_games + 3) / 4, 128, 0, s>>>(num_games, boards, lines, err);
  strat_config c = {};
  c.num_games = num_games; c.two_square = two_square ? 1 : 0;
  const Params P = make_params(c);  // the mask depends on num_games and two_square only (no chasing rule: no move log)
  k_legal_mask<false><<<batches(num_games), 32, 0, s>>>(P, lines, mask);
  if (status) k_copy<int><<<1, 1, 0, s>>>(err, status, (size_t)1);
  return launch_status();
}
