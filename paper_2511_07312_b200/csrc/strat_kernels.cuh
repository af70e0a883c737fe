// strat_kernels.cuh - single-purpose kernels: reset, import/export, legal mask, sampler, step, encode, on-chip rollouts, replay ring, determinise, reductions
// Part of libstrat.so (one translation unit: strat.cu includes these in order).
#pragma once

namespace {
using namespace strat;

// Warp-cooperative auto-reset of the games flagged in `rs` (bit = lane = game of the batch):
// the result equals setup_game (C2: descending Fisher-Yates over the listed multiset, one
// Philox stream per side).  The 2 x 10 Philox blocks of a game are drawn by 20 lanes at once,
// the sequential swaps run on a 40-byte row of shared memory, and the bit planes are built
// with warp ballots (lane = cell of a 32-cell word).  Attempt 0 of both sides is produced
// here; a side that fails the mobility test (R#5, p ~ 2e-6) sends that game through the
// thread-per-game setup_game, which redraws.  `scratch` >= 3,200 words.
__device__ __forceinline__ void coop_setup(const Params& P, int first, uint32_t rs, Game& g, uint32_t* scratch, int lane) {
  const uint32_t full = 0xffffffffu;
  uint32_t* sD = scratch;                                        // [32][2][40] draws
  uint8_t* sA = reinterpret_cast<uint8_t*>(scratch + 32 * 80);  // [32][2][40] piece types
  for (uint32_t m = rs; m; m &= m - 1) {
    int owner = __ffs((int)m) - 1;
    uint32_t epoch = __shfl_sync(full, g.epoch, owner);
    if (P.pool) {  // custom setups (R#30): lanes 0/1 draw the two pool entries, all lanes copy the 80 types
      uint32_t idx = 0;
      if (lane < 2) {
        uint32_t o[4];
        philox(P.game_base + (uint32_t)(first + owner), epoch, 0u, lane ? TAG_SETUP_BLUE : TAG_SETUP_RED, P.key0, P.key1, o);
        idx = bounded(o[0], (uint32_t)P.pool_size);
      }
      uint32_t i0 = __shfl_sync(full, idx, 0), i1 = __shfl_sync(full, idx, 1);
      for (int i = lane; i < 80; i += 32)
        sA[owner * 80 + i] = i < 40 ? P.pool[(size_t)i0 * 40 + i] : P.pool[((size_t)P.pool_size + i1) * 40 + (i - 40)];
      continue;
    }
    if (lane < 20) {
      int side = lane >= 10 ? 1 : 0, blk = lane - 10 * side;
      uint32_t o[4];
      philox(P.game_base + (uint32_t)(first + owner), epoch, (uint32_t)blk, side ? TAG_SETUP_BLUE : TAG_SETUP_RED,
             P.key0, P.key1, o);
      uint32_t* d = sD + owner * 80 + side * 40 + 4 * blk;
      d[0] = o[0]; d[1] = o[1]; d[2] = o[2]; d[3] = o[3];
    }
    for (int i = lane; i < 80; i += 32) sA[owner * 80 + i] = (uint8_t)multiset_type(P.variant, i < 40 ? i : i - 40);
  }
  __syncwarp();
  if (((rs >> lane) & 1u) && !P.pool) {
    for (int side = 0; side < 2; ++side) {
      uint8_t* A = sA + lane * 80 + side * 40;
      const uint32_t* D = sD + lane * 80 + side * 40;
      for (int i = 39; i >= 1; --i) {
        int j = (int)bounded(D[39 - i], (uint32_t)(i + 1));
        uint8_t t = A[i]; A[i] = A[j]; A[j] = t;
      }
    }
  }
  __syncwarp();
  for (uint32_t m = rs; m; m &= m - 1) {
    int owner = __ffs((int)m) - 1;
    const uint8_t* A = sA + owner * 80;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      int c = 32 * w + lane;
      uint32_t t = c < 40 ? A[c] : (c >= 60 && c < 100) ? A[c - 20] : 0u;
      uint32_t b0 = __ballot_sync(full, t & 1u), b1 = __ballot_sync(full, t & 2u), b2 = __ballot_sync(full, t & 4u),
               b3 = __ballot_sync(full, t & 8u), bo = __ballot_sync(full, t != 0u && c >= 60);
      if (lane == owner) { g.t0.w[w] = b0; g.t1.w[w] = b1; g.t2.w[w] = b2; g.t3.w[w] = b3; g.own.w[w] = bo; }
    }
  }
  if ((rs >> lane) & 1u) {
    g.mvd = g.rev = bb_zero();
    hist_clear(g);
    g.done = 0; g.reason = 0; g.result = 0; g.ply = 0; g.battleless = 0; g.chase = 0; g.logn = 0;
    if (!P.pool && (!side_can_ever_move(g, 0) || !side_can_ever_move(g, 1))) setup_game(P, (uint32_t)(first + lane), g);
  }
  __syncwarp();
}

// Warp-cooperative (re)start of the S2 trackers of the games flagged in `rs` (bit = lane = game of
// the batch), whose new state the flagged lanes hold in g: the 100 cell records by all lanes
// (16 bytes each: start square = the square itself, no history), the rest by the game's lane.
__device__ __forceinline__ void coop_track_start(const Params& P, int first, uint32_t rs, const Game& g, int lane) {
  for (uint32_t m = rs; m; m &= m - 1) {
    int owner = __ffs((int)m) - 1;
    uint4* blk = reinterpret_cast<uint4*>(P.track + (size_t)(first + owner) * kTrackWords);
    for (int c = lane; c < 100; c += 32) __stcg(blk + c, make_uint4((uint32_t)c << 22, 0u, 0u, 0u));
  }
  if ((rs >> lane) & 1u) track_start_tail(game_track(P, (uint32_t)(first + lane)), g);
}

// Trackers of every game (re)started from its current line: after a reset, an import, a restore.
// One warp per game.
__global__ void __launch_bounds__(128) k_track_start(Params P, const uint32_t* __restrict__ lines) {
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int gi = blockIdx.x * 4 + warp;
  if (gi >= P.num_games) return;
  Game g;
  load_game_global(lines, gi, g, nullptr);  // every lane reads the same line
  uint4* blk = reinterpret_cast<uint4*>(P.track + (size_t)gi * kTrackWords);
  for (int c = lane; c < 100; c += 32) __stcg(blk + c, make_uint4((uint32_t)c << 22, 0u, 0u, 0u));
  if (lane == 0) track_start_tail(game_track(P, (uint32_t)gi), g);
}

// ------------------------------------------------------------------ kernels
__global__ void __launch_bounds__(32) k_reset(Params P, uint32_t* __restrict__ lines) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, P.num_games - first);
  if (lane < ng) {
    Game g; g.epoch = 0;
    setup_game(P, (uint32_t)(first + lane), g);
    write_game(s_state, lane, g);
  }
  __syncwarp();
  store_lines(lines, first, ng, s_state, lane);
}

// canonical uint8[N][128] -> device lines.  One warp per game; the seven bit planes are
// packed with warp ballots (lane = cell within a 32-cell word).
// A side with more than kMaxScouts Scouts (no variant of the game has that) is refused with BAD_STATE:
// the mask-free sampler of the on-chip rollouts keeps a list of at most that many (count_actions).
__global__ void __launch_bounds__(128) k_import(int n, const uint8_t* __restrict__ canon, uint32_t* __restrict__ lines,
                                                int* __restrict__ err) {
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int g = blockIdx.x * 4 + warp;
  if (g >= n) return;
  uint32_t cw = reinterpret_cast<const uint32_t*>(canon + (size_t)g * 128)[lane];  // bytes 4l..4l+3
  uint32_t mine = 0;
  int scouts_red = 0, scouts_blue = 0;
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    int cell = 32 * r + lane;
    uint32_t w = __shfl_sync(0xffffffffu, cw, (cell >> 2) & 31);
    uint32_t b = cell < 100 ? (w >> (8 * (cell & 3))) & 0xFFu : 0u;
    uint32_t t = b & 15u;
    bool piece = t >= 1 && t <= 12;
    scouts_red += __popc(__ballot_sync(0xffffffffu, t == (uint32_t)T_SCOUT && !(b & 16u)));
    scouts_blue += __popc(__ballot_sync(0xffffffffu, t == (uint32_t)T_SCOUT && (b & 16u)));
#pragma unroll
    for (int p = 0; p < 7; ++p) {
      bool bit = p < 4 ? (piece && ((t >> p) & 1u)) : (piece && ((b >> p) & 1u));  // p=4 owner(bit4),5 moved,6 revealed
      uint32_t word = __ballot_sync(0xffffffffu, bit);
      if (lane == 4 * p + r) mine = word;
    }
  }
  // meta: history pairs ride in the spare bits of words 3,7,11,15; flags in word 19
  uint32_t hw = __shfl_sync(0xffffffffu, cw, 25 + (lane >> 2));  // canonical bytes 100+4p.. for lane 4p+3
  uint32_t fw = __shfl_sync(0xffffffffu, cw, 30);
  if ((lane & 3) == 3 && lane < 16) {
    uint32_t f0 = hw & 0xFFu, t0 = (hw >> 8) & 0xFFu, f1 = (hw >> 16) & 0xFFu, t1 = hw >> 24;
    uint32_t e0 = f0 == 0xFFu ? kHistNone : (f0 | (t0 << 7));
    uint32_t e1 = f1 == 0xFFu ? kHistNone : (f1 | (t1 << 7));
    mine |= (e0 | (e1 << 14)) << 4;
  }
  if (lane == 19) {
    uint32_t fl = fw & 0xFFu;
    int32_t res = (int32_t)(int8_t)((fw >> 8) & 0xFFu);
    mine |= ((fl & 1u) | (((fl >> 2) & 7u) << 1) | ((uint32_t)(res + 1) << 4)) << 4;
  }
  uint32_t w29 = __shfl_sync(0xffffffffu, cw, 29), w31 = __shfl_sync(0xffffffffu, cw, 31);
  if (lane == 28) mine = w29;  // ply | battleless<<16 : same bytes as canonical 116..119
  if (lane == 29) mine = w31;  // epoch
  if (lane == 30) mine = fw >> 16;  // chase ages: canonical bytes 122..123
  if (lane == 31) mine = 0;
  lines[(size_t)g * kLineWords + lane] = mine;
  if (lane == 0 && (scouts_red > kMaxScouts || scouts_blue > kMaxScouts)) raise_error(err, STRAT_BAD_STATE);
}

// device lines -> canonical.  One warp per game; lane l < 25 assembles cells 4l..4l+3.
__global__ void __launch_bounds__(128) k_export(int n, const uint32_t* __restrict__ lines, uint8_t* __restrict__ canon) {
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int g = blockIdx.x * 4 + warp;
  if (g >= n) return;
  uint32_t lw = lines[(size_t)g * kLineWords + lane];
  uint32_t out = 0;
  int r = (lane >> 3) & 3, sh = 4 * (lane & 7);  // cells 4l..4l+3 sit in word r of each plane, bits sh..sh+3
  uint32_t nib[7];
#pragma unroll
  for (int p = 0; p < 7; ++p) nib[p] = (__shfl_sync(0xffffffffu, lw, 4 * p + r) >> sh) & 0xFu;
  if (lane < 25) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      uint32_t b = 0;
#pragma unroll
      for (int p = 0; p < 7; ++p) b |= ((nib[p] >> k) & 1u) << p;
      int cell = 4 * lane + k;
      if (is_lake_cell(cell)) b = 15;
      out |= b << (8 * k);
    }
  }
  uint32_t hw = __shfl_sync(0xffffffffu, lw, 4 * ((lane - 25) & 3) + 3) >> 4;   // history pair for lanes 25..28
  uint32_t fw = __shfl_sync(0xffffffffu, lw, 19) >> 4;
  uint32_t w28 = __shfl_sync(0xffffffffu, lw, 28), w29 = __shfl_sync(0xffffffffu, lw, 29);
  uint32_t w30 = __shfl_sync(0xffffffffu, lw, 30);
  if (lane >= 25 && lane < 29) {
    uint32_t e0 = hw & 0x3FFFu, e1 = (hw >> 14) & 0x3FFFu;
    uint32_t b0 = e0 == kHistNone ? 0xFFFFu : ((e0 & 127u) | ((e0 >> 7) << 8));
    uint32_t b1 = e1 == kHistNone ? 0xFFFFu : ((e1 & 127u) | ((e1 >> 7) << 8));
    out = b0 | (b1 << 16);
  }
  if (lane == 29) out = w28;
  if (lane == 30) {
    uint32_t done = fw & 1u, reason = (fw >> 1) & 7u;
    int32_t res = (int32_t)((fw >> 4) & 3u) - 1;
    out = (done | (reason << 2)) | (((uint32_t)res & 0xFFu) << 8) | ((w30 & 0xFFFFu) << 16);
  }
  if (lane == 31) out = w29;
  reinterpret_cast<uint32_t*>(canon + (size_t)g * 128)[lane] = out;
}

template <bool kChase>
__global__ void __launch_bounds__(32) k_legal_mask(Params P, const uint32_t* __restrict__ lines, uint32_t* __restrict__ mask) {
  __shared__ __align__(16) uint32_t s_mask[kBatch * kMaskWords];  // 14.5 KB: 15 one-warp CTAs per SM, one wave at 65,536 games
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, P.num_games - first);
  zero_smem16(s_mask, kMaskBytes, lane);
  __syncwarp();
  if (lane < ng) {
    Game g; load_game_global(lines, first + lane, g, nullptr);
    int cnt[4];
    if (!g.done) legal_mask_row(g, g.ply & 1u, rules_of<kChase>(P), s_mask + lane * kMaskWords, cnt,
                                kChase ? game_log(P, (uint32_t)(first + lane)) : nullptr);
  }
  __syncwarp();
  store_mask(mask, first, ng, s_mask, lane);
}

// One warp per game: lanes load the 113 mask words coalesced, count with popc, locate the
// r-th set bit with warp-shuffle prefix sums.
__global__ void __launch_bounds__(128) k_sample_uniform(Params P, const uint32_t* __restrict__ lines,
                                                        const uint32_t* __restrict__ mask, int16_t* __restrict__ actions) {
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int g = blockIdx.x * 4 + warp;
  if (g >= P.num_games) return;
  const uint32_t* row = mask + (size_t)g * kMaskWords;
  uint32_t w[4]; int cnt[4], incl[4], tot[4];
  int n = 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    int wi = 32 * k + lane;
    w[k] = wi < kMaskWords ? row[wi] : 0u;
    cnt[k] = __popc(w[k]);
    int x = cnt[k];
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, off); if (lane >= off) x += y; }
    incl[k] = x;
    tot[k] = __shfl_sync(0xffffffffu, x, 31);
    n += tot[k];
  }
  int action = -1;
  if (n > 0) {
    uint32_t meta = lane < 2 ? lines[(size_t)g * kLineWords + 28 + lane] : 0u;
    uint32_t w28 = __shfl_sync(0xffffffffu, meta, 0), epoch = __shfl_sync(0xffffffffu, meta, 1);
    uint32_t o[4];
    philox(P.game_base + (uint32_t)g, epoch, w28 & 0xFFFFu, TAG_ACTION, P.key0, P.key1, o);
    int r = (int)bounded(o[0], (uint32_t)n);
    int base = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      int excl = base + incl[k] - cnt[k];  // set bits before this lane's word
      bool mine = r >= excl && r < excl + cnt[k];
      uint32_t owner = __ballot_sync(0xffffffffu, mine);
      int a = (32 * k + lane) * 32 + (mine ? nth_set_bit(w[k], r - excl) : 0);
      if (owner) action = __shfl_sync(0xffffffffu, a, __ffs((int)owner) - 1);
      base += tot[k];
    }
  }
  if (lane == 0) actions[g] = (int16_t)action;
}

template <bool kChase, bool kTrack>
__global__ void __launch_bounds__(32) k_step(Params P, uint32_t* __restrict__ lines, const int16_t* __restrict__ actions,
                                             int8_t* __restrict__ reward, uint8_t* __restrict__ done, int* __restrict__ err,
                                             HistSlot hs) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  __shared__ __align__(16) uint32_t s_scratch[3200];  // warp-cooperative auto-reset
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, P.num_games - first);
  load_lines(lines, first, ng, s_state, lane);
  if (hs.lines) store_lines(hs.lines, first, ng, s_state, lane);  // the state this step starts from
  __syncwarp();
  Game g;
  bool reset_me = false;
  if (lane < ng) {
    read_game(s_state, lane, g);
    int a = (int)actions[first + lane];
    StepOut o = step_game<true, true, kChase, kTrack>(P, (uint32_t)(first + lane), g, a);
    if (o.illegal) raise_error(err, STRAT_ILLEGAL_ACTION);
    reward[first + lane] = (int8_t)o.reward;
    done[first + lane] = (uint8_t)o.done;
    if (hs.lines) { hs.act[first + lane] = (int16_t)a; hs.rew[first + lane] = (int8_t)o.reward; hs.done[first + lane] = (uint8_t)o.done; }
    reset_me = o.needs_reset;
  }
  uint32_t rs = __ballot_sync(0xffffffffu, reset_me);
  if (rs && P.pin) { if (reset_me) reset_game(P, (uint32_t)(first + lane), g); __syncwarp(); }  // owner lanes' tracker writes first
  else if (rs) coop_setup(P, first, rs, g, s_scratch, lane);
  if (kTrack && rs && P.track) coop_track_start(P, first, rs, g, lane);
  if (lane < ng) write_game(s_state, lane, g);
  __syncwarp();
  store_lines(lines, first, ng, s_state, lane);
}

__global__ void __launch_bounds__(32) k_encode_obs(Params P, const uint32_t* __restrict__ lines, uint16_t* __restrict__ obs) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  __shared__ __align__(16) uint32_t s_bits[kBatch * kBitsRowWords];  // 17,792 B
  __shared__ __align__(16) uint4 s_lut[256];
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, P.num_games - first);
  fill_lut(s_lut, lane, 32);
  load_lines(lines, first, ng, s_state, lane);
  if (lane < ng) {
    Game g; read_game(s_state, lane, g);
    encode_bits(g, s_bits + lane * kBitsRowWords);
  }
  __syncwarp();
  expand_obs(obs, first, ng, s_bits, s_lut, lane);
}

// `plies` plies of uniform-random legal play with the board in registers.  The 3600-bit mask is
// never built: the r-th legal action is found from the move bitboards (count_actions /
// choose_action).  All 32 lanes run the ply loop together and meet at a __syncwarp after every
// phase whose length differs from game to game (the Scout ray loops above all), so that the
// selection and the step run with the warp converged instead of once per group of lanes.
constexpr int kScoutScratch = 17;  // 16 words per game, odd stride
#ifndef STRAT_ROLLOUT_MIN_CTAS
#define STRAT_ROLLOUT_MIN_CTAS 16
#endif
template <bool kChase>
__global__ void __launch_bounds__(32, STRAT_ROLLOUT_MIN_CTAS) k_rollout_uniform(Params P, uint32_t* __restrict__ lines, int plies, int* __restrict__ err) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  __shared__ uint32_t s_scouts[kBatch * kScoutScratch];
  const uint32_t full = 0xffffffffu;
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, P.num_games - first);
  load_lines(lines, first, ng, s_state, lane);
  Game g;
  bool live = lane < ng;  // still playing: a frozen game (no auto-reset) or a fault ends the lane's rollout
  if (live) read_game(s_state, lane, g);
  uint32_t* scouts = s_scouts + lane * kScoutScratch;
  const uint16_t* glog = kChase ? game_log(P, (uint32_t)(first + lane)) : nullptr;
  // Without the chasing rule "the opponent has no legal move" is not tested after a move: the next ply's move
  // generation says so (no action at all), and the game is closed then as the step would have closed it
  // (finish_no_move).  One move generation per ply instead of two; the states after every ply are the same.
  constexpr bool kDefer = !kChase;
  bool pending = false;
  for (int t = 0; t < plies; ++t) {
    live = live && !g.done;
    if (!__any_sync(full, live)) break;
    ActionSet A;
    uint32_t u = 0;
    if (live) {
      count_actions(g, g.ply & 1u, rules_of<kChase>(P), scouts, A);
      if (kDefer && pending && A.n == 0) {  // rare: the previous ply ended the game
        finish_no_move<kChase>(P, (uint32_t)(first + lane), g);
        live = !g.done;
        if (live) count_actions(g, g.ply & 1u, rules_of<kChase>(P), scouts, A);  // auto-reset: a fresh game
      }
      if (live) u = action_draw(P, (uint32_t)(first + lane), g);
    }
    pending = false;
    const int kmax = (int)__reduce_max_sync(full, live ? (unsigned)A.ns : 0u);  // also reconverges the warp
    int a = -1;
    if (live) a = choose_action(g, g.ply & 1u, rules_of<kChase>(P), A, u, scouts, glog, kmax);
    __syncwarp();
    if (live) {
      StepOut o = step_game<false, false, kChase, false, kDefer>(P, (uint32_t)(first + lane), g, a);
      pending = o.nomove_pending;
      if (o.illegal) {
        raise_error(err, STRAT_ILLEGAL_ACTION);
        live = false;
      }
    }
    __syncwarp();
  }
  if (kDefer && pending && live && !g.done && !has_legal_move(g, g.ply & 1u, rules_of<kChase>(P)))
    finish_no_move<kChase>(P, (uint32_t)(first + lane), g);  // the test the last ply left open
  if (lane < ng) write_game(s_state, lane, g);
  __syncwarp();
  store_lines(lines, first, ng, s_state, lane);
}

// ---- replay ring
template <typename T>
__global__ void k_copy(const T* __restrict__ src, T* __restrict__ dst, size_t count) {
  size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += stride) dst[i] = src[i];
}
// Ring position p (index into the capacity-sized ring) -> push-order number -> rows.
struct RingMap { uint32_t filled; uint64_t capacity, base /* oldest live record's number */, rows, obs_rows; };
// A gather that sits between two fused steps of a self-play loop without separating them
// (strat_replay_sample_chained).  It is launched with the programmatic-serialisation attribute and lets
// the NEXT fused step start at once (launch_dependents).  In the regular loop (step, commit, gather,
// step, ...) it does not wait for the step before it as a whole either: a record pushed by the step
// with version v, game g, is complete once that step has published batch g/32 (f_state >= v: mask,
// action, reward, done) and the step before it the batch's observation (f_obs >= v - 1), so only the
// few records of the newest blocks wait, each for its own batch, and the gather runs alongside the
// step that feeds it.  Records of steps up to `vouch` are known to be complete (an earlier gather
// waited for that grid).  Otherwise (use_flags = 0) it waits for everything before it in the stream.
// The CTA that finishes last publishes the gather's number in *done_flag: the next gather waits for
// it before it overwrites the minibatch, the fused step after the next one before it overwrites rows
// this gather may still read.
struct GatherChain {
  uint32_t* counter; uint32_t* done_flag; uint32_t number;
  int use_flags; const uint32_t* f_state; const uint32_t* f_obs;
  uint32_t newest_version, vouch; uint32_t block; uint64_t newest_block;
};
// Returns false (nothing copied) if the record's producer has not published it yet and may_defer is set.
__device__ __forceinline__ bool replay_gather_one(int j, int lane, uint32_t k0, uint32_t k1, uint32_t d0, uint32_t d1,
                                                  const RingMap& map, const uint16_t* __restrict__ r_obs,
                                                  const uint32_t* __restrict__ r_mask, const int16_t* __restrict__ r_act,
                                                  const int8_t* __restrict__ r_rew, const uint8_t* __restrict__ r_done,
                                                  uint16_t* __restrict__ obs, uint32_t* __restrict__ mask,
                                                  int16_t* __restrict__ act, int8_t* __restrict__ rew, uint8_t* __restrict__ done,
                                                  const GatherChain& chain, bool may_defer = false) {
  uint32_t o[4];
  philox((uint32_t)(j >> 2), d0, d1, TAG_SAMPLE, k0, k1, o);
  uint32_t u = (j & 3) == 0 ? o[0] : (j & 3) == 1 ? o[1] : (j & 3) == 2 ? o[2] : o[3];
  uint64_t idx = bounded(u, map.filled);
  uint64_t seq = map.base + (idx + map.capacity - map.base % map.capacity) % map.capacity;
  size_t p = (size_t)(seq % map.rows), po = (size_t)(seq % map.obs_rows);
  if (chain.use_flags) {
    const uint64_t blk = seq / chain.block;
    const uint32_t need = chain.newest_version - (uint32_t)(chain.newest_block - blk);  // version of the step that pushed it
    if ((int32_t)(need - chain.vouch) > 0) {
      const uint32_t b = (uint32_t)(seq - blk * chain.block) / (uint32_t)kBatch;
      int ready = 1;
      if (lane == 0) {
        if (may_defer) {
          ready = (int32_t)(ld_acquire(chain.f_state + b) - need) >= 0 && (int32_t)(ld_acquire(chain.f_obs + b) - (need - 1u)) >= 0;
        } else {
          while ((int32_t)(ld_acquire(chain.f_state + b) - need) < 0) __nanosleep(64);
          while ((int32_t)(ld_acquire(chain.f_obs + b) - (need - 1u)) < 0) __nanosleep(64);
        }
      }
      ready = __shfl_sync(0xffffffffu, ready, 0);
      __syncwarp();  // the other lanes' loads of the record come after lane 0's acquire (a shuffle alone orders no memory)
      if (!ready) return false;
    }
  }
  // all loads of the record are issued before the first store: a warp that copied chunk by chunk would
  // pay one trip to HBM (microseconds while the fused steps saturate it) for every 512 bytes
  uint32_t mw[4];
  if (mask) {
#pragma unroll
    for (int k = 0; k < 4; ++k) mw[k] = 32 * k + lane < kMaskWords ? __ldcg(r_mask + p * kMaskWords + 32 * k + lane) : 0u;
  }
  if (obs) {
    const uint4* s = reinterpret_cast<const uint4*>(r_obs + po * STRAT_OBS_ELEMS);
    uint4* d = reinterpret_cast<uint4*>(obs + (size_t)j * STRAT_OBS_ELEMS);
    uint4 v[6];
#pragma unroll
    for (int h = 0; h < 3; ++h) {  // 550 chunks = 3 x 6 x 32 - 26
#pragma unroll
      for (int k = 0; k < 6; ++k) {
        int q = 32 * (6 * h + k) + lane;
        if (q < kObsChunks) v[k] = __ldcs(s + q);
      }
#pragma unroll
      for (int k = 0; k < 6; ++k) {
        int q = 32 * (6 * h + k) + lane;
        if (q < kObsChunks) __stcs(d + q, v[k]);  // evict-first: normal-priority lines between the streaming output
                                                    // of the fused steps get written back out of order (measured)
      }
    }
  }
  if (mask) {
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (32 * k + lane < kMaskWords) mask[(size_t)j * kMaskWords + 32 * k + lane] = mw[k];
  }
  if (lane == 0) {
    if (act) act[j] = __ldcg(r_act + p);
    if (rew) rew[j] = __ldcg(r_rew + p);
    if (done) done[j] = __ldcg(r_done + p);
  }
  return true;
}

// one warp per batch element: draw the record index, gather the record.
template <bool kChained>
__global__ void __launch_bounds__(128, 8) k_replay_sample(uint32_t k0, uint32_t k1, uint32_t d0, uint32_t d1, int batch,
                                                          RingMap map, const uint16_t* __restrict__ r_obs,
                                                          const uint32_t* __restrict__ r_mask, const int16_t* __restrict__ r_act,
                                                          const int8_t* __restrict__ r_rew, const uint8_t* __restrict__ r_done,
                                                          uint16_t* __restrict__ obs, uint32_t* __restrict__ mask,
                                                          int16_t* __restrict__ act, int8_t* __restrict__ rew, uint8_t* __restrict__ done,
                                                          GatherChain chain) {
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (kChained) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (!chain.use_flags) asm volatile("griddepcontrol.wait;" ::: "memory");
    if (threadIdx.x == 0)  // the minibatch buffers are the previous gather's too
      while ((int32_t)(ld_acquire(chain.done_flag) - (chain.number - 1u)) < 0) __nanosleep(64);
    __syncthreads();
    // records whose producer (the fused step running alongside) has not published them yet are taken
    // last, so that what is left to do when that step ends is one record's copy, not a warp's whole share
    uint32_t deferred = 0u;
    int slot = 0;
    for (int j = blockIdx.x * 4 + warp; j < batch; j += gridDim.x * 4, ++slot)
      if (!replay_gather_one(j, lane, k0, k1, d0, d1, map, r_obs, r_mask, r_act, r_rew, r_done, obs, mask, act, rew, done,
                             chain, slot < 32))
        deferred |= 1u << slot;
    slot = 0;
    for (int j = blockIdx.x * 4 + warp; j < batch && deferred; j += gridDim.x * 4, ++slot)
      if ((deferred >> slot) & 1u) {
        deferred &= ~(1u << slot);
        replay_gather_one(j, lane, k0, k1, d0, d1, map, r_obs, r_mask, r_act, r_rew, r_done, obs, mask, act, rew, done, chain);
      }
    __syncthreads();
    if (threadIdx.x == 0) {
      __threadfence();
      uint32_t* counter = chain.counter + (chain.number & 1u);  // consecutive gathers never overlap (the wait above)
      if (atomicAdd(counter, 1u) == gridDim.x - 1u) {  // the last CTA: the whole minibatch is out
        *counter = 0u;
        __threadfence();
        atomicMax(chain.done_flag, chain.number);
      }
    }
    return;
  }
  int j = blockIdx.x * 4 + warp;
  if (j >= batch) return;
  replay_gather_one(j, lane, k0, k1, d0, d1, map, r_obs, r_mask, r_act, r_rew, r_done, obs, mask, act, rew, done, chain);
}

// ---- search-shaped batch
__global__ void __launch_bounds__(32) k_determinise(int num_out, int samples_per_root, uint32_t k0, uint32_t k1, uint32_t out_base,
                                                    const uint32_t* __restrict__ roots, uint32_t* __restrict__ out,
                                                    const uint16_t* __restrict__ root_logs, uint16_t* __restrict__ out_logs,
                                                    int* __restrict__ err) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, num_out - first);
  const bool keep_log = root_logs && out_logs;  // both environments run the chasing rule: its memory is copied too
  if (lane < ng) {
    int G = first + lane, r = G / samples_per_root;
    if (keep_log) copy_game_log(root_logs + (size_t)r * kLogPlies, out_logs + (size_t)G * kLogPlies);
    uint32_t W[32];
    const uint4* p = reinterpret_cast<const uint4*>(roots + (size_t)r * kLineWords);
#pragma unroll
    for (int k = 0; k < 8; ++k) { uint4 v = __ldg(p + k); W[4 * k] = v.x; W[4 * k + 1] = v.y; W[4 * k + 2] = v.z; W[4 * k + 3] = v.w; }
    Game root, g;
    unpack_line(W, root);
    if (!determinise_game(root, k0, k1, out_base + (uint32_t)G, keep_log, g)) raise_error(err, STRAT_BAD_STATE);
    write_game(s_state, lane, g);
  }
  __syncwarp();
  store_lines(out, first, ng, s_state, lane);
}

__global__ void __launch_bounds__(256) k_reduce_returns(const uint32_t* __restrict__ lines, const uint8_t* __restrict__ root_side,
                                                        int samples_per_root, int32_t* __restrict__ out) {
  __shared__ int s_sum[8], s_win[8], s_loss[8];
  int r = blockIdx.x;
  int sign = root_side[r] == 0 ? 1 : -1;
  int sum = 0, win = 0, loss = 0;
  for (int s = threadIdx.x; s < samples_per_root; s += blockDim.x) {
    uint32_t f = lines[((size_t)r * samples_per_root + s) * kLineWords + 19] >> 4;
    int ret = (f & 1u) ? ((int)((f >> 4) & 3u) - 1) * sign : 0;
    sum += ret; win += ret > 0; loss += ret < 0;
  }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) {
    sum += __shfl_down_sync(0xffffffffu, sum, off);
    win += __shfl_down_sync(0xffffffffu, win, off);
    loss += __shfl_down_sync(0xffffffffu, loss, off);
  }
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) { s_sum[warp] = sum; s_win[warp] = win; s_loss[warp] = loss; }
  __syncthreads();
  if (threadIdx.x == 0) {
    int a = 0, b = 0, c = 0;
    for (int k = 0; k < 8; ++k) { a += s_sum[k]; b += s_win[k]; c += s_loss[k]; }
    out[3 * r] = a; out[3 * r + 1] = b; out[3 * r + 2] = c;
  }
}

// Scalar queries of Table S1 from the state lines of one time step.
__global__ void __launch_bounds__(256) k_line_info(int n, const uint32_t* __restrict__ lines, int32_t* __restrict__ info) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  const uint32_t* L = lines + (size_t)g * kLineWords;
  uint32_t w28 = L[28], f = L[19] >> 4;
  uint32_t ply = w28 & 0xFFFFu, done = f & 1u, reason = (f >> 1) & 7u;
  int4 v = make_int4((int)(ply & 1u), (int)ply, (int)(w28 >> 16), (int)(done | (reason << 2)));
  reinterpret_cast<int4*>(info)[g] = v;
}

// ComputeTwoSquareRuleApplies and ComputeIsUnknownPiece of one time step.
// two_square[g] = 1 iff the two-square rule takes at least one move away from the acting player
// (the shortest banned distance would be legal without the rule; longer ones follow, R#6);
// unknown[g][c] = 1 iff square c holds a piece of the opponent whose type the acting player has
// not seen.  Thread per game; either output may be null.
__global__ void __launch_bounds__(128) k_line_flags(Params P, const uint32_t* __restrict__ lines,
                                                    uint8_t* __restrict__ two_square, uint8_t* __restrict__ unknown) {
  int gi = blockIdx.x * blockDim.x + threadIdx.x;
  if (gi >= P.num_games) return;
  Game g;
  load_game_global(lines, gi, g, nullptr);
  int side = g.ply & 1u;
  if (two_square) {
    uint8_t applies = 0;
    if (!g.done && P.two_square) {
      Ban b = two_square_ban(g, side, 1);
      if (b.from >= 0 && b.k <= 9) {
        Moves m; single_step_moves(g, side, 0, m);  // the moves without the rule
        applies = move_in_moves(m, b.from * 36 + b.dir * 9 + b.k - 1) ? 1 : 0;
      }
    }
    two_square[gi] = applies;
  }
  if (unknown) {
    BB occ = occupied(g);
    BB hidden = bb_andn(bb_andn(occ, owned_by(g, occ, side)), g.rev);
    uint32_t* out = reinterpret_cast<uint32_t*>(unknown + (size_t)gi * 100);  // 100 B per game: 4-B aligned
#pragma unroll 5
    for (int c4 = 0; c4 < 25; ++c4) {
      uint32_t nib = (bb_word(hidden, (4 * c4) >> 5) >> ((4 * c4) & 31)) & 0xFu;  // cells 4c4..4c4+3 never straddle a word
      out[c4] = (nib & 1u) | ((nib & 2u) << 7) | ((nib & 4u) << 14) | ((nib & 8u) << 21);
    }
  }
}

// GetTerminatedSince: for a game that is finished at time step t, the number of
// steps since the action that ended it = the run of consecutive steps t-1, t-2, ... whose done
// byte has bit 0 set (a frozen game keeps reporting it, R#15), looked up in the ring's done
// arrays; 0 for a live game.  `depth` = how many steps before t are still in the ring.
__global__ void __launch_bounds__(256) k_terminated_since(int n, const uint32_t* __restrict__ lines_t,
                                                          const uint8_t* __restrict__ ring_done, int length, int64_t t,
                                                          int depth, int32_t* __restrict__ out) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  int since = 0;
  if ((lines_t[(size_t)g * kLineWords + 19] >> 4) & 1u) {
    for (int j = 1; j <= depth; ++j) {
      size_t slot = (size_t)((t - j) % length);
      if (!(ring_done[slot * (size_t)n + g] & 1u)) break;
      since = j;
    }
  }
  out[g] = since;
}

// Validates a custom setup pool (R#30): type codes 0..12, at most kMaxScouts Scouts and a side that
// can move.  One thread per setup; raises BAD_ARG on the environment's sticky error word.
__global__ void __launch_bounds__(128) k_check_pool(const uint8_t* __restrict__ pool, int K, int* __restrict__ err) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 2 * K) return;
  int side = i >= K ? 1 : 0;
  const uint8_t* A = pool + (size_t)i * 40;
  Game g;
  g.t0 = g.t1 = g.t2 = g.t3 = g.own = g.mvd = g.rev = bb_zero();
  bool ok = true;
  int scouts = 0;
  for (int k = 0; k < 40; ++k) {
    if (A[k] > 12) ok = false;
    else if (A[k]) put_piece(g, (side ? 60 : 0) + k, A[k], side);
    scouts += A[k] == T_SCOUT ? 1 : 0;
  }
  if (!ok || scouts > kMaxScouts || !side_can_ever_move(g, side)) raise_error(err, STRAT_BAD_ARG);
}

// A state copied in from elsewhere (history ring) has no move log here: it remembers 8 plies.
__global__ void __launch_bounds__(256) k_clear_logn(int n, uint32_t* __restrict__ lines) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g < n) lines[(size_t)g * kLineWords + 31] = 0;
}

// The plies that led to loaded states: plies uint8[n][63][2] (from, to), most recent first,
// 0xFF = unknown.  K = the leading known ones (both squares < 100: a malformed entry would otherwise become a
// log entry that collides with a real ply in the chasing rule's walk); ply b back goes to log entry (K - b) mod 64 and word
// 31 of the line becomes K, exactly what K played plies would have left.
__global__ void __launch_bounds__(256) k_load_plies(int n, const uint8_t* __restrict__ plies, uint32_t* __restrict__ lines,
                                                    uint16_t* __restrict__ logs) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  const uint8_t* p = plies + (size_t)g * (2 * (kLogPlies - 1));
  int K = 0;  // an entry that names no square (0xFF = unknown, or anything else >= 100) ends the known plies
  while (K < kLogPlies - 1 && p[2 * K] < 100u && p[2 * K + 1] < 100u) ++K;
  uint16_t* glog = logs + (size_t)g * kLogPlies;
  for (int b = 1; b <= K; ++b)
    glog[(K - b) & (kLogPlies - 1)] = (uint16_t)((uint32_t)p[2 * (b - 1)] | ((uint32_t)p[2 * (b - 1) + 1] << 7));
  lines[(size_t)g * kLineWords + 31] = (uint32_t)K;
}

// Move logs of the states at time step t of a board-history ring, rebuilt from the actions the ring
// holds (GetPlayedActions): ply b back of game g = the action applied at step t - b, as long
// as that step is still in the ring and did not end a game.  Entries are placed where the state's
// own counter (word 31 of its line) expects them; plies older than the last restart come from the
// pinned log when there is one (same entry index: a restart copies the pinned log), everything
// else is marked unknown, which ends the chasing rule's walk back.
__global__ void __launch_bounds__(256) k_rebuild_logs(int n, const uint32_t* __restrict__ lines_t, const int16_t* __restrict__ act,
                                                      const uint8_t* __restrict__ done, int length, long long t, long long oldest,
                                                      const uint16_t* __restrict__ pin_logs, uint16_t* __restrict__ logs) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  uint32_t logn = lines_t[(size_t)g * kLineWords + 31];
  int known = (int)min(logn, (uint32_t)(kLogPlies - 1));
  uint16_t* glog = logs + (size_t)g * kLogPlies;
  bool in_game = true;
  for (int b = 1; b <= known; ++b) {
    uint32_t idx = (logn - (uint32_t)b) & (uint32_t)(kLogPlies - 1);
    uint32_t e = kHistNone;
    if (in_game && t - b >= oldest) {
      size_t row = (size_t)((t - b) % length) * (size_t)n + (size_t)g;
      int a = act[row];
      if ((done[row] & 1u) == 0 && a >= 0) {  // bit 0 = the game ended with this action
        int from = a / 36, r = a - 36 * from, dir = r / 9, dist = r - 9 * dir + 1;
        int to = from + (dir == 0 ? 10 : dir == 1 ? 1 : dir == 2 ? -10 : -1) * dist;
        e = (uint32_t)from | ((uint32_t)to << 7);
      } else {
        in_game = false;  // step t - b ended a game: the state at t - b + 1 was a fresh or pinned one
      }
    }
    if (e == kHistNone && !in_game && pin_logs) e = pin_logs[(size_t)g * kLogPlies + idx];
    glog[idx] = (uint16_t)e;
  }
}

// ------------------------------------------------------------------ S2 information state
// ComputeInfostateTensor in the paper's own form: bf16 [N][487][10][10] = 97,400 bytes per game,
// HBM-write bound.  One warp per game.  Build: the 48,700 cells of a game as a bit stream A
// (bit set = 1.0) in shared memory, filled by the lanes with shared-memory atomics from the
// game's line and tracker block - lane = square for the per-piece channels, lane = plane for the
// whole-board ones.  The 58 channels that hold other values (type posteriors 12-35, the two
// fractions 41-42, the -1.0 of the 32 move channels) get two more bit streams B and C over those
// planes only, each with one bf16 value per plane.  Store: four cells (one nibble of the
// streams, never straddling a plane: 100 = 25 nibbles) per lane and 8-byte streaming store, 256
// contiguous bytes per warp instruction (a game is 8-byte, not 16-byte, aligned: 97,400 = 8 x 12,175).
constexpr int kInfoPlanes = STRAT_INFO_PLANES;
constexpr int kInfoNibbles = kInfoPlanes * 25;               // 12,175 per game
constexpr int kInfoAWords = (kInfoPlanes * 100 + 31) / 32 + 1;  // 1,523
constexpr int kInfoSpecial = 58;                              // planes 12-35, 41-42, 455-486
constexpr int kInfoBWords = (kInfoSpecial * 100 + 31) / 32 + 1;  // 183

__device__ __forceinline__ void info_set(uint32_t* stream, int plane, int cell) {
  int bit = 100 * plane + cell;
  atomicOr(stream + (bit >> 5), 1u << (bit & 31));
}
__device__ __forceinline__ void info_place(uint32_t* stream, int plane, const BB& b) {  // a whole 100-bit plane
  int o = 100 * plane, w = o >> 5, sh = o & 31;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint32_t v = b.w[i];
    if (!v) continue;
    atomicOr(stream + w + i, v << sh);
    if (sh) atomicOr(stream + w + i + 1, v >> (32 - sh));
  }
}
// Round-to-nearest-even bf16 of the IEEE double quotient num / den (> 0): DESIGN.md reading I8.
__device__ __forceinline__ uint32_t bf16_of_ratio(long long num, long long den) {
  if (num <= 0 || den <= 0) return 0u;
  unsigned long long b = (unsigned long long)__double_as_longlong((double)num / (double)den);
  int e = (int)((b >> 52) & 0x7FFull) - 1023;
  unsigned long long man = b & 0xFFFFFFFFFFFFFull;
  unsigned long long keep = man >> 45, rem = man & ((1ull << 45) - 1ull), half = 1ull << 44;
  if (rem > half || (rem == half && (keep & 1ull))) ++keep;
  if (keep == 128ull) { keep = 0; ++e; }
  return ((uint32_t)(e + 127) << 7) | (uint32_t)keep;
}

// One staged game: the three bit streams and the plane values (what the storer needs).
struct InfoStage { uint32_t* A; uint32_t* Bs; uint32_t* Cs; uint32_t* val; };
__device__ __forceinline__ InfoStage info_stage(uint32_t* base) {
  InfoStage s; s.A = base; s.Bs = base + kInfoAWords; s.Cs = s.Bs + kInfoBWords; s.val = s.Cs + kInfoBWords;
  return s;
}
// builder warp: game gi -> bit streams + values in `st`; trk / sline = its private staging
__device__ __forceinline__ void info_build(const Params& P, const uint32_t* __restrict__ lines, int gi, const InfoStage& st,
                                           uint32_t* trk, uint32_t* sline, int lane) {
  uint32_t* A = st.A; uint32_t* Bs = st.Bs; uint32_t* Cs = st.Cs; uint32_t* val = st.val;
  // ---- stage the game's line and tracker block, clear the streams
  for (int j = lane; j < (kInfoAWords + 2 * kInfoBWords + kInfoSpecial + 1) / 4; j += 32)
    reinterpret_cast<uint4*>(A)[j] = make_uint4(0u, 0u, 0u, 0u);
  {
    const uint4* src = reinterpret_cast<const uint4*>(P.track + (size_t)gi * kTrackWords);
    uint4* dst = reinterpret_cast<uint4*>(trk);
#pragma unroll
    for (int k = 0; k < 4; ++k) dst[32 * k + lane] = __ldcg(src + 32 * k + lane);
    sline[lane] = __ldcg(lines + (size_t)gi * kLineWords + lane);
  }
  __syncwarp();
  Game g;
  unpack_line(sline, g);
  const int side = (int)(g.ply & 1u);
  const BB occ = occupied(g), mine = owned_by(g, occ, side), enemy = bb_andn(occ, mine);
  // ---- lane = square: what the piece on it is and has done
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const int c = 32 * r + lane;
    if (c >= 100) break;
    if (!bb_test(occ, c)) {
      if (!is_lake_cell(c)) info_set(A, 38, c);                     // empty (R#17: lakes are not squares)
      continue;
    }
    const bool own = bb_test(mine, c) != 0, rev = bb_test(g.rev, c) != 0, mvd = bb_test(g.mvd, c) != 0;
    const int t = type_at(g, c);
    if (own) info_set(A, t - 1, c);                                 // 0-11
    if (rev) info_set(A, (own ? 24 : 12) + t - 1, c);               // a revealed piece: probability 1 (12-35)
    else info_set(A, own ? 36 : 37, c);                             // hidden pieces
    if (mvd) info_set(A, own ? 39 : 40, c);                         // pieces that moved
    const uint32_t r0 = trk[4 * c], r1 = trk[4 * c + 1], r2 = trk[4 * c + 2], r3 = trk[4 * c + 3];
    const int a = own ? 43 : 76, b = own ? 251 : 303;
    for (uint32_t w = r0 & 0x3FFFFFu; w; w &= w - 1) info_set(A, a + __ffs((int)w) - 1, c);            // threat, evasion
    for (uint32_t w = r1 & 0x7FFu; w; w &= w - 1) info_set(A, a + 22 + __ffs((int)w) - 1, c);          // active adjacency
    for (uint32_t w = (r1 >> 11) & 0x1FFFu; w; w &= w - 1) info_set(A, b + __ffs((int)w) - 1, c);      // protected
    for (uint32_t w = r2 & 0x3FFFFFFu; w; w &= w - 1) info_set(A, b + 13 + __ffs((int)w) - 1, c);      // against, by
    for (uint32_t w = r3 & 0x1FFFu; w; w &= w - 1) info_set(A, b + 39 + __ffs((int)w) - 1, c);         // been protected against
    info_set(A, 355 + (int)((r0 >> 22) & 127u), c);                 // P:606 start square
  }
  // ---- lane = plane: type posteriors (reading I7), fractions, moves
  if (lane < 24) {
    // lanes 0-11: the opponent's pieces as the player sees them (12-23); 12-23: the player's, as the opponent does (24-35)
    const int t = lane % 12 + 1;
    const BB hid = bb_andn(lane < 12 ? enemy : mine, g.rev);
    const BB hid_unmoved = bb_andn(hid, g.mvd), hid_moved = bb_and(hid, g.mvd);
    const BB imm = bb_and(g.t3, bb_or(g.t2, bb_and(g.t1, g.t0)));
    const int u = bb_popc(hid_unmoved), m = bb_popc(hid_moved), I = bb_popc(bb_and(hid, imm)), M = u + m - I;
    const int ct = bb_popc(type_is(g, hid, t));
    const bool immovable = t == T_FLAG || t == T_BOMB;
    const int free_unmoved = u - I > 0 ? u - I : 0;
    uint32_t vu = immovable ? bf16_of_ratio(ct, u) : bf16_of_ratio((long long)free_unmoved * ct, (long long)u * M);
    uint32_t vm = immovable ? 0u : bf16_of_ratio(ct, M);
    if (vu) info_place(Bs, lane, hid_unmoved);
    if (vm) info_place(Cs, lane, hid_moved);
    val[lane] = vu | (vm << 16);
  } else if (lane < 26) {
    BB all; all.w[0] = all.w[1] = all.w[2] = 0xFFFFFFFFu; all.w[3] = 0xFu;
    uint32_t v = lane == 24 ? bf16_of_ratio((long long)g.ply, (long long)P.ply_cap)
                            : (P.max_battleless > 0 ? bf16_of_ratio((long long)g.battleless, (long long)P.max_battleless) : 0u);
    if (v) info_place(Bs, lane, all);
    val[lane] = v;
  }
  {  // move j = ply t-1-j: +1.0 on the destination (stream A), -1.0 on the source (stream B)
    const int slot = (int)((g.ply - 1u - (uint32_t)lane) & 31u);
    const uint32_t e = (trk[kTrkMoves + (slot >> 1)] >> (16 * (slot & 1))) & 0xFFFFu;
    if (e != kHistNone) {
      info_set(A, 455 + lane, (int)(e >> 7));
      info_set(Bs, 26 + lane, (int)(e & 127u));
    }
    val[26 + lane] = 0xBF80u;
  }
  // ---- captured pieces by start square and causes of death
  {
    const int n = min((int)trk[kTrkDeaths], kTrkMaxDeaths);
    for (int k = lane; k < n; k += 32) {
      const uint32_t e = trk[kTrkDeathList + k];
      const int start = (int)(e & 127u), t = (int)((e >> 7) & 15u), owner = (int)((e >> 11) & 1u), sq = (int)((e >> 12) & 127u),
                cause = (int)((e >> 19) & 7u);
      const int j = t <= 10 ? t - 1 : t == T_BOMB ? 10 : -1;
      if (j >= 0) info_set(A, (owner == side ? 109 : 120) + j, start);
      if (cause) info_set(A, (owner == side ? 131 : 191) + 10 * (cause - 1) + t - 1, sq);
    }
  }
}
// storer warp: the staged game -> 97,400 bytes of bf16
__device__ __forceinline__ void info_store(uint16_t* __restrict__ out, int gi, const InfoStage& st, int lane) {
  const uint32_t* A = st.A; const uint32_t* Bs = st.Bs; const uint32_t* Cs = st.Cs; const uint32_t* val = st.val;
  // ---- store: nibble n of the streams -> cells 4n..4n+3 of the game, two nibbles (16 bytes) per
  // lane and streaming store.  `out` is 8-byte aligned and a game is 97,400 B = 8 mod 16, so every
  // other game starts at 8 mod 16: such a game's first nibble goes out alone, the others' last one.
  // Which games those are is read off the game's address (`out` itself may be a slice that starts at
  // 8 mod 16).  Bits -> bf16 in registers: two bits spread to bit 0 and bit 16, times 0x3F80 (or
  // times the plane's value).
  uint16_t* gout = out + (size_t)gi * (kInfoPlanes * 100);
  const int odd = (int)((reinterpret_cast<uintptr_t>(gout) >> 3) & 1u);
  uint4* dst = reinterpret_cast<uint4*>(gout + 4 * odd);  // pair k = nibbles 2k+odd, 2k+odd+1
  auto spread = [](uint32_t t) { return (t & 1u) | ((t & 2u) << 15); };
  auto nib_value = [&](int n) -> uint2 {  // any nibble, valued planes included
    const uint32_t t = (A[n >> 3] >> (4 * (n & 7))) & 15u;
    uint2 v = make_uint2(spread(t) * 0x3F80u, spread(t >> 2) * 0x3F80u);
    const int shift = n < 300 ? -1 : n < 900 ? 300 : n < 1025 ? -1 : n < 1075 ? 1025 - 600 : n < 11375 ? -1 : 11375 - 650;
    if (shift >= 0) {
      const int nn = n - shift;  // nibble of the compact valued streams: planes 12-35 -> 0-23, 41-42 -> 24-25, 455-486 -> 26-57
      const uint32_t vv = val[nn / 25];
      const uint32_t tb = (Bs[nn >> 3] >> (4 * (nn & 7))) & 15u, tc = (Cs[nn >> 3] >> (4 * (nn & 7))) & 15u;
      v.x |= spread(tb) * (vv & 0xFFFFu) | spread(tc) * (vv >> 16);
      v.y |= spread(tb >> 2) * (vv & 0xFFFFu) | spread(tc >> 2) * (vv >> 16);
    }
    return v;
  };
  auto plain_pairs = [&](int ka, int kb) {  // pairs ka..kb-1 whose two nibbles lie in 0/1 planes
#pragma unroll 4
    for (int k = ka + lane; k < kb; k += 32) {
      const int bit = 8 * k + 4 * odd;
      const uint32_t t = __funnelshift_r(A[bit >> 5], A[(bit >> 5) + 1], bit & 31);
      __stcs(dst + k, make_uint4(spread(t) * 0x3F80u, spread(t >> 2) * 0x3F80u, spread(t >> 4) * 0x3F80u,
                                 spread(t >> 6) * 0x3F80u));
    }
  };
  auto any_pairs = [&](int ka, int kb) {
    for (int k = ka + lane; k < kb; k += 32) {
      const uint2 lo = nib_value(2 * k + odd), hi = nib_value(2 * k + odd + 1);
      __stcs(dst + k, make_uint4(lo.x, lo.y, hi.x, hi.y));
    }
  };
  {
    // plain nibble ranges [0,300) [900,1025) [1075,11375): pair k is plain iff lo <= 2k+odd and 2k+odd+1 < hi
    const int a0 = 0, b0 = (300 - 2 - odd) / 2 + 1, a1 = (900 - odd + 1) / 2, b1 = (1025 - 2 - odd) / 2 + 1,
              a2 = (1075 - odd + 1) / 2, b2 = (11375 - 2 - odd) / 2 + 1, pairs = (kInfoNibbles - 1) / 2;
    plain_pairs(a0, b0); any_pairs(b0, a1); plain_pairs(a1, b1); any_pairs(b1, a2); plain_pairs(a2, b2); any_pairs(b2, pairs);
    if (lane == 0) {
      const int n = odd ? 0 : kInfoNibbles - 1;
      __stcs(reinterpret_cast<uint2*>(gout) + n, nib_value(n));
    }
  }
}

// CTA = one BUILDER warp + one STORER warp handing a staged game back and forth (full / empty mbarriers, as
// in the fused step); twenty such pairs per SM, so the HBM write stream of an SM never waits for a build.  Games are handed out by a
// ticket counter, not by a fixed stride: the SMs do not all drain their stores at the same rate, and a
// persistent grid with equal shares ends on its slowest SM (plain streaming stores on this GPU: 6.2 TB/s
// with equal shares, 7.2-7.4 TB/s when every CTA fetches its next piece of work as it finishes one).
// The counter cleans up after itself like the fused step's: atomicInc wraps to 0 after exactly
// num_games draws (num_games - grid successful ones and one failing draw per CTA).
constexpr int kInfoStageWords = kInfoAWords + 2 * kInfoBWords + kInfoSpecial + 1;  // 1,948
// One stage and 20 CTAs per SM (48 registers, 10 KB of shared memory): 1.064 ms at 65,536 games; two stages
// with 12 CTAs 1.085 ms, one stage with 12 / 16 CTAs 1.108 / 1.082 ms.
#ifndef STRAT_INFO_STAGES
#define STRAT_INFO_STAGES 1
#endif
#ifndef STRAT_INFO_CTAS
#define STRAT_INFO_CTAS 20
#endif
constexpr int kInfoStages = STRAT_INFO_STAGES;
constexpr int kInfoCtasPerSm = STRAT_INFO_CTAS;
constexpr int kInfoCtaWords = kInfoStages * kInfoStageWords + kTrackWords + kLineWords;      // 4,440 words = 17,760 B with two stages
static_assert(kInfoStageWords % 4 == 0, "16-byte aligned stages");
__global__ void __launch_bounds__(64, kInfoCtasPerSm) k_encode_infostate(Params P, const uint32_t* __restrict__ lines,
                                                         uint16_t* __restrict__ out, uint32_t* __restrict__ ticket) {
  __shared__ __align__(16) uint32_t s_info[kInfoCtaWords];
  __shared__ __align__(8) uint64_t s_full[kInfoStages], s_empty[kInfoStages];
  __shared__ int s_game[kInfoStages];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0)
    for (int s = 0; s < kInfoStages; ++s) { mbar_init(&s_full[s], 32); mbar_init(&s_empty[s], 32); }
  __syncthreads();
  int gi = blockIdx.x;  // grid <= num_games
  for (int it = 0;; ++it) {
    const int stage = it % kInfoStages, round = it / kInfoStages;
    const InfoStage st = info_stage(s_info + stage * kInfoStageWords);
    if (warp == 0) {
      if (round > 0) mbar_wait(&s_empty[stage], (uint32_t)(round - 1) & 1u);
      if (it > 0) {
        uint32_t tk = 0;
        if (lane == 0) tk = atomicInc(ticket, (uint32_t)P.num_games - 1u);
        tk = __shfl_sync(0xffffffffu, tk, 0);
        gi = tk < (uint32_t)(P.num_games - (int)gridDim.x) ? (int)(gridDim.x + tk) : -1;
      }
      if (lane == 0) s_game[stage] = gi;
      if (gi >= 0) {
        info_build(P, lines, gi, st, s_info + kInfoStages * kInfoStageWords, s_info + kInfoStages * kInfoStageWords + kTrackWords, lane);
        __syncwarp();
      }
      mbar_arrive(&s_full[stage]);
      if (gi < 0) break;
    } else {
      mbar_wait(&s_full[stage], (uint32_t)round & 1u);
      gi = s_game[stage];
      if (gi < 0) break;
      info_store(out, gi, st, lane);
      mbar_arrive(&s_empty[stage]);
    }
  }
}

__global__ void k_set_int(int* p, int v) { *p = v; }

// Measurement aid (strat_probe_write): a constant streamed out in pieces of `chunk16` 16-byte vectors with the
// store instruction of the step kernels' outputs.  Persistent CTAs; pieces by ticket (self-resetting
// counter, as above) or by a fixed stride.
__global__ void __launch_bounds__(128) k_probe_write(uint4* __restrict__ dst, uint32_t pieces, uint32_t chunk16,
                                                     uint32_t* __restrict__ ticket, int dynamic) {
  __shared__ uint32_t s_piece;
  const uint4 v = make_uint4(0x3F803F80u, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u);
  uint32_t c = blockIdx.x;
  for (;;) {
    uint4* q = dst + (size_t)c * chunk16;
    for (uint32_t i = threadIdx.x; i < chunk16; i += blockDim.x) st_stream(q + i, v);
    if (dynamic) {
      __syncthreads();
      if (threadIdx.x == 0) {
        uint32_t tk = atomicInc(ticket, pieces - 1u);
        s_piece = tk < pieces - gridDim.x ? gridDim.x + tk : 0xFFFFFFFFu;
      }
      __syncthreads();
      c = s_piece;
    } else {
      c += gridDim.x;
    }
    if (c >= pieces) break;
  }
}


}  // namespace
