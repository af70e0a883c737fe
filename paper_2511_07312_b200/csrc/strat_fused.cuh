// strat_fused.cuh - the fused hot path: persistent, warp-specialised step with cross-launch overlap
// Part of libstrat.so (one translation unit: strat.cu includes these in order).
#pragma once

namespace {
using namespace strat;

// ---- the fused hot path, warp-specialised and persistent -------------------------------
// One CTA = one LOGIC warp + one STORE warp sharing two staging buffers.  The logic warp
// walks batches of 32 games (thread per game): state line straight from global into
// registers, mask rows into the stage, mask/action/reward/done/state out, then the new
// state's 4400-bit observation stream into the same stage.  The store warp expands finished
// stages to bf16 and streams them out.  The two are decoupled by mbarriers, so on every SM
// observation stores of batch i flow while batch i+1 is still in its (latency-bound) rule
// logic; with one-warp CTAs all resident warps ran logic, then stores, in lockstep.
// Staging buffers per CTA and resident CTAs per SM (measured on B200, CUDA events, 65,536 / 262,144 games;
// "back to back" = 2,000 overlapped launches, "alone" = one launch with the GPU to itself):
//   strat_rollout_step   ONE stage, 8 CTAs per SM (128 registers): 83.0 / 342 us back to back, 121 / 381 us
//                        alone.  A CTA's logic and its stores then alternate and the SM's other seven CTAs
//                        fill the gaps; drawing no batch ahead of the stores keeps the SMs, which do not all
//                        drain stores at one rate, in balance.  (Two stages, 3 CTAs per SM and two launches
//                        co-resident, round 1's choice: 85.5 / 352 and 121 / 386 us.  One stage with 2..7
//                        CTAs: the same back to back, but 185..127 us alone.)
//   with chase_rule      the same shape (the rule code fits 128 registers too): 84.7 us back to back, 124 us alone
//                        (two stages, 3 CTAs: 87.0 us).
//   with the S2 trackers two stages, 3 CTAs per SM and two launches co-resident, as strat_rollout_step had them
//                        in round 1: its logic warp waits for the tracker record from HBM and is what bounds
//                        the step; one stage with 8 CTAs is 3 % faster back to back (113 us) and 2 % slower
//                        alone (154 against 151 us), and alone is how the 487-channel pipeline runs it.
//   strat_step_observe   TWO stages, 3 CTAs per SM: it never overlaps its neighbours in the stream (it waits
//                        for its actions' producer), its launch is short (~14 batches per SM) and what
//                        counts is how evenly the SMs finish: 2 -> 102.5 us, 3 -> 102.4 us, 4 -> 104.5 us,
//                        6 -> 109.6 us; one stage with 6 CTAs 112.7 us.  Tried and dropped: the logic warp
//                        helping to store the CTA's last batch (drawing the next ticket before the hand-over,
//                        to know which batch is the last, unbalances the SMs by more than the help gains:
//                        106.5 us); drawing the last tickets only when the store warp has nothing left (no
//                        change).
template <bool kExternal, bool kTrack> struct WsShape { static constexpr int kStages = (kExternal || kTrack) ? 2 : 1; };
constexpr int kWsCtasPerSm = 8;          // strat_rollout_step, also with chase_rule
constexpr int kWsTrackCtasPerSm = 3;     // ... with the S2 trackers (infostate)
constexpr int kWsExternalCtasPerSm = 3;  // strat_step_observe
constexpr int kWsStageWords = kBatch * kBitsRowWords;  // 4448 words = 17,792 B (mask rows need 3,616)

// Per-batch version flags in global memory: consecutive launches of the fused step overlap
// (programmatic dependent launch), ordered batch by batch instead of kernel by kernel.
// whole warp: returns once *flag == want (lane 0 polls; the barrier orders the other lanes)
__device__ __forceinline__ void flag_wait(const uint32_t* flag, uint32_t want, int lane) {
  if (lane == 0)
    while (ld_acquire(flag) != want) __nanosleep(64);
  __syncwarp();
}
// whole warp: publish this warp's prior global writes, then set the flag.  kPublish = false: nobody reads the
// flag while this grid runs (strat_step_observe: the launches around it wait for whole grids), so it is only
// kept up to date for later launches and the warp does not wait for its stores to drain - with a handful of
// batches per CTA all store warps would do that at the same moments and the write stream would stall there
// (measured: the number of batches being stored dropped to a third every ~25 us).
template <bool kPublish = true>
__device__ __forceinline__ void flag_set(uint32_t* flag, uint32_t v, int lane) {
  __syncwarp();
  if (lane == 0) {
    // release is cumulative over the lanes the barrier above ordered before it; a sequentially consistent
    // __threadfence() in front of it (round 1) only cost time: 86.3 -> 85.7 us per overlapped step
    if (kPublish) st_release(flag, v);
    else asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(flag), "r"(v) : "memory");
  }
}
// nibble -> 4 bf16 (0x3F80 where the bit is set); 16 entries x 8 B = one bank row, so the
// two LDS.64 per 16-byte chunk never conflict.
__device__ __forceinline__ void fill_lut16(uint2* lut, int tid) {
  if (tid < 16) {
    uint2 v;
    v.x = ((tid & 1) ? 0x3F80u : 0u) | ((tid & 2) ? 0x3F800000u : 0u);
    v.y = ((tid & 4) ? 0x3F80u : 0u) | ((tid & 8) ? 0x3F800000u : 0u);
    lut[tid] = v;
  }
}
__device__ __forceinline__ void expand_obs16(uint16_t* __restrict__ obs, int first_game, int ng,
                                             const uint32_t* s_bits, const uint2* lut, int lane) {
  for (int gi = 0; gi < ng; ++gi) {
    const uint8_t* row = reinterpret_cast<const uint8_t*>(s_bits + gi * kBitsRowWords);
    uint4* dst = reinterpret_cast<uint4*>(obs + (size_t)(first_game + gi) * STRAT_OBS_ELEMS);
#pragma unroll
    for (int k = 0; k < 17; ++k) {
      uint32_t b = row[32 * k + lane];
      uint2 lo = lut[b & 15u], hi = lut[b >> 4];
      st_stream(dst + 32 * k + lane, make_uint4(lo.x, lo.y, hi.x, hi.y));
    }
    if (lane < kObsChunks - 544) {
      uint32_t b = row[544 + lane];
      uint2 lo = lut[b & 15u], hi = lut[b >> 4];
      st_stream(dst + 544 + lane, make_uint4(lo.x, lo.y, hi.x, hi.y));
    }
  }
}
__device__ __forceinline__ void store_game_global(uint32_t* __restrict__ lines, int game, const Game& g) {
  uint32_t W[32];
  pack_line(g, W);
  uint4* p = reinterpret_cast<uint4*>(lines + (size_t)game * kLineWords);
  const uint64_t pol = lines_policy();
#pragma unroll
  for (int k = 0; k < 8; ++k) st_line16(p + k, make_uint4(W[4 * k], W[4 * k + 1], W[4 * k + 2], W[4 * k + 3]), pol);
}

// kExternal = false (strat_rollout_step): mask of the state -> uniform legal action -> step ->
//   observation of the new state; `actions` is an output.
// kExternal = true (strat_step_observe): `actions` is the caller's input (validated) -> step ->
//   mask AND observation of the new state: the data-collection loop of PAPER.md:232, 461-462
//   (ApplyActions, then ComputeLegalActionMask + ComputeInfostateTensor for the next policy call).
template <bool kExternal, bool kChase, bool kTrack>
__global__ void __launch_bounds__(64, kExternal ? kWsExternalCtasPerSm : kTrack ? 2 * kWsTrackCtasPerSm : kWsCtasPerSm)
k_rollout_step(Params P, uint32_t* __restrict__ lines, uint32_t* __restrict__ mask,
                                                        int16_t* __restrict__ actions, int8_t* __restrict__ reward,
                                                        uint8_t* __restrict__ done, uint16_t* __restrict__ obs,
                                                        uint32_t* __restrict__ ticket, uint32_t* __restrict__ f_state,
                                                        uint32_t* __restrict__ f_obs, uint32_t version, HistSlot hs,
                                                        int* __restrict__ err, int wait_prior,
                                                        const uint32_t* __restrict__ gather_flag, uint32_t gather_number) {
  constexpr int kWsStages = WsShape<kExternal, kTrack>::kStages;
  __shared__ __align__(16) uint32_t s_stage[kWsStages][kWsStageWords];
  __shared__ __align__(8) uint2 s_lut[16];
  // strat_step_observe runs 3 CTAs per SM and has shared memory to spare: a byte -> 8 x bf16 table (one
  // LDS.128 per 16 bytes stored instead of two LDS.64 plus the nibble arithmetic) lets its store warps,
  // of which an SM has only three, issue a batch faster (isolated launch at 65,536 games: 102.4 -> 100.4 us;
  // 32-byte stores on top of it were slower, 103.2 us)
  __shared__ __align__(16) uint4 s_lut256[kExternal ? 256 : 1];
  __shared__ __align__(8) uint64_t s_full[kWsStages], s_empty[kWsStages];
  __shared__ int s_batch[kWsStages];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nbatches = (P.num_games + kBatch - 1) / kBatch;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < kWsStages; ++s) { mbar_init(&s_full[s], 32); mbar_init(&s_empty[s], 32); }
  }
  fill_lut16(s_lut, threadIdx.x);
  if (kExternal) fill_lut(s_lut256, threadIdx.x, 64);
  __syncthreads();
  // Let the next launch of this kernel become resident now: it orders itself behind this one
  // batch by batch through f_state / f_obs.  wait_prior (host, launch_fused): this launch does not directly
  // continue its own environment's chain of fused steps - no flags tie it to what runs before it - so it
  // waits for that as a whole.
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (wait_prior) asm volatile("griddepcontrol.wait;" ::: "memory");
  if (warp == 0) {
    // in a self-play loop with chained gathers (strat_replay_sample_chained): the rows this step writes
    // may still be read by the gather before the last one; wait until that one has finished (it has)
    if (gather_flag) {
      if (lane == 0)
        while ((int32_t)(ld_acquire(gather_flag) - gather_number) < 0) __nanosleep(64);
      __syncwarp();
    }
    // ------------------------------------------------ logic warp (thread per game)
    // batches: the first one is the CTA's own index, the rest are drawn from this launch's
    // ticket counter.  atomicInc wraps to 0 after exactly nbatches draws (nbatches - grid
    // successful ones + one failing draw per CTA), so the counter cleans up after itself.
    int b = blockIdx.x;
    for (int it = 0;; ++it) {
      const int stage = it % kWsStages, round = it / kWsStages;
      uint32_t* work = s_stage[stage];
      if (round > 0) mbar_wait(&s_empty[stage], (uint32_t)(round - 1) & 1u);
      if (it > 0) {
        uint32_t tk = 0;
        if (lane == 0) tk = atomicInc(ticket, (uint32_t)nbatches - 1u);
        tk = __shfl_sync(0xffffffffu, tk, 0);
        b = tk < (uint32_t)(nbatches - (int)gridDim.x) ? (int)(gridDim.x + tk) : -1;
      }
      if (b < 0) {
        if (lane == 0) s_batch[stage] = -1;
        mbar_arrive(&s_full[stage]);
        break;
      }
      const int first = b * kBatch, ng = min(kBatch, P.num_games - first);
      flag_wait(f_state + b, version - 1u, lane);  // the previous launch is done with this batch's state
      if (!kExternal) zero_smem16(work, kMaskBytes, lane);
      Game g;
      int n = 0, cnt[4] = {0, 0, 0, 0};
      if (lane < ng) load_game_global(lines, first + lane, g, hs.lines);
      __syncwarp();
      bool reset_me = false;
      if (!kExternal) {
        if (lane < ng && !g.done) n = legal_mask_row(g, g.ply & 1u, rules_of<kChase>(P), work + lane * kMaskWords, cnt,
                                                       kChase ? game_log(P, (uint32_t)(first + lane)) : nullptr);
        __syncwarp();
        if (mask) store_mask(mask, first, ng, work, lane);
        if (lane < ng) {
          int a = -1;
          if (n > 0) a = pick_action(work + lane * kMaskWords, cnt, n, action_draw(P, (uint32_t)(first + lane), g));
          StepOut o = step_game<false, true, kChase, kTrack>(P, (uint32_t)(first + lane), g, a);  // a comes from this state's mask
          if (o.illegal) raise_error(err, STRAT_ILLEGAL_ACTION);
          // write-once outputs leave the L2 first (evict-first), like the mask rows and the observations:
          // lines of normal priority in between would be written back out of order, long after their neighbours
          if (actions) __stcs(actions + first + lane, (int16_t)a);
          if (reward) __stcs(reward + first + lane, (int8_t)o.reward);
          if (done) __stcs(done + first + lane, (uint8_t)o.done);
          if (hs.lines) { __stcs(hs.act + first + lane, (int16_t)a); __stcs(hs.rew + first + lane, (int8_t)o.reward); __stcs(hs.done + first + lane, (uint8_t)o.done); }
          reset_me = o.needs_reset;
        }
        uint32_t rs = __ballot_sync(0xffffffffu, reset_me);  // also: every lane is done with its mask row
        if (rs && P.pin) { if (reset_me) reset_game(P, (uint32_t)(first + lane), g); __syncwarp(); }  // owner lanes' tracker writes first
        else if (rs) coop_setup(P, first, rs, g, work, lane);
        if (kTrack && rs && P.track) coop_track_start(P, first, rs, g, lane);
        if (lane < ng) store_game_global(lines, first + lane, g);
        flag_set(f_state + b, version, lane);  // state, mask, action, reward, done of this batch are out
      } else {
        // caller's actions: the observation of the NEW state goes out first (it is 95 % of the bytes and
        // only needs the step), its legal mask is built afterwards while the store warp is already writing
        if (lane < ng) {
          int a = (int)actions[first + lane];
          StepOut o = step_game<true, true, kChase, kTrack>(P, (uint32_t)(first + lane), g, a);
          if (o.illegal) raise_error(err, STRAT_ILLEGAL_ACTION);
          __stcs(reward + first + lane, (int8_t)o.reward);
          __stcs(done + first + lane, (uint8_t)o.done);
          if (hs.lines) { __stcs(hs.act + first + lane, (int16_t)a); __stcs(hs.rew + first + lane, (int8_t)o.reward); __stcs(hs.done + first + lane, (uint8_t)o.done); }
          reset_me = o.needs_reset;
        }
        uint32_t rs = __ballot_sync(0xffffffffu, reset_me);
        if (rs && P.pin) { if (reset_me) reset_game(P, (uint32_t)(first + lane), g); __syncwarp(); }  // owner lanes' tracker writes first
        else if (rs) coop_setup(P, first, rs, g, work, lane);  // borrows the stage; the bit streams overwrite it
        if (kTrack && rs && P.track) coop_track_start(P, first, rs, g, lane);
        if (lane < ng) store_game_global(lines, first + lane, g);
        __syncwarp();
        if (lane < ng) encode_bits(g, work + lane * kBitsRowWords);
        __syncwarp();
        if (lane == 0) s_batch[stage] = b;
        mbar_arrive(&s_full[stage]);
        if (mask) {  // mask rows in the OTHER stage's buffer, once the store warp has emptied it
          const int ostage = (it + 1) % kWsStages, oround = (it + 1) / kWsStages;
          uint32_t* mwork = s_stage[ostage];
          if (oround > 0) mbar_wait(&s_empty[ostage], (uint32_t)(oround - 1) & 1u);
          zero_smem16(mwork, kMaskBytes, lane);
          __syncwarp();
          if (lane < ng && !g.done)  // of the NEW state
            legal_mask_row(g, g.ply & 1u, rules_of<kChase>(P), mwork + lane * kMaskWords, cnt,
                           kChase ? game_log(P, (uint32_t)(first + lane)) : nullptr);
          __syncwarp();
          store_mask(mask, first, ng, mwork, lane);
        }
        flag_set<false>(f_state + b, version, lane);  // state, reward, done, mask of this batch are out
        continue;
      }
      __syncwarp();  // the stage becomes bit streams
      if (lane < ng) encode_bits(g, work + lane * kBitsRowWords);
      __syncwarp();
      if (lane == 0) s_batch[stage] = b;
      mbar_arrive(&s_full[stage]);
    }
  } else {
    // ------------------------------------------------ store warp (lane per 16-byte chunk)
    for (int it = 0;; ++it) {
      const int stage = it % kWsStages, round = it / kWsStages;
      mbar_wait(&s_full[stage], (uint32_t)round & 1u);
      const int b = s_batch[stage];
      if (b < 0) break;
      const int first = b * kBatch, ng = min(kBatch, P.num_games - first);
      flag_wait(f_obs + b, version - 1u, lane);  // write-after-write on a reused obs buffer
      if (kExternal) expand_obs(obs, first, ng, s_stage[stage], s_lut256, lane);
      else expand_obs16(obs, first, ng, s_stage[stage], s_lut, lane);
      flag_set<!kExternal>(f_obs + b, version, lane);
      mbar_arrive(&s_empty[stage]);
    }
  }
}


}  // namespace
