// strat.cu — sm_100a kernels and the C ABI of libstrat.so (include/strat.h).
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
#include <new>

#include "../../include/strat.h"
#include "strat_game.cuh"

namespace {
using namespace strat;

constexpr int kBatch = 32;             // games per warp/CTA
constexpr int kStateStride = 144;      // bytes between games' staged lines (16-B aligned, conflict-free LDS.128)
constexpr int kMaskRowBytes = kMaskWords * 4;        // 452
constexpr int kBitsRowWords = 139;                   // 138 used; odd stride -> conflict-free
constexpr int kObsChunks = 550;                      // 16-B chunks per game observation
constexpr int kStateBytes = kBatch * kStateStride;   // 4608
constexpr int kMaskBytes = kBatch * kMaskRowBytes;   // 14464

// ------------------------------------------------------------------ small PTX helpers
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void st_stream(uint4* p, uint4 v) { __stcs(p, v); }  // write-once outputs

// ------------------------------------------------------------------ warp-cooperative I/O
// 32 (or `ng`) device lines, contiguous in global memory, into the padded staging area.
__device__ __forceinline__ void load_lines(const uint32_t* __restrict__ lines, int first_game, int ng,
                                           uint8_t* s_state, int lane) {
  const uint4* src = reinterpret_cast<const uint4*>(lines + (size_t)first_game * kLineWords);
  for (int j = lane; j < ng * 8; j += 32) cp_async16(s_state + (j >> 3) * kStateStride + (j & 7) * 16, src + j);
  cp_async_wait_all();
  __syncwarp();
}
__device__ __forceinline__ void store_lines(uint32_t* __restrict__ lines, int first_game, int ng,
                                            const uint8_t* s_state, int lane) {
  uint4* dst = reinterpret_cast<uint4*>(lines + (size_t)first_game * kLineWords);
  for (int j = lane; j < ng * 8; j += 32)
    dst[j] = *reinterpret_cast<const uint4*>(s_state + (j >> 3) * kStateStride + (j & 7) * 16);
}
__device__ __forceinline__ void read_game(const uint8_t* s_state, int lane, Game& g) {
  uint32_t W[32];
  const uint4* p = reinterpret_cast<const uint4*>(s_state + lane * kStateStride);
#pragma unroll
  for (int k = 0; k < 8; ++k) { uint4 v = p[k]; W[4 * k] = v.x; W[4 * k + 1] = v.y; W[4 * k + 2] = v.z; W[4 * k + 3] = v.w; }
  unpack_line(W, g);
}
__device__ __forceinline__ void write_game(uint8_t* s_state, int lane, const Game& g) {
  uint32_t W[32];
  pack_line(g, W);
  uint4* p = reinterpret_cast<uint4*>(s_state + lane * kStateStride);
#pragma unroll
  for (int k = 0; k < 8; ++k) p[k] = make_uint4(W[4 * k], W[4 * k + 1], W[4 * k + 2], W[4 * k + 3]);
}
__device__ __forceinline__ void zero_smem16(void* s, int bytes, int lane) {
  uint4* p = reinterpret_cast<uint4*>(s);
  for (int j = lane; j < bytes / 16; j += 32) p[j] = make_uint4(0, 0, 0, 0);
}
// mask rows of `ng` games: shared (rows of 113 words, no padding) -> global, 16 B at a time.
// first_game is a multiple of 32, so the global address is 16-byte aligned (32*452 = 16*904).
__device__ __forceinline__ void store_mask(uint32_t* __restrict__ mask, int first_game, int ng,
                                           const uint32_t* s_mask, int lane) {
  uint32_t* dst = mask + (size_t)first_game * kMaskWords;
  int words = ng * kMaskWords;
  int vec = words >> 2;
  const uint4* s4 = reinterpret_cast<const uint4*>(s_mask);
  uint4* d4 = reinterpret_cast<uint4*>(dst);
  for (int j = lane; j < vec; j += 32) d4[j] = s4[j];
  for (int j = (vec << 2) + lane; j < words; j += 32) dst[j] = s_mask[j];
}
// bf16 expansion table: entry e = 8 bf16 values (0x3F80 where bit set), element 0 lowest.
__device__ __forceinline__ void fill_lut(uint4* lut, int tid, int nthreads) {
  for (int e = tid; e < 256; e += nthreads) {
    uint4 v;
    v.x = ((e & 1) ? 0x3F80u : 0u) | ((e & 2) ? 0x3F800000u : 0u);
    v.y = ((e & 4) ? 0x3F80u : 0u) | ((e & 8) ? 0x3F800000u : 0u);
    v.z = ((e & 16) ? 0x3F80u : 0u) | ((e & 32) ? 0x3F800000u : 0u);
    v.w = ((e & 64) ? 0x3F80u : 0u) | ((e & 128) ? 0x3F800000u : 0u);
    lut[e] = v;
  }
}
// Observation of `ng` games from their bit streams: lane l writes chunk 32k+l, so every
// STG.128 of the warp covers 512 contiguous, sector-aligned bytes (8800 = 275 sectors).
__device__ __forceinline__ void expand_obs(uint16_t* __restrict__ obs, int first_game, int ng,
                                           const uint32_t* s_bits, const uint4* lut, int lane) {
  for (int gi = 0; gi < ng; ++gi) {
    const uint8_t* row = reinterpret_cast<const uint8_t*>(s_bits + gi * kBitsRowWords);
    uint4* dst = reinterpret_cast<uint4*>(obs + (size_t)(first_game + gi) * STRAT_OBS_ELEMS);
#pragma unroll
    for (int k = 0; k < 17; ++k) st_stream(dst + 32 * k + lane, lut[row[32 * k + lane]]);
    if (lane < kObsChunks - 544) st_stream(dst + 544 + lane, lut[row[544 + lane]]);
  }
}

__device__ __forceinline__ void raise_error(int* err, int code) { atomicCAS(err, 0, code); }

// One time step of the board-history ring (strat_history): where a state-advancing kernel
// records the state it starts from and the transition it makes.  lines == nullptr: no history.
struct HistSlot { uint32_t* lines; int16_t* act; int8_t* rew; uint8_t* done; };

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
__global__ void __launch_bounds__(128) k_import(int n, const uint8_t* __restrict__ canon, uint32_t* __restrict__ lines) {
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int g = blockIdx.x * 4 + warp;
  if (g >= n) return;
  uint32_t cw = reinterpret_cast<const uint32_t*>(canon + (size_t)g * 128)[lane];  // bytes 4l..4l+3
  uint32_t mine = 0;
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    int cell = 32 * r + lane;
    uint32_t w = __shfl_sync(0xffffffffu, cw, (cell >> 2) & 31);
    uint32_t b = cell < 100 ? (w >> (8 * (cell & 3))) & 0xFFu : 0u;
    uint32_t t = b & 15u;
    bool piece = t >= 1 && t <= 12;
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
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  __shared__ __align__(16) uint32_t s_mask[kBatch * kMaskWords];
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, P.num_games - first);
  zero_smem16(s_mask, kMaskBytes, lane);
  load_lines(lines, first, ng, s_state, lane);
  if (lane < ng) {
    Game g; read_game(s_state, lane, g);
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

template <bool kChase>
__global__ void __launch_bounds__(32) k_step(Params P, uint32_t* __restrict__ lines, const int16_t* __restrict__ actions,
                                             int8_t* __restrict__ reward, uint8_t* __restrict__ done, int* __restrict__ err,
                                             HistSlot hs) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, P.num_games - first);
  load_lines(lines, first, ng, s_state, lane);
  if (hs.lines) store_lines(hs.lines, first, ng, s_state, lane);  // the state this step starts from
  __syncwarp();
  if (lane < ng) {
    Game g; read_game(s_state, lane, g);
    int a = (int)actions[first + lane];
    StepOut o = step_game<true, false, kChase>(P, (uint32_t)(first + lane), g, a);
    if (o.illegal) raise_error(err, STRAT_ILLEGAL_ACTION);
    reward[first + lane] = (int8_t)o.reward;
    done[first + lane] = (uint8_t)o.done;
    if (hs.lines) { hs.act[first + lane] = (int16_t)a; hs.rew[first + lane] = (int8_t)o.reward; hs.done[first + lane] = (uint8_t)o.done; }
    write_game(s_state, lane, g);
  }
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

// ---- the fused hot path, warp-specialised and persistent -------------------------------
// One CTA = one LOGIC warp + one STORE warp sharing two staging buffers.  The logic warp
// walks batches of 32 games (thread per game): state line straight from global into
// registers, mask rows into the stage, mask/action/reward/done/state out, then the new
// state's 4400-bit observation stream into the same stage.  The store warp expands finished
// stages to bf16 and streams them out.  The two are decoupled by mbarriers, so on every SM
// observation stores of batch i flow while batch i+1 is still in its (latency-bound) rule
// logic; with one-warp CTAs all resident warps ran logic, then stores, in lockstep.
#ifdef STRAT_PROF  // developer build only (_work/): per-phase cycle counters
__device__ unsigned long long g_prof[32];
__device__ unsigned long long g_trace[8192 * 6];
__device__ __forceinline__ unsigned long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
__device__ __forceinline__ unsigned smid() { unsigned r; asm volatile("mov.u32 %0, %smid;" : "=r"(r)); return r; }
#define TRACE(b, k, v) do { if (lane == 0 && (b) < 8192) g_trace[(b) * 6 + (k)] = (v); } while (0)
#define PROF_T(v) long long v = clock64()
#define PROF_ADD(slot, a, b) do { if (lane == 0) atomicAdd(&g_prof[slot], (unsigned long long)((b) - (a))); } while (0)
#else
#define PROF_T(v)
#define PROF_ADD(slot, a, b)
#define TRACE(b, k, v)
#endif
constexpr int kWsStages = 2;
// Resident CTAs per SM of ONE launch.  Two consecutive launches are co-resident (6 CTAs x 35.7 KB
// of shared memory per SM): the later one trails the earlier one batch by batch, so the HBM
// write stream never drains between steps.  Measured on B200 at 65,536 games: 2 -> 88.8 us,
// 3 -> 87.8 us, 4 -> 90.3 us, 6 -> 93.1 us per step.
#ifndef STRAT_WS_CTAS_PER_SM
#define STRAT_WS_CTAS_PER_SM 3
#endif
constexpr int kWsCtasPerSm = STRAT_WS_CTAS_PER_SM;
constexpr int kWsStageWords = kBatch * kBitsRowWords;  // 4448 words = 17,792 B (mask rows need 3,616)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
  uint32_t a = smem_u32(b), ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(a), "r"(parity) : "memory");
  } while (!ok);
}
// Per-batch version flags in global memory: consecutive launches of the fused step overlap
// (programmatic dependent launch), ordered batch by batch instead of kernel by kernel.
__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(uint32_t* p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// whole warp: returns once *flag == want (lane 0 polls; the barrier orders the other lanes)
__device__ __forceinline__ void flag_wait(const uint32_t* flag, uint32_t want, int lane) {
  if (lane == 0)
    while (ld_acquire(flag) != want) __nanosleep(64);
  __syncwarp();
}
// whole warp: publish this warp's prior global writes, then set the flag
__device__ __forceinline__ void flag_set(uint32_t* flag, uint32_t v, int lane) {
  __syncwarp();
  if (lane == 0) { __threadfence(); st_release(flag, v); }
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
__device__ __forceinline__ void load_game_global(const uint32_t* __restrict__ lines, int game, Game& g,
                                                 uint32_t* __restrict__ hist_lines) {
  uint32_t W[32];
  const uint4* p = reinterpret_cast<const uint4*>(lines + (size_t)game * kLineWords);
#pragma unroll
  for (int k = 0; k < 8; ++k) { uint4 v = __ldcg(p + k); W[4 * k] = v.x; W[4 * k + 1] = v.y; W[4 * k + 2] = v.z; W[4 * k + 3] = v.w; }
  if (hist_lines) {  // board-history ring: the state this step starts from
    uint4* q = reinterpret_cast<uint4*>(hist_lines + (size_t)game * kLineWords);
#pragma unroll
    for (int k = 0; k < 8; ++k) __stcg(q + k, make_uint4(W[4 * k], W[4 * k + 1], W[4 * k + 2], W[4 * k + 3]));
  }
  unpack_line(W, g);
}
__device__ __forceinline__ void store_game_global(uint32_t* __restrict__ lines, int game, const Game& g) {
  uint32_t W[32];
  pack_line(g, W);
  uint4* p = reinterpret_cast<uint4*>(lines + (size_t)game * kLineWords);
#pragma unroll
  for (int k = 0; k < 8; ++k) __stcg(p + k, make_uint4(W[4 * k], W[4 * k + 1], W[4 * k + 2], W[4 * k + 3]));
}

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
  if ((rs >> lane) & 1u) {
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
    if (!side_can_ever_move(g, 0) || !side_can_ever_move(g, 1)) setup_game(P, (uint32_t)(first + lane), g);
  }
  __syncwarp();
}

// kExternal = false (strat_rollout_step): mask of the state -> uniform legal action -> step ->
//   observation of the new state; `actions` is an output.
// kExternal = true (strat_step_observe): `actions` is the caller's input (validated) -> step ->
//   mask AND observation of the new state: the data-collection loop of PAPER.md:232, 461-462
//   (ApplyActions, then ComputeLegalActionMask + ComputeInfostateTensor for the next policy call).
template <bool kExternal, bool kChase>
__global__ void __launch_bounds__(64) k_rollout_step(Params P, uint32_t* __restrict__ lines, uint32_t* __restrict__ mask,
                                                        int16_t* __restrict__ actions, int8_t* __restrict__ reward,
                                                        uint8_t* __restrict__ done, uint16_t* __restrict__ obs,
                                                        uint32_t* __restrict__ ticket, uint32_t* __restrict__ f_state,
                                                        uint32_t* __restrict__ f_obs, uint32_t version, HistSlot hs,
                                                        int* __restrict__ err) {
  __shared__ __align__(16) uint32_t s_stage[kWsStages][kWsStageWords];
  __shared__ __align__(8) uint2 s_lut[16];
  __shared__ __align__(8) uint64_t s_full[kWsStages], s_empty[kWsStages];
  __shared__ int s_batch[kWsStages];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nbatches = (P.num_games + kBatch - 1) / kBatch;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < kWsStages; ++s) { mbar_init(&s_full[s], 32); mbar_init(&s_empty[s], 32); }
  }
  fill_lut16(s_lut, threadIdx.x);
  __syncthreads();
  // Let the next launch of this kernel become resident now: it orders itself behind this one
  // batch by batch through f_state / f_obs (it never calls griddepcontrol.wait).
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (warp == 0) {
    // ------------------------------------------------ logic warp (thread per game)
    // batches: the first one is the CTA's own index, the rest are drawn from this launch's
    // ticket counter.  atomicInc wraps to 0 after exactly nbatches draws (nbatches - grid
    // successful ones + one failing draw per CTA), so the counter cleans up after itself.
    int b = blockIdx.x;
    for (int it = 0;; ++it) {
      const int stage = it % kWsStages, round = it / kWsStages;
      uint32_t* work = s_stage[stage];
      PROF_T(t0);
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
      PROF_T(t1);
      TRACE(b, 0, gtime()); TRACE(b, 4, smid()); TRACE(b, 5, blockIdx.x);
      zero_smem16(work, kMaskBytes, lane);
      Game g;
      int n = 0, cnt[4] = {0, 0, 0, 0};
      if (lane < ng) load_game_global(lines, first + lane, g, hs.lines);
      __syncwarp();
      PROF_T(t2);
      bool reset_me = false;
      if (!kExternal) {
        if (lane < ng && !g.done) n = legal_mask_row(g, g.ply & 1u, rules_of<kChase>(P), work + lane * kMaskWords, cnt,
                                                       kChase ? game_log(P, (uint32_t)(first + lane)) : nullptr);
        __syncwarp();
        PROF_T(t3);
        if (mask) store_mask(mask, first, ng, work, lane);
        PROF_T(t4);
        if (lane < ng) {
          int a = -1;
          if (n > 0) a = pick_action(work + lane * kMaskWords, cnt, n, action_draw(P, (uint32_t)(first + lane), g));
          StepOut o = step_game<false, true, kChase>(P, (uint32_t)(first + lane), g, a);  // a comes from this state's mask
          if (o.illegal) raise_error(err, STRAT_ILLEGAL_ACTION);
          if (actions) actions[first + lane] = (int16_t)a;
          if (reward) reward[first + lane] = (int8_t)o.reward;
          if (done) done[first + lane] = (uint8_t)o.done;
          if (hs.lines) { hs.act[first + lane] = (int16_t)a; hs.rew[first + lane] = (int8_t)o.reward; hs.done[first + lane] = (uint8_t)o.done; }
          reset_me = o.needs_reset;
        }
        uint32_t rs = __ballot_sync(0xffffffffu, reset_me);  // also: every lane is done with its mask row
        if (rs && P.pin) { if (reset_me) reset_game(P, (uint32_t)(first + lane), g); }
        else if (rs) coop_setup(P, first, rs, g, work, lane);
        if (lane < ng) store_game_global(lines, first + lane, g);
        flag_set(f_state + b, version, lane);  // state, mask, action, reward, done of this batch are out
        PROF_ADD(2, t2, t3); PROF_ADD(3, t3, t4);
      } else {
        if (lane < ng) {
          int a = (int)actions[first + lane];
          StepOut o = step_game<true, true, kChase>(P, (uint32_t)(first + lane), g, a);
          if (o.illegal) raise_error(err, STRAT_ILLEGAL_ACTION);
          reward[first + lane] = (int8_t)o.reward;
          done[first + lane] = (uint8_t)o.done;
          if (hs.lines) { hs.act[first + lane] = (int16_t)a; hs.rew[first + lane] = (int8_t)o.reward; hs.done[first + lane] = (uint8_t)o.done; }
          reset_me = o.needs_reset;
        }
        uint32_t rs = __ballot_sync(0xffffffffu, reset_me);
        if (rs && P.pin) { if (reset_me) reset_game(P, (uint32_t)(first + lane), g); }
        else if (rs) {  // the cooperative reset borrows the stage: clear its scratch again afterwards
          coop_setup(P, first, rs, g, work, lane);
          zero_smem16(work, kMaskBytes, lane);
          __syncwarp();
        }
        if (lane < ng) {
          store_game_global(lines, first + lane, g);
          if (!g.done)  // of the NEW state
            legal_mask_row(g, g.ply & 1u, rules_of<kChase>(P), work + lane * kMaskWords, cnt,
                           kChase ? game_log(P, (uint32_t)(first + lane)) : nullptr);
        }
        __syncwarp();
        if (mask) store_mask(mask, first, ng, work, lane);
        flag_set(f_state + b, version, lane);  // state, reward, done, mask of this batch are out
      }
      __syncwarp();  // the stage becomes bit streams
      PROF_T(t5);
      if (lane < ng) encode_bits(g, work + lane * kBitsRowWords);
      __syncwarp();
      PROF_T(t6);
      if (lane == 0) s_batch[stage] = b;
      mbar_arrive(&s_full[stage]);
      TRACE(b, 1, gtime());
      PROF_ADD(0, t0, t1); PROF_ADD(1, t1, t2); PROF_ADD(4, t2, t5);
      PROF_ADD(5, t5, t6); PROF_ADD(6, t0, t6); PROF_ADD(7, 0, 1);
    }
  } else {
    // ------------------------------------------------ store warp (lane per 16-byte chunk)
    for (int it = 0;; ++it) {
      const int stage = it % kWsStages, round = it / kWsStages;
      PROF_T(t0);
      mbar_wait(&s_full[stage], (uint32_t)round & 1u);
      const int b = s_batch[stage];
      if (b < 0) break;
      const int first = b * kBatch, ng = min(kBatch, P.num_games - first);
      flag_wait(f_obs + b, version - 1u, lane);  // write-after-write on a reused obs buffer
      PROF_T(t1);
      TRACE(b, 2, gtime());
      expand_obs16(obs, first, ng, s_stage[stage], s_lut, lane);
      flag_set(f_obs + b, version, lane);
      TRACE(b, 3, gtime());
      PROF_T(t2);
      mbar_arrive(&s_empty[stage]);
      PROF_ADD(8, t0, t1); PROF_ADD(9, t1, t2); PROF_ADD(10, 0, 1);
    }
  }
}

// `plies` plies of uniform-random legal play with the board in registers.  The 3600-bit mask is
// never built: the r-th legal action is found from the move bitboards (sample_action_direct).
constexpr int kScoutScratch = 9;  // 8 words per game, odd stride
template <bool kChase>
__global__ void __launch_bounds__(32) k_rollout_uniform(Params P, uint32_t* __restrict__ lines, int plies, int* __restrict__ err) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  __shared__ uint32_t s_scouts[kBatch * kScoutScratch];
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, P.num_games - first);
  load_lines(lines, first, ng, s_state, lane);
  if (lane < ng) {
    Game g; read_game(s_state, lane, g);
    for (int t = 0; t < plies; ++t) {
      if (g.done) break;  // auto_reset keeps games live; otherwise the game is frozen for good
      int a = sample_action_direct(g, g.ply & 1u, rules_of<kChase>(P), action_draw(P, (uint32_t)(first + lane), g),
                                   s_scouts + lane * kScoutScratch, kChase ? game_log(P, (uint32_t)(first + lane)) : nullptr);
      if (step_game<false, false, kChase>(P, (uint32_t)(first + lane), g, a).illegal) {
        raise_error(err, STRAT_ILLEGAL_ACTION);
        break;
      }
    }
    write_game(s_state, lane, g);
  }
  __syncwarp();
  store_lines(lines, first, ng, s_state, lane);
}

// ---- replay ring
template <typename T>
__global__ void k_copy(const T* __restrict__ src, T* __restrict__ dst, size_t count) {
  size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += stride) dst[i] = src[i];
}
// one warp per batch element: draw the record index, gather the record.
__global__ void __launch_bounds__(128) k_replay_sample(uint32_t k0, uint32_t k1, uint32_t d0, uint32_t d1, int batch,
                                                       uint32_t filled, const uint16_t* __restrict__ r_obs,
                                                       const uint32_t* __restrict__ r_mask, const int16_t* __restrict__ r_act,
                                                       const int8_t* __restrict__ r_rew, const uint8_t* __restrict__ r_done,
                                                       uint16_t* __restrict__ obs, uint32_t* __restrict__ mask,
                                                       int16_t* __restrict__ act, int8_t* __restrict__ rew, uint8_t* __restrict__ done) {
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int j = blockIdx.x * 4 + warp;
  if (j >= batch) return;
  uint32_t o[4];
  philox((uint32_t)(j >> 2), d0, d1, TAG_SAMPLE, k0, k1, o);
  uint32_t u = (j & 3) == 0 ? o[0] : (j & 3) == 1 ? o[1] : (j & 3) == 2 ? o[2] : o[3];
  size_t p = bounded(u, filled);
  if (obs) {
    const uint4* s = reinterpret_cast<const uint4*>(r_obs + p * STRAT_OBS_ELEMS);
    uint4* d = reinterpret_cast<uint4*>(obs + (size_t)j * STRAT_OBS_ELEMS);
    for (int q = lane; q < kObsChunks; q += 32) d[q] = __ldcs(s + q);
  }
  if (mask)
    for (int q = lane; q < kMaskWords; q += 32) mask[(size_t)j * kMaskWords + q] = r_mask[p * kMaskWords + q];
  if (lane == 0) {
    if (act) act[j] = r_act[p];
    if (rew) rew[j] = r_rew[p];
    if (done) done[j] = r_done[p];
  }
}

// ---- search-shaped batch
__global__ void __launch_bounds__(32) k_determinise(int num_out, int samples_per_root, uint32_t k0, uint32_t k1, uint32_t out_base,
                                                    const uint32_t* __restrict__ roots, uint32_t* __restrict__ out,
                                                    int* __restrict__ err) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, num_out - first);
  if (lane < ng) {
    int G = first + lane, r = G / samples_per_root;
    uint32_t W[32];
    const uint4* p = reinterpret_cast<const uint4*>(roots + (size_t)r * kLineWords);
#pragma unroll
    for (int k = 0; k < 8; ++k) { uint4 v = __ldg(p + k); W[4 * k] = v.x; W[4 * k + 1] = v.y; W[4 * k + 2] = v.z; W[4 * k + 3] = v.w; }
    Game root, g;
    unpack_line(W, root);
    if (!determinise_game(root, k0, k1, out_base + (uint32_t)G, g)) raise_error(err, STRAT_BAD_STATE);
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

// ---- one search step without networks (S3.7)
// Steps 1-2: slot G = r*rollouts + c*L + l of the output environment = root r, opponent
// configuration c (one DETERMINISE stream per configuration), l-th legal action applied (the
// forced first move).  Thread per slot; the root's mask row lives in shared memory.
template <bool kChase>
__global__ void __launch_bounds__(32) k_search_expand(Params Pr, Params Po, int rollouts, uint32_t k0, uint32_t k1,
                                                      const uint32_t* __restrict__ roots, uint32_t* __restrict__ out,
                                                      int* __restrict__ err) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  __shared__ __align__(16) uint32_t s_mask[kBatch * kMaskWords];
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, Po.num_games - first);
  zero_smem16(s_mask, kMaskBytes, lane);
  __syncwarp();
  if (lane < ng) {
    int G = first + lane, r = G / rollouts, s = G - r * rollouts;
    uint32_t W[32];
    const uint4* p = reinterpret_cast<const uint4*>(roots + (size_t)r * kLineWords);
#pragma unroll
    for (int k = 0; k < 8; ++k) { uint4 v = __ldg(p + k); W[4 * k] = v.x; W[4 * k + 1] = v.y; W[4 * k + 2] = v.z; W[4 * k + 3] = v.w; }
    Game root, g;
    unpack_line(W, root);
    uint32_t* row = s_mask + lane * kMaskWords;
    int cnt[4] = {0, 0, 0, 0};
    int L = root.done ? 0 : legal_mask_row(root, root.ply & 1u, rules_of<kChase>(Pr), row, cnt,
                                           kChase ? game_log(Pr, (uint32_t)r) : nullptr);
    int C = L > 0 ? max(1, rollouts / L) : 0;
    int used = min(C * L, rollouts);
    if (s >= used) {  // unused slot: the root, frozen
      g = root; g.done = 1; g.reason = 0; g.result = 0;
    } else {
      int c = s / L, l = s - c * L;
      if (!determinise_game(root, k0, k1, Po.game_base + (uint32_t)(r * rollouts + c), g)) raise_error(err, STRAT_BAD_STATE);
      step_game<false, false, kChase>(Po, (uint32_t)G, g, pick_rank(row, cnt, l));
    }
    write_game(s_state, lane, g);
  }
  __syncwarp();
  store_lines(out, first, ng, s_state, lane);
}

// Steps 3-4: per root, qhat(a) = mean over configurations of the value of the game that started
// with a (its result from the searcher's side, 0 while it runs), the magnet policy rho
// and eq. (8).  One CTA per root; float32 arithmetic.
constexpr int kPolicyThreads = 128;
template <bool kChase>
__global__ void __launch_bounds__(kPolicyThreads) k_search_policy(Params Pr, int rollouts, const uint32_t* __restrict__ roots,
                                                                  const uint32_t* __restrict__ games,
                                                                  const float* __restrict__ pi_theta, float alpha, float beta,
                                                                  float* __restrict__ qhat, float* __restrict__ rho,
                                                                  float* __restrict__ pi_search) {
  __shared__ __align__(16) uint32_t s_row[kMaskWords + 3];
  __shared__ int16_t s_legal[STRAT_NUM_ACTIONS];
  __shared__ int s_q[STRAT_NUM_ACTIONS];      // value sums, then (as float) the logits
  __shared__ int s_cell[100];
  __shared__ int s_L, s_pieces, s_sign;
  __shared__ float s_red[kPolicyThreads / 32];
  const int tid = threadIdx.x, r = blockIdx.x;
  float* q = qhat + (size_t)r * STRAT_NUM_ACTIONS;
  float* rh = rho + (size_t)r * STRAT_NUM_ACTIONS;
  float* ps = pi_search + (size_t)r * STRAT_NUM_ACTIONS;
  for (int a = tid; a < STRAT_NUM_ACTIONS; a += kPolicyThreads) { q[a] = 0.f; rh[a] = 0.f; ps[a] = 0.f; s_q[a] = 0; }
  for (int w = tid; w < kMaskWords + 3; w += kPolicyThreads) s_row[w] = 0;
  if (tid < 100) s_cell[tid] = 0;
  __syncthreads();
  if (tid == 0) {
    uint32_t W[32];
    const uint4* p = reinterpret_cast<const uint4*>(roots + (size_t)r * kLineWords);
#pragma unroll
    for (int k = 0; k < 8; ++k) { uint4 v = __ldg(p + k); W[4 * k] = v.x; W[4 * k + 1] = v.y; W[4 * k + 2] = v.z; W[4 * k + 3] = v.w; }
    Game root;
    unpack_line(W, root);
    int cnt[4] = {0, 0, 0, 0};
    int L = root.done ? 0 : legal_mask_row(root, root.ply & 1u, rules_of<kChase>(Pr), s_row, cnt,
                                           kChase ? game_log(Pr, (uint32_t)r) : nullptr);
    int k = 0, pieces = 0;
    for (int w = 0; w < kMaskWords; ++w)
      for (uint32_t b = s_row[w]; b; b &= b - 1) {
        int a = 32 * w + __ffs((int)b) - 1;
        s_legal[k++] = (int16_t)a;
        if (s_cell[a / 36]++ == 0) ++pieces;
      }
    s_L = L; s_pieces = pieces; s_sign = (root.ply & 1u) ? -1 : 1;
  }
  __syncthreads();
  const int L = s_L;
  if (L == 0) return;
  const int C = max(1, rollouts / L), used = min(C * L, rollouts);
  for (int s = tid; s < used; s += kPolicyThreads) {
    uint32_t f = games[((size_t)r * rollouts + s) * kLineWords + 19] >> 4;
    int v = (f & 1u) ? ((int)((f >> 4) & 3u) - 1) * s_sign : 0;
    if (v) atomicAdd(&s_q[s % L], v);
  }
  __syncthreads();
  float* logit = reinterpret_cast<float*>(s_q);
  float mx = -INFINITY;
  for (int l = tid; l < L; l += kPolicyThreads) {
    int a = s_legal[l];
    int n = (used - l + L - 1) / L;  // games that started with this action
    float qv = n ? (float)s_q[l] / (float)n : 0.f;
    float rv = 1.0f / ((float)s_pieces * (float)s_cell[a / 36]);
    float pv = pi_theta ? pi_theta[(size_t)r * STRAT_NUM_ACTIONS + a] : 1.0f / (float)L;
    q[a] = qv; rh[a] = rv;
    float lg = (qv + alpha * logf(rv) + beta * logf(pv)) / (alpha + beta);
    logit[l] = lg;
    mx = fmaxf(mx, lg);
  }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, off));
  if ((tid & 31) == 0) s_red[tid >> 5] = mx;
  __syncthreads();
  mx = fmaxf(fmaxf(s_red[0], s_red[1]), fmaxf(s_red[2], s_red[3]));
  __syncthreads();
  float z = 0.f;
  for (int l = tid; l < L; l += kPolicyThreads) { float e = expf(logit[l] - mx); logit[l] = e; z += e; }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) z += __shfl_xor_sync(0xffffffffu, z, off);
  if ((tid & 31) == 0) s_red[tid >> 5] = z;
  __syncthreads();
  z = (s_red[0] + s_red[1]) + (s_red[2] + s_red[3]);
  for (int l = tid; l < L; l += kPolicyThreads) ps[s_legal[l]] = logit[l] / z;
}

// A state copied in from elsewhere (history ring) has no move log here: it remembers 8 plies.
__global__ void __launch_bounds__(256) k_clear_logn(int n, uint32_t* __restrict__ lines) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g < n) lines[(size_t)g * kLineWords + 31] = 0;
}

__global__ void k_set_int(int* p, int v) { *p = v; }

// ------------------------------------------------------------------ host side
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline bool cfg_ok(const strat_config* c) {
  return c && c->num_games >= 1 && (c->variant == 0 || c->variant == 1) && c->max_plies >= 0 &&
         c->max_battleless >= 0 && (c->chase_rule == 0 || c->chase_rule == 1);
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
  P.pin = nullptr;
  return P;
}
inline int launch_status() { return cudaGetLastError() == cudaSuccess ? STRAT_OK : STRAT_CUDA_ERROR; }
inline int batches(int n) { return (n + kBatch - 1) / kBatch; }
// A launch cannot start before every CTA of the previous one has started, and each launch in
// flight holds at least one of the <= 32 x SMs resident CTA slots, so far fewer than kTicketRing
// launches are ever in flight and two launches never share a ticket counter.
constexpr int kTicketRing = 8192;
inline size_t sync_words(int n) { return (size_t)kTicketRing + 2 * (size_t)batches(n); }

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
// records [0,n) of the source go to ring positions (head+i) mod capacity: at most two runs.
template <typename T>
void push_array(const T* src, T* ring, size_t per_rec, int64_t head, int64_t cap, int64_t n, cudaStream_t s) {
  int64_t first = n < cap - head ? n : cap - head;
  copy_elems<T>(src, ring + (size_t)head * per_rec, (size_t)first * per_rec, s);
  copy_elems<T>(src + (size_t)first * per_rec, ring, (size_t)(n - first) * per_rec, s);
}

}  // namespace

struct strat_env {
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
};

// Circular buffer of `length` time steps: per step N device lines + N x
// (action i16, reward i8, done u8).
struct strat_history {
  int32_t num_games, length;
  int64_t cur;                 // CurrentStep: state updates recorded so far
  uint32_t* lines; int16_t* act; int8_t* rew; uint8_t* done;
  const strat_env* env;        // attached environment (live state = time step cur)
  strat::Params P;             // its rule parameters, kept for queries after a detach
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
}  // namespace

struct strat_replay {
  int64_t per_slot, slots, capacity, head, filled;
  uint16_t* obs; uint32_t* mask; int16_t* action; int8_t* reward; uint8_t* done;
};

namespace {
// Launch of the fused step.  Programmatic dependent launch: the launch may become resident while
// the previous launch in the stream is still running IF that one is also a fused step (the only
// kernel that executes griddepcontrol.launch_dependents); behind any other kernel the attribute
// changes nothing.  Ordering against the previous fused step is per batch (f_state / f_obs).
template <bool kExternal>
int launch_fused(strat_env* env, uint32_t* mask, int16_t* actions, int8_t* reward, uint8_t* done, uint16_t* obs,
                 void* stream) {
  const int nb = batches(env->P.num_games);
  // a launch that follows a policy kernel has the GPU to itself: one more CTA per SM
  const int per_sm = kExternal ? kWsCtasPerSm + 1 : kWsCtasPerSm;
  const int grid = nb < env->num_sms * per_sm ? nb : env->num_sms * per_sm;
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)grid); lc.blockDim = dim3(64); lc.dynamicSmemBytes = 0; lc.stream = (cudaStream_t)stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = 1;
  const uint32_t version = env->version + 1;
  auto kernel = env->P.chase_rule ? k_rollout_step<kExternal, true> : k_rollout_step<kExternal, false>;
  if (cudaLaunchKernelEx(&lc, kernel, env->P, env->lines, mask, actions, reward, done, obs,
                         env->tickets + (version % kTicketRing), env->f_state, env->f_obs, version,
                         hist_slot(env->hist), env->err) != cudaSuccess)
    return STRAT_CUDA_ERROR;
  env->version = version;
  if (env->hist) env->hist->cur += 1;
  return STRAT_OK;
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
    default: return "unknown error";
  }
}

size_t strat_workspace_bytes(const strat_config* cfg) {
  if (!cfg_ok(cfg)) return 0;
  return align_up((size_t)cfg->num_games * STRAT_LINE_BYTES, 256) + 256 + align_up(sync_words(cfg->num_games) * 4, 256) +
         (cfg->chase_rule ? (size_t)cfg->num_games * kLogPlies * 2 : 0);  // move logs: the chasing rule's memory
}

int strat_create(const strat_config* cfg, void* workspace_dev, size_t bytes, void* stream, strat_env** out) {
  if (!cfg_ok(cfg) || !workspace_dev || !out || bytes < strat_workspace_bytes(cfg) ||
      ((uintptr_t)workspace_dev & 255) != 0)
    return STRAT_BAD_ARG;
  if (cudaSetDevice(cfg->device) != cudaSuccess) return STRAT_CUDA_ERROR;
  strat_env* e = new (std::nothrow) strat_env;
  if (!e) return STRAT_BAD_ARG;
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
  if (cfg->chase_rule)
    e->P.movelog = reinterpret_cast<uint16_t*>(reinterpret_cast<uint8_t*>(e->tickets) + align_up(sync_words(cfg->num_games) * 4, 256));
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
  delete env;
  return STRAT_OK;
}

int strat_reset(strat_env* env, uint64_t seed, void* stream) {
  if (!env) return STRAT_BAD_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  env->cfg.seed = seed;
  const uint32_t* pin = env->P.pin;
  uint16_t* movelog = env->P.movelog;
  env->P = make_params(env->cfg);
  env->P.pin = pin;
  env->P.movelog = movelog;
  k_set_int<<<1, 1, 0, s>>>(env->err, 0);
  k_reset<<<batches(env->P.num_games), 32, 0, s>>>(env->P, env->lines);
  return launch_status();
}

int strat_reset_from(strat_env* env, const uint8_t* boards, void* stream) {
  if (!env || !boards) return STRAT_BAD_ARG;
  int n = env->P.num_games;
  k_import<<<(n + 3) / 4, 128, 0, (cudaStream_t)stream>>>(n, boards, env->lines);
  return launch_status();
}

int strat_pin_reset_state(strat_env* env, void* pin_lines_dev, const uint8_t* boards, void* stream) {
  if (!env) return STRAT_BAD_ARG;
  if (!boards) { env->P.pin = nullptr; return STRAT_OK; }
  if (!pin_lines_dev || ((uintptr_t)pin_lines_dev & 15) != 0) return STRAT_BAD_ARG;
  int n = env->P.num_games;
  k_import<<<(n + 3) / 4, 128, 0, (cudaStream_t)stream>>>(n, boards, reinterpret_cast<uint32_t*>(pin_lines_dev));
  env->P.pin = reinterpret_cast<const uint32_t*>(pin_lines_dev);
  return launch_status();
}

int strat_get_boards(const strat_env* env, uint8_t* boards, void* stream) {
  if (!env || !boards) return STRAT_BAD_ARG;
  int n = env->P.num_games;
  k_export<<<(n + 3) / 4, 128, 0, (cudaStream_t)stream>>>(n, env->lines, boards);
  return launch_status();
}

int strat_legal_mask(const strat_env* env, uint32_t* mask, void* stream) {
  if (!env || !mask) return STRAT_BAD_ARG;
  if (env->P.chase_rule) k_legal_mask<true><<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, mask);
  else k_legal_mask<false><<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, mask);
  return launch_status();
}

int strat_sample_uniform(const strat_env* env, const uint32_t* mask, int16_t* actions, void* stream) {
  if (!env || !mask || !actions) return STRAT_BAD_ARG;
  int n = env->P.num_games;
  k_sample_uniform<<<(n + 3) / 4, 128, 0, (cudaStream_t)stream>>>(env->P, env->lines, mask, actions);
  return launch_status();
}

int strat_step(strat_env* env, const int16_t* actions, int8_t* reward, uint8_t* done, void* stream) {
  if (!env || !actions || !reward || !done) return STRAT_BAD_ARG;
  if (env->P.chase_rule)
    k_step<true><<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, actions, reward, done,
                                                                             env->err, hist_slot(env->hist));
  else
    k_step<false><<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, actions, reward, done,
                                                                              env->err, hist_slot(env->hist));
  if (env->hist) env->hist->cur += 1;
  return launch_status();
}

int strat_encode_obs(const strat_env* env, uint16_t* obs, void* stream) {
  if (!env || !obs) return STRAT_BAD_ARG;
  k_encode_obs<<<batches(env->P.num_games), 32, 0, (cudaStream_t)stream>>>(env->P, env->lines, obs);
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
  if (env->hist) return STRAT_BAD_STATE;  // on-chip plies are not recorded
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
  k_set_int<<<1, 1, 0, (cudaStream_t)stream>>>(env->err, 0);
  return launch_status();
}

// ---- replay ring
int strat_replay_layout(int32_t per_slot, int32_t slots, size_t off[5]) {
  if (per_slot <= 0 || slots <= 0 || !off) return STRAT_BAD_ARG;
  size_t C = (size_t)per_slot * (size_t)slots, p = 0;
  off[0] = p; p += align_up(C * STRAT_OBS_ELEMS * 2, 256);
  off[1] = p; p += align_up(C * STRAT_MASK_WORDS * 4, 256);
  off[2] = p; p += align_up(C * 2, 256);
  off[3] = p; p += align_up(C, 256);
  off[4] = p;
  return STRAT_OK;
}

size_t strat_replay_bytes(int32_t per_slot, int32_t slots) {
  size_t off[5];
  if (strat_replay_layout(per_slot, slots, off) != STRAT_OK) return 0;
  return off[4] + align_up((size_t)per_slot * (size_t)slots, 256);
}

int strat_replay_create(void* mem_dev, size_t bytes, int32_t per_slot, int32_t slots, strat_replay** out) {
  size_t need = strat_replay_bytes(per_slot, slots);
  if (!mem_dev || !out || need == 0 || bytes < need || ((uintptr_t)mem_dev & 255) != 0) return STRAT_BAD_ARG;
  strat_replay* r = new (std::nothrow) strat_replay;
  if (!r) return STRAT_BAD_ARG;
  size_t off[5];
  strat_replay_layout(per_slot, slots, off);
  uint8_t* b = reinterpret_cast<uint8_t*>(mem_dev);
  r->per_slot = per_slot; r->slots = slots; r->capacity = (int64_t)per_slot * slots; r->head = 0; r->filled = 0;
  r->obs = reinterpret_cast<uint16_t*>(b + off[0]); r->mask = reinterpret_cast<uint32_t*>(b + off[1]);
  r->action = reinterpret_cast<int16_t*>(b + off[2]); r->reward = reinterpret_cast<int8_t*>(b + off[3]);
  r->done = b + off[4];
  *out = r;
  return STRAT_OK;
}

int strat_replay_destroy(strat_replay* r) { delete r; return STRAT_OK; }

int strat_replay_push(strat_replay* r, const uint16_t* obs, const uint32_t* mask, const int16_t* action,
                      const int8_t* reward, const uint8_t* done, int32_t n, void* stream) {
  if (!r || !obs || !mask || !action || !reward || !done || n < 0 || n > r->capacity) return STRAT_BAD_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  push_array<uint16_t>(obs, r->obs, STRAT_OBS_ELEMS, r->head, r->capacity, n, s);
  push_array<uint32_t>(mask, r->mask, STRAT_MASK_WORDS, r->head, r->capacity, n, s);
  push_array<int16_t>(action, r->action, 1, r->head, r->capacity, n, s);
  push_array<int8_t>(reward, r->reward, 1, r->head, r->capacity, n, s);
  push_array<uint8_t>(done, r->done, 1, r->head, r->capacity, n, s);
  r->head = (r->head + n) % r->capacity;
  r->filled = r->filled + n > r->capacity ? r->capacity : r->filled + n;
  return launch_status();
}

int strat_replay_reserve(strat_replay* r, int32_t n, int32_t ahead, uint16_t** obs, uint32_t** mask) {
  if (!r || !obs || !mask || n <= 0 || n > r->capacity || r->capacity % n != 0 || r->head % n != 0 || ahead < 0)
    return STRAT_BAD_ARG;
  size_t first = (size_t)((r->head + (int64_t)ahead * n) % r->capacity);
  *obs = r->obs + first * STRAT_OBS_ELEMS;
  *mask = r->mask + first * STRAT_MASK_WORDS;
  return STRAT_OK;
}

int strat_replay_commit(strat_replay* r, const int16_t* action, const int8_t* reward, const uint8_t* done, int32_t n,
                        void* stream) {
  if (!r || !action || !reward || !done || n <= 0 || n > r->capacity || r->capacity % n != 0 || r->head % n != 0)
    return STRAT_BAD_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  copy_elems<int16_t>(action, r->action + r->head, (size_t)n, s);
  copy_elems<int8_t>(reward, r->reward + r->head, (size_t)n, s);
  copy_elems<uint8_t>(done, r->done + r->head, (size_t)n, s);
  r->head = (r->head + n) % r->capacity;
  r->filled = r->filled + n > r->capacity ? r->capacity : r->filled + n;
  return launch_status();
}

int strat_replay_sample(const strat_replay* r, uint64_t seed, uint64_t draw_index, int32_t batch, uint16_t* obs,
                        uint32_t* mask, int16_t* action, int8_t* reward, uint8_t* done, void* stream) {
  if (!r || batch < 0) return STRAT_BAD_ARG;
  if (r->filled == 0) return STRAT_BAD_STATE;
  if (batch == 0) return STRAT_OK;
  k_replay_sample<<<(batch + 3) / 4, 128, 0, (cudaStream_t)stream>>>(
      (uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)draw_index, (uint32_t)(draw_index >> 32), batch,
      (uint32_t)r->filled, r->obs, r->mask, r->action, r->reward, r->done, obs, mask, action, reward, done);
  return launch_status();
}

int strat_replay_state(const strat_replay* r, int64_t* head, int64_t* filled) {
  if (!r) return STRAT_BAD_ARG;
  if (head) *head = r->head;
  if (filled) *filled = r->filled;
  return STRAT_OK;
}

// ---- board-history ring (Table S1)
size_t strat_history_bytes(int32_t num_games, int32_t length) {
  if (num_games <= 0 || length <= 0) return 0;
  size_t n = (size_t)num_games, T = (size_t)length;
  return align_up(T * n * STRAT_LINE_BYTES, 256) + align_up(T * n * 2, 256) + 2 * align_up(T * n, 256);
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
  h->done = b;
  *out = h;
  return STRAT_OK;
}

int strat_history_destroy(strat_history* h) {
  if (h && h->env) const_cast<strat_env*>(h->env)->hist = nullptr;
  delete h;
  return STRAT_OK;
}

int strat_history_attach(strat_env* env, strat_history* h) {
  if (!env) return STRAT_BAD_ARG;
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
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !mask) return STRAT_BAD_ARG;
  Params P = h->env ? h->env->P : h->P;
  if (t != h->cur) P.movelog = nullptr;  // a past state is judged with the 8 plies its line remembers
  if (P.chase_rule) k_legal_mask<true><<<batches(h->num_games), 32, 0, (cudaStream_t)stream>>>(P, L, mask);
  else k_legal_mask<false><<<batches(h->num_games), 32, 0, (cudaStream_t)stream>>>(P, L, mask);
  return launch_status();
}

int strat_history_encode_obs(const strat_history* h, int64_t t, uint16_t* obs, void* stream) {
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !obs) return STRAT_BAD_ARG;
  const Params& P = h->env ? h->env->P : h->P;
  k_encode_obs<<<batches(h->num_games), 32, 0, (cudaStream_t)stream>>>(P, L, obs);
  return launch_status();
}

int strat_history_get_boards(const strat_history* h, int64_t t, uint8_t* boards, void* stream) {
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !boards) return STRAT_BAD_ARG;
  k_export<<<(h->num_games + 3) / 4, 128, 0, (cudaStream_t)stream>>>(h->num_games, L, boards);
  return launch_status();
}

int strat_history_transition(const strat_history* h, int64_t t, const int16_t** actions, const int8_t** reward,
                             const uint8_t** done) {
  if (!h || t < 0 || t >= h->cur || t < h->cur - h->length) return STRAT_BAD_ARG;
  size_t off = (size_t)(t % h->length) * (size_t)h->num_games;
  if (actions) *actions = h->act + off;
  if (reward) *reward = h->rew + off;
  if (done) *done = h->done + off;
  return STRAT_OK;
}

int strat_history_info(const strat_history* h, int64_t t, int32_t* info, void* stream) {
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !info || ((uintptr_t)info & 15) != 0) return STRAT_BAD_ARG;
  k_line_info<<<(h->num_games + 255) / 256, 256, 0, (cudaStream_t)stream>>>(h->num_games, L, info);
  return launch_status();
}

int strat_history_restore(const strat_history* h, int64_t t, strat_env* env, void* stream) {
  const uint32_t* L = hist_lines_at(h, t);
  if (!L || !env || env->P.num_games != h->num_games) return STRAT_BAD_ARG;
  if (L != env->lines) {
    copy_elems<uint32_t>(L, env->lines, (size_t)h->num_games * kLineWords, (cudaStream_t)stream);
    k_clear_logn<<<(h->num_games + 255) / 256, 256, 0, (cudaStream_t)stream>>>(h->num_games, env->lines);
  }
  return launch_status();
}

// ---- search-shaped batch
int strat_determinise(const strat_env* roots, int32_t samples_per_root, uint64_t seed, strat_env* out, void* stream) {
  if (!roots || !out || samples_per_root <= 0 ||
      (int64_t)roots->P.num_games * samples_per_root != (int64_t)out->P.num_games)
    return STRAT_BAD_ARG;
  k_determinise<<<batches(out->P.num_games), 32, 0, (cudaStream_t)stream>>>(
      out->P.num_games, samples_per_root, (uint32_t)seed, (uint32_t)(seed >> 32), out->P.game_base, roots->lines,
      out->lines, out->err);
  return launch_status();
}

int strat_search_expand(const strat_env* roots, int32_t rollouts, uint64_t seed, strat_env* out, void* stream) {
  if (!roots || !out || rollouts <= 0 || (int64_t)roots->P.num_games * rollouts != (int64_t)out->P.num_games ||
      out->P.auto_reset || out->hist)
    return STRAT_BAD_ARG;
  auto kernel = roots->P.chase_rule ? k_search_expand<true> : k_search_expand<false>;
  kernel<<<batches(out->P.num_games), 32, 0, (cudaStream_t)stream>>>(roots->P, out->P, rollouts, (uint32_t)seed,
                                                                     (uint32_t)(seed >> 32), roots->lines, out->lines, out->err);
  return launch_status();
}

int strat_search_policy(const strat_env* roots, const strat_env* games, int32_t rollouts, const float* pi_theta,
                        float alpha, float beta, float* qhat, float* rho, float* pi_search, void* stream) {
  if (!roots || !games || rollouts <= 0 || (int64_t)roots->P.num_games * rollouts != (int64_t)games->P.num_games ||
      !qhat || !rho || !pi_search || !(alpha + beta > 0.f))
    return STRAT_BAD_ARG;
  auto kernel = roots->P.chase_rule ? k_search_policy<true> : k_search_policy<false>;
  kernel<<<roots->P.num_games, kPolicyThreads, 0, (cudaStream_t)stream>>>(roots->P, rollouts, roots->lines, games->lines,
                                                                         pi_theta, alpha, beta, qhat, rho, pi_search);
  return launch_status();
}

int strat_reduce_returns(const strat_env* games, const uint8_t* root_side, int32_t samples_per_root, int32_t* out,
                         void* stream) {
  if (!games || !root_side || !out || samples_per_root <= 0 || games->P.num_games % samples_per_root != 0)
    return STRAT_BAD_ARG;
  int R = games->P.num_games / samples_per_root;
  k_reduce_returns<<<R, 256, 0, (cudaStream_t)stream>>>(games->lines, root_side, samples_per_root, out);
  return launch_status();
}

#ifdef STRAT_PROF
int strat_debug_prof(unsigned long long* out_host, int clear) {
  if (cudaMemcpyFromSymbol(out_host, g_prof, sizeof(g_prof)) != cudaSuccess) return STRAT_CUDA_ERROR;
  if (clear) { unsigned long long z[32] = {0}; cudaMemcpyToSymbol(g_prof, z, sizeof(z)); }
  return STRAT_OK;
}
int strat_debug_trace(unsigned long long* out_host) {
  return cudaMemcpyFromSymbol(out_host, g_trace, sizeof(g_trace)) == cudaSuccess ? STRAT_OK : STRAT_CUDA_ERROR;
}
#endif

}  // extern "C"
