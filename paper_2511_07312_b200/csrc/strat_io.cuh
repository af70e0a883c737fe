// strat_io.cuh - batch constants, PTX helpers, warp-cooperative I/O between global and shared memory
// Part of libstrat.so (one translation unit: strat.cu includes these in order).
#pragma once

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
// State lines are the only data a step reads back (the next step, 128 B per game): they are kept in the
// L2 with the evict_last policy, next to gigabytes of evict-first output that stream through it.
#ifndef STRAT_LINES_POLICY
#define STRAT_LINES_POLICY 1
#endif
__device__ __forceinline__ uint64_t lines_policy() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ uint4 ld_line16(const uint4* p, uint64_t pol) {
  uint4 v;
#if STRAT_LINES_POLICY
  asm volatile("ld.global.cg.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(pol) : "memory");
#else
  v = __ldcg(p);
#endif
  return v;
}
__device__ __forceinline__ void st_line16(uint4* p, uint4 v, uint64_t pol) {
#if STRAT_LINES_POLICY
  asm volatile("st.global.cg.L2::cache_hint.v4.u32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(pol) : "memory");
#else
  __stcg(p, v);
#endif
}

// ------------------------------------------------------------------ flags in global memory (between overlapping launches)
__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(uint32_t* p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ------------------------------------------------------------------ mbarriers (producer / consumer warps of one CTA)
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
  for (int j = lane; j < vec; j += 32) st_stream(d4 + j, s4[j]);  // evict-first like the observations
  for (int j = (vec << 2) + lane; j < words; j += 32) __stcs(dst + j, s_mask[j]);
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

// One game's line straight from global memory into registers (each lane reads its own 128 B =
// four full sectors; ld.global.cg because consecutive fused steps overlap on the device).
__device__ __forceinline__ void load_game_global(const uint32_t* __restrict__ lines, int game, Game& g,
                                                 uint32_t* __restrict__ hist_lines) {
  uint32_t W[32];
  const uint4* p = reinterpret_cast<const uint4*>(lines + (size_t)game * kLineWords);
  const uint64_t pol = lines_policy();
#pragma unroll
  for (int k = 0; k < 8; ++k) { uint4 v = ld_line16(p + k, pol); W[4 * k] = v.x; W[4 * k + 1] = v.y; W[4 * k + 2] = v.z; W[4 * k + 3] = v.w; }
  if (hist_lines) {  // board-history ring: the state this step starts from
    uint4* q = reinterpret_cast<uint4*>(hist_lines + (size_t)game * kLineWords);
#pragma unroll
    for (int k = 0; k < 8; ++k) __stcs(q + k, make_uint4(W[4 * k], W[4 * k + 1], W[4 * k + 2], W[4 * k + 3]));  // write-once: evict-first
  }
  unpack_line(W, g);
}
__device__ __forceinline__ void raise_error(int* err, int code) { atomicCAS(err, 0, code); }

// One time step of the board-history ring (strat_history): where a state-advancing kernel
// records the state it starts from and the transition it makes.  lines == nullptr: no history.
struct HistSlot { uint32_t* lines; int16_t* act; int8_t* rew; uint8_t* done; };


}  // namespace
