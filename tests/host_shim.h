// Host stand-ins for the primitives paper_2511_07312_b200/csrc/strat_game.cuh is written in, so that the
// per-game rule code can be compiled for a CPU and compared with the oracle by the CPU-only test run
// (tests/host_harness.cpp, tests/test_device_logic_on_host.py).  Test infrastructure: nothing in the product
// includes or links this.
#pragma once
#include <stdint.h>
#define STRAT_PRIMITIVES_PROVIDED
#define SD static inline
static inline int sd_popc(uint32_t x) { return __builtin_popcount(x); }
static inline int sd_ffs(uint32_t x) { return __builtin_ffs((int)x); }
static inline int sd_clz(uint32_t x) { return x ? __builtin_clz(x) : 32; }
static inline uint32_t sd_mulhi(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) >> 32); }
static inline uint32_t sd_fsr(uint32_t lo, uint32_t hi, int s) { return (uint32_t)((((uint64_t)hi << 32) | lo) >> s); }
static inline uint32_t sd_fsl(uint32_t lo, uint32_t hi, int s) { return (uint32_t)(((((uint64_t)hi << 32) | lo) << s) >> 32); }
static inline int min(int a, int b) { return a < b ? a : b; }
static inline int max(int a, int b) { return a > b ? a : b; }
#define STRAT_UNROLL
static inline uint16_t sd_ldlog(const uint16_t* p) { return *p; }
static inline void sd_stlog(uint16_t* p, uint16_t v) { *p = v; }
static inline uint32_t sd_ld32(const uint32_t* p) { return *p; }
static inline void sd_st32(uint32_t* p, uint32_t v) { *p = v; }
static inline void sd_or32(uint32_t* p, uint32_t v) { *p |= v; }
static inline void sd_st16(uint32_t* words, int half, uint32_t v) { reinterpret_cast<uint16_t*>(words)[half] = (uint16_t)v; }
static inline void sd_ld128(const uint32_t* p, uint32_t& a, uint32_t& b, uint32_t& c, uint32_t& d) { a = p[0]; b = p[1]; c = p[2]; d = p[3]; }
static inline void sd_st128(uint32_t* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) { p[0] = a; p[1] = b; p[2] = c; p[3] = d; }
