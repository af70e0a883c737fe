// strat_game.cuh — per-game Stratego logic on 100-bit bitboards, one thread per game.
//
// The device keeps each game as ONE 128-byte line in a bit-sliced form: seven 100-bit
// planes (type bits T0..T3, owner, moved, revealed) in four 32-bit words each, with the
// 8-ply history, flags and counters packed into the spare bits (layout below).  Every
// rule then becomes a handful of 32-bit logic ops on whole boards instead of loops over
// cells: legal single-step moves are four shifted ANDs, the 28 board planes of the
// observation are LOP3 combinations of the seven state planes.
//
// Rules follow PAPER.md:208-212 (movement, battle, win/draw, two-square rule) with the
// readings R#1..R#23 listed in DESIGN.md.
#pragma once
#include <stdint.h>

// The bit and memory primitives the rule code is written in (SD, STRAT_UNROLL, sd_*).  A test harness may
// supply its own before including this file (STRAT_PRIMITIVES_PROVIDED: tests/host_shim.h runs the rule code
// on a CPU against the oracle); the library itself only ever uses the device definitions below.
#ifndef STRAT_PRIMITIVES_PROVIDED
#define STRAT_UNROLL _Pragma("unroll")
#define SD __device__ __forceinline__
SD int sd_popc(uint32_t x) { return __popc(x); }
SD int sd_ffs(uint32_t x) { return __ffs((int)x); }
SD int sd_clz(uint32_t x) { return __clz((int)x); }
SD uint32_t sd_mulhi(uint32_t a, uint32_t b) { return __umulhi(a, b); }
SD uint32_t sd_fsr(uint32_t lo, uint32_t hi, int s) { return __funnelshift_r(lo, hi, s); }
SD uint32_t sd_fsl(uint32_t lo, uint32_t hi, int s) { return __funnelshift_l(lo, hi, s); }
// move-log accesses go to L2: consecutive launches of the fused step overlap on the device
SD uint16_t sd_ldlog(const uint16_t* p) { return __ldcg(p); }
SD void sd_stlog(uint16_t* p, uint16_t v) { __stcg(p, v); }
SD uint32_t sd_ld32(const uint32_t* p) { return __ldcg(p); }
SD void sd_st32(uint32_t* p, uint32_t v) { __stcg(p, v); }
// tracker bits are OR-ed in at the L2 without reading them back (RED.OR: nothing to wait for)
SD void sd_or32(uint32_t* p, uint32_t v) { atomicOr(p, v); }
SD void sd_st16(uint32_t* words, int half, uint32_t v) { __stcg(reinterpret_cast<uint16_t*>(words) + half, (uint16_t)v); }
SD void sd_ld128(const uint32_t* p, uint32_t& a, uint32_t& b, uint32_t& c, uint32_t& d) {
  uint4 v = __ldcg(reinterpret_cast<const uint4*>(p)); a = v.x; b = v.y; c = v.z; d = v.w;
}
SD void sd_st128(uint32_t* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) { __stcg(reinterpret_cast<uint4*>(p), make_uint4(a, b, c, d)); }
#endif

namespace strat {

constexpr int kLineWords = 32;
constexpr int kMaskWords = 113;
constexpr int kObsStreamWords = 138;  // 4400 bits
constexpr int T_SPY = 1, T_SCOUT = 2, T_MINER = 3, T_MARSHAL = 10, T_FLAG = 11, T_BOMB = 12;
constexpr int REASON_FLAG = 1, REASON_NOMOVE_WIN = 2, REASON_NOMOVE_DRAW = 3, REASON_PLY_CAP = 4,
              REASON_BATTLELESS = 5;
constexpr uint32_t TAG_SETUP_RED = 0, TAG_SETUP_BLUE = 1, TAG_ACTION = 2, TAG_SAMPLE = 3, TAG_DETERMINISE = 4;
constexpr uint32_t kHistNone = 0x3FFF;
constexpr int kLogPlies = 64;  // move-log entries per game; the chasing rule looks back 63 plies at most
constexpr int kMaxBans = 63;
constexpr int kMaxScouts = 8;  // per side; imports and setup pools with more are refused (count_actions' list)

struct Params {  // per-environment constants handed to every kernel by value
  uint32_t key0, key1;     // Philox key = seed
  uint32_t game_base;      // global index of local game 0
  int32_t num_games;
  int32_t variant;
  int32_t ply_cap;         // effective: 1..65535
  int32_t max_battleless;  // 0 = off
  int32_t auto_reset;
  int32_t two_square;
  int32_t chase_rule;      // continuous-chasing rule (R#28)
  uint16_t* movelog;       // [num_games][64] plies played since the state was loaded (chase_rule only), or null
  const uint8_t* pool;     // custom setups [2][pool_size][40] type codes (red, then blue), or null (R#30)
  int32_t pool_size;
  const uint32_t* pin;     // device lines [num_games][32] a finished game restarts from, or null (R#27)
  const uint16_t* pin_log; // [num_games][64] move logs that belong to the pinned lines, or null
  uint32_t* track;         // [num_games][512] trackers of the paper's information state (S2), or null
};

// Rule switches handed to the move generators: bit 0 two-square rule, bit 1 chasing rule.
constexpr int RULE_TWO_SQUARE = 1, RULE_CHASE = 2;
// kChase = false compiles the (rare, register-hungry) chasing-rule paths out of a kernel.
template <bool kChase> SD int rules_of(const Params& P) {
  return (P.two_square ? RULE_TWO_SQUARE : 0) | ((kChase && P.chase_rule) ? RULE_CHASE : 0);
}

// The move log of one game (chasing rule's memory), or null when the environment keeps none.
SD uint16_t* game_log(const Params& P, uint32_t local_game) {
  return P.movelog ? P.movelog + (size_t)local_game * 64 : nullptr;
}
// A state that is copied, pinned or restored takes the plies that led to it along.
SD void copy_game_log(const uint16_t* src, uint16_t* dst) {
  const uint32_t* s = reinterpret_cast<const uint32_t*>(src);
  uint32_t* d = reinterpret_cast<uint32_t*>(dst);
  STRAT_UNROLL
  for (int k = 0; k < kLogPlies / 2; k += 4) {
    uint32_t a, b, c, e;
    sd_ld128(s + k, a, b, c, e);
    sd_st128(d + k, a, b, c, e);
  }
}

// ------------------------------------------------------------------ 100-bit boards
struct BB { uint32_t w[4]; };  // cell c -> word c>>5, bit c&31; w[3] uses bits 0..3

constexpr uint32_t col_word(int col, int i) {
  uint32_t m = 0;
  for (int r = 0; r < 10; ++r) {
    int c = 10 * r + col;
    if ((c >> 5) == i) m |= 1u << (c & 31);
  }
  return m;
}
constexpr uint32_t lake_word(int i) {
  uint32_t m = 0;
  const int L[8] = {42, 43, 46, 47, 52, 53, 56, 57};
  for (int k = 0; k < 8; ++k)
    if ((L[k] >> 5) == i) m |= 1u << (L[k] & 31);
  return m;
}
// Board constants as literals (device code cannot index host constexpr arrays); the
// static_asserts tie them to the geometry.
#define STRAT_LAKE_W1 0x0330CC00u   /* cells 42,43,46,47,52,53,56,57 all lie in word 1 */
static_assert(lake_word(0) == 0 && lake_word(1) == STRAT_LAKE_W1 && lake_word(2) == 0 && lake_word(3) == 0, "lakes");
static_assert(col_word(0, 0) == 0x40100401u && col_word(0, 1) == 0x10040100u && col_word(0, 2) == 0x04010040u &&
              col_word(0, 3) == 0u, "col 0");
static_assert(col_word(9, 0) == 0x20080200u && col_word(9, 1) == 0x08020080u && col_word(9, 2) == 0x02008020u &&
              col_word(9, 3) == 0x8u, "col 9");
enum BoardConst { kLake, kNotLake, kNotCol0, kNotCol9 };
SD bool is_lake_cell(int c) { return (c >> 5) == 1 && ((STRAT_LAKE_W1 >> (c & 31)) & 1u); }

SD BB bb_zero() { BB r; r.w[0] = r.w[1] = r.w[2] = r.w[3] = 0; return r; }
SD BB bb_and(BB a, BB b) { BB r;
STRAT_UNROLL
for (int i = 0; i < 4; ++i) r.w[i] = a.w[i] & b.w[i]; return r; }
SD BB bb_or(BB a, BB b) { BB r;
STRAT_UNROLL
for (int i = 0; i < 4; ++i) r.w[i] = a.w[i] | b.w[i]; return r; }
SD BB bb_andn(BB a, BB b) { BB r;
STRAT_UNROLL
for (int i = 0; i < 4; ++i) r.w[i] = a.w[i] & ~b.w[i]; return r; }  // a & ~b
SD BB bb_const(BoardConst k) {
  BB r;
  if (k == kLake)         { r.w[0] = 0u;           r.w[1] = STRAT_LAKE_W1;  r.w[2] = 0u;           r.w[3] = 0u; }
  else if (k == kNotLake) { r.w[0] = 0xFFFFFFFFu;  r.w[1] = ~STRAT_LAKE_W1; r.w[2] = 0xFFFFFFFFu;  r.w[3] = 0xFu; }
  else if (k == kNotCol0) { r.w[0] = ~0x40100401u; r.w[1] = ~0x10040100u;   r.w[2] = ~0x04010040u; r.w[3] = 0xFu; }
  else                    { r.w[0] = ~0x20080200u; r.w[1] = ~0x08020080u;   r.w[2] = ~0x02008020u; r.w[3] = 0x7u; }
  return r;
}
SD bool bb_any(BB a) { return (a.w[0] | a.w[1] | a.w[2] | a.w[3]) != 0; }
SD int bb_popc(BB a) { return sd_popc(a.w[0]) + sd_popc(a.w[1]) + sd_popc(a.w[2]) + sd_popc(a.w[3]); }
// r[c] = a[c+S]
template <int S> SD BB bb_down(BB a) {
  BB r;
  r.w[0] = sd_fsr(a.w[0], a.w[1], S); r.w[1] = sd_fsr(a.w[1], a.w[2], S);
  r.w[2] = sd_fsr(a.w[2], a.w[3], S); r.w[3] = a.w[3] >> S;
  return r;
}
// r[c] = a[c-S]
template <int S> SD BB bb_up(BB a) {
  BB r;
  r.w[3] = sd_fsl(a.w[2], a.w[3], S) & 0xFu; r.w[2] = sd_fsl(a.w[1], a.w[2], S);
  r.w[1] = sd_fsl(a.w[0], a.w[1], S); r.w[0] = a.w[0] << S;
  return r;
}
SD uint32_t bb_word(const BB& a, int i) {
  uint32_t x = a.w[0];
  x = i == 1 ? a.w[1] : x; x = i == 2 ? a.w[2] : x; x = i == 3 ? a.w[3] : x;
  return x;
}
SD uint32_t bb_test(const BB& a, int c) { return (bb_word(a, c >> 5) >> (c & 31)) & 1u; }
// single-cell selector: m[i] = bit of cell c in word i
struct CellSel { uint32_t m[4]; };
SD CellSel cell_sel(int c) {
  CellSel s; uint32_t bit = 1u << (c & 31); int wi = c >> 5;
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i) s.m[i] = wi == i ? bit : 0u;
  return s;
}
SD void bb_put(BB& a, const CellSel& s, uint32_t v) {  // set cell to v (0/1)
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i) a.w[i] = (a.w[i] & ~s.m[i]) | (v ? s.m[i] : 0u);
}
SD uint32_t bb_get(const BB& a, const CellSel& s) {
  return ((a.w[0] & s.m[0]) | (a.w[1] & s.m[1]) | (a.w[2] & s.m[2]) | (a.w[3] & s.m[3])) != 0;
}

// ------------------------------------------------------------------ Philox4x32-10
SD void philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4]) {
STRAT_UNROLL
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = sd_mulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = sd_mulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
SD uint32_t bounded(uint32_t u, uint32_t n) { return sd_mulhi(u, n); }

// ------------------------------------------------------------------ game state
// Device line, 32 words:  word 4p+i = plane p (0 T0, 1 T1, 2 T2, 3 T3, 4 owner, 5 moved,
// 6 revealed), cells 32i..32i+31.  Word 4p+3 holds cells 96..99 in bits 0..3 and 28 spare
// bits: planes 0..3 carry history entries 2p (bits 4..17) and 2p+1 (bits 18..31), an entry
// being from | to<<7 (0x3FFF = none); plane 4 carries flags (bit 4 done, bits 5..7 reason,
// bits 8..9 result+1).  Word 28 = ply | battleless<<16, word 29 = epoch, word 30 = chase age of
// red | blue<<8 (R#28), word 31 = plies in the game's move log (device only; a line that is
// imported or copied to another environment starts with 0).
struct Game {
  BB t0, t1, t2, t3, own, mvd, rev;
  uint32_t h[4];
  uint32_t done, reason;
  int32_t result;
  uint32_t ply, battleless, epoch;
  uint32_t chase;  // chase age of red | blue << 8: positions of the player's running chase (0 = none)
  uint32_t logn;   // plies appended to this game's move log since the state was set up / loaded
};

SD void unpack_line(const uint32_t* W, Game& g) {
  BB* pl[7] = {&g.t0, &g.t1, &g.t2, &g.t3, &g.own, &g.mvd, &g.rev};
  STRAT_UNROLL
  for (int p = 0; p < 7; ++p) {
    STRAT_UNROLL
    for (int i = 0; i < 3; ++i) pl[p]->w[i] = W[4 * p + i];
    pl[p]->w[3] = W[4 * p + 3] & 0xFu;
  }
  STRAT_UNROLL
  for (int p = 0; p < 4; ++p) g.h[p] = W[4 * p + 3] >> 4;
  uint32_t f = W[19] >> 4;
  g.done = f & 1u; g.reason = (f >> 1) & 7u; g.result = (int32_t)((f >> 4) & 3u) - 1;
  g.ply = W[28] & 0xFFFFu; g.battleless = W[28] >> 16; g.epoch = W[29]; g.chase = W[30] & 0xFFFFu; g.logn = W[31];
}
SD void pack_line(const Game& g, uint32_t* W) {
  const BB* pl[7] = {&g.t0, &g.t1, &g.t2, &g.t3, &g.own, &g.mvd, &g.rev};
  STRAT_UNROLL
  for (int p = 0; p < 7; ++p)
    STRAT_UNROLL
    for (int i = 0; i < 4; ++i) W[4 * p + i] = pl[p]->w[i];
  STRAT_UNROLL
  for (int p = 0; p < 4; ++p) W[4 * p + 3] |= g.h[p] << 4;
  W[19] |= (g.done | (g.reason << 1) | ((uint32_t)(g.result + 1) << 4)) << 4;
  W[28] = g.ply | (g.battleless << 16); W[29] = g.epoch; W[30] = g.chase; W[31] = g.logn;
}
SD uint32_t hist_entry(const Game& g, int j) {  // selects, not an indexed load: g stays in registers
  const int k = j >> 1;
  uint32_t w = g.h[0];
  w = k == 1 ? g.h[1] : w; w = k == 2 ? g.h[2] : w; w = k == 3 ? g.h[3] : w;
  return (w >> (14 * (j & 1))) & 0x3FFFu;
}
SD void hist_push(Game& g, uint32_t e) {
  uint32_t carry = e;
  STRAT_UNROLL
  for (int p = 0; p < 4; ++p) {
    uint32_t out = g.h[p] >> 14;
    g.h[p] = ((g.h[p] << 14) | carry) & 0x0FFFFFFFu;
    carry = out;
  }
}
SD void hist_clear(Game& g) {
STRAT_UNROLL
for (int p = 0; p < 4; ++p) g.h[p] = 0x0FFFFFFFu; }

SD BB occupied(const Game& g) { return bb_or(bb_or(g.t0, g.t1), bb_or(g.t2, g.t3)); }
SD BB owned_by(const Game& g, BB occ, int side) {
  BB r;
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i) r.w[i] = occ.w[i] & (side ? g.own.w[i] : ~g.own.w[i]); return r;
}

// ------------------------------------------------------------------ two-square rule
// P:212 / R#6.  The side's last three moves are history entries first, first+2, first+4
// (first = 1 when it is that side's turn, else 0).  If they are consecutive moves of one
// piece along one line whose crossed boundaries intersect, moves of that piece (now at
// `from`) in direction `dir` of distance >= k are banned.
struct Ban { int from, dir, k; };
SD Ban two_square_ban(const Game& g, int side, int enabled) {
  Ban b; b.from = -1; b.dir = 0; b.k = 99;
  if (!enabled) return b;
  int first = ((int)(g.ply & 1u) == side) ? 1 : 0;
  uint32_t e3 = hist_entry(g, first), e2 = hist_entry(g, first + 2), e1 = hist_entry(g, first + 4);
  if (e3 == kHistNone || e2 == kHistNone || e1 == kHistNone) return b;
  int p0 = e1 & 127, p1 = e1 >> 7, f2 = e2 & 127, p2 = e2 >> 7, f3 = e3 & 127, p3 = e3 >> 7;
  if (p1 != f2 || p2 != f3) return b;
  int r0 = p0 / 10, r1 = p1 / 10, r2 = p2 / 10, r3 = p3 / 10;
  int c0 = p0 - 10 * r0, c1 = p1 - 10 * r1, c2 = p2 - 10 * r2, c3 = p3 - 10 * r3;
  bool same_row = r0 == r1 && r1 == r2 && r2 == r3;
  bool same_col = c0 == c1 && c1 == c2 && c2 == c3;
  if (!same_row && !same_col) return b;
  int x0 = same_row ? c0 : r0, x1 = same_row ? c1 : r1, x2 = same_row ? c2 : r2, x3 = same_row ? c3 : r3;
  int lo = max(max(min(x0, x1), min(x1, x2)), min(x2, x3));
  int hi = min(min(max(x0, x1), max(x1, x2)), max(x2, x3));
  if (lo >= hi) return b;
  b.from = p3;
  if (x3 > x2) { b.dir = same_row ? 3 : 2; b.k = x3 - hi + 1; }
  else         { b.dir = same_row ? 1 : 0; b.k = lo - x3 + 1; }
  return b;
}

// ------------------------------------------------------------------ continuous-chasing rule
// P:212-218 / R#28.  threat = a move to an empty square that ends next to an opponent's piece;
// evade = the piece threatened on the previous ply moves, to an empty square, away from the
// piece that threatened it; a player's chase = its threats alternating with the opponent's
// evades; g.chase holds each player's chase age (positions since its first threat, 0 = none).
SD uint32_t chase_age(const Game& g, int side) { return (g.chase >> (8 * side)) & 0xFFu; }
SD bool cells_adjacent(int a, int b) {
  int ra = a / 10, rb = b / 10, dr = ra - rb, dc = (a - 10 * ra) - (b - 10 * rb);
  return dr * dr + dc * dc == 1;
}
SD BB neighbours_of(int c) {
  CellSel s = cell_sel(c);
  BB one; one.w[0] = s.m[0]; one.w[1] = s.m[1]; one.w[2] = s.m[2]; one.w[3] = s.m[3];
  return bb_or(bb_or(bb_up<10>(one), bb_down<10>(one)),
               bb_or(bb_and(bb_up<1>(one), bb_const(kNotCol0)), bb_and(bb_down<1>(one), bb_const(kNotCol9))));
}
// The moves of `side` that the chasing rule bans in this position (at most one per earlier
// position of the chase: it can be recreated by at most one move).
// A position is the type and owner on every square.  Earlier positions are rebuilt by taking
// the logged plies back on copies of the five type/owner planes (no battle happens inside a
// chase); position t-b is recreated by the move c->a iff it differs from the current one on
// exactly the squares {c, a}, with the current piece of c standing on a.
// Returned: action indices (the caller still checks that they are otherwise legal).
SD int chase_banned_actions(const Game& g, int side, BB mine, BB enemy, const uint16_t* glog, int banned[kMaxBans]) {
  int age = (int)chase_age(g, side);
  if (age < 2) return 0;
  int first = ((int)(g.ply & 1u) == side) ? 1 : 0;
  uint32_t eprev = hist_entry(g, first);  // this player's previous ply
  int back = min(age - 1, kMaxBans), nb = 0;
  int logged = glog ? (int)min(g.logn, (uint32_t)(kLogPlies - 1)) : 0;
  BB k[5] = {g.t0, g.t1, g.t2, g.t3, g.own};
  for (int b = 1; b <= back; ++b) {
    // plies 1..8 back are in the line's history, older ones in the game's move log
    uint32_t e = b <= 8 ? hist_entry(g, b - 1)
               : b <= logged ? (uint32_t)sd_ldlog(glog + ((g.logn - (uint32_t)b) & (kLogPlies - 1))) : kHistNone;
    if (e == kHistNone) break;
    CellSel sf = cell_sel((int)(e & 127u)), st = cell_sel((int)(e >> 7));
    STRAT_UNROLL
    for (int p = 0; p < 5; ++p) { uint32_t v = bb_get(k[p], st); bb_put(k[p], st, 0); bb_put(k[p], sf, v); }
    uint32_t d[4];
    STRAT_UNROLL
    for (int i = 0; i < 4; ++i)
      d[i] = (k[0].w[i] ^ g.t0.w[i]) | (k[1].w[i] ^ g.t1.w[i]) | (k[2].w[i] ^ g.t2.w[i]) | (k[3].w[i] ^ g.t3.w[i]) |
             (k[4].w[i] ^ g.own.w[i]);
    if (sd_popc(d[0]) + sd_popc(d[1]) + sd_popc(d[2]) + sd_popc(d[3]) != 2) continue;
    int s1 = -1, s2 = -1;
    STRAT_UNROLL
    for (int i = 0; i < 4; ++i) {
      uint32_t w = d[i];
      while (w) { int sq = 32 * i + sd_ffs(w) - 1; w &= w - 1; if (s1 < 0) s1 = sq; else s2 = sq; }
    }
    // c = the square that holds a piece now and is empty in the earlier position; a = the reverse
    bool occ1 = bb_test(g.t0, s1) | bb_test(g.t1, s1) | bb_test(g.t2, s1) | bb_test(g.t3, s1);
    int c = occ1 ? s1 : s2, a = occ1 ? s2 : s1;
    CellSel sc = cell_sel(c), sa = cell_sel(a);
    bool ok = bb_test(mine, c) != 0;
    uint32_t cur_a = 0, old_c = 0, same = 1;
    const BB* cur[5] = {&g.t0, &g.t1, &g.t2, &g.t3, &g.own};
    STRAT_UNROLL
    for (int p = 0; p < 5; ++p) {
      if (p < 4) { cur_a |= bb_get(*cur[p], sa); old_c |= bb_get(k[p], sc); }
      same &= (bb_get(*cur[p], sc) == bb_get(k[p], sa)) ? 1u : 0u;
    }
    if (!ok || cur_a || old_c || !same) continue;
    int ra = a / 10, rc = c / 10, qa = a - 10 * ra, qc = c - 10 * rc;
    int dir, dist;
    if (qa == qc) { dir = ra > rc ? 0 : 2; dist = ra > rc ? ra - rc : rc - ra; }
    else if (ra == rc) { dir = qa > qc ? 1 : 3; dist = qa > qc ? qa - qc : qc - qa; }
    else continue;
    if (!bb_any(bb_and(neighbours_of(a), enemy))) continue;                                  // not a threat
    if (eprev != kHistNone && c == (int)(eprev >> 7) && a == (int)(eprev & 127u)) continue;  // the return move
    banned[nb++] = c * 36 + dir * 9 + dist - 1;
  }
  return nb;
}

// ------------------------------------------------------------------ move generation
struct Moves {
  BB d[4];      // d[dir][c] = piece of `side` at c may move one square in dir (after bans)
  BB scouts;    // own Scouts
  BB empty;     // empty non-lake squares
  BB ok;        // squares a piece of `side` may land on (empty or enemy, not lake)
  Ban ban;
};
SD void single_step_moves(const Game& g, int side, int rules, Moves& m) {
  BB occ = occupied(g);
  BB mine = owned_by(g, occ, side);
  BB notlake = bb_const(kNotLake);
  m.ok = bb_andn(notlake, mine);
  m.empty = bb_andn(notlake, occ);
  // immovable types: Flag 1011, Bomb 1100  ->  T3 & (T2 | (T1 & T0))
  BB imm = bb_and(g.t3, bb_or(g.t2, bb_and(g.t1, g.t0)));
  BB movable = bb_andn(mine, imm);
  m.scouts = bb_andn(bb_andn(bb_andn(bb_and(mine, g.t1), g.t0), g.t2), g.t3);
  m.d[0] = bb_and(movable, bb_down<10>(m.ok));
  m.d[2] = bb_and(movable, bb_up<10>(m.ok));
  m.d[1] = bb_and(bb_and(movable, bb_down<1>(m.ok)), bb_const(kNotCol9));
  m.d[3] = bb_and(bb_and(movable, bb_up<1>(m.ok)), bb_const(kNotCol0));
  m.ban = two_square_ban(g, side, rules & RULE_TWO_SQUARE);
  if (m.ban.from >= 0 && m.ban.k <= 1) {
    CellSel s = cell_sel(m.ban.from);
    STRAT_UNROLL
    for (int d = 0; d < 4; ++d)
      if (d == m.ban.dir)
      STRAT_UNROLL
      for (int i = 0; i < 4; ++i) m.d[d].w[i] &= ~s.m[i];
  }
}
// GetHasLegalMovement: a banned distance bans every longer one (R#6), so a side
// has a legal move iff it has a legal single-step move - unless the chasing rule takes moves
// away one by one (has_legal_move below then counts them).
SD bool has_single_step_move(const Moves& m) {
  return bb_any(bb_or(bb_or(m.d[0], m.d[1]), bb_or(m.d[2], m.d[3])));
}

// ---- Scout rays without loops: pull the Scout's row and column out of the boards as 10-bit
// lines and count empties with ffs/clz.
SD uint32_t row_bits(const BB& a, int r) {  // bit i = cell 10r+i
  int pos = 10 * r, wi = pos >> 5, sh = pos & 31;  // wi in 0..2
  uint32_t lo = wi == 0 ? a.w[0] : wi == 1 ? a.w[1] : a.w[2];
  uint32_t hi = wi == 0 ? a.w[1] : wi == 1 ? a.w[2] : a.w[3];
  return sd_fsr(lo, hi, sh) & 0x3FFu;
}
SD uint32_t col_bits(const BB& a, int q) {  // bit i = cell 10i+q
  // shift the board down by q, keep column 0, then squeeze the stride-10 bits together with
  // one multiply per word (all partial products land on distinct bits)
  uint32_t s0 = sd_fsr(a.w[0], a.w[1], q), s1 = sd_fsr(a.w[1], a.w[2], q), s2 = sd_fsr(a.w[2], a.w[3], q);
  uint32_t x0 = ((s0 & 0x40100401u) * 0x08040201u) >> 27;  // cells 0,10,20,30   -> rows 0..3
  uint32_t x1 = ((s1 & 0x10040100u) * 0x00100804u) >> 28;  // cells 40,50,60     -> rows 4..6
  uint32_t x2 = ((s2 & 0x04010040u) * 0x00402010u) >> 28;  // cells 70,80,90     -> rows 7..9
  return x0 | (x1 << 4) | (x2 << 7);
}
// e = empty squares of a 10-cell line, k = squares the mover may land on; from coordinate x.
SD int ray_up(uint32_t e, uint32_t k, int x) {
  uint32_t blockers = ((~e & 0x3FFu) >> (x + 1)) | (1u << (9 - x));  // + board-edge sentinel
  int ne = sd_ffs(blockers) - 1;                                       // consecutive empties
  return ne + (int)((k >> (x + 1 + ne)) & 1u);                         // + capture of the blocker
}
SD int ray_down(uint32_t e, uint32_t k, int x) {
  uint32_t blockers = ~e & ((1u << x) - 1u);
  int p = 31 - sd_clz(blockers);                                       // nearest blocker, -1 if none
  return (x - 1 - p) + (int)(((k << 1) >> (p + 1)) & 1u);
}
// Longest legal distance of a Scout at c=(r,q) in each direction (0 if none), bans applied.
SD void scout_rays(const Moves& m, int c, int r, int q, int len[4]) {
  uint32_t er = row_bits(m.empty, r), kr = row_bits(m.ok, r);
  uint32_t ec = col_bits(m.empty, q), kc = col_bits(m.ok, q);
  len[0] = ray_up(ec, kc, r); len[1] = ray_up(er, kr, q);
  len[2] = ray_down(ec, kc, r); len[3] = ray_down(er, kr, q);
  if (m.ban.from == c) {
    STRAT_UNROLL
    for (int d = 0; d < 4; ++d)
      if (d == m.ban.dir) len[d] = min(len[d], m.ban.k - 1);
  }
}

// Is action a legal by movement, lakes, blocking and the two-square rule (all in m)?
SD bool move_in_moves(const Moves& m, int a) {
  if (a < 0 || a >= 3600) return false;
  int from = a / 36, rem = a - 36 * from, d = rem / 9, dist = rem - 9 * d + 1;
  if (!bb_test(m.d[d], from)) return false;
  if (dist == 1) return true;
  if (!bb_test(m.scouts, from)) return false;
  int r = from / 10, q = from - 10 * r;
  int len[4];
  scout_rays(m, from, r, q, len);
  int ld = d == 0 ? len[0] : d == 1 ? len[1] : d == 2 ? len[2] : len[3];
  return dist <= ld;
}
// Distinct actions of banned[0..nb) that are legal in m, compacted in place; returns their number.
SD int keep_legal_banned(const Moves& m, int banned[kMaxBans], int nb) {
  int k = 0;
  for (int i = 0; i < nb; ++i) {
    bool dup = false;
    for (int j = 0; j < k; ++j) dup |= banned[j] == banned[i];
    if (!dup && move_in_moves(m, banned[i])) banned[k++] = banned[i];
  }
  return k;
}
SD bool has_legal_move(const Game& g, int side, int rules, const uint16_t* glog = nullptr) {
  Moves m; single_step_moves(g, side, rules, m);
  if (!has_single_step_move(m)) return false;
  if (!(rules & RULE_CHASE) || chase_age(g, side) < 2) return true;
  BB occ = occupied(g), mine = owned_by(g, occ, side);
  int banned[kMaxBans];
  int nb = chase_banned_actions(g, side, mine, bb_andn(occ, mine), glog, banned);
  if (nb == 0) return true;
  nb = keep_legal_banned(m, banned, nb);
  int total = 0;  // every legal move without the chasing rule
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i) {
    uint32_t sc = m.scouts.w[i];
    total += sd_popc(m.d[0].w[i] & ~sc) + sd_popc(m.d[1].w[i] & ~sc) + sd_popc(m.d[2].w[i] & ~sc) + sd_popc(m.d[3].w[i] & ~sc);
    uint32_t ss = (m.d[0].w[i] | m.d[1].w[i] | m.d[2].w[i] | m.d[3].w[i]) & sc;
    while (ss) {
      int b = sd_ffs(ss) - 1; ss &= ss - 1;
      int c = 32 * i + b, r = c / 10, q = c - 10 * r, len[4];
      scout_rays(m, c, r, q, len);
      total += len[0] + len[1] + len[2] + len[3];
    }
  }
  return total > nb;
}

SD void mask_or_field(uint32_t* row, int c, uint64_t field) {  // the 36 action bits of cell c
  int pos = 36 * c, wi = pos >> 5, sh = pos & 31;
  field <<= sh;  // 36 + 28 <= 64
  row[wi] |= (uint32_t)field;
  uint32_t hi = (uint32_t)(field >> 32);
  if (hi) row[wi + 1] |= hi;
}

// Legal mask of `side` into `row` (113 words, already zero).  Returns the number of legal
// actions and, in cnt[i], how many of them start from cells 32i..32i+31 (= mask words
// 36i..36i+35; used by pick_action).  a = from*36 + dir*9 + dist-1.
SD int legal_mask_row(const Game& g, int side, int rules, uint32_t* row, int cnt[4], const uint16_t* glog = nullptr) {
  Moves m; single_step_moves(g, side, rules, m);
  // pieces that move one square: four bits per piece, no branches
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i) {
    uint32_t sc = m.scouts.w[i];
    uint32_t d0 = m.d[0].w[i] & ~sc, d1 = m.d[1].w[i] & ~sc, d2 = m.d[2].w[i] & ~sc, d3 = m.d[3].w[i] & ~sc;
    cnt[i] = sd_popc(d0) + sd_popc(d1) + sd_popc(d2) + sd_popc(d3);
    uint32_t any = d0 | d1 | d2 | d3;
    while (any) {
      int b = sd_ffs(any) - 1;
      any &= any - 1;
      uint32_t f = ((d0 >> b) & 1u) | (((d1 >> b) & 1u) << 9) | (((d2 >> b) & 1u) << 18) | (((d3 >> b) & 1u) << 27);
      mask_or_field(row, 32 * i + b, (uint64_t)f);
    }
  }
  // Scouts: up to nine bits per direction
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i) {
    uint32_t ss = (m.d[0].w[i] | m.d[1].w[i] | m.d[2].w[i] | m.d[3].w[i]) & m.scouts.w[i];
    while (ss) {
      int b = sd_ffs(ss) - 1;
      ss &= ss - 1;
      int c = 32 * i + b, r = c / 10, q = c - 10 * r;
      int len[4];
      scout_rays(m, c, r, q, len);
      cnt[i] += len[0] + len[1] + len[2] + len[3];
      uint64_t field = (uint64_t)((1u << len[0]) - 1u) | ((uint64_t)((1u << len[1]) - 1u) << 9) |
                       ((uint64_t)((1u << len[2]) - 1u) << 18) | ((uint64_t)((1u << len[3]) - 1u) << 27);
      mask_or_field(row, c, field);
    }
  }
  if ((rules & RULE_CHASE) && chase_age(g, side) >= 2) {  // rare: take the chase-banned threats out
    BB occ = occupied(g), mine = owned_by(g, occ, side);
    int banned[kMaxBans];
    int nb = chase_banned_actions(g, side, mine, bb_andn(occ, mine), glog, banned);
    for (int i = 0; i < nb; ++i) {
      uint32_t bit = 1u << (banned[i] & 31);
      int w = banned[i] >> 5, grp = (banned[i] / 36) >> 5;
      if (row[w] & bit) {
        row[w] &= ~bit;
        STRAT_UNROLL
        for (int k = 0; k < 4; ++k) cnt[k] -= (k == grp) ? 1 : 0;
      }
    }
  }
  return cnt[0] + cnt[1] + cnt[2] + cnt[3];
}

// r-th (from 0) set bit of a word
SD int nth_set_bit(uint32_t w, int r) {
  int pos = 0;
STRAT_UNROLL
  for (int s = 16; s >= 1; s >>= 1) {
    int c = sd_popc(w & (((1u << s) - 1u) << pos));
    if (r >= c) { r -= c; pos += s; }
  }
  return pos;
}
// SampleRandomLegalAction, C3a: the r-th set bit of the row, r = bounded(u, n).
// cnt[i] = set bits in mask words 36i..36i+35, so only one 36-word stretch is scanned.
SD int pick_rank(const uint32_t* row, const int cnt[4], int r) {
  int w0 = 0;
  if (r >= cnt[0]) { r -= cnt[0]; w0 = 36; if (r >= cnt[1]) { r -= cnt[1]; w0 = 72; if (r >= cnt[2]) { r -= cnt[2]; w0 = 108; } } }
  for (int w = w0; w < kMaskWords; ++w) {
    int c = sd_popc(row[w]);
    if (r < c) return 32 * w + nth_set_bit(row[w], r);
    r -= c;
  }
  return -1;
}
SD int pick_action(const uint32_t* row, const int cnt[4], int n, uint32_t u) {
  if (n == 0) return -1;
  return pick_rank(row, cnt, (int)bounded(u, (uint32_t)n));
}
// r-th (from 0) legal action in ascending order, given the per-group counts, the non-Scout
// direction bits D[group][dir] and two words per Scout that can move:
//   scouts[2k]   = cell | len0<<7 | len1<<11 | len2<<15 | len3<<19
//   scouts[2k+1] = start | total<<16 | group<<24, start = rank, inside its 32-cell group, of the
//                  Scout's first action, total = its number of actions.
// Either r falls into a Scout's interval, or it is the (r - Scout actions before it)-th action of
// the non-Scout pieces, whose cell is found by a 5-step binary search on the four direction
// planes.  No walk over the pieces and no early exit: the lanes of a warp stay converged.
// kmax >= ns bounds the Scout loop (a kernel passes the largest ns of its warp).
SD int select_action(const uint32_t (&D)[4][4], const int cnt[4], const uint32_t* scouts, int ns, int r, int kmax = 8) {
  int gi = 0;
  if (r >= cnt[0]) { r -= cnt[0]; gi = 1; if (r >= cnt[1]) { r -= cnt[1]; gi = 2; if (r >= cnt[2]) { r -= cnt[2]; gi = 3; } } }
  int before = 0, hit_k = -1, hit_q = 0;
  for (int k = 0; k < kmax; ++k) {
    uint32_t w = k < ns ? scouts[2 * k + 1] : 0xFF000000u;  // group 255: never matches
    int start = (int)(w & 0xFFFFu), tot = (int)((w >> 16) & 0xFFu);
    bool valid = (int)(w >> 24) == gi;
    int q = r - start;
    before += (valid && q >= tot) ? tot : 0;
    bool inside = valid && q >= 0 && q < tot;
    hit_k = inside ? k : hit_k;
    hit_q = inside ? q : hit_q;
  }
  r -= before;
  uint32_t d0 = gi == 0 ? D[0][0] : gi == 1 ? D[1][0] : gi == 2 ? D[2][0] : D[3][0];
  uint32_t d1 = gi == 0 ? D[0][1] : gi == 1 ? D[1][1] : gi == 2 ? D[2][1] : D[3][1];
  uint32_t d2 = gi == 0 ? D[0][2] : gi == 1 ? D[1][2] : gi == 2 ? D[2][2] : D[3][2];
  uint32_t d3 = gi == 0 ? D[0][3] : gi == 1 ? D[1][3] : gi == 2 ? D[2][3] : D[3][3];
  // non-Scout pieces: smallest bit b with (actions of cells 0..b) > r
  int b = 0;
  STRAT_UNROLL
  for (int s = 16; s >= 1; s >>= 1) {
    uint32_t below = (1u << (b + s)) - 1u;  // cells 0 .. b+s-1
    int c = sd_popc(d0 & below) + sd_popc(d1 & below) + sd_popc(d2 & below) + sd_popc(d3 & below);
    b += c <= r ? s : 0;
  }
  uint32_t below = (1u << b) - 1u;
  int q = r - (sd_popc(d0 & below) + sd_popc(d1 & below) + sd_popc(d2 & below) + sd_popc(d3 & below));
  int l0 = (d0 >> b) & 1, l1 = (d1 >> b) & 1, l2 = (d2 >> b) & 1, cell = 32 * gi + b;
  // a Scout was hit: its ray lengths take the place of the one-step bits
  uint32_t e = hit_k >= 0 ? scouts[2 * hit_k] : 0u;
  bool hit = hit_k >= 0;
  l0 = hit ? (int)((e >> 7) & 15u) : l0; l1 = hit ? (int)((e >> 11) & 15u) : l1; l2 = hit ? (int)((e >> 15) & 15u) : l2;
  q = hit ? hit_q : q;
  cell = hit ? (int)(e & 127u) : cell;
  int dir = (q >= l0 ? 1 : 0) + (q >= l0 + l1 ? 1 : 0) + (q >= l0 + l1 + l2 ? 1 : 0);
  int qd = q - (dir > 0 ? l0 : 0) - (dir > 1 ? l1 : 0) - (dir > 2 ? l2 : 0);
  return cell * 36 + dir * 9 + qd;
}
// SampleRandomLegalAction without materialising the 3600-bit mask (on-chip rollouts): equal to
// pick_action(legal_mask_row(...)) for the same draw u.  Actions ascend with the from-cell, then
// the direction, then the distance, so the r-th legal action follows from per-cell counts (1 per
// open direction; a Scout's ray lengths).  Two phases, so that a kernel can let its lanes
// reconverge (__syncwarp) between the Scout loops, whose trip counts differ from game to game,
// and the selection: count_actions fills an ActionSet, choose_action picks from it.
// `scouts` = 16 words of per-thread scratch (two per Scout that can move).
struct ActionSet {
  uint32_t D[4][4];  // non-Scout pieces: D[group][dir] bit b = cell 32*group+b may step in dir
  int cnt[4];        // legal actions per 32-cell group of from-cells
  int ns, n;         // Scouts with moves, all legal actions (before chasing-rule bans)
  Moves m;
};
SD void count_actions(const Game& g, int side, int rules, uint32_t* scouts, ActionSet& A) {
  single_step_moves(g, side, rules, A.m);
  const Moves& m = A.m;
  int ns = 0;
  // 1. non-Scout counts, and the list of Scouts that can move (ascending cells) with the number of
  //    non-Scout actions before each inside its 32-cell group - a short loop per group
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i) {
    uint32_t sc = m.scouts.w[i];
    STRAT_UNROLL
    for (int d = 0; d < 4; ++d) A.D[i][d] = m.d[d].w[i] & ~sc;
    A.cnt[i] = sd_popc(A.D[i][0]) + sd_popc(A.D[i][1]) + sd_popc(A.D[i][2]) + sd_popc(A.D[i][3]);
    uint32_t ss = (m.d[0].w[i] | m.d[1].w[i] | m.d[2].w[i] | m.d[3].w[i]) & sc;
    while (ss && ns < kMaxScouts) {
      int bit = sd_ffs(ss) - 1;
      ss &= ss - 1;
      uint32_t below = (1u << bit) - 1u;
      int pre = sd_popc(A.D[i][0] & below) + sd_popc(A.D[i][1] & below) + sd_popc(A.D[i][2] & below) +
                sd_popc(A.D[i][3] & below);
      scouts[2 * ns] = (uint32_t)(32 * i + bit);
      scouts[2 * ns + 1] = (uint32_t)pre;
      ++ns;
    }
  }
  // 2. one pass over that list (its length, not the number of Scouts per 32-cell group, sets the
  //    number of passes a warp makes): ray lengths and the rank of each Scout's first action
  int grp = -1, scout_actions = 0;
  for (int k = 0; k < ns; ++k) {
    int c = (int)scouts[2 * k], i = c >> 5, r = c / 10, q = c - 10 * r;
    int len[4];
    scout_rays(m, c, r, q, len);
    scout_actions = i == grp ? scout_actions : 0;  // ranks are relative to the 32-cell group
    grp = i;
    int start = (int)scouts[2 * k + 1] + scout_actions;  // < 32*4 + 8*36
    int tot = len[0] + len[1] + len[2] + len[3];
    scouts[2 * k] = (uint32_t)c | ((uint32_t)len[0] << 7) | ((uint32_t)len[1] << 11) | ((uint32_t)len[2] << 15) |
                    ((uint32_t)len[3] << 19);
    scouts[2 * k + 1] = (uint32_t)start | ((uint32_t)tot << 16) | ((uint32_t)i << 24);
    scout_actions += tot;
    STRAT_UNROLL
    for (int j = 0; j < 4; ++j) A.cnt[j] += j == i ? tot : 0;
  }
  A.ns = ns;
  A.n = A.cnt[0] + A.cnt[1] + A.cnt[2] + A.cnt[3];
}
SD int choose_action(const Game& g, int side, int rules, const ActionSet& A, uint32_t u, const uint32_t* scouts,
                     const uint16_t* glog = nullptr, int kmax = 8) {
  if (A.n == 0) return -1;
  if ((rules & RULE_CHASE) && chase_age(g, side) >= 2) {  // rare: skip the chase-banned threats
    BB occ = occupied(g), mine = owned_by(g, occ, side);
    int banned[kMaxBans];
    int nb = chase_banned_actions(g, side, mine, bb_andn(occ, mine), glog, banned);
    nb = keep_legal_banned(A.m, banned, nb);
    if (nb > 0) {
      if (A.n == nb) return -1;
      int r = (int)bounded(u, (uint32_t)(A.n - nb));
      // the r-th action that is not banned: skip the banned ones at or below it (fixed point)
      for (int ra = r;;) {
        int a = select_action(A.D, A.cnt, scouts, A.ns, ra, kmax);
        int below = 0;
        for (int i = 0; i < nb; ++i) below += banned[i] <= a ? 1 : 0;
        if (r + below == ra) return a;
        ra = r + below;
      }
    }
  }
  return select_action(A.D, A.cnt, scouts, A.ns, (int)bounded(u, (uint32_t)A.n), kmax);
}
SD uint32_t action_draw(const Params& P, uint32_t local_game, const Game& g) {
  uint32_t o[4];
  philox(P.game_base + local_game, g.epoch, g.ply, TAG_ACTION, P.key0, P.key1, o);
  return o[0];
}

// Is action a legal for the side to move?  (step validates what it is given)
SD bool action_is_legal(const Game& g, int side, int rules, int a, const uint16_t* glog = nullptr) {
  Moves m; single_step_moves(g, side, rules, m);
  if (!move_in_moves(m, a)) return false;
  if ((rules & RULE_CHASE) && chase_age(g, side) >= 2) {
    BB occ = occupied(g), mine = owned_by(g, occ, side);
    int banned[kMaxBans];
    int nb = chase_banned_actions(g, side, mine, bb_andn(occ, mine), glog, banned);
    for (int i = 0; i < nb; ++i)
      if (banned[i] == a) return false;
  }
  return true;
}

// ------------------------------------------------------------------ setup (C2)
SD void put_piece(Game& g, int c, int type, int owner) {
  CellSel s = cell_sel(c);
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i) {
    g.t0.w[i] |= (type & 1) ? s.m[i] : 0u; g.t1.w[i] |= (type & 2) ? s.m[i] : 0u;
    g.t2.w[i] |= (type & 4) ? s.m[i] : 0u; g.t3.w[i] |= (type & 8) ? s.m[i] : 0u;
    g.own.w[i] |= owner ? s.m[i] : 0u;
  }
}
SD uint32_t multiset_type(int variant, int i) {
  if (variant == 0) {
    // Flag, Bomb x6, Spy, Scout x8, Miner x5, Sergeant x4, Lieutenant x4, Captain x4,
    // Major x3, Colonel x2, General, Marshal  (BASELINE.json configs[0] order)
    return i < 1 ? 11 : i < 7 ? 12 : i < 8 ? 1 : i < 16 ? 2 : i < 21 ? 3 : i < 25 ? 4 : i < 29 ? 5
         : i < 33 ? 6 : i < 36 ? 7 : i < 38 ? 8 : i < 39 ? 9 : 10;
  }
  // Barrage: Flag, Marshal, General, Miner, Scout, Scout, Spy, Bomb, 32 empties
  return i == 0 ? 11 : i == 1 ? 10 : i == 2 ? 9 : i == 3 ? 3 : i == 4 ? 2 : i == 5 ? 2 : i == 6 ? 1
       : i == 7 ? 12 : 0;
}
// R#5: can this side ever move: a movable own piece next to a non-lake square without an own
// piece (depends on the side's own pieces only).
SD bool side_can_ever_move(const Game& t, int side) {
  BB occ = occupied(t);
  BB mine = owned_by(t, occ, side);
  BB ok = bb_andn(bb_const(kNotLake), mine);
  BB imm = bb_and(t.t3, bb_or(t.t2, bb_and(t.t1, t.t0)));
  BB mv = bb_andn(mine, imm);
  BB can = bb_or(bb_or(bb_and(mv, bb_down<10>(ok)), bb_and(mv, bb_up<10>(ok))),
                 bb_or(bb_and(bb_and(mv, bb_down<1>(ok)), bb_const(kNotCol9)),
                       bb_and(bb_and(mv, bb_up<1>(ok)), bb_const(kNotCol0))));
  return bb_any(can);
}
// Fresh game for (global game, g.epoch): both sides by descending Fisher-Yates over the
// listed multiset, redrawn until the side can ever move (R#4, R#5).
SD void setup_game(const Params& P, uint32_t local_game, Game& g) {
  g.t0 = g.t1 = g.t2 = g.t3 = g.own = g.mvd = g.rev = bb_zero();
  hist_clear(g);
  g.done = 0; g.reason = 0; g.result = 0; g.ply = 0; g.battleless = 0; g.chase = 0; g.logn = 0;
  uint32_t gidx = P.game_base + local_game;
  if (P.pool) {  // R#30: each side's setup = pool entry bounded(first draw of its SETUP stream, K)
    for (int side = 0; side < 2; ++side) {
      uint32_t o[4];
      philox(gidx, g.epoch, 0u, side ? TAG_SETUP_BLUE : TAG_SETUP_RED, P.key0, P.key1, o);
      const uint8_t* A = P.pool + ((size_t)side * P.pool_size + bounded(o[0], (uint32_t)P.pool_size)) * 40;
      for (int i = 0; i < 40; ++i)
        if (A[i]) put_piece(g, (side ? 60 : 0) + i, A[i], side);
    }
    return;
  }
  for (int side = 0; side < 2; ++side) {
    for (uint32_t attempt = 0;; ++attempt) {
      uint8_t A[40];
      for (int i = 0; i < 40; ++i) A[i] = (uint8_t)multiset_type(P.variant, i);
      uint32_t o[4] = {0, 0, 0, 0};
      for (int i = 39; i >= 1; --i) {
        int d = 39 - i;
        if ((d & 3) == 0) philox(gidx, g.epoch, (attempt << 8) | (uint32_t)(d >> 2),
                                 side ? TAG_SETUP_BLUE : TAG_SETUP_RED, P.key0, P.key1, o);
        uint32_t u = (d & 3) == 0 ? o[0] : (d & 3) == 1 ? o[1] : (d & 3) == 2 ? o[2] : o[3];
        int j = (int)bounded(u, (uint32_t)(i + 1));
        uint8_t t = A[i]; A[i] = A[j]; A[j] = t;
      }
      Game trial = g;
      int base = side ? 60 : 0;
      for (int i = 0; i < 40; ++i)
        if (A[i]) put_piece(trial, base + i, A[i], side);
      if (side_can_ever_move(trial, side)) { g = trial; break; }
    }
  }
}

// Auto-reset of a finished game whose epoch has already been advanced: a fresh setup, or the
// game's pinned line with the slot's own epoch (R#27).
SD void reset_game(const Params& P, uint32_t local_game, Game& g) {
  if (P.pin) {
    uint32_t W[32], epoch = g.epoch;
    STRAT_UNROLL
    for (int k = 0; k < 32; ++k) W[k] = P.pin[(size_t)local_game * kLineWords + k];
    unpack_line(W, g);
    g.epoch = epoch;
    // the plies that led to the pinned state restart with it; word 31 of the pinned line counts them
    uint16_t* glog = game_log(P, local_game);
    if (glog && P.pin_log) copy_game_log(P.pin_log + (size_t)local_game * kLogPlies, glog);
    else g.logn = 0;
  } else {
    setup_game(P, local_game, g);
  }
}

// ------------------------------------------------------------------ step (C4)
// +1 attacker wins, -1 attacker loses, 0 both removed (Ext. Data Fig. 3b)
SD int battle(int att, int def) {
  if (def == T_FLAG) return 1;
  if (def == T_BOMB) return att == T_MINER ? 1 : -1;
  if (att == T_SPY && def == T_MARSHAL) return 1;
  return att > def ? 1 : att < def ? -1 : 0;
}

// ------------------------------------------------------------------ S2 trackers
// What the paper's 487-channel information state needs beyond the board: one 2 KB block per game.
//   words 4c..4c+3  record of the piece standing on square c (it travels with the piece):
//       w0  bits 0-10 has threatened (Spy..Marshal revealed, bit 10 = a hidden piece)
//           bits 11-21 has evaded (same keys)
//           bits 22-28 the square the piece started on
//       w1  bits 0-10 has been actively adjacent to (same keys)
//           bits 11-23 has protected: own piece Spy..Marshal, Bomb (revealed), bit 11 an empty
//                      square, bit 12 a hidden piece
//       w2  bits 0-12 has protected against (types, bit 11 unused, bit 12 hidden)
//           bits 13-25 has been protected by
//       w3  bits 0-12 has been protected against
//   word 400        number of pieces captured so far
//   words 401..492  one entry per captured piece: start square | type << 7 | owner << 11 |
//                   square of the battle << 12 | cause of death (1..6) << 19
//   words 493..508  the last 32 plies, from | to << 7 in 16 bits (0x3FFF = unknown), ply p in
//                   entry p & 31
constexpr int kTrackWords = 512;
constexpr int kTrkDeaths = 400, kTrkDeathList = 401, kTrkMaxDeaths = 92, kTrkMoves = 493;

SD uint32_t* game_track(const Params& P, uint32_t local_game) {
  return P.track ? P.track + (size_t)local_game * kTrackWords : nullptr;
}
SD int type_at(const Game& g, int c) {
  return (int)(bb_test(g.t0, c) | (bb_test(g.t1, c) << 1) | (bb_test(g.t2, c) << 2) | (bb_test(g.t3, c) << 3));
}
// Thread-level (re)start of a game's trackers: the squares the pieces stand on are their start
// squares, the recent moves are the ones the line remembers (reading I9).
SD void track_start_tail(uint32_t* trk, const Game& g) {
  sd_st32(trk + kTrkDeaths, 0u);
  // ring slot s holds the ply p with (p & 31) == s among the last 32: ply - 1 - j with
  // j = (ply - 1 - s) & 31, known only if the line's 8-ply history has it (0x3FFF = unknown)
  for (int w = 0; w < 16; ++w) {
    uint32_t v = 0;
    STRAT_UNROLL
    for (int h = 0; h < 2; ++h) {
      int j = (int)((g.ply - 1u - (uint32_t)(2 * w + h)) & 31u);
      uint32_t e = j < 8 ? hist_entry(g, j) : kHistNone;
      v |= e << (16 * h);
    }
    sd_st32(trk + kTrkMoves + w, v);
  }
}
SD void track_start(uint32_t* trk, const Game& g) {
  for (int c = 0; c < 100; ++c) {
    sd_st32(trk + 4 * c, (uint32_t)c << 22); sd_st32(trk + 4 * c + 1, 0u);
    sd_st32(trk + 4 * c + 2, 0u); sd_st32(trk + 4 * c + 3, 0u);
  }
  track_start_tail(trk, g);
}
// The seven state bits of square c: type (bits 0-3), owner (4), moved (5), revealed (6).
SD uint32_t cell_bits(const Game& g, int c) {
  const int wi = c >> 5, sh = c & 31;
  return ((bb_word(g.t0, wi) >> sh) & 1u) | (((bb_word(g.t1, wi) >> sh) & 1u) << 1) | (((bb_word(g.t2, wi) >> sh) & 1u) << 2) |
         (((bb_word(g.t3, wi) >> sh) & 1u) << 3) | (((bb_word(g.own, wi) >> sh) & 1u) << 4) |
         (((bb_word(g.mvd, wi) >> sh) & 1u) << 5) | (((bb_word(g.rev, wi) >> sh) & 1u) << 6);
}
SD uint32_t key11_of(uint32_t b) {  // b = cell_bits of a piece
  uint32_t t = b & 15u;
  return !(b & 64u) ? 1u << 10 : t <= 10u ? 1u << (t - 1u) : 0u;
}
SD uint32_t key13_of(uint32_t b) {
  uint32_t t = b & 15u;
  return !(b & 64u) ? 1u << 12 : t <= 10u ? 1u << (t - 1u) : t == (uint32_t)T_BOMB ? 1u << 10 : 0u;
}
// The trackers' share of one ply, judged on the position BEFORE the move (g is unchanged).
// pt / tt = type of the moving piece / of what stands on the target square (0 = empty).
// Written for one thread per game next to 31 other games: the mover's record is the only thing
// read (one 16-byte load), every other update is an OR at the L2, and the only loops run over
// the (few) pieces that stand next to an enemy.
SD void track_ply(uint32_t* trk, const Game& g, int two_square, int side, int from, int to, int dist, int pt, int tt) {
  const BB occ = occupied(g), mine = owned_by(g, occ, side), enemy = bb_andn(occ, mine);
  // everything the ply reads from the block, in one trip: the mover's record, the target's first word (its
  // start square, needed if it dies) and the number of pieces captured so far
  uint32_t r0, r1, r2, r3;
  sd_ld128(trk + 4 * from, r0, r1, r2, r3);
  const uint32_t d0 = sd_ld32(trk + 4 * to);
  const uint32_t deaths = sd_ld32(trk + kTrkDeaths);
  // (i) active adjacency: every legal one-square capture that is not the move played.
  // att[d] = own movable pieces with an enemy on the next square in direction d.
  {
    const BB movable = bb_andn(mine, bb_and(g.t3, bb_or(g.t2, bb_and(g.t1, g.t0))));
    BB att[4];
    att[0] = bb_and(movable, bb_down<10>(enemy));
    att[1] = bb_and(bb_and(movable, bb_down<1>(enemy)), bb_const(kNotCol9));
    att[2] = bb_and(movable, bb_up<10>(enemy));
    att[3] = bb_and(bb_and(movable, bb_up<1>(enemy)), bb_const(kNotCol0));
    const Ban ban = two_square_ban(g, side, two_square);
    const int skip_from = ban.from >= 0 && ban.k <= 1 ? ban.from : -1;  // that capture is not legal: no chance to attack
    const CellSel sb = cell_sel(skip_from >= 0 ? skip_from : 0), sf = cell_sel(from);
    const bool played = tt != 0 && dist == 1;
    const int pdir = to - from == 10 ? 0 : to - from == 1 ? 1 : to - from == -10 ? 2 : 3;
    STRAT_UNROLL
    for (int d = 0; d < 4; ++d)
      STRAT_UNROLL
      for (int i = 0; i < 4; ++i) {
        if (skip_from >= 0 && ban.dir == d) att[d].w[i] &= ~sb.m[i];
        if (played && pdir == d) att[d].w[i] &= ~sf.m[i];
      }
    // next to a HIDDEN enemy piece: the key is the same for all of them, no square needs a look
    const BB hid = bb_andn(enemy, g.rev);
    BB ph;
    {
      BB h0 = bb_down<10>(hid), h1 = bb_down<1>(hid), h2 = bb_up<10>(hid), h3 = bb_up<1>(hid);
      STRAT_UNROLL
      for (int i = 0; i < 4; ++i)
        ph.w[i] = (att[0].w[i] & h0.w[i]) | (att[1].w[i] & h1.w[i]) | (att[2].w[i] & h2.w[i]) | (att[3].w[i] & h3.w[i]);
    }
    if (bb_get(ph, sf)) r1 |= 1u << 10;  // the mover's record is in registers and is written back below
    STRAT_UNROLL
    for (int i = 0; i < 4; ++i) {
      uint32_t w = ph.w[i] & ~sf.m[i];
      while (w) { int p = 32 * i + sd_ffs(w) - 1; w &= w - 1; sd_or32(trk + 4 * p + 1, 1u << 10); }
    }
    // next to a REVEALED enemy piece: walk those enemies (few), their type is the key
    const BB seen = bb_and(enemy, g.rev);
    BB qs;
    {
      BB a0 = bb_up<10>(att[0]), a1 = bb_up<1>(att[1]), a2 = bb_down<10>(att[2]), a3 = bb_down<1>(att[3]);  // targets of the attackers
      STRAT_UNROLL
      for (int i = 0; i < 4; ++i) qs.w[i] = seen.w[i] & (a0.w[i] | a1.w[i] | a2.w[i] | a3.w[i]);
    }
    STRAT_UNROLL
    for (int i = 0; i < 4; ++i) {
      uint32_t w = qs.w[i];
      while (w) {
        int q = 32 * i + sd_ffs(w) - 1; w &= w - 1;
        uint32_t key = key11_of(cell_bits(g, q));
        STRAT_UNROLL
        for (int d = 0; d < 4; ++d) {
          const int p = q - (d == 0 ? 10 : d == 1 ? 1 : d == 2 ? -10 : -1);
          if (p < 0 || p > 99 || !bb_test(att[d], p)) continue;
          if (p == from) r1 |= key; else if (key) sd_or32(trk + 4 * p + 1, key);
        }
      }
    }
  }
  if (tt == 0) {
    // the previous ply, if it was a move to an empty square, may have threatened
    const uint32_t e0 = hist_entry(g, 0);
    const int x = (int)(e0 >> 7);
    const bool prev = e0 != kHistNone && g.battleless > 0 && bb_test(enemy, x);
    const uint32_t bA = prev ? cell_bits(g, x) : 0u;
    const uint32_t kA11 = key11_of(bA), kA13 = key13_of(bA);
    // (ii) evasion
    if (prev && cells_adjacent(from, x) && !cells_adjacent(to, x)) r0 |= kA11 << 11;
    const uint32_t kC13 = (bb_test(g.rev, from) || dist >= 2) ? (pt <= 10 ? 1u << (pt - 1) : 0u) : 1u << 12;  // what C shows after this move
    const int tr = to / 10, tq = to - 10 * tr;
    STRAT_UNROLL
    for (int d = 0; d < 4; ++d) {  // the four squares next to the new square
      const bool on = d == 0 ? tr < 9 : d == 1 ? tq < 9 : d == 2 ? tr > 0 : tq > 0;
      const int q = to + (d == 0 ? 10 : d == 1 ? 1 : d == 2 ? -10 : -1);
      if (!on || q == from) continue;
      const uint32_t b = cell_bits(g, q);
      const bool piece = (b & 15u) != 0u, theirs = piece && (int)((b >> 4) & 1u) != side;
      if (theirs) r0 |= key11_of(b);                                       // (iv) threat
      if (prev && cells_adjacent(q, x)) {                                  // (iii) protection
        if (piece && !theirs) {
          r1 |= key13_of(b) << 11; r2 |= kA13;
          if (kC13) sd_or32(trk + 4 * q + 2, kC13 << 13);
          if (kA13) sd_or32(trk + 4 * q + 3, kA13);
        } else if (!piece && !is_lake_cell(q)) {
          r1 |= 1u << (11 + 11); r2 |= kA13;                              // ... of an empty square
        }
      }
    }
    sd_st128(trk + 4 * to, r0, r1, r2, r3);
  } else {
    // (v) captures and causes of death; "revealed at the time of the attack" = before this battle
    const bool d_rev = bb_test(g.rev, to) != 0;
    const int out = battle(pt, tt);
    const bool d_dies = out >= 0 && tt != T_FLAG, c_dies = out <= 0;
    uint32_t n = deaths;  // one thread owns the block: a plain store, no atomic to wait for
    sd_st32(trk + kTrkDeaths, deaths + (d_dies ? 1u : 0u) + (c_dies ? 1u : 0u));
    if (d_dies) {
      uint32_t cause = tt <= 10 ? (d_rev ? (out > 0 ? 4u : 5u) : 6u) : 0u;
      if (n < (uint32_t)kTrkMaxDeaths)
        sd_st32(trk + kTrkDeathList + n, ((d0 >> 22) & 127u) | ((uint32_t)tt << 7) | ((uint32_t)(side ^ 1) << 11) |
                                             ((uint32_t)to << 12) | (cause << 19));
      ++n;
    }
    if (c_dies) {
      uint32_t cause = d_rev ? (out < 0 ? 1u : 2u) : 3u;
      if (n < (uint32_t)kTrkMaxDeaths)
        sd_st32(trk + kTrkDeathList + n, ((r0 >> 22) & 127u) | ((uint32_t)pt << 7) | ((uint32_t)side << 11) |
                                             ((uint32_t)to << 12) | (cause << 19));
    }
    if (out > 0) sd_st128(trk + 4 * to, r0, r1, r2, r3);
  }
  // the ply itself
  sd_st16(trk + kTrkMoves, (int)(g.ply & 31u), (uint32_t)from | ((uint32_t)to << 7));
}

struct StepOut { int reward; uint32_t done; bool illegal; bool needs_reset; bool nomove_pending; };

// kValidate = false only when `a` was just drawn from this state's own legal mask.
// kDeferReset: the caller performs the auto-reset itself (epoch is already advanced) when
// o.needs_reset is set; the result must equal reset_game(P, local_game, g).
// kDeferNoMove (on-chip rollouts): "the opponent has no legal move" is left open (o.nomove_pending) unless
// a draw by ply cap or battleless count is due, whose rank in R#12 needs the answer now.  The caller learns
// it from the next ply's own move generation and closes the game with finish_no_move: the opponent's move
// set is computed once per ply instead of twice.
template <bool kValidate, bool kDeferReset = false, bool kChase = false, bool kTrack = false, bool kDeferNoMove = false>
SD StepOut step_game(const Params& P, uint32_t local_game, Game& g, int a) {
  StepOut o; o.illegal = false; o.needs_reset = false; o.nomove_pending = false;
  if (g.done) { o.reward = 0; o.done = 1u | (g.reason << 2); return o; }  // R#15: frozen
  int side = g.ply & 1u;
  // a live game without a legal move (only a hand-built line can be one: play ends such games)
  // has no action to take: the "action" -1 is illegal like any other
  if (!kValidate && a < 0) { o.reward = 0; o.done = 0; o.illegal = true; return o; }
  uint16_t* glog = kChase ? game_log(P, local_game) : nullptr;
  if (kValidate && !action_is_legal(g, side, rules_of<kChase>(P), a, glog)) { o.reward = 0; o.done = 0; o.illegal = true; return o; }
  int from = a / 36, rem = a - 36 * from, d = rem / 9, dist = rem - 9 * d + 1;
  int to = from + dist * (d == 0 ? 10 : d == 1 ? 1 : d == 2 ? -10 : -1);
  CellSel sf = cell_sel(from), st = cell_sel(to);
  int pt = bb_get(g.t0, sf) | (bb_get(g.t1, sf) << 1) | (bb_get(g.t2, sf) << 2) | (bb_get(g.t3, sf) << 3);
  uint32_t prev = bb_get(g.rev, sf);
  int tt = bb_get(g.t0, st) | (bb_get(g.t1, st) << 1) | (bb_get(g.t2, st) << 2) | (bb_get(g.t3, st) << 3);
  if (kTrack && P.track)  // S2 trackers, judged on the position before the move
    track_ply(game_track(P, local_game), g, P.two_square, side, from, to, dist, pt, tt);
  if (kChase && P.chase_rule) {  // chase state machine (R#28), judged on the position before the move
    uint32_t ap = chase_age(g, side), aq = chase_age(g, side ^ 1);
    if (tt != 0) {
      ap = aq = 0;  // a battle ends every chase
    } else {
      BB occ0 = occupied(g);
      BB enemy0 = bb_andn(occ0, owned_by(g, occ0, side));
      bool threat = bb_any(bb_and(neighbours_of(to), enemy0));
      if (aq > 0) {  // the opponent's previous ply was a threat by the piece now on x
        uint32_t e0 = hist_entry(g, 0);
        bool evade = e0 != kHistNone && cells_adjacent(from, (int)(e0 >> 7)) && !cells_adjacent(to, (int)(e0 >> 7));
        aq = evade ? (aq < 255u ? aq + 1u : 255u) : 0u;
      }
      ap = threat ? (ap > 0 ? (ap < 255u ? ap + 1u : 255u) : 1u) : 0u;
    }
    g.chase = side == 0 ? (ap | (aq << 8)) : (aq | (ap << 8));
    if (glog) sd_stlog(glog + (g.logn & (uint32_t)(kLogPlies - 1)), (uint16_t)((uint32_t)from | ((uint32_t)to << 7)));
    g.logn += 1;
  }
  hist_push(g, (uint32_t)from | ((uint32_t)to << 7));
  bool flag_captured = false;
  int outcome = 1;  // plain move = the mover arrives
  // the battle is decided first, without branches on the lanes' different cases
  const bool fight = tt != 0;
  g.battleless = fight ? 0u : g.battleless + 1u;
  prev = fight ? 1u : (prev | (dist >= 2 ? 1u : 0u));  // battle: both revealed; R#10: a long move shows a Scout
  outcome = fight ? battle(pt, tt) : 1;
  flag_captured = tt == T_FLAG;
  // One pass over the seven planes: the origin square empties in every case; the target takes the mover's
  // bits (outcome > 0), is cleared (both removed) or stays as it is but revealed (the defender wins; R#11:
  // its moved bit is unchanged).
  {
    const bool win = outcome > 0, stays = outcome < 0;
    const uint32_t bits = win ? ((uint32_t)pt | ((uint32_t)side << 4) | (1u << 5) | (prev << 6)) : 0u;
    BB* planes[7] = {&g.t0, &g.t1, &g.t2, &g.t3, &g.own, &g.mvd, &g.rev};
    STRAT_UNROLL
    for (int i = 0; i < 4; ++i) {
      const uint32_t tm = stays ? 0u : st.m[i];   // target word mask, void when the defender stays
      const uint32_t clr = ~(sf.m[i] | tm);
      STRAT_UNROLL
      for (int p = 0; p < 7; ++p) planes[p]->w[i] = (planes[p]->w[i] & clr) | (((bits >> p) & 1u) ? tm : 0u);
      g.rev.w[i] |= stays ? st.m[i] : 0u;
    }
  }
  g.ply += 1;
  int mover_result = side == 0 ? 1 : -1;
  // terminal tests in R#12 order
  const bool draw_due = (int)g.ply >= P.ply_cap || (P.max_battleless > 0 && (int)g.battleless >= P.max_battleless);
  if (flag_captured) { g.done = 1; g.reason = REASON_FLAG; g.result = mover_result; }
  else if (kDeferNoMove && !draw_due) { o.nomove_pending = true; }
  else if (!has_legal_move(g, side ^ 1, rules_of<kChase>(P), glog)) {
    g.done = 1;
    if (!has_legal_move(g, side, rules_of<kChase>(P), glog)) { g.reason = REASON_NOMOVE_DRAW; g.result = 0; }
    else { g.reason = REASON_NOMOVE_WIN; g.result = mover_result; }
  }
  else if ((int)g.ply >= P.ply_cap) { g.done = 1; g.reason = REASON_PLY_CAP; g.result = 0; }
  else if (P.max_battleless > 0 && (int)g.battleless >= P.max_battleless) {
    g.done = 1; g.reason = REASON_BATTLELESS; g.result = 0;
  }
  o.reward = g.done ? g.result : 0;
  o.done = g.done | ((uint32_t)side << 1) | ((g.done ? g.reason : 0u) << 2);
  if (g.done && P.auto_reset) {  // R#16
    g.epoch += 1;
    if (kDeferReset) o.needs_reset = true;
    else { reset_game(P, local_game, g); if (kTrack && P.track) track_start(game_track(P, local_game), g); }
  }
  return o;
}

// Closes a game whose side to move was found to have no legal move (step_game<..., kDeferNoMove> left the
// test open): exactly what step_game does in that case, auto-reset included.
template <bool kChase>
SD void finish_no_move(const Params& P, uint32_t local_game, Game& g) {
  const int side = (int)(g.ply & 1u);             // cannot move; the previous mover is side ^ 1
  const int mover_result = side == 1 ? 1 : -1;
  g.done = 1;
  if (!has_legal_move(g, side ^ 1, rules_of<kChase>(P), kChase ? game_log(P, local_game) : nullptr)) { g.reason = REASON_NOMOVE_DRAW; g.result = 0; }
  else { g.reason = REASON_NOMOVE_WIN; g.result = mover_result; }
  if (P.auto_reset) { g.epoch += 1; reset_game(P, local_game, g); }
}

// ------------------------------------------------------------------ observation bits (C5)
// The 44 planes as one 4400-bit stream (plane p at bit 100p) = 138 words.  Byte q of the
// stream is exactly the 8 bf16 values of the q-th 16-byte chunk of the game's observation.
SD BB type_is(const Game& g, BB base, int v) {
  BB r;
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i)
    r.w[i] = base.w[i] & ((v & 1) ? g.t0.w[i] : ~g.t0.w[i]) & ((v & 2) ? g.t1.w[i] : ~g.t1.w[i]) &
             ((v & 4) ? g.t2.w[i] : ~g.t2.w[i]) & ((v & 8) ? g.t3.w[i] : ~g.t3.w[i]);
  return r;
}
SD BB hist_plane(uint32_t e, int which) {
  if (e == kHistNone) return bb_zero();
  CellSel s = cell_sel(which ? (int)(e >> 7) : (int)(e & 127));
  BB r;
  STRAT_UNROLL
  for (int i = 0; i < 4; ++i) r.w[i] = s.m[i]; return r;
}
// append `count` (<= 8) planes starting at stream bit 100*first_plane (a multiple of 800 bits
// = 25 words, so every shift below is a compile-time constant once unrolled)
template <int COUNT> SD void pack_planes(const BB (&pl)[8], uint32_t* out) {
  constexpr int NW = (COUNT * 100 + 31) / 32;
  uint32_t o[NW];
STRAT_UNROLL
  for (int k = 0; k < NW; ++k) o[k] = 0;
STRAT_UNROLL
  for (int p = 0; p < COUNT; ++p)
STRAT_UNROLL
    for (int i = 0; i < 4; ++i) {
      const int nb = i == 3 ? 4 : 32, pos = 100 * p + 32 * i, wi = pos >> 5, sh = pos & 31;
      o[wi] |= pl[p].w[i] << sh;
      if (sh != 0 && sh + nb > 32) o[wi + 1] |= pl[p].w[i] >> (32 - sh);
    }
STRAT_UNROLL
  for (int k = 0; k < NW; ++k) out[k] = o[k];
}
SD void encode_bits(const Game& g, uint32_t* out /* 138 words */) {
  int side = g.ply & 1u;
  BB occ = occupied(g);
  BB mine = owned_by(g, occ, side);
  BB enemy = bb_andn(occ, mine);
  BB seen = bb_and(enemy, g.rev);
  BB pl[8];
STRAT_UNROLL
  for (int k = 0; k < 8; ++k) pl[k] = type_is(g, mine, k + 1);                  // planes 0-7
  pack_planes<8>(pl, out);
STRAT_UNROLL
  for (int k = 0; k < 4; ++k) pl[k] = type_is(g, mine, k + 9);                  // 8-11
STRAT_UNROLL
  for (int k = 0; k < 4; ++k) pl[4 + k] = type_is(g, seen, k + 1);              // 12-15
  pack_planes<8>(pl, out + 25);
STRAT_UNROLL
  for (int k = 0; k < 8; ++k) pl[k] = type_is(g, seen, k + 5);                  // 16-23
  pack_planes<8>(pl, out + 50);
  BB hidden = bb_andn(enemy, g.rev);
  pl[0] = bb_and(hidden, g.mvd);                                                 // 24
  pl[1] = bb_andn(hidden, g.mvd);                                                // 25
  pl[2] = bb_const(kLake);                                                       // 26
  pl[3] = bb_andn(bb_const(kNotLake), occ);                                      // 27
  pl[4] = hist_plane(hist_entry(g, 0), 0); pl[5] = hist_plane(hist_entry(g, 0), 1);   // 28,29
  pl[6] = hist_plane(hist_entry(g, 1), 0); pl[7] = hist_plane(hist_entry(g, 1), 1);   // 30,31
  pack_planes<8>(pl, out + 75);
STRAT_UNROLL
  for (int j = 0; j < 4; ++j) {                                                  // 32-39
    pl[2 * j] = hist_plane(hist_entry(g, 2 + j), 0); pl[2 * j + 1] = hist_plane(hist_entry(g, 2 + j), 1);
  }
  pack_planes<8>(pl, out + 100);
STRAT_UNROLL
  for (int j = 0; j < 2; ++j) {                                                  // 40-43
    pl[2 * j] = hist_plane(hist_entry(g, 6 + j), 0); pl[2 * j + 1] = hist_plane(hist_entry(g, 6 + j), 1);
  }
  pack_planes<4>(pl, out + 125);
}

// ------------------------------------------------------------------ canonical <-> device line
SD void import_canonical(const uint8_t* L, Game& g) {
  g.t0 = g.t1 = g.t2 = g.t3 = g.own = g.mvd = g.rev = bb_zero();
  for (int c = 0; c < 100; ++c) {
    uint32_t b = L[c], t = b & 15u;
    if (t == 0 || t == 15) continue;
    put_piece(g, c, (int)t, (b >> 4) & 1u);
    CellSel s = cell_sel(c);
    STRAT_UNROLL
    for (int i = 0; i < 4; ++i) {
      g.mvd.w[i] |= (b & 0x20u) ? s.m[i] : 0u; g.rev.w[i] |= (b & 0x40u) ? s.m[i] : 0u;
    }
  }
  STRAT_UNROLL
  for (int p = 0; p < 4; ++p) {
    uint32_t e[2];
    STRAT_UNROLL
    for (int k = 0; k < 2; ++k) {
      uint32_t f = L[100 + 2 * (2 * p + k)], t = L[101 + 2 * (2 * p + k)];
      e[k] = (f == 0xFF) ? kHistNone : (f | (t << 7));
    }
    g.h[p] = e[0] | (e[1] << 14);
  }
  g.ply = L[116] | ((uint32_t)L[117] << 8);
  g.battleless = L[118] | ((uint32_t)L[119] << 8);
  g.done = L[120] & 1u; g.reason = (L[120] >> 2) & 7u; g.result = (int32_t)(int8_t)L[121];
  g.chase = L[122] | ((uint32_t)L[123] << 8);
  g.logn = 0;
  g.epoch = L[124] | ((uint32_t)L[125] << 8) | ((uint32_t)L[126] << 16) | ((uint32_t)L[127] << 24);
}
SD void export_canonical(const Game& g, uint8_t* L) {
  for (int c = 0; c < 100; ++c) {
    uint32_t t = bb_test(g.t0, c) | (bb_test(g.t1, c) << 1) | (bb_test(g.t2, c) << 2) | (bb_test(g.t3, c) << 3);
    uint32_t b = t | (bb_test(g.own, c) << 4) | (bb_test(g.mvd, c) << 5) | (bb_test(g.rev, c) << 6);
    if (is_lake_cell(c)) b = 15;
    L[c] = (uint8_t)b;
  }
  STRAT_UNROLL
  for (int j = 0; j < 8; ++j) {
    uint32_t e = hist_entry(g, j);
    L[100 + 2 * j] = e == kHistNone ? 0xFF : (uint8_t)(e & 127);
    L[101 + 2 * j] = e == kHistNone ? 0xFF : (uint8_t)(e >> 7);
  }
  L[116] = (uint8_t)g.ply; L[117] = (uint8_t)(g.ply >> 8);
  L[118] = (uint8_t)g.battleless; L[119] = (uint8_t)(g.battleless >> 8);
  L[120] = (uint8_t)(g.done | (g.reason << 2)); L[121] = (uint8_t)(int8_t)g.result;
  L[122] = (uint8_t)g.chase; L[123] = (uint8_t)(g.chase >> 8);
  L[124] = (uint8_t)g.epoch; L[125] = (uint8_t)(g.epoch >> 8); L[126] = (uint8_t)(g.epoch >> 16);
  L[127] = (uint8_t)(g.epoch >> 24);
}

// ------------------------------------------------------------------ determinise (C7)
// Re-type the hidden pieces of the searcher's opponent with a uniformly random arrangement
// consistent with the public history (R#22): each hidden Bomb/Flag, in ascending order of its
// original square, draws a free hidden square, redrawing while that square holds a moved piece;
// the movable types are then shuffled (descending Fisher-Yates) and dealt to the remaining
// free squares.  One DETERMINISE draw stream per output game.  Returns draws used, 0 on the
// 4096-draw safety cap.
struct DrawStream {
  uint32_t gidx, k0, k1, o[4];
  int d;
};
SD uint32_t next_draw(DrawStream& s) {
  if ((s.d & 3) == 0) philox(s.gidx, 0u, (uint32_t)(s.d >> 2), TAG_DETERMINISE, s.k0, s.k1, s.o);
  int k = s.d & 3;
  ++s.d;
  return k == 0 ? s.o[0] : k == 1 ? s.o[1] : k == 2 ? s.o[2] : s.o[3];
}
SD int determinise_game(const Game& root, uint32_t k0, uint32_t k1, uint32_t gidx, bool keep_log, Game& out) {
  out = root;
  if (!keep_log) out.logn = 0;  // the copy's environment keeps no move log: it remembers the 8 plies of its line
  int searcher = root.ply & 1u;
  BB occ = occupied(root);
  BB enemy = bb_andn(occ, owned_by(root, occ, searcher));
  BB hidden = bb_andn(enemy, root.rev);
  uint8_t freeSq[40], T[40], Tm[40];  // freeSq bit 7: the piece on that square has moved
  int n = 0;
  for (int i = 0; i < 4; ++i) {
    uint32_t w = hidden.w[i];
    while (w && n < 40) {
      int b = sd_ffs(w) - 1; w &= w - 1;
      int c = 32 * i + b;
      freeSq[n] = (uint8_t)(c | (bb_test(root.mvd, c) << 7));
      T[n] = (uint8_t)(bb_test(root.t0, c) | (bb_test(root.t1, c) << 1) | (bb_test(root.t2, c) << 2) |
                       (bb_test(root.t3, c) << 3));
      ++n;
    }
  }
  DrawStream ds; ds.gidx = gidx; ds.k0 = k0; ds.k1 = k1; ds.d = 0;
  ds.o[0] = ds.o[1] = ds.o[2] = ds.o[3] = 0;
  int m = n, k = 0;
  for (int j = 0; j < n; ++j) {
    int t = T[j];
    if (t != T_BOMB && t != T_FLAG) { Tm[k++] = (uint8_t)t; continue; }
    for (;;) {
      if (ds.d >= 4096) return 0;
      int idx = (int)bounded(next_draw(ds), (uint32_t)m);
      int sq = freeSq[idx];
      if (sq & 0x80) continue;  // a moved piece cannot be a Bomb or the Flag
      CellSel s = cell_sel(sq);
      bb_put(out.t0, s, t & 1); bb_put(out.t1, s, (t >> 1) & 1); bb_put(out.t2, s, (t >> 2) & 1); bb_put(out.t3, s, (t >> 3) & 1);
      freeSq[idx] = freeSq[m - 1];
      --m;
      break;
    }
  }
  for (int i = k - 1; i >= 1; --i) {
    if (ds.d >= 4096) return 0;
    int j = (int)bounded(next_draw(ds), (uint32_t)(i + 1));
    uint8_t t = Tm[i]; Tm[i] = Tm[j]; Tm[j] = t;
  }
  for (int i = 0; i < k; ++i) {
    CellSel s = cell_sel(freeSq[i] & 0x7F);
    int t = Tm[i];
    bb_put(out.t0, s, t & 1); bb_put(out.t1, s, (t >> 1) & 1); bb_put(out.t2, s, (t >> 2) & 1); bb_put(out.t3, s, (t >> 3) & 1);
  }
  return ds.d > 0 ? ds.d : 1;
}

}  // namespace strat
