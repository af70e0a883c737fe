// Test harness: the per-game device logic (strat_game.cuh) compiled for the HOST on top of
// tests/host_shim.h, so that the CPU-only test run can compare it with the oracle.  Test
// infrastructure only: nothing in the product loads this; there is no CPU path in the library.
#include <cstdint>
#include <cstring>
#include "host_shim.h"
#include "../paper_2511_07312_b200/csrc/strat_game.cuh"

using namespace strat;

static Params make(int variant, uint64_t seed, int max_plies, int auto_reset, int two_square, int chase, uint64_t game_base) {
  Params P;
  memset(&P, 0, sizeof P);
  P.key0 = (uint32_t)seed; P.key1 = (uint32_t)(seed >> 32);
  P.game_base = (uint32_t)game_base; P.num_games = 1; P.variant = variant;
  P.ply_cap = (max_plies >= 1 && max_plies <= 65535) ? max_plies : 65535;
  P.max_battleless = 0; P.auto_reset = auto_reset; P.two_square = two_square; P.chase_rule = chase;
  return P;
}

extern "C" {
// fresh game (global index gidx, epoch 0) -> canonical line
void hh_reset(int variant, uint64_t seed, uint32_t gidx, uint8_t* line) {
  Params P = make(variant, seed, 0, 0, 1, 0, 0);
  Game g; g.epoch = 0;
  setup_game(P, gidx, g);
  export_canonical(g, line);
}
int hh_legal_mask(const uint8_t* line, int two_square, int chase, uint32_t* row) {
  Game g; import_canonical(line, g);
  memset(row, 0, 113 * 4);
  int cnt[4] = {0, 0, 0, 0};
  if (g.done) return 0;
  return legal_mask_row(g, g.ply & 1, (two_square ? RULE_TWO_SQUARE : 0) | (chase ? RULE_CHASE : 0), row, cnt, nullptr);
}
// r-th legal action two ways: from the mask row, and mask-free (count_actions / choose_action)
int hh_pick(const uint8_t* line, int two_square, int chase, uint32_t u, int* mask_free) {
  Game g; import_canonical(line, g);
  uint32_t row[113]; memset(row, 0, sizeof row);
  int cnt[4] = {0, 0, 0, 0}, rules = (two_square ? RULE_TWO_SQUARE : 0) | (chase ? RULE_CHASE : 0);
  if (g.done) { *mask_free = -1; return -1; }
  int n = legal_mask_row(g, g.ply & 1, rules, row, cnt, nullptr);
  uint32_t scouts[16];
  ActionSet A;
  count_actions(g, g.ply & 1, rules, scouts, A);
  *mask_free = choose_action(g, g.ply & 1, rules, A, u, scouts, nullptr, 8);
  return pick_action(row, cnt, n, u);
}
// one validated step of game `gidx` (auto-reset inside, like strat_step)
void hh_step(const uint8_t* line, int variant, uint64_t seed, uint32_t gidx, int max_plies, int auto_reset,
             int two_square, int chase, int action, uint8_t* line_out, int* reward, int* done, int* illegal) {
  Params P = make(variant, seed, max_plies, auto_reset, two_square, chase, 0);
  Game g; import_canonical(line, g);
  StepOut o = step_game<true, false, true>(P, gidx, g, action);
  export_canonical(g, line_out);
  *reward = o.reward; *done = (int)o.done; *illegal = o.illegal ? 1 : 0;
}
// S2 trackers: start a game's 512-word tracker block from a line ...
void hh_track_start(const uint8_t* line, uint32_t* trk) {
  Game g; import_canonical(line, g);
  track_start(trk, g);
}
// ... and one validated, tracked step of game `gidx` (auto-reset inside restarts the trackers)
void hh_track_step(const uint8_t* line, uint32_t* trk, int variant, uint64_t seed, uint32_t gidx, int max_plies,
                   int auto_reset, int action, uint8_t* line_out, int* illegal) {
  Params P = make(variant, seed, max_plies, auto_reset, 1, 0, gidx);
  P.track = trk;
  Game g; import_canonical(line, g);
  StepOut o = step_game<true, false, false, true>(P, 0u, g, action);
  export_canonical(g, line_out);
  *illegal = o.illegal ? 1 : 0;
}
// observation as 4400 bf16 bit patterns
void hh_encode(const uint8_t* line, uint16_t* obs) {
  Game g; import_canonical(line, g);
  uint32_t bits[139]; memset(bits, 0, sizeof bits);
  encode_bits(g, bits);
  for (int i = 0; i < 4400; ++i) obs[i] = ((bits[i >> 5] >> (i & 31)) & 1u) ? 0x3F80 : 0;
}
}
