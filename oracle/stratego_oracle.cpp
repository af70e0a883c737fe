// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, single-threaded CPU implementation of the batched Stratego
// environment step of arxiv 2511.07312 ("Ataraxos"), written from the rules
// text of the paper.  It shares no code, header, table or helper with the CUDA
// path under paper_2511_07312_b200/csrc/ and neither imports the other.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this library.
//
// Citations: P:NNN = /root/reference/PAPER.md line NNN.  BJ = BASELINE.json.
// R#n = reading n of the paper listed in DESIGN.md ("Readings").
//
// Parity status of each function (what pins it, see tests/test_oracle_*.py):
//   philox4x32_10      pinned: Random123 known-answer vectors.
//   battle             pinned: rules text P:208-210 enumerated as a 120-entry table.
//   setup              pinned: multiset, chi-square marginals, count 1.41e33.
//   legal moves        pinned: hand-worked positions E1-E5, closed form at ply 0,
//                      mirror/rotation metamorphic maps, naive Python enumerator.
//   two-square (non-Scout) pinned: BJ wording "A->B,B->A,A->B then B->A illegal".
//   two-square (Scout overlap reading R#6)   PARITY UNPINNED against the paper
//                      (P:246 only says "special care"); fixed by worked example E5.
//   step / terminal    pinned: invariants, worked endings.
//   reveal-on-long-Scout-move (R#10), reward timing (R#13), absolute
//   orientation (R#1), setup rejection (R#5): PARITY UNPINNED (paper silent).
//   encode             pinned: partition property, start-position counts,
//                      information-state property.
//   replay ring        pinned: FIFO content, chi-square of indices.
//   determinise        pinned: multiset/constraint/obs-equality properties, chi-square of
//                      Bomb/Flag placement over the unmoved squares.
//   continuous chasing (R#28) pinned: hand-worked chase around a 2x2 block, state-machine
//                      cases, independent snapshot checker.  The mechanics the paper leaves
//                      open (what ends a chase, the length of its memory) are PARITY UNPINNED against it.
//   search step (R#29)  pinned: expansion structure, hand-computed rho and equal-value limit,
//                      per-action averaging, KKT conditions of eq. (7) at the eq. (8) output.
//                      The stand-ins for the networks are this build's (R#29), not the paper's.
//   setup pool (R#30)   pinned: every dealt side is a pool entry, entries are used uniformly
//                      (chi-square), the two sides draw independently.
//   pinned reset (R#27) pinned: a restarted game equals its pinned line byte for byte except
//                      the epoch; the reading itself (epoch keeps counting) is PARITY UNPINNED
//                      against the paper (P:252-254 gives no detail).
//
//   information state S2 (P:482-610, 487 channels; readings I1-I9 in DESIGN.md):
//                      pinned: hand-built mini-games for every channel group (threat, evasion,
//                      declined attack, protection of a piece and of an empty square, each of
//                      the six causes of death, captures by start square), channel sums fixed by
//                      the piece counts, start-square and move channels against the played
//                      moves, information-state property, channels 12-35 against the empirical
//                      marginals of the (independent) determinisation sampler and by hand.
//                      The READING of channels 12-35 ("assuming the setup and moves were
//                      selected uniformly at random": taken as uniform over the
//                      arrangements consistent with revealed / moved, the likelihood of the
//                      observed moves ignored) and the mechanics the paper leaves open (what
//                      counts as a threat / protection of an empty square, the square a piece
//                      "died in", ten type channels per cause of death) are PARITY UNPINNED
//                      against the paper's own simulator.
//
// Layouts:
//   canonical line, 128 B per game:
//     0..99   cell bytes: bits0-3 type (0 empty, 1 Spy,2 Scout,3 Miner,4 Sergeant,
//             5 Lieutenant,6 Captain,7 Major,8 Colonel,9 General,10 Marshal,
//             11 Flag,12 Bomb, 15 lake)  [type order P:499], bit4 owner (0 red,
//             1 blue), bit5 moved, bit6 revealed
//     100..115 history entry j = (from,to) of ply t-1-j, 0xFF,0xFF if none
//     116..117 ply (LE u16)   118..119 battleless count (LE u16)
//     120 flags: bit0 done, bits2-4 reason (1 flag,2 no-move win,3 no-move draw,
//             4 ply cap,5 battleless)    121 result (int8, red's)
//     122..123 chase age of red / blue (R#28; 0 unless chase_rule is on)
//     124..127 epoch (LE u32)
//   cell c = 10*row + col; red home rows 0-3, blue home rows 6-9;
//   lakes {42,43,52,53,46,47,56,57} (BJ configs[0]: c5-d6, g5-h6).
//   action a = from*36 + dir*9 + (dist-1); dir 0:+row 1:+col 2:-row 3:-col.
//   mask bit a -> word a>>5, bit a&31; 113 words per game.

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <new>

namespace {

constexpr int kCells = 100;
constexpr int kLine = 128;
constexpr int kMaskWords = 113;
constexpr int kPlanes = 44;
constexpr int kObs = kPlanes * kCells;  // 4400 bf16 per game
constexpr int kInfoPlanes = 487;        // 455 board/history channels + 32 move channels
constexpr int kInfo = kInfoPlanes * kCells;

constexpr int T_EMPTY = 0, T_SPY = 1, T_SCOUT = 2, T_MINER = 3, T_MARSHAL = 10,
              T_FLAG = 11, T_BOMB = 12, T_LAKE = 15;
constexpr uint8_t B_OWNER = 0x10, B_MOVED = 0x20, B_REVEALED = 0x40;

constexpr int ORC_OK = 0, ORC_BAD_ARG = -1, ORC_BAD_STATE = -2, ORC_ILLEGAL_ACTION = -4;

enum { TAG_SETUP_RED = 0, TAG_SETUP_BLUE = 1, TAG_ACTION = 2, TAG_SAMPLE = 3, TAG_DETERMINISE = 4 };
enum { REASON_NONE = 0, REASON_FLAG = 1, REASON_NOMOVE_WIN = 2, REASON_NOMOVE_DRAW = 3,
       REASON_PLY_CAP = 4, REASON_BATTLELESS = 5 };

struct Config {  // mirrors the field order of the product's strat_config on purpose
                 // (same C-ABI shape), but is declared independently.
  int32_t num_games;
  int32_t variant;  // 0 classic, 1 barrage
  uint64_t seed;
  int32_t max_plies;       // 0 = none (hard cap 65535, the u16 ply field)
  int32_t max_battleless;  // 0 = off
  int32_t auto_reset;
  int32_t two_square;
  int32_t device;  // unused here
  int32_t chase_rule;      // 1: apply the continuous-chasing rule (R#28)
  uint64_t game_base;  // global index of game 0 (RNG keying under sharding)
  int32_t infostate;   // 1: keep the per-piece trackers of the paper's information state (S2)
  int32_t reserved;
};

// ---- trackers of the paper's information state.  Everything a channel of S2 needs
// beyond the board itself.  A piece is identified by the square it started the game on
// (P:606 needs that anyway); its history bits travel with that identity.
// Keys: a set over "the other piece at the time" = revealed type Spy..Marshal (bits 0-9),
// revealed Bomb (bit 10, protection groups only), bit 11 = empty square (channel 262) / padding
// (channels 275, 288, 301: never set), bit 12 = that piece was not revealed.  The three 11-wide
// groups (threat, evasion, active adjacency) use bits 0-9 and bit 12.
struct PieceTrack {
  uint16_t threatened;       // P:519-520 "has ever threatened a piece of the opponent which ... was"
  uint16_t evaded;           // P:526-527 "has ever evaded a threat from an opponent's piece which ... was"
  uint16_t adjacent;         // P:533-534 "has ever been actively adjacent to an opponent's piece which ... was"
  uint16_t protected_piece;  // P:576-578 "has ever protected a piece of the player which ... / an empty square"
  uint16_t protected_against;
  uint16_t was_protected_by;
  uint16_t was_protected_against;
};
struct Track {
  int id_at[kCells];             // start square of the piece standing on each square, -1 if none
  PieceTrack piece[kCells];      // by start square
  int start_type[kCells];        // what stood on each square when the game started (0 = nothing)
  int start_owner[kCells];
  bool captured[kCells];         // by start square
  bool died[2][6][10][kCells];   // [owner][cause 1..6][type Spy..Marshal][square of the battle]
  int moves[32][2];              // most recent first; [j][0] = -1 if there is no such move
};

struct Game {
  uint8_t cell[kCells];
  uint8_t hist[8][2];
  int ply;
  int battleless;
  bool done;
  int reason;
  int result;  // red's
  uint32_t epoch;
  // Two-square state machine: "tracking the last four positions occupied
  // by the last-acting piece for each player".
  int chain_len[2];
  int chain[2][4];
  // Continuous-chasing state machine (R#28): number of positions of the player's
  // running chase, counted from the one right after its first threat; 0 = not chasing.
  int chase_age[2];
  // Move log of the chasing rule's memory: the last 64 plies played since this state was
  // set up or loaded (circular by logn).  Not part of the canonical line: a loaded state
  // remembers the 8 plies its line carries.
  int logn;
  uint8_t log[64][2];
};

// "The distribution from which the initial board is sampled can be customized"; in the
// paper's training a pool of 1,000 network-generated setups per player per GPU.  K setups
// per side, 40 type codes each (entry i of a red setup -> cell i, of a blue one -> cell 60+i).
struct SetupPool {
  int K = 0;
  std::vector<uint8_t> side[2];
};

struct Env {
  Config cfg;
  std::vector<Game> g;
  std::vector<Track> track;  // one per game when cfg.infostate, else empty
  int error;
  SetupPool pool;
  // "Reset Behaviour and Support for Search": terminated boards restart from a
  // custom non-initial state instead of a fresh setup.  Empty = not pinned.
  std::vector<uint8_t> pin;
  // "the continuous chasing rule needs to be tested against the history of board states that leads
  // to the non-initial reset state": per game up to 63 plies (from,to) that led to the
  // pinned state, most recent first, 0xFF = unknown.  Empty = the 8 plies of the line only.
  std::vector<uint8_t> pin_plies;
};

// ---------------------------------------------------------------- geometry
bool is_lake(int c) {
  return c == 42 || c == 43 || c == 52 || c == 53 || c == 46 || c == 47 || c == 56 || c == 57;
}
int type_of(uint8_t b) { return b & 15; }
int owner_of(uint8_t b) { return (b >> 4) & 1; }
bool is_piece(uint8_t b) { return type_of(b) >= 1 && type_of(b) <= 12; }
bool is_movable_type(int t) { return t >= 1 && t <= 10; }
const int DROW[4] = {1, 0, -1, 0};
const int DCOL[4] = {0, 1, 0, -1};

// ---------------------------------------------------------------- C1 RNG
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw 2011, "Parallel random numbers: as
// easy as 1, 2, 3").  BJ north_star: "Philox4x32-10-seeded".
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Draw d of a stream instance = word d&3 of block d>>2 (R#3).
uint32_t stream_draw(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2_base, uint32_t tag, int d) {
  uint32_t ctr[4] = {c0, c1, c2_base + (uint32_t)(d >> 2), tag};
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t out[4];
  philox4x32_10(ctr, key, out);
  return out[d & 3];
}

// Bounded integer in [0,n): (u*n) >> 32 (R#3; no rejection, deterministic).
uint32_t bounded(uint32_t u, uint32_t n) { return (uint32_t)(((uint64_t)u * n) >> 32); }

// ---------------------------------------------------------------- C2 setup
// BJ configs[0]: Flag 1, Bomb 6, Spy 1, Scout 8, Miner 5, Sergeant 4, Lieutenant 4,
// Captain 4, Major 3, Colonel 2, General 1, Marshal 1, in that listed order.
// BJ configs[1]: Flag, Marshal, General, Miner, Scout x2, Spy, Bomb, then 32 empties.
void multiset(int variant, int A[40]) {
  int n = 0;
  if (variant == 0) {
    const int types[12] = {11, 12, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10};
    const int count[12] = {1, 6, 1, 8, 5, 4, 4, 4, 3, 2, 1, 1};
    for (int k = 0; k < 12; ++k)
      for (int i = 0; i < count[k]; ++i) A[n++] = types[k];
  } else {
    const int b[8] = {11, 10, 9, 3, 2, 2, 1, 12};
    for (int k = 0; k < 8; ++k) A[n++] = b[k];
    while (n < 40) A[n++] = 0;
  }
}

// R#5: a side's setup is redrawn until it owns a movable piece with an on-board,
// non-lake 4-neighbour not holding one of its own pieces.
bool side_can_ever_move(const uint8_t cell[kCells], int side) {
  for (int c = 0; c < kCells; ++c) {
    uint8_t b = cell[c];
    if (!is_piece(b) || owner_of(b) != side || !is_movable_type(type_of(b))) continue;
    int r = c / 10, q = c % 10;
    for (int d = 0; d < 4; ++d) {
      int rr = r + DROW[d], qq = q + DCOL[d];
      if (rr < 0 || rr > 9 || qq < 0 || qq > 9) continue;
      int t = rr * 10 + qq;
      if (is_lake(t)) continue;
      if (is_piece(cell[t]) && owner_of(cell[t]) == side) continue;
      return true;
    }
  }
  return false;
}

// Returns the number of attempts used (1 unless the first permutation left the side immobile).
int setup_side(const Config& cfg, uint32_t gidx, uint32_t epoch, int side, uint8_t cell[kCells]) {
  for (uint32_t attempt = 0;; ++attempt) {
    int A[40];
    multiset(cfg.variant, A);
    // Descending Fisher-Yates (R#4): for i = 39..1: j = bounded(draw[39-i], i+1).
    for (int i = 39; i >= 1; --i) {
      uint32_t u = stream_draw(cfg.seed, gidx, epoch, attempt << 8,
                               side == 0 ? TAG_SETUP_RED : TAG_SETUP_BLUE, 39 - i);
      int j = (int)bounded(u, (uint32_t)(i + 1));
      int tmp = A[i]; A[i] = A[j]; A[j] = tmp;
    }
    int base = side == 0 ? 0 : 60;
    for (int i = 0; i < 40; ++i)
      cell[base + i] = A[i] == 0 ? 0 : (uint8_t)(A[i] | (side ? B_OWNER : 0));
    if (side_can_ever_move(cell, side)) return (int)attempt + 1;
  }
}

void clear_dynamic(Game& gm) {
  memset(gm.hist, 0xFF, sizeof gm.hist);
  gm.ply = 0; gm.battleless = 0; gm.done = false; gm.reason = 0; gm.result = 0;
  gm.chain_len[0] = gm.chain_len[1] = 0;
  gm.chase_age[0] = gm.chase_age[1] = 0;
  gm.logn = 0;
}

void new_game(const Config& cfg, uint32_t gidx, Game& gm, const SetupPool* pool = nullptr) {  // epoch already set
  memset(gm.cell, 0, sizeof gm.cell);
  for (int c = 0; c < kCells; ++c)
    if (is_lake(c)) gm.cell[c] = T_LAKE;
  clear_dynamic(gm);
  if (pool && pool->K > 0) {  // R#30: each side's setup = pool entry bounded(first draw of its SETUP stream, K)
    for (int side = 0; side < 2; ++side) {
      uint32_t u = stream_draw(cfg.seed, gidx, gm.epoch, 0, side == 0 ? TAG_SETUP_RED : TAG_SETUP_BLUE, 0);
      const uint8_t* A = &pool->side[side][(size_t)bounded(u, (uint32_t)pool->K) * 40];
      int base = side == 0 ? 0 : 60;
      for (int i = 0; i < 40; ++i) gm.cell[base + i] = A[i] == 0 ? 0 : (uint8_t)(A[i] | (side ? B_OWNER : 0));
    }
    return;
  }
  // Each side depends on its own pieces only, so the order of the two is immaterial.
  setup_side(cfg, gidx, gm.epoch, 0, gm.cell);
  setup_side(cfg, gidx, gm.epoch, 1, gm.cell);
}

// ---------------------------------------------------------------- C3 legal moves
// Two-square rule: "prohibits a piece from crossing the same square
// boundary on more than three consecutive turns of its owner".  Reading R#6: the
// candidate move of the chain's piece is banned iff the chain holds four positions
// (three consecutive moves of that piece), the three moves and the candidate lie on
// one row or column, and the four of them cross at least one common boundary.
bool two_square_banned(const Game& gm, int side, int from, int to) {
  if (gm.chain_len[side] != 4) return false;
  const int* p = gm.chain[side];
  if (p[3] != from) return false;
  int pos[5] = {p[0], p[1], p[2], p[3], to};
  bool same_row = true, same_col = true;
  for (int i = 1; i < 5; ++i) {
    if (pos[i] / 10 != pos[0] / 10) same_row = false;
    if (pos[i] % 10 != pos[0] % 10) same_col = false;
  }
  if (!same_row && !same_col) return false;
  // Coordinate along the line; boundary b lies between coordinates b and b+1.
  int x[5];
  for (int i = 0; i < 5; ++i) x[i] = same_row ? pos[i] % 10 : pos[i] / 10;
  for (int b = 0; b < 9; ++b) {
    bool all = true;
    for (int m = 0; m < 4; ++m) {
      int lo = x[m] < x[m + 1] ? x[m] : x[m + 1];
      int hi = x[m] < x[m + 1] ? x[m + 1] : x[m];
      if (!(lo <= b && b < hi)) all = false;
    }
    if (all) return true;
  }
  return false;
}

// ---- continuous-chasing rule (reading R#28)
bool adjacent(int a, int b) {
  int dr = a / 10 - b / 10, dc = a % 10 - b % 10;
  return (dr == 0 && (dc == 1 || dc == -1)) || (dc == 0 && (dr == 1 || dr == -1));
}
// "a threat [is] an action that moves a piece adjacent to a piece of the opponent";
// a move onto an opponent's piece is a battle, not a threat.
bool is_threat(const Game& gm, int side, int from, int to) {
  if (gm.cell[to] != 0) return false;
  for (int d = 0; d < 4; ++d) {
    int rr = to / 10 + DROW[d], qq = to % 10 + DCOL[d];
    if (rr < 0 || rr > 9 || qq < 0 || qq > 9) continue;
    int c = rr * 10 + qq;
    if (c == from) continue;  // the square the piece leaves
    if (is_piece(gm.cell[c]) && owner_of(gm.cell[c]) != side) return true;
  }
  return false;
}
// "An evade is an action that moves a piece that was threatened on the previous turn away
// from the piece that threatened it", "to an empty square".  The opponent's
// chase_age > 0 says its previous ply was a threat; the threatening piece stands on that
// ply's destination square.
bool is_evade(const Game& gm, int side, int from, int to) {
  if (gm.chase_age[side ^ 1] == 0 || gm.hist[0][0] == 0xFF) return false;
  if (gm.cell[to] != 0) return false;
  int x = gm.hist[0][1];
  return adjacent(from, x) && !adjacent(to, x);
}
// "a player who is chasing may not make a threat that would result in a position that has
// already taken place during the chase, unless that threat would return the moved piece to the
// square it occupied prior to the previous turn of the chasing player".  A position is
// the type and owner of the piece on every square.  The chase's earlier positions are rebuilt
// by taking back the logged plies one by one (no battle happens inside a chase); the state
// remembers the 8 plies of its line and up to 63 plies played since it was loaded (R#28).
bool chase_banned(const Game& gm, int side, int from, int to) {
  int age = gm.chase_age[side];
  if (age < 2) return false;
  if (!is_threat(gm, side, from, to)) return false;
  int first = ((gm.ply & 1) == side) ? 1 : 0;  // history entry of this player's previous ply
  if (gm.hist[first][0] != 0xFF && from == gm.hist[first][1] && to == gm.hist[first][0]) return false;
  uint8_t R[kCells], K[kCells];
  for (int c = 0; c < kCells; ++c) R[c] = K[c] = (uint8_t)(gm.cell[c] & 0x1F);
  R[to] = R[from]; R[from] = 0;
  // look-back b = 1 takes the last ply back, b = 2 the one before, ...: plies 1..8 are in the
  // line's history, plies up to 63 in the move log if that many were played since the load
  for (int b = 1; b <= age - 1; ++b) {
    int f, g;
    if (b <= 8) {
      if (gm.hist[b - 1][0] == 0xFF) break;
      f = gm.hist[b - 1][0]; g = gm.hist[b - 1][1];
    } else if (b <= gm.logn && b <= 63) {
      f = gm.log[(gm.logn - b) & 63][0]; g = gm.log[(gm.logn - b) & 63][1];
    } else {
      break;
    }
    K[f] = K[g]; K[g] = 0;  // take the ply back
    if (memcmp(R, K, kCells) == 0) return true;
  }
  return false;
}

// Is (from,dir,dist) a legal move for `side` on this board?  P:210: movable pieces
// move one square in a cardinal direction onto an empty square or an opponent's
// piece; Scouts any number of squares "so long as the movement does not jump over a
// lake or an occupied square".
bool move_is_legal(const Game& gm, const Config& cfg, int side, int from, int dir, int dist) {
  uint8_t b = gm.cell[from];
  if (!is_piece(b) || owner_of(b) != side) return false;
  int t = type_of(b);
  if (!is_movable_type(t)) return false;          // Bomb and Flag never move
  if (dist >= 2 && t != T_SCOUT) return false;
  int r = from / 10, q = from % 10;
  for (int k = 1; k <= dist; ++k) {
    int rr = r + DROW[dir] * k, qq = q + DCOL[dir] * k;
    if (rr < 0 || rr > 9 || qq < 0 || qq > 9) return false;
    int c = rr * 10 + qq;
    if (is_lake(c)) return false;
    if (k < dist) {
      if (gm.cell[c] != 0) return false;          // may not jump
    } else {
      if (is_piece(gm.cell[c]) && owner_of(gm.cell[c]) == side) return false;
    }
  }
  int to = (r + DROW[dir] * dist) * 10 + (q + DCOL[dir] * dist);
  if (cfg.two_square && two_square_banned(gm, side, from, to)) return false;
  if (cfg.chase_rule && chase_banned(gm, side, from, to)) return false;
  return true;
}

// Number of legal moves of `side` (as if it were its turn), optionally setting mask bits.
int gen_moves(const Game& gm, const Config& cfg, int side, uint32_t* mask) {
  int n = 0;
  for (int from = 0; from < kCells; ++from)
    for (int dir = 0; dir < 4; ++dir)
      for (int dist = 1; dist <= 9; ++dist)
        if (move_is_legal(gm, cfg, side, from, dir, dist)) {
          int a = from * 36 + dir * 9 + (dist - 1);
          if (mask) mask[a >> 5] |= 1u << (a & 31);
          ++n;
        }
  return n;
}

// ---------------------------------------------------------------- C4 battle
// P:208-210 + Extended Data Fig. 3b as spelled out in BJ north_star: equal ranks both
// removed, Spy attacking Marshal wins, Miner defuses Bomb, every other attacker on a
// Bomb is lost, capturing the Flag ends the game.  +1 attacker wins, -1 loses, 0 tie.
int battle(int att, int def) {
  if (def == T_FLAG) return +1;
  if (def == T_BOMB) return att == T_MINER ? +1 : -1;
  if (att == T_SPY && def == T_MARSHAL) return +1;
  if (att > def) return +1;   // "higher numbered piece defeats the lower"
  if (att < def) return -1;
  return 0;
}

// ---------------------------------------------------------------- S2 trackers
// Key of "the other piece at the time": its type if it was revealed, else "not revealed".
// Returns the bit, or 0 when the case has no channel (a revealed Bomb in the 11-wide groups of
// P:519-534, whose channels run Spy..Marshal + hidden; a revealed Flag anywhere).
uint16_t key_of(uint8_t b, bool with_bomb) {
  if (!(b & B_REVEALED)) return (uint16_t)(1u << 12);
  int t = type_of(b);
  if (t >= 1 && t <= 10) return (uint16_t)(1u << (t - 1));
  if (t == T_BOMB && with_bomb) return (uint16_t)(1u << 10);
  return 0;
}

// A fresh game, or a state loaded from a canonical line: the squares the pieces stand on now are
// their start squares, nothing has happened to them yet, and the recent moves are what the
// line's history remembers (reading I9).
void track_init(const Game& gm, Track& tk) {
  for (int c = 0; c < kCells; ++c) {
    bool p = is_piece(gm.cell[c]);
    tk.id_at[c] = p ? c : -1;
    tk.piece[c] = PieceTrack{0, 0, 0, 0, 0, 0, 0};
    tk.start_type[c] = p ? type_of(gm.cell[c]) : 0;
    tk.start_owner[c] = p ? owner_of(gm.cell[c]) : 0;
    tk.captured[c] = false;
  }
  memset(tk.died, 0, sizeof tk.died);
  for (int j = 0; j < 32; ++j) {
    bool have = j < 8 && gm.hist[j][0] != 0xFF;
    tk.moves[j][0] = have ? gm.hist[j][0] : -1;
    tk.moves[j][1] = have ? gm.hist[j][1] : -1;
  }
}

// The trackers' share of one ply, judged on the position BEFORE the move (gm is not yet
// changed).  `side` moves its piece from `from` to `to` (`dist` squares).
void track_ply(const Game& gm, const Config& cfg, Track& tk, int side, int from, int to, int dist) {
  const uint8_t C = gm.cell[from];
  const int idC = tk.id_at[from];
  // (i) Active adjacency: "the player controlling the former has had the chance to
  // attack the latter, but opted not to": every one-square capture that was legal for the
  // mover's side in this position and is not the move played (reading I3).
  for (int p = 0; p < kCells; ++p) {
    if (!is_piece(gm.cell[p]) || owner_of(gm.cell[p]) != side) continue;
    for (int d = 0; d < 4; ++d) {
      int rr = p / 10 + DROW[d], qq = p % 10 + DCOL[d];
      if (rr < 0 || rr > 9 || qq < 0 || qq > 9) continue;
      int q = rr * 10 + qq;
      if (!is_piece(gm.cell[q]) || owner_of(gm.cell[q]) == side) continue;
      if (p == from && q == to) continue;  // the attack that was made
      if (!move_is_legal(gm, cfg, side, p, d, 1)) continue;
      tk.piece[tk.id_at[p]].adjacent |= key_of(gm.cell[q], false);
    }
  }
  // The previous ply, if it was a move to an empty square, may have been a threat by the piece A
  // that now stands on x; battleless > 0 says that ply was not a battle.
  bool prev = gm.hist[0][0] != 0xFF && gm.battleless > 0;
  int x = prev ? gm.hist[0][1] : -1;
  if (prev && (!is_piece(gm.cell[x]) || owner_of(gm.cell[x]) == side)) prev = false;  // hand-built lines only
  const bool battle_ply = gm.cell[to] != 0;
  if (!battle_ply) {  // threats, evasions and protections are moves to empty squares (readings I1, I2, I4)
    const uint8_t Cafter = (uint8_t)(C | B_MOVED | (dist >= 2 ? B_REVEALED : 0));  // what C shows after this move (R#10)
    if (prev) {
      const uint8_t A = gm.cell[x];
      // (ii) Evasion: "a piece that was threatened in the immediately preceding move is
      // moved away from the threatening piece, to an empty square".
      if (adjacent(from, x) && !adjacent(to, x)) tk.piece[idC].evaded |= key_of(A, false);
      // (iii) Protection: A threatened B; C moves "to become adjacent to B".
      for (int b = 0; b < kCells; ++b) {
        if (b == from || !is_piece(gm.cell[b]) || owner_of(gm.cell[b]) != side) continue;
        if (!adjacent(b, x) || !adjacent(b, to) || adjacent(b, from)) continue;
        tk.piece[idC].protected_piece |= key_of(gm.cell[b], true);
        tk.piece[idC].protected_against |= key_of(A, true);
        tk.piece[tk.id_at[b]].was_protected_by |= key_of(Cafter, true);
        tk.piece[tk.id_at[b]].was_protected_against |= key_of(A, true);
      }
      // "We extend the same terminology to the case in which B is an empty square":
      // a square that was empty when A moved next to it, still is, and is next to C's new square
      // (reading I4; the square C leaves was not empty when A came, so it does not count).
      for (int e = 0; e < kCells; ++e) {
        if (e == to || gm.cell[e] != 0) continue;  // occupied squares and lakes
        if (!adjacent(e, x) || !adjacent(e, to)) continue;
        tk.piece[idC].protected_piece |= (uint16_t)(1u << 11);
        tk.piece[idC].protected_against |= key_of(A, true);
      }
    }
    // (iv) Threat: "a movement of one's piece so as to make the piece adjacent to a piece of
    // the opponent.  The opponent's piece is considered threatened."
    for (int d = 0; d < 4; ++d) {
      int rr = to / 10 + DROW[d], qq = to % 10 + DCOL[d];
      if (rr < 0 || rr > 9 || qq < 0 || qq > 9) continue;
      int q = rr * 10 + qq;
      if (q == from || !is_piece(gm.cell[q]) || owner_of(gm.cell[q]) == side) continue;
      tk.piece[idC].threatened |= key_of(gm.cell[q], false);
    }
    tk.id_at[to] = idC; tk.id_at[from] = -1;
  } else {
    // (v) Captures and causes of death.  "revealed at the time of the attack" = before
    // this battle reveals both.  The square a piece died in = the square of the battle (reading I5).
    const uint8_t D = gm.cell[to];
    const int idD = tk.id_at[to];
    const bool d_rev = (D & B_REVEALED) != 0;
    const int tc = type_of(C), td = type_of(D), out = battle(tc, td);
    if (out >= 0 && td != T_FLAG) {  // the defender dies (the Flag's capture ends the game: no channel)
      tk.captured[idD] = true;
      int cause = d_rev ? (out > 0 ? 4 : 5) : 6;
      if (td >= 1 && td <= 10) tk.died[side ^ 1][cause - 1][td - 1][to] = true;  // ten type channels per cause (reading I6)
    }
    if (out <= 0) {  // the attacker dies
      tk.captured[idC] = true;
      int cause = d_rev ? (out < 0 ? 1 : 2) : 3;
      tk.died[side][cause - 1][tc - 1][to] = true;
    }
    tk.id_at[from] = -1;
    if (out > 0) tk.id_at[to] = idC; else if (out == 0) tk.id_at[to] = -1;
  }
  for (int j = 31; j >= 1; --j) { tk.moves[j][0] = tk.moves[j - 1][0]; tk.moves[j][1] = tk.moves[j - 1][1]; }
  tk.moves[0][0] = from; tk.moves[0][1] = to;
}

int effective_ply_cap(const Config& cfg) {
  return (cfg.max_plies >= 1 && cfg.max_plies <= 65535) ? cfg.max_plies : 65535;
}

void read_line(const uint8_t* L, Game& gm);  // canonical line -> game (defined below)
void load_plies(Game& gm, const uint8_t* plies);  // plies that led to a loaded state (defined below)

void step_game(Env* e, int gi, int action, int8_t* reward, uint8_t* done_out) {
  Game& gm = e->g[gi];
  const Config& cfg = e->cfg;
  if (gm.done) {  // R#15: frozen
    *reward = 0;
    *done_out = (uint8_t)(1 | (gm.reason << 2));
    return;
  }
  int side = gm.ply & 1;  // red moves first
  bool ok = action >= 0 && action < 3600;
  int from = 0, dir = 0, dist = 1;
  if (ok) {
    from = action / 36; dir = (action % 36) / 9; dist = action % 9 + 1;
    ok = move_is_legal(gm, cfg, side, from, dir, dist);
  }
  if (!ok) {
    if (e->error == 0) e->error = ORC_ILLEGAL_ACTION;
    *reward = 0; *done_out = 0;
    return;
  }
  int to = (from / 10 + DROW[dir] * dist) * 10 + (from % 10 + DCOL[dir] * dist);
  if (cfg.infostate) track_ply(gm, cfg, e->track[gi], side, from, to, dist);  // S2 trackers, on the position before the move
  // 0. chase state machine (R#28), judged on the position before the move.
  if (cfg.chase_rule) {
    bool fight = gm.cell[to] != 0;
    bool threat = is_threat(gm, side, from, to), evade = is_evade(gm, side, from, to);
    int q = side ^ 1;
    if (fight) {
      gm.chase_age[0] = gm.chase_age[1] = 0;
    } else {
      if (gm.chase_age[q] > 0) gm.chase_age[q] = evade ? (gm.chase_age[q] < 255 ? gm.chase_age[q] + 1 : 255) : 0;
      if (threat) gm.chase_age[side] = gm.chase_age[side] > 0 ? (gm.chase_age[side] < 255 ? gm.chase_age[side] + 1 : 255) : 1;
      else gm.chase_age[side] = 0;
    }
  }
  // 1. two-square chain of the mover.
  if (gm.chain_len[side] > 0 && gm.chain[side][gm.chain_len[side] - 1] == from) {
    if (gm.chain_len[side] == 4) {
      for (int i = 0; i < 3; ++i) gm.chain[side][i] = gm.chain[side][i + 1];
      gm.chain_len[side] = 3;
    }
    gm.chain[side][gm.chain_len[side]++] = to;
  } else {
    gm.chain[side][0] = from; gm.chain[side][1] = to; gm.chain_len[side] = 2;
  }
  for (int j = 7; j >= 1; --j) { gm.hist[j][0] = gm.hist[j - 1][0]; gm.hist[j][1] = gm.hist[j - 1][1]; }
  gm.hist[0][0] = (uint8_t)from; gm.hist[0][1] = (uint8_t)to;
  if (cfg.chase_rule) {  // the chasing rule's memory
    gm.log[gm.logn & 63][0] = (uint8_t)from; gm.log[gm.logn & 63][1] = (uint8_t)to;
    gm.logn += 1;
  }
  // 2. mover's bits.
  uint8_t P = gm.cell[from] | B_MOVED;
  if (dist >= 2) P |= B_REVEALED;  // R#10
  uint8_t T = gm.cell[to];
  bool flag_captured = false;
  if (T == 0) {                    // 3. plain move
    gm.cell[to] = P; gm.cell[from] = 0;
    gm.battleless += 1;
  } else {                         // 4. battle: both revealed
    gm.battleless = 0;
    P |= B_REVEALED; T |= B_REVEALED;
    int out = battle(type_of(P), type_of(T));
    if (out > 0) {
      if (type_of(T) == T_FLAG) flag_captured = true;
      gm.cell[to] = P; gm.cell[from] = 0;
    } else if (out < 0) {
      gm.cell[from] = 0; gm.cell[to] = T;   // R#11: defender's moved bit unchanged
      gm.chain_len[side] = 0;
    } else {
      gm.cell[from] = 0; gm.cell[to] = 0;
      gm.chain_len[side] = 0;
    }
  }
  // 5. terminal tests, R#12 order.
  gm.ply += 1;
  int mover_result = side == 0 ? +1 : -1;
  if (flag_captured) {
    gm.done = true; gm.reason = REASON_FLAG; gm.result = mover_result;
  } else if (gen_moves(gm, cfg, gm.ply & 1, nullptr) == 0) {
    gm.done = true;
    if (gen_moves(gm, cfg, side, nullptr) == 0) { gm.reason = REASON_NOMOVE_DRAW; gm.result = 0; }
    else { gm.reason = REASON_NOMOVE_WIN; gm.result = mover_result; }
  } else if (gm.ply >= effective_ply_cap(cfg)) {
    gm.done = true; gm.reason = REASON_PLY_CAP; gm.result = 0;
  } else if (cfg.max_battleless > 0 && gm.battleless >= cfg.max_battleless) {
    gm.done = true; gm.reason = REASON_BATTLELESS; gm.result = 0;
  }
  // 6. outputs (R#13, R#14).
  *reward = gm.done ? (int8_t)gm.result : 0;
  *done_out = (uint8_t)((gm.done ? 1 : 0) | (side << 1) | ((gm.done ? gm.reason : 0) << 2));
  if (gm.done && cfg.auto_reset) {  // R#16
    uint32_t epoch = gm.epoch + 1;
    if (!e->pin.empty()) {  // R#27: the pinned line with the slot's own epoch counter
      read_line(&e->pin[(size_t)gi * kLine], gm);
      if (!e->pin_plies.empty()) load_plies(gm, &e->pin_plies[(size_t)gi * 126]);
      gm.epoch = epoch;
    } else {
      gm.epoch = epoch;
      new_game(cfg, (uint32_t)(cfg.game_base + (uint64_t)gi), gm, &e->pool);
    }
    if (cfg.infostate) track_init(gm, e->track[gi]);
  }
}

// ---------------------------------------------------------------- canonical line
void write_line(const Game& gm, uint8_t* L) {
  memset(L, 0, kLine);
  memcpy(L, gm.cell, kCells);
  for (int j = 0; j < 8; ++j) { L[100 + 2 * j] = gm.hist[j][0]; L[101 + 2 * j] = gm.hist[j][1]; }
  L[116] = (uint8_t)(gm.ply & 255); L[117] = (uint8_t)(gm.ply >> 8);
  L[118] = (uint8_t)(gm.battleless & 255); L[119] = (uint8_t)(gm.battleless >> 8);
  L[120] = (uint8_t)((gm.done ? 1 : 0) | (gm.reason << 2));
  L[121] = (uint8_t)(int8_t)gm.result;
  L[122] = (uint8_t)gm.chase_age[0]; L[123] = (uint8_t)gm.chase_age[1];
  L[124] = (uint8_t)gm.epoch; L[125] = (uint8_t)(gm.epoch >> 8);
  L[126] = (uint8_t)(gm.epoch >> 16); L[127] = (uint8_t)(gm.epoch >> 24);
}

// Rebuild one player's chain by replaying that player's moves found in the 8-ply
// history window, oldest first (the chain needs the last three only).  Pieces that
// died leave a cell their owner cannot move from next, so plain replay is exact.
void rebuild_chains(Game& gm) {
  gm.chain_len[0] = gm.chain_len[1] = 0;
  for (int j = 7; j >= 0; --j) {
    // Entries are taken as given (existence = the 0xFF marker only); entry j is the move
    // of ply t-1-j, so its mover is the parity of that number (also when a hand-built
    // line carries more history than plies).
    int side = (gm.ply - 1 - j) & 1;
    if (gm.hist[j][0] == 0xFF) {
      // an unknown ply of that player: its "consecutive turns" are interrupted (R#24)
      gm.chain_len[side] = 0;
      continue;
    }
    int from = gm.hist[j][0], to = gm.hist[j][1];
    if (gm.chain_len[side] > 0 && gm.chain[side][gm.chain_len[side] - 1] == from) {
      if (gm.chain_len[side] == 4) {
        for (int i = 0; i < 3; ++i) gm.chain[side][i] = gm.chain[side][i + 1];
        gm.chain_len[side] = 3;
      }
      gm.chain[side][gm.chain_len[side]++] = to;
    } else {
      gm.chain[side][0] = from; gm.chain[side][1] = to; gm.chain_len[side] = 2;
    }
  }
  // A chain whose last position no longer holds a piece of that player is dead.
  for (int s = 0; s < 2; ++s) {
    if (gm.chain_len[s] == 0) continue;
    uint8_t b = gm.cell[gm.chain[s][gm.chain_len[s] - 1]];
    if (!is_piece(b) || owner_of(b) != s) gm.chain_len[s] = 0;
  }
}

void read_line(const uint8_t* L, Game& gm) {
  memcpy(gm.cell, L, kCells);
  for (int j = 0; j < 8; ++j) { gm.hist[j][0] = L[100 + 2 * j]; gm.hist[j][1] = L[101 + 2 * j]; }
  gm.ply = L[116] | (L[117] << 8);
  gm.battleless = L[118] | (L[119] << 8);
  gm.done = (L[120] & 1) != 0;
  gm.reason = (L[120] >> 2) & 7;
  gm.result = (int8_t)L[121];
  gm.chase_age[0] = L[122]; gm.chase_age[1] = L[123];
  gm.logn = 0;
  gm.epoch = (uint32_t)L[124] | ((uint32_t)L[125] << 8) | ((uint32_t)L[126] << 16) | ((uint32_t)L[127] << 24);
  rebuild_chains(gm);
}

// The plies that led to a loaded state, `plies` = [63][2] most recent first: the state then
// remembers K = the number of leading known plies, exactly as if they had been played here.
void load_plies(Game& gm, const uint8_t* plies) {
  int K = 0;
  while (K < 63 && plies[2 * K] != 0xFF) ++K;
  gm.logn = K;
  for (int b = 1; b <= K; ++b) {
    gm.log[(K - b) & 63][0] = plies[2 * (b - 1)];
    gm.log[(K - b) & 63][1] = plies[2 * (b - 1) + 1];
  }
}

// ---------------------------------------------------------------- C5 encode
// BJ configs[0]: 12 own-type planes, 12 revealed-opponent-type planes, hidden opponent
// moved / unmoved, lake, empty, from/to planes of the last 8 plies; type order P:499.
void encode_game(const Game& gm, uint16_t* obs) {
  const uint16_t ONE = 0x3F80;  // bf16 1.0
  for (int i = 0; i < kObs; ++i) obs[i] = 0;
  int p = gm.ply & 1;
  for (int c = 0; c < kCells; ++c) {
    uint8_t b = gm.cell[c];
    int plane;
    if (type_of(b) == T_LAKE) plane = 26;
    else if (b == 0) plane = 27;                       // R#17: empty excludes lakes
    else if (owner_of(b) == p) plane = type_of(b) - 1;
    else if (b & B_REVEALED) plane = 12 + type_of(b) - 1;
    else if (b & B_MOVED) plane = 24;
    else plane = 25;
    obs[plane * kCells + c] = ONE;
  }
  for (int j = 0; j < 8; ++j) {
    if (gm.hist[j][0] == 0xFF) continue;
    obs[(28 + 2 * j) * kCells + gm.hist[j][0]] = ONE;
    obs[(29 + 2 * j) * kCells + gm.hist[j][1]] = ONE;
  }
}

// ---------------------------------------------------------------- S2 information state
// Round-to-nearest-even bf16 of the IEEE double quotient num/den (reading I8: the real-valued
// channels are that quotient, rounded once).
uint16_t bf16_of_ratio(long long num, long long den) {
  if (num == 0 || den == 0) return 0;
  double x = (double)num / (double)den;
  uint16_t sign = 0;
  if (x < 0) { sign = 0x8000; x = -x; }
  int e = 0;
  double m = frexp(x, &e);            // x = m * 2^e, m in [0.5, 1)
  double q = nearbyint(m * 256.0);    // 8 significant bits, ties to even (default rounding mode)
  if (q >= 256.0) { q = 128.0; e += 1; }
  int biased = e - 1 + 127;           // value = (q / 128) * 2^(e-1)
  return (uint16_t)(sign | (biased << 7) | ((int)q - 128));
}

// Channels 12-23 / 24-35: "probability that it belongs to the opponent and has type
// T ..., assuming the setup and moves were selected uniformly at random".  Reading I7: uniform
// over the arrangements of the owner's still-hidden pieces on their squares that are consistent
// with what the viewer has seen - revealed pieces are known, a piece that has moved is neither
// Bomb nor Flag.  With u unmoved and m moved hidden squares, c_T hidden pieces of type T,
// I = c_Flag + c_Bomb and M = u + m - I movable ones:
//   unmoved square:  P(T) = c_T / u  for T in {Flag, Bomb},  (u - I) c_T / (u M)  otherwise;
//   moved square:    P(T) = 0        for T in {Flag, Bomb},  c_T / M              otherwise.
// `owner` = whose pieces are being guessed; planes = 12 channels (Spy..Marshal, Flag, Bomb).
void type_posterior(const Game& gm, int owner, uint16_t* planes) {
  int c[13] = {0}, u = 0, m = 0;
  for (int s = 0; s < kCells; ++s) {
    uint8_t b = gm.cell[s];
    if (!is_piece(b) || owner_of(b) != owner || (b & B_REVEALED)) continue;
    c[type_of(b)] += 1;
    if (b & B_MOVED) ++m; else ++u;
  }
  int I = c[T_FLAG] + c[T_BOMB], M = u + m - I;
  int free_unmoved = u - I > 0 ? u - I : 0;  // a hand-built line may mark a Bomb as moved
  for (int s = 0; s < kCells; ++s) {
    uint8_t b = gm.cell[s];
    if (!is_piece(b) || owner_of(b) != owner) continue;
    if (b & B_REVEALED) { planes[(type_of(b) - 1) * kCells + s] = 0x3F80; continue; }
    for (int t = 1; t <= 12; ++t) {
      bool immovable = t == T_FLAG || t == T_BOMB;
      uint16_t v;
      if (b & B_MOVED) v = immovable ? 0 : bf16_of_ratio(c[t], M);
      else v = immovable ? bf16_of_ratio(c[t], u) : bf16_of_ratio((long long)free_unmoved * c[t], (long long)u * M);
      planes[(t - 1) * kCells + s] = v;
    }
  }
}

void encode_infostate(const Game& gm, const Config& cfg, const Track& tk, uint16_t* out) {
  const uint16_t ONE = 0x3F80, MINUS_ONE = 0xBF80;
  for (int i = 0; i < kInfo; ++i) out[i] = 0;
  const int p = gm.ply & 1;  // "the player" = the acting player
  auto set = [&](int channel, int square) { out[channel * kCells + square] = ONE; };
  // ---- basic piece properties
  for (int s = 0; s < kCells; ++s) {
    uint8_t b = gm.cell[s];
    if (type_of(b) == T_LAKE) continue;
    if (b == 0) { set(38, s); continue; }                      // empty (lakes are not squares: R#17)
    bool mine = owner_of(b) == p;
    if (mine) set(type_of(b) - 1, s);                          // 0-11
    if (!(b & B_REVEALED)) set(mine ? 36 : 37, s);             // hidden pieces
    if (b & B_MOVED) set(mine ? 39 : 40, s);                   // pieces that moved
  }
  type_posterior(gm, p ^ 1, out + 12 * kCells);                // 12-23: the opponent's pieces, as the player sees them
  type_posterior(gm, p, out + 24 * kCells);                    // 24-35: the player's pieces, as the opponent sees them
  uint16_t f41 = bf16_of_ratio(gm.ply, effective_ply_cap(cfg));
  uint16_t f42 = cfg.max_battleless > 0 ? bf16_of_ratio(gm.battleless, cfg.max_battleless) : 0;
  for (int s = 0; s < kCells; ++s) { out[41 * kCells + s] = f41; out[42 * kCells + s] = f42; }
  // ---- per-piece history, for the player's pieces then for the opponent's
  for (int s = 0; s < kCells; ++s) {
    if (!is_piece(gm.cell[s])) continue;
    const PieceTrack& t = tk.piece[tk.id_at[s]];
    bool mine = owner_of(gm.cell[s]) == p;
    int a = mine ? 43 : 76;     // threat / evasion / active adjacency: 10 types + hidden each
    const uint16_t g11[3] = {t.threatened, t.evaded, t.adjacent};
    for (int k = 0; k < 3; ++k) {
      for (int j = 0; j < 10; ++j)
        if (g11[k] & (1u << j)) set(a + 11 * k + j, s);
      if (g11[k] & (1u << 12)) set(a + 11 * k + 10, s);
    }
    int b = mine ? 251 : 303;   // protections: 13 channels each (11 types, empty square / padding, not revealed)
    const uint16_t g13[4] = {t.protected_piece, t.protected_against, t.was_protected_by, t.was_protected_against};
    for (int k = 0; k < 4; ++k)
      for (int j = 0; j < 13; ++j)
        if (g13[k] & (1u << j)) set(b + 13 * k + j, s);
    set(355 + tk.id_at[s], s);  // the piece on s started from square id
  }
  // ---- captured pieces by start square: Spy..Marshal, Bomb
  for (int s = 0; s < kCells; ++s) {
    if (!tk.captured[s]) continue;
    int t = tk.start_type[s];
    int j = t >= 1 && t <= 10 ? t - 1 : t == T_BOMB ? 10 : -1;
    if (j >= 0) set((tk.start_owner[s] == p ? 109 : 120) + j, s);
  }
  // ---- causes of death
  for (int o = 0; o < 2; ++o)
    for (int c = 0; c < 6; ++c)
      for (int t = 0; t < 10; ++t)
        for (int s = 0; s < kCells; ++s)
          if (tk.died[o][c][t][s]) set((o == p ? 131 : 191) + 10 * c + t, s);
  // ---- the most recent 32 moves: +1 on the destination, -1 on the source
  for (int j = 0; j < 32; ++j) {
    if (tk.moves[j][0] < 0) continue;
    out[(455 + j) * kCells + tk.moves[j][1]] = ONE;
    out[(455 + j) * kCells + tk.moves[j][0]] = MINUS_ONE;
  }
}

// ---------------------------------------------------------------- C6 replay ring
struct Replay {
  int64_t per_slot, slots, capacity, head, filled;
  std::vector<uint16_t> obs;
  std::vector<uint32_t> mask;
  std::vector<int16_t> action;
  std::vector<int8_t> reward;
  std::vector<uint8_t> done;
};

}  // namespace

// ======================================================================= C ABI
extern "C" {

int orc_create(const Config* cfg, Env** out) {
  if (!cfg || !out || cfg->num_games <= 0 || (cfg->variant != 0 && cfg->variant != 1)) return ORC_BAD_ARG;
  Env* e = new (std::nothrow) Env;
  if (!e) return ORC_BAD_ARG;
  e->cfg = *cfg;
  e->g.resize((size_t)cfg->num_games);
  e->error = 0;
  if (cfg->infostate) e->track.resize((size_t)cfg->num_games);
  for (int i = 0; i < cfg->num_games; ++i) {
    e->g[i].epoch = 0;
    new_game(e->cfg, (uint32_t)(cfg->game_base + (uint64_t)i), e->g[i]);
    if (cfg->infostate) track_init(e->g[i], e->track[i]);
  }
  *out = e;
  return ORC_OK;
}

int orc_destroy(Env* e) { delete e; return ORC_OK; }

int orc_reset(Env* e, uint64_t seed) {
  if (!e) return ORC_BAD_ARG;
  e->cfg.seed = seed;
  e->error = 0;
  for (int i = 0; i < e->cfg.num_games; ++i) {
    e->g[i].epoch = 0;
    new_game(e->cfg, (uint32_t)(e->cfg.game_base + (uint64_t)i), e->g[i], &e->pool);
    if (e->cfg.infostate) track_init(e->g[i], e->track[i]);
  }
  return ORC_OK;
}

// pool = [2][K][40] type codes (red setups, then blue setups); nullptr / K = 0: uniform permutations
// again.  A setup must hold type codes 0..12 and leave its side able to move (else BAD_ARG).
int orc_set_setup_pool(Env* e, const uint8_t* pool, int32_t K) {
  if (!e) return ORC_BAD_ARG;
  if (!pool || K <= 0) { e->pool.K = 0; e->pool.side[0].clear(); e->pool.side[1].clear(); return ORC_OK; }
  for (int side = 0; side < 2; ++side)
    for (int k = 0; k < K; ++k) {
      const uint8_t* A = pool + ((size_t)side * K + k) * 40;
      uint8_t cell[kCells];
      memset(cell, 0, sizeof cell);
      for (int c = 0; c < kCells; ++c)
        if (is_lake(c)) cell[c] = T_LAKE;
      for (int i = 0; i < 40; ++i) {
        if (A[i] > 12) return ORC_BAD_ARG;
        cell[(side ? 60 : 0) + i] = A[i] == 0 ? 0 : (uint8_t)(A[i] | (side ? B_OWNER : 0));
      }
      if (!side_can_ever_move(cell, side)) return ORC_BAD_ARG;
    }
  e->pool.K = K;
  e->pool.side[0].assign(pool, pool + (size_t)K * 40);
  e->pool.side[1].assign(pool + (size_t)K * 40, pool + (size_t)2 * K * 40);
  return ORC_OK;
}

int orc_reset_from(Env* e, const uint8_t* boards) {
  if (!e || !boards) return ORC_BAD_ARG;
  for (int i = 0; i < e->cfg.num_games; ++i) {
    read_line(boards + (size_t)i * kLine, e->g[i]);
    if (e->cfg.infostate) track_init(e->g[i], e->track[i]);  // reading I9: the loaded position is where the trackers start
  }
  return ORC_OK;
}

// The same with the plies that led to each state: plies uint8[N][63][2] (from,to), most recent
// first, 0xFF,0xFF = unknown.  The first 8 repeat the line's own history.
int orc_reset_from_with_plies(Env* e, const uint8_t* boards, const uint8_t* plies) {
  int rc = orc_reset_from(e, boards);
  if (rc != ORC_OK || !plies) return rc;
  for (int i = 0; i < e->cfg.num_games; ++i) load_plies(e->g[i], plies + (size_t)i * 126);
  return ORC_OK;
}

// boards == nullptr unpins.
int orc_pin_reset_state(Env* e, const uint8_t* boards) {
  if (!e) return ORC_BAD_ARG;
  if (boards) e->pin.assign(boards, boards + (size_t)e->cfg.num_games * kLine);
  else e->pin.clear();
  e->pin_plies.clear();
  return ORC_OK;
}
int orc_pin_reset_state_with_plies(Env* e, const uint8_t* boards, const uint8_t* plies) {
  int rc = orc_pin_reset_state(e, boards);
  if (rc == ORC_OK && boards && plies) e->pin_plies.assign(plies, plies + (size_t)e->cfg.num_games * 126);
  return rc;
}

int orc_get_boards(const Env* e, uint8_t* boards) {
  if (!e || !boards) return ORC_BAD_ARG;
  for (int i = 0; i < e->cfg.num_games; ++i) write_line(e->g[i], boards + (size_t)i * kLine);
  return ORC_OK;
}

int orc_legal_mask(const Env* e, uint32_t* mask) {
  if (!e || !mask) return ORC_BAD_ARG;
  for (int i = 0; i < e->cfg.num_games; ++i) {
    uint32_t* m = mask + (size_t)i * kMaskWords;
    for (int w = 0; w < kMaskWords; ++w) m[w] = 0;
    const Game& gm = e->g[i];
    if (!gm.done) gen_moves(gm, e->cfg, gm.ply & 1, m);  // R#15: finished -> zero mask
  }
  return ORC_OK;
}

// C3a (P:480 SampleRandomLegalAction): r-th set bit, r = bounded(u, popcount),
// u = word 0 of the ACTION block keyed by (global game, epoch, ply).
int orc_sample_uniform(const Env* e, const uint32_t* mask, int16_t* actions) {
  if (!e || !mask || !actions) return ORC_BAD_ARG;
  for (int i = 0; i < e->cfg.num_games; ++i) {
    const uint32_t* m = mask + (size_t)i * kMaskWords;
    int n = 0;
    for (int a = 0; a < 3600; ++a) n += (m[a >> 5] >> (a & 31)) & 1;
    if (n == 0) { actions[i] = -1; continue; }
    const Game& gm = e->g[i];
    uint32_t u = stream_draw(e->cfg.seed, (uint32_t)(e->cfg.game_base + (uint64_t)i), gm.epoch,
                             (uint32_t)gm.ply, TAG_ACTION, 0);
    int r = (int)bounded(u, (uint32_t)n);
    int16_t chosen = -1;
    for (int a = 0; a < 3600; ++a)
      if ((m[a >> 5] >> (a & 31)) & 1) {
        if (r == 0) { chosen = (int16_t)a; break; }
        --r;
      }
    actions[i] = chosen;
  }
  return ORC_OK;
}

int orc_step(Env* e, const int16_t* actions, int8_t* reward, uint8_t* done) {
  if (!e || !actions || !reward || !done) return ORC_BAD_ARG;
  for (int i = 0; i < e->cfg.num_games; ++i) step_game(e, i, actions[i], &reward[i], &done[i]);
  return ORC_OK;
}

int orc_encode_obs(const Env* e, uint16_t* obs) {
  if (!e || !obs) return ORC_BAD_ARG;
  for (int i = 0; i < e->cfg.num_games; ++i) encode_game(e->g[i], obs + (size_t)i * kObs);
  return ORC_OK;
}

// ComputeInfostateTensor in the paper's own form (P:462, S2 P:482-610): bf16 [N][487][10][10].
int orc_encode_infostate(const Env* e, uint16_t* out) {
  if (!e || !out) return ORC_BAD_ARG;
  if (!e->cfg.infostate) return ORC_BAD_STATE;
  for (int i = 0; i < e->cfg.num_games; ++i) encode_infostate(e->g[i], e->cfg, e->track[i], out + (size_t)i * kInfo);
  return ORC_OK;
}
uint16_t orc_bf16_of_ratio(int64_t num, int64_t den) { return bf16_of_ratio(num, den); }

int orc_check(Env* e) {
  if (!e) return ORC_BAD_ARG;
  int err = e->error;
  return err;
}

int orc_clear_error(Env* e) { if (!e) return ORC_BAD_ARG; e->error = 0; return ORC_OK; }

// ---- replay ring (C6, BJ configs[3]; R#19, R#20)
int orc_replay_create(int32_t per_slot, int32_t slots, Replay** out) {
  if (!out || per_slot <= 0 || slots <= 0) return ORC_BAD_ARG;
  Replay* r = new (std::nothrow) Replay;
  if (!r) return ORC_BAD_ARG;
  r->per_slot = per_slot; r->slots = slots; r->capacity = (int64_t)per_slot * slots;
  r->head = 0; r->filled = 0;
  r->obs.assign((size_t)r->capacity * kObs, 0);
  r->mask.assign((size_t)r->capacity * kMaskWords, 0);
  r->action.assign((size_t)r->capacity, 0);
  r->reward.assign((size_t)r->capacity, 0);
  r->done.assign((size_t)r->capacity, 0);
  *out = r;
  return ORC_OK;
}

int orc_replay_destroy(Replay* r) { delete r; return ORC_OK; }

int orc_replay_push(Replay* r, const uint16_t* obs, const uint32_t* mask, const int16_t* action,
                    const int8_t* reward, const uint8_t* done, int32_t n) {
  if (!r || n < 0 || n > r->capacity) return ORC_BAD_ARG;
  for (int i = 0; i < n; ++i) {
    int64_t p = (r->head + i) % r->capacity;
    memcpy(&r->obs[(size_t)p * kObs], obs + (size_t)i * kObs, kObs * sizeof(uint16_t));
    memcpy(&r->mask[(size_t)p * kMaskWords], mask + (size_t)i * kMaskWords, kMaskWords * sizeof(uint32_t));
    r->action[(size_t)p] = action[i];
    r->reward[(size_t)p] = reward[i];
    r->done[(size_t)p] = done[i];
  }
  r->head = (r->head + n) % r->capacity;
  r->filled = r->filled + n > r->capacity ? r->capacity : r->filled + n;
  return ORC_OK;
}

// Physical record index of batch element j (C6 / R#20): bounded(draw j, filled); SAMPLE stream:
// c0 = block j>>2, (c1,c2) = draw_index lo,hi, word j&3.
static int64_t sample_index(uint64_t seed, uint64_t draw_index, int j, int64_t filled) {
  uint32_t ctr[4] = {(uint32_t)(j >> 2), (uint32_t)draw_index, (uint32_t)(draw_index >> 32), TAG_SAMPLE};
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t o[4];
  philox4x32_10(ctr, key, o);
  return (int64_t)bounded(o[j & 3], (uint32_t)filled);
}
// The indices alone (full-size rings do not fit in host memory; the tests gather on their own).
int orc_sample_indices(uint64_t seed, uint64_t draw_index, int32_t batch, int64_t filled, int64_t* indices) {
  if (!indices || batch < 0 || filled <= 0 || filled > 0xFFFFFFFFll) return ORC_BAD_ARG;
  for (int j = 0; j < batch; ++j) indices[j] = sample_index(seed, draw_index, j, filled);
  return ORC_OK;
}

// Element j reads physical record sample_index(j).  `indices` (optional) receives the indices.
int orc_replay_sample(const Replay* r, uint64_t seed, uint64_t draw_index, int32_t batch,
                      uint16_t* obs, uint32_t* mask, int16_t* action, int8_t* reward, uint8_t* done,
                      int64_t* indices) {
  if (!r || batch < 0) return ORC_BAD_ARG;
  if (r->filled == 0) return ORC_BAD_STATE;
  for (int j = 0; j < batch; ++j) {
    int64_t p = sample_index(seed, draw_index, j, r->filled);
    if (indices) indices[j] = p;
    if (obs) memcpy(obs + (size_t)j * kObs, &r->obs[(size_t)p * kObs], kObs * sizeof(uint16_t));
    if (mask) memcpy(mask + (size_t)j * kMaskWords, &r->mask[(size_t)p * kMaskWords], kMaskWords * sizeof(uint32_t));
    if (action) action[j] = r->action[(size_t)p];
    if (reward) reward[j] = r->reward[(size_t)p];
    if (done) done[j] = r->done[(size_t)p];
  }
  return ORC_OK;
}

// Raw record p of the ring (tests compare ring contents).
int orc_replay_read(const Replay* r, int64_t p, uint16_t* obs, uint32_t* mask, int16_t* action,
                    int8_t* reward, uint8_t* done) {
  if (!r || p < 0 || p >= r->capacity) return ORC_BAD_ARG;
  memcpy(obs, &r->obs[(size_t)p * kObs], kObs * sizeof(uint16_t));
  memcpy(mask, &r->mask[(size_t)p * kMaskWords], kMaskWords * sizeof(uint32_t));
  *action = r->action[(size_t)p]; *reward = r->reward[(size_t)p]; *done = r->done[(size_t)p];
  return ORC_OK;
}

int64_t orc_replay_head(const Replay* r) { return r ? r->head : -1; }
int64_t orc_replay_filled(const Replay* r) { return r ? r->filled : -1; }

// ---- C7 determinise (BJ configs[4]): for output game G = r*S + s, re-type the searcher's
// opponent's unrevealed pieces with a uniformly random arrangement of their multiset that is
// consistent with the public history (no Bomb or Flag on a piece that has moved).
// Reading R#22: BJ says "permuted uniformly with rejection of any permutation that places a
// Bomb or Flag on a moved piece".  Rejecting whole permutations accepts with probability
// 3.9e-6 .. 2.6e-2 on the 16 ply-200 roots of config 4 (measured), i.e. up to ~250,000
// attempts per sample, so the rejection is applied per placed piece instead, which yields the
// same uniform distribution over consistent arrangements:
//   1. each hidden Bomb/Flag, in ascending order of its original square, draws a square
//      uniformly among the hidden squares still free, redrawing while that square holds a
//      moved piece (rejection);
//   2. the remaining (movable) types, in ascending order of their original squares, are
//      shuffled by descending Fisher-Yates and dealt to the free squares in their list order.
// The free-square list starts as the hidden squares ascending; taking entry i replaces it by
// the last entry.  One DETERMINISE stream per output game: draw d = word d&3 of block d>>2,
// counter (global G, 0, block).  More than 4096 draws -> BAD_STATE.  `attempts` (optional,
// [R*S]) receives the number of draws used.
static int determinise_one(const Game& root, uint64_t seed, uint32_t gidx, Game& out, int* draws) {
  int searcher = root.ply & 1;
  int H[40], T[40], n = 0;
  for (int c = 0; c < kCells; ++c) {
    uint8_t b = root.cell[c];
    if (is_piece(b) && owner_of(b) != searcher && !(b & B_REVEALED)) {
      if (n >= 40) return ORC_BAD_STATE;
      H[n] = c; T[n] = type_of(b); ++n;
    }
  }
  Game gm = root;
  int freeSq[40], m = n, d = 0;
  for (int i = 0; i < n; ++i) freeSq[i] = H[i];
  // 1. Bombs and Flag onto unmoved squares
  for (int j = 0; j < n; ++j) {
    if (T[j] != T_BOMB && T[j] != T_FLAG) continue;
    for (;;) {
      if (d >= 4096) return ORC_BAD_STATE;
      uint32_t u = stream_draw(seed, gidx, 0, 0, TAG_DETERMINISE, d++);
      int idx = (int)bounded(u, (uint32_t)m);
      int sq = freeSq[idx];
      if (root.cell[sq] & B_MOVED) continue;  // rejection
      gm.cell[sq] = (uint8_t)((root.cell[sq] & 0xF0) | T[j]);
      freeSq[idx] = freeSq[m - 1];
      --m;
      break;
    }
  }
  // 2. movable types over the remaining squares
  int Tm[40], k = 0;
  for (int j = 0; j < n; ++j)
    if (T[j] != T_BOMB && T[j] != T_FLAG) Tm[k++] = T[j];
  if (k != m) return ORC_BAD_STATE;
  for (int i = k - 1; i >= 1; --i) {
    if (d >= 4096) return ORC_BAD_STATE;
    uint32_t u = stream_draw(seed, gidx, 0, 0, TAG_DETERMINISE, d++);
    int j = (int)bounded(u, (uint32_t)(i + 1));
    int tmp = Tm[i]; Tm[i] = Tm[j]; Tm[j] = tmp;
  }
  for (int i = 0; i < k; ++i) gm.cell[freeSq[i]] = (uint8_t)((root.cell[freeSq[i]] & 0xF0) | Tm[i]);
  if (draws) *draws = d;
  out = gm;  // the copy remembers what the root remembers (its move log travels with it)
  return ORC_OK;
}

int orc_determinise(const Env* roots, int32_t samples_per_root, uint64_t seed, Env* out, int32_t* attempts) {
  if (!roots || !out || samples_per_root <= 0) return ORC_BAD_ARG;
  int R = roots->cfg.num_games;
  if ((int64_t)R * samples_per_root != out->cfg.num_games) return ORC_BAD_ARG;
  for (int r = 0; r < R; ++r)
    for (int s = 0; s < samples_per_root; ++s) {
      int G = r * samples_per_root + s, d = 0;
      int rc = determinise_one(roots->g[r], seed, (uint32_t)(out->cfg.game_base + (uint64_t)G), out->g[G], &d);
      if (rc != ORC_OK) return rc;
      if (attempts) attempts[G] = d;
      if (out->cfg.infostate) track_init(out->g[G], out->track[G]);  // reading I9: the trackers start with the copy
    }
  return ORC_OK;
}

// Per-root reduction of rollout returns (R#23): return = red's result from the
// searcher's perspective, 0 if the game is unfinished.  out[r] = {sum, wins, losses}.
int orc_reduce_returns(const Env* games, const uint8_t* root_side, int32_t samples_per_root, int32_t* out) {
  if (!games || !root_side || !out || samples_per_root <= 0) return ORC_BAD_ARG;
  if (games->cfg.num_games % samples_per_root) return ORC_BAD_ARG;
  int R = games->cfg.num_games / samples_per_root;
  for (int r = 0; r < R; ++r) {
    int sum = 0, wins = 0, losses = 0;
    for (int s = 0; s < samples_per_root; ++s) {
      const Game& gm = games->g[(size_t)r * samples_per_root + s];
      int ret = gm.done ? gm.result * (root_side[r] == 0 ? +1 : -1) : 0;
      sum += ret; if (ret > 0) ++wins; if (ret < 0) ++losses;
    }
    out[3 * r] = sum; out[3 * r + 1] = wins; out[3 * r + 2] = losses;
  }
  return ORC_OK;
}

// ---- one search step without networks (S3.7; R29)
// Legal actions of the root's side to move, ascending.
static int legal_list(const Env* e, const Game& gm, int* list) {
  if (gm.done) return 0;
  uint32_t m[kMaskWords];
  for (int w = 0; w < kMaskWords; ++w) m[w] = 0;
  gen_moves(gm, e->cfg, gm.ply & 1, m);
  int L = 0;
  for (int a = 0; a < 3600; ++a)
    if (m[a >> 5] & (1u << (a & 31))) list[L++] = a;
  return L;
}
// Steps 1-2: "samples roughly 1,000 / (number of legal actions) possible
// configurations of the types of the hidden pieces", "at least one rollout for each combination
// of legal move and sampled opponent configuration.  After the initial move, which is forced,
// ...".  Root r with L legal actions gets C = max(1, rollouts / L) configurations (the
// determinisation sampler of C7 stands in for the belief network); slot r*rollouts + c*L + l
// holds configuration c with the l-th legal action applied; the other slots are frozen.
int orc_search_expand(const Env* roots, int32_t rollouts, uint64_t seed, Env* out) {
  if (!roots || !out || rollouts <= 0) return ORC_BAD_ARG;
  int R = roots->cfg.num_games;
  if ((int64_t)R * rollouts != out->cfg.num_games || out->cfg.auto_reset || out->cfg.infostate) return ORC_BAD_ARG;
  std::vector<int> list(3600);
  for (int r = 0; r < R; ++r) {
    const Game& root = roots->g[r];
    int L = legal_list(roots, root, list.data());
    int C = L > 0 ? (rollouts / L > 1 ? rollouts / L : 1) : 0;
    int64_t used = (int64_t)C * L < rollouts ? (int64_t)C * L : rollouts;
    for (int s = 0; s < rollouts; ++s) {
      int G = r * rollouts + s;
      if (s >= used) {  // unused slot: a frozen game
        out->g[G] = root;
        out->g[G].done = true; out->g[G].reason = 0; out->g[G].result = 0;
        continue;
      }
      int c = s / L, l = s % L;
      uint32_t gidx = (uint32_t)(out->cfg.game_base + (uint64_t)r * rollouts + (uint64_t)c);  // one stream per configuration
      int rc = determinise_one(root, seed, gidx, out->g[G], nullptr);
      if (rc != ORC_OK) return rc;
      int8_t rew; uint8_t dn;
      step_game(out, G, list[l], &rew, &dn);  // the forced first move
    }
  }
  return ORC_OK;
}
// Steps 3-4: qhat(a) = average value over the configurations of the games that
// started with a - the value is the game's result from the searcher's side once the rollouts
// are over, 0 if it is still running (stand-in for the move network's value head) - and
//   pi_search = argmax <qhat, pi> - alpha KL(pi, rho) - beta KL(pi, pi_theta)
//             \propto [ exp(qhat) rho^alpha pi_theta^beta ]^(1/(alpha+beta))              (7), (8)
// with rho the magnet policy "that selects a movable piece uniformly at random and then selects
// a legal move for this piece uniformly at random" and pi_theta the caller's
// prior over the 3600 actions (nullptr = uniform over the legal ones).  All in double.
// `values` (float32 [R*rollouts], or nullptr): P:865-866 step 3 averages "the value output of the move
// network at the positions reached by the rollouts".  values[r*rollouts + s] is that output for game s of
// root r, from the SEARCHER's side (the player to move at the root).  A game that has ended has a known
// value, its result; the caller's value counts for the games still running (with nullptr those count 0:
// the stand-in of DESIGN.md R29).
int orc_search_policy_values(const Env* roots, const Env* games, int32_t rollouts, const float* pi_theta,
                             const float* values, double alpha, double beta, float* qhat, float* rho, float* pi_search);
int orc_search_policy(const Env* roots, const Env* games, int32_t rollouts, const float* pi_theta, double alpha,
                      double beta, float* qhat, float* rho, float* pi_search) {
  return orc_search_policy_values(roots, games, rollouts, pi_theta, nullptr, alpha, beta, qhat, rho, pi_search);
}
int orc_search_policy_values(const Env* roots, const Env* games, int32_t rollouts, const float* pi_theta,
                             const float* values, double alpha, double beta, float* qhat, float* rho, float* pi_search) {
  if (!roots || !games || rollouts <= 0 || !qhat || !rho || !pi_search || !(alpha + beta > 0)) return ORC_BAD_ARG;
  int R = roots->cfg.num_games;
  if ((int64_t)R * rollouts != games->cfg.num_games) return ORC_BAD_ARG;
  std::vector<int> list(3600);
  for (int r = 0; r < R; ++r) {
    float* q = qhat + (size_t)r * 3600; float* rh = rho + (size_t)r * 3600; float* ps = pi_search + (size_t)r * 3600;
    for (int a = 0; a < 3600; ++a) q[a] = rh[a] = ps[a] = 0.0f;
    const Game& root = roots->g[r];
    int L = legal_list(roots, root, list.data());
    if (L == 0) continue;
    int C = rollouts / L > 1 ? rollouts / L : 1;
    int64_t used = (int64_t)C * L < rollouts ? (int64_t)C * L : rollouts;
    int sign = (root.ply & 1) == 0 ? +1 : -1;
    int per_cell[kCells] = {0}, pieces = 0;
    for (int l = 0; l < L; ++l) per_cell[list[l] / 36] += 1;
    for (int c = 0; c < kCells; ++c) pieces += per_cell[c] > 0;
    std::vector<double> logit(L);
    double mx = -1e300;
    // A prior without mass on any legal action of this root says nothing here (KL(pi, pi_theta) is
    // infinite for every pi, eq. 7 has no maximiser): the root is treated as if no prior were given
    // (R29).
    const float* prior = pi_theta;
    if (prior) {
      bool any = false;
      for (int l = 0; l < L; ++l) any = any || prior[(size_t)r * 3600 + list[l]] > 0.0f;
      if (!any) prior = nullptr;
    }
    for (int l = 0; l < L; ++l) {
      double sum = 0;
      int cnt = 0;
      for (int64_t s = l; s < used; s += L) {
        const Game& gm = games->g[(size_t)r * rollouts + (size_t)s];
        if (gm.done) sum += gm.result * sign;
        else if (values) sum += (double)values[(size_t)r * rollouts + (size_t)s];
        ++cnt;
      }
      double qv = cnt ? sum / cnt : 0.0;
      double rv = 1.0 / ((double)pieces * per_cell[list[l] / 36]);
      double pv = prior ? (double)prior[(size_t)r * 3600 + list[l]] : 1.0 / L;
      q[list[l]] = (float)qv; rh[list[l]] = (float)rv;
      logit[l] = (qv + alpha * log(rv) + beta * log(pv)) / (alpha + beta);
      if (logit[l] > mx) mx = logit[l];
    }
    double z = 0;
    for (int l = 0; l < L; ++l) z += exp(logit[l] - mx);
    for (int l = 0; l < L; ++l) ps[list[l]] = (float)(exp(logit[l] - mx) / z);
  }
  return ORC_OK;
}

// ---- probes used by the pins only
// Global game indices in [start, start+count) whose setup at `epoch` needs a redraw (R#5) for
// either side; used once by tests/golden/make_setup_redraw_cases.py to find test cases for a
// path that random play reaches about twice in a million setups.
int orc_find_setup_redraws(const Config* cfg, uint32_t epoch, uint32_t start, uint32_t count, uint32_t* out, int max_out) {
  if (!cfg || !out) return ORC_BAD_ARG;
  int n = 0;
  uint8_t cell[kCells];
  for (uint32_t i = 0; i < count && n < max_out; ++i) {
    memset(cell, 0, sizeof cell);
    for (int c = 0; c < kCells; ++c)
      if (is_lake(c)) cell[c] = T_LAKE;
    int a0 = setup_side(*cfg, start + i, epoch, 0, cell);
    int a1 = setup_side(*cfg, start + i, epoch, 1, cell);
    if (a0 > 1 || a1 > 1) out[n++] = start + i;
  }
  return n;
}
void orc_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }
int orc_battle(int att, int def) { return battle(att, def); }
int orc_is_lake(int c) { return is_lake(c) ? 1 : 0; }
void orc_multiset(int variant, int32_t out[40]) { int A[40]; multiset(variant, A); for (int i = 0; i < 40; ++i) out[i] = A[i]; }
// chain of player `side` of game gi: returns length, fills pos[4].
int orc_chain(const Env* e, int gi, int side, int32_t pos[4]) {
  const Game& gm = e->g[gi];
  for (int i = 0; i < gm.chain_len[side]; ++i) pos[i] = gm.chain[side][i];
  return gm.chain_len[side];
}
// Number of legal moves of `side` as if it were its turn (GetHasLegalMovement).
int orc_count_moves(const Env* e, int gi, int side) { return gen_moves(e->g[gi], e->cfg, side, nullptr); }

}  // extern "C"
