/* strat.h — C ABI of libstrat.so: the batched Stratego environment step on one B200.
 *
 * The hot path of arxiv 2511.07312's self-play/search pipeline (PAPER.md:226-240,
 * "StrategoRolloutBuffer": N parallel games, ApplyActions, ComputeLegalActionMask,
 * ComputeInfostateTensor, ComputeRewardP10, SampleRandomLegalAction — Table S1,
 * PAPER.md:455-480), in the I/O layouts BASELINE.json fixes.  Every call below runs
 * hand-written sm_100a kernels; there is no CPU path.
 *
 * Conventions
 *   - Every function returns 0 (STRAT_OK) or a negative error code; no exceptions.
 *   - Pointers are DEVICE pointers unless the name ends in `_host`.  The caller owns
 *     all device memory, including the library's own state: size it with
 *     strat_workspace_bytes / strat_replay_bytes, allocate (e.g. a torch.uint8 tensor)
 *     and pass it to *_create.  The library never allocates device memory and never
 *     synchronises, except in strat_check and the *_host entry points
 *     (third desideratum: no dynamic allocation after construction).
 *   - `stream` is a cudaStream_t passed as void* (0 = default stream).  Calls are
 *     asynchronous with respect to the host.
 *   - Device-detected faults (an illegal action for a live game) set a sticky device
 *     error word and leave that game unchanged; strat_check reads it.
 *   - Handles are not thread-safe: calls on one environment / ring / history come from one
 *     host thread at a time, and consecutive calls on one environment use one stream (or are
 *     ordered by the caller with events).  Different environments are independent.
 *
 * Layouts (BASELINE.json configs[0])
 *   cell c = 10*row + col, row 0 = red's back row; lakes {42,43,46,47,52,53,56,57}.
 *   canonical line uint8[128] per game (what reset_from / get_boards exchange):
 *     0..99    cell byte: bits0-3 type (0 empty, 1 Spy, 2 Scout, 3 Miner, 4 Sergeant,
 *              5 Lieutenant, 6 Captain, 7 Major, 8 Colonel, 9 General, 10 Marshal,
 *              11 Flag, 12 Bomb, 15 lake; order of PAPER.md:499), bit4 owner (0 red,
 *              1 blue), bit5 moved, bit6 revealed
 *     100..115 history: entry j = (from,to) of ply t-1-j; 0xFF,0xFF if none
 *     116..117 ply (LE u16)      118..119 plies since the last battle (LE u16)
 *     120      bit0 done, bits2-4 reason (1 Flag captured, 2 opponent has no move,
 *              3 neither has a move (draw), 4 ply cap (draw), 5 battleless cap (draw))
 *     121      result for red (int8: +1, -1, 0)
 *     122..123 chase age of red / blue: positions of the player's running chase, counted
 *              from the one right after its first threat (0 = not chasing; always 0 unless
 *              chase_rule is on; R28)
 *     124..127 epoch (LE u32): number of auto-resets of this game slot
 *   action  a = from*36 + dir*9 + (dist-1); dir 0:+row 1:+col 2:-row 3:-col; dist 1..9
 *   mask    uint32[N][113]; bit a -> word a>>5, bit a&31; bits 3600..3615 are zero
 *   obs     bf16 (as uint16) [N][44][10][10], values 0x0000 / 0x3F80, for the side to
 *           move: 0-11 own type k+1; 12-23 revealed opponent type k-11; 24 hidden
 *           opponent, moved; 25 hidden opponent, unmoved; 26 lake; 27 empty non-lake;
 *           28+2j / 29+2j from / to square of ply t-1-j, j = 0..7
 *   reward  int8[N]: red's result on the terminating step, else 0
 *   done    uint8[N]: bit0 game ended on this step, bit1 player who acted (0 red),
 *           bits2-4 reason as above
 *   RNG     Philox4x32-10, key = seed, counter = (c0,c1,c2,tag): setup tag 0 red /
 *           1 blue (global game, epoch, attempt<<8 | block); action tag 2 (global game,
 *           epoch, ply), word 0; sample tag 3 (block, draw_index lo, hi); determinise
 *           tag 4 (global output game, attempt, block).  Bounded draw = (u*n)>>32.
 */
#ifndef STRAT_H_
#define STRAT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define STRAT_OK 0
#define STRAT_BAD_ARG (-1)
#define STRAT_BAD_STATE (-2)
#define STRAT_CUDA_ERROR (-3)
#define STRAT_ILLEGAL_ACTION (-4)
#define STRAT_TOO_LARGE (-5)   /* more games than the built-in scratch of strat_legal_mask_static holds */

#define STRAT_LINE_BYTES 128
#define STRAT_MASK_WORDS 113
#define STRAT_OBS_PLANES 44
#define STRAT_OBS_ELEMS 4400
#define STRAT_NUM_ACTIONS 3600
#define STRAT_INFO_PLANES 487   /* the paper's own information state */
#define STRAT_INFO_ELEMS 48700

typedef struct strat_config {
  int32_t num_games;      /* N >= 1 */
  int32_t variant;        /* 0 classic (40 pieces a side), 1 Barrage (8 a side) */
  uint64_t seed;          /* Philox key */
  int32_t max_plies;      /* draw after this many plies; 0 = none (hard cap 65535) */
  int32_t max_battleless; /* draw after this many plies without a battle; 0 = off */
  int32_t auto_reset;     /* 1: a finished game restarts inside the same step */
  int32_t two_square;     /* 1: apply the two-square rule */
  int32_t device;         /* CUDA device ordinal */
  int32_t chase_rule;     /* 1: apply the continuous-chasing rule (R28: a
                             chasing player may not make a threat that recreates a position of
                             the chase, except by moving straight back; memory: 63 plies played in
                             this environment + the 8 plies a loaded line carries), 0: off */
  uint64_t game_base;     /* global index of game 0 (RNG keying when games are sharded);
                             game_base + num_games <= 2^32 (the RNG counter word is 32 bits) */
  int32_t infostate;      /* 1: keep, per game, the trackers the paper's 487-channel information state
                             needs (threats, evasions, active adjacencies, protections,
                             captures, causes of death, start squares, the last 32 moves): 2 KB more
                             workspace per game, updated by strat_step / strat_rollout_step /
                             strat_step_observe; strat_encode_infostate then works.  0: off */
  int32_t reserved;       /* 0 */
} strat_config;

typedef struct strat_env strat_env;       /* host handle; state lives in the workspace */
typedef struct strat_replay strat_replay; /* host handle; ring lives in caller memory */

const char* strat_error_string(int code);

/* ---- environment ---------------------------------------------------------------- */

/* Bytes of device workspace an environment of this configuration needs. 0 on bad cfg. */
size_t strat_workspace_bytes(const strat_config* cfg);

/* Bind an environment to `workspace_dev` (>= strat_workspace_bytes, 256-B aligned).
 * Launches the initial reset (seeded setups; BASELINE.json configs[0,1])
 * on `stream`.  The handle is freed by strat_destroy; the workspace stays the caller's. */
int strat_create(const strat_config* cfg, void* workspace_dev, size_t bytes, void* stream,
                 strat_env** out);
int strat_destroy(strat_env* env);

/* Two environments that are used on ONE stream and exchange output buffers (one's fused step
 * writes what the other's reads or overwrites): afterwards their fused steps are ordered against
 * each other as plain stream order.  Without it only consecutive fused steps of the SAME
 * environment overlap (ordered batch by batch), and a fused step is ordered against everything
 * else the library was asked to do with its environment; fused steps of two unrelated
 * environments issued back to back on one stream may overlap on the device.  `b` joins the group of
 * `a`; a group grows one lone environment at a time: STRAT_BAD_STATE if `b` already shares its
 * ordering with other environments (they would be left unordered against the group of `a`). */
int strat_share_chain(strat_env* a, strat_env* b);

/* All games: new Philox key, epoch 0, ply 0, fresh setups. */
int strat_reset(strat_env* env, uint64_t seed, void* stream);

/* Load / store all games as canonical lines uint8[N][128] (device pointers).
 * reset_from is the "reset to a non-initial state" of PAPER.md:252-254.  A line that gives one
 * side more than 8 Scouts (no variant of the game does: BASELINE.json configs[0,1] list 8 and 2)
 * raises STRAT_BAD_STATE on the sticky error word (strat_check); so does a pinned line. */
int strat_reset_from(strat_env* env, const uint8_t* boards, void* stream);
/* The same with the plies that led to each state ("the continuous chasing rule needs
 * to be tested against the history of board states that leads to the non-initial reset state"):
 * plies uint8[N][63][2] (device) = (from, to) squares, most recent first, 0xFF,0xFF = unknown; the
 * leading known ones become the game's move log, as if they had been played here (the first 8
 * repeat the line's own history); an entry with a square >= 100 counts as unknown.  Without chase_rule nothing remembers plies: same as
 * strat_reset_from. */
int strat_reset_from_with_plies(strat_env* env, const uint8_t* boards, const uint8_t* plies, void* stream);
int strat_get_boards(const strat_env* env, uint8_t* boards, void* stream);

/* Customised initial-board distribution ("The distribution from which the initial
 * board is sampled can be customized"; the paper trains from a pool of 1,000 network-generated
 * setups per player per GPU).  pool_dev: uint8[2][K][40] type codes on the device
 * (K red setups, then K blue setups; entry i of a red setup goes to cell i, of a blue one to cell
 * 60+i; 0 = empty), caller-owned and read until replaced.  From the next reset / auto-reset on,
 * each side of a fresh game is pool entry bounded(first draw of the side's setup stream, K),
 * independently for the two sides (R30).  A setup with a type code above 12, with more
 * than 8 Scouts or with no piece that can ever move raises STRAT_BAD_ARG on the sticky error word (strat_check).
 * pool_dev == NULL: uniform permutations of the multiset again. */
int strat_set_setup_pool(strat_env* env, const uint8_t* pool_dev, int32_t K, void* stream);

/* "Pin" the simulation (Reset Behaviour and Support for Search): while a pin
 * is set, a game that terminates (auto_reset = 1) restarts from ITS pinned state instead of a
 * fresh setup; only the slot's epoch counter keeps counting up, so every restart plays a new
 * action stream.  boards: canonical uint8[N][128] (device); pin_lines_dev: N*128 bytes of
 * caller-owned device memory (16-B aligned) that the library fills and keeps reading until
 * the pin is removed (boards == NULL).  The current state of the games is not touched. */
int strat_pin_reset_state(strat_env* env, void* pin_lines_dev, const uint8_t* boards, void* stream);
/* The same with the plies that led to each pinned state (layout as in strat_reset_from_with_plies):
 * a restart from the pin restarts with them in its move log.  pin_logs_dev: N*128
 * more bytes of caller-owned device memory (16-B aligned), kept like pin_lines_dev. */
int strat_pin_reset_state_with_plies(strat_env* env, void* pin_lines_dev, void* pin_logs_dev, const uint8_t* boards,
                                     const uint8_t* plies, void* stream);

/* ComputeLegalActionMask for the acting player (rules PAPER.md:210-212).
 * mask: uint32[N][113].  Finished games get an all-zero mask. */
int strat_legal_mask(const strat_env* env, uint32_t* mask, void* stream);

/* SampleRandomLegalAction: the r-th set bit of each game's mask,
 * r = bounded(Philox action draw, popcount).  actions: int16[N], -1 where the mask is empty. */
int strat_sample_uniform(const strat_env* env, const uint32_t* mask, int16_t* actions, void* stream);

/* ApplyActions: one action per game; battle by rank with the Spy,
 * Bomb/Miner and Flag cases; terminal tests; auto-reset.
 * reward int8[N], done uint8[N] describe the step just taken (also for a game that was
 * auto-reset inside the call).  A finished game without auto-reset is left frozen. */
int strat_step(strat_env* env, const int16_t* actions, int8_t* reward, uint8_t* done, void* stream);

/* ComputeInfostateTensor in BASELINE.json's 44-plane bf16 form.
 * obs: uint16[N][4400]. */
int strat_encode_obs(const strat_env* env, uint16_t* obs, void* stream);

/* ComputeInfostateTensor in the paper's own form (S2): bf16 (as
 * uint16) [N][487][10][10] for the acting player ("the player"; the other one is "the opponent"),
 * absolute board coordinates.  Needs strat_config.infostate = 1 (else STRAT_BAD_STATE).  `out`
 * must be 8-byte aligned.  Channels (values 0 / 1.0 unless stated; T runs Spy..Marshal, Flag, Bomb
 * as far as the count says; readings I1-I9 in DESIGN.md):
 *     0-11   the player's piece of type T               12-23  probability that the square holds an
 *    24-35   the same from the opponent's side                  opponent's piece of type T: 1.0 for a
 *    36/37   hidden piece of the player / the opponent          revealed one, else uniform over the
 *    38      empty (not a lake)                                 arrangements of the hidden types on the
 *    39/40   player's / opponent's piece that has moved         hidden squares with no Bomb or Flag on a
 *    41      ply / ply cap       42  plies since the last       piece that has moved (bf16, rounded once
 *            battle / max_battleless (0 if that rule is off)    from the double quotient)
 *    43-52, 53   the player's piece has threatened a revealed T (Spy..Marshal) / a hidden piece
 *    54-63, 64   ... has evaded a threat from ...        65-74, 75  ... was actively adjacent to ...
 *    76-108      the same three groups for the opponent's pieces
 *   109-119  start square of a captured piece of the player, T = Spy..Marshal, Bomb;  120-130 opponent's
 *   131-190  a piece of the player of type T (Spy..Marshal) died on this square by cause 1..6:
 *            131 + 10*(cause-1) + T-1;  191-250 the opponent's
 *   251-263  the player's piece has protected a revealed T (Spy..Marshal, Bomb) / an empty square / a
 *            hidden piece;  264-276 has protected against (.., 275 padding, 276 hidden);  277-289 has
 *            been protected by;  290-302 has been protected against;  303-354 the opponent's
 *   355-454  channel 355+k: the piece on this square started the game on square k
 *   455-486  move t-1-j (j = 0..31): +1.0 on its destination, -1.0 on its source
 * The trackers start with the game (reset, auto-reset) or with a loaded position
 * (strat_reset_from, a pinned restart, strat_history_restore: the squares the pieces stand on
 * then count as their start squares, the line's 8-ply history as the known moves).
 * Calls for one environment on different streams may run at the same time (each takes a work
 * counter of its own); they read the state, so order them against the steps as usual. */
int strat_encode_infostate(const strat_env* env, uint16_t* out, void* stream);

/* One fused pass of the hot path: legal mask -> uniform legal action -> step -> encode of
 * the new state.  Produces exactly what strat_legal_mask, strat_sample_uniform,
 * strat_step, strat_encode_obs produce when called in that order.  Any output pointer
 * except `obs` may be NULL (that output is then not written).
 * Consecutive calls of this function for one environment on one stream overlap on the device,
 * ordered batch by batch; everything else in the stream (strat_step_observe included: it waits for
 * the producer of its actions, and what follows it waits for it) sees plain stream order.  They cannot be captured into a CUDA graph (STRAT_BAD_STATE while `stream` is
 * capturing): each launch carries a host-side launch counter. */
int strat_rollout_step(strat_env* env, uint32_t* mask, int16_t* actions, int8_t* reward,
                       uint8_t* done, uint16_t* obs, void* stream);

/* The data-collection loop with an external policy in one pass (PAPER.md:232 ApplyActions, then
 * the two queries the next policy call needs): applies `actions` (validated
 * like strat_step), then writes the legal mask and the observation of the NEW state.  Produces
 * exactly what strat_step, strat_legal_mask, strat_encode_obs produce in that order.
 * `mask` may be NULL. */
int strat_step_observe(strat_env* env, const int16_t* actions, int8_t* reward, uint8_t* done, uint32_t* mask,
                       uint16_t* obs, void* stream);

/* Same, with HOST destination buffers (pinned memory recommended): runs the fused step
 * into `scratch_dev` (>= strat_host_scratch_bytes(cfg) bytes, caller-owned), copies the
 * five outputs to the host pointers on `stream` and synchronises the stream. */
size_t strat_host_scratch_bytes(const strat_config* cfg);
int strat_rollout_step_host(strat_env* env, void* scratch_dev, uint32_t* mask_host,
                            int16_t* actions_host, int8_t* reward_host, uint8_t* done_host,
                            uint16_t* obs_host, void* stream);

/* The RL-loop shape with a host-side policy (PAPER.md:232 ApplyActions + Table S1 queries):
 * copies int16[N] actions from `actions_host` to the device, runs strat_step_observe and
 * copies reward, done, mask and obs to the host pointers; synchronises the stream.
 * `scratch_dev` as for strat_rollout_step_host. */
int strat_step_host(strat_env* env, void* scratch_dev, const int16_t* actions_host, int8_t* reward_host,
                    uint8_t* done_host, uint32_t* mask_host, uint16_t* obs_host, void* stream);

/* `plies` plies of uniform-random legal play with the boards kept on chip (search-shaped
 * rollouts, BASELINE.json configs[4]).  Equal to `plies` repetitions
 * of legal_mask + sample_uniform + step; nothing but the state is written. */
int strat_rollout_uniform(strat_env* env, int32_t plies, void* stream);

/* Synchronise the device and return the sticky error word (0 if none). */
int strat_check(strat_env* env);
int strat_clear_error(strat_env* env, void* stream);

/* ---- device replay ring (BASELINE.json configs[3]) -------------------------------- */
/* capacity = per_slot * slots records of (obs 8800 B, mask 452 B, action i16, reward i8,
 * done u8) = 9256 B, stored as five arrays (a "slot" is a contiguous run of per_slot records of
 * each array; R19).  Ring position p in [0, capacity) is where the p-th, (p+capacity)-th,
 * ... pushed record goes; head = position of the next record, filled = live records.
 *
 * Two kinds of ring:
 *   plain    (strat_replay_create): every array has exactly `capacity` rows, position p = row p;
 *            filled by strat_replay_push (copying).
 *   in-place (strat_replay_create_in_place, block = records per push, capacity % block == 0): the
 *            fused step writes the records itself (strat_replay_reserve / _reserve_rows / _commit).
 *            In self-play record t = (obs_t, mask_t, a_t, r_t, done_t): step t produces mask_t,
 *            a_t, r_t, done_t of the block being completed AND obs_{t+1} of the block after it.
 *            So that what is written ahead never lands in a record that is still live (a record
 *            pairing a new observation with a 32-steps-old mask and action), the four small arrays
 *            have capacity + block rows and the observation array capacity + 2*block rows: the
 *            record with push-order number s lives in row s % rows (s % obs_rows for its
 *            observation); strat_replay_locate maps a ring position to its rows.
 * strat_replay_layout returns the byte offset of each array inside the caller's memory:
 * {obs, mask, action, reward, done} (block = 0 for a plain ring). */
size_t strat_replay_bytes(int32_t per_slot, int32_t slots);
size_t strat_replay_bytes_in_place(int32_t per_slot, int32_t slots, int32_t block);
int strat_replay_layout(int32_t per_slot, int32_t slots, int32_t block, size_t offsets[5]);
int strat_replay_create(void* mem_dev, size_t bytes, int32_t per_slot, int32_t slots, strat_replay** out);
int strat_replay_create_in_place(void* mem_dev, size_t bytes, int32_t per_slot, int32_t slots, int32_t block,
                                 strat_replay** out);
int strat_replay_destroy(strat_replay* r);
/* Append n records in order at positions (head+i) mod capacity; head += n; filled = min(filled+n, capacity). */
int strat_replay_push(strat_replay* r, const uint16_t* obs, const uint32_t* mask, const int16_t* action,
                      const int8_t* reward, const uint8_t* done, int32_t n, void* stream);
/* In-place push (in-place rings only; STRAT_BAD_ARG on a plain ring, if n does not divide the
 * row counts, or if records were pushed that are not a multiple of n): the addresses of the obs
 * and mask rows of the n records `ahead` blocks after the next one to be committed (ahead = 0:
 * the records the next commit appends; ahead = 1: the block after it), so that
 * strat_rollout_step / strat_encode_obs / strat_legal_mask write them where they belong.
 * strat_replay_commit then appends action/reward/done for those n records and advances head. */
int strat_replay_reserve(strat_replay* r, int32_t n, int32_t ahead, uint16_t** obs, uint32_t** mask);
/* The action / reward / done rows of the n records the next commit appends, so that the step
 * writes them in place as well; strat_replay_commit(r, NULL, NULL, NULL, n, stream) then only
 * advances head (no copy kernel). */
int strat_replay_reserve_rows(strat_replay* r, int32_t n, int16_t** action, int8_t** reward, uint8_t** done);
int strat_replay_commit(strat_replay* r, const int16_t* action, const int8_t* reward, const uint8_t* done,
                        int32_t n, void* stream);
/* Uniform minibatch with replacement: element j = the record at ring position
 * bounded(sample draw j, filled).  STRAT_BAD_STATE on an empty ring. */
int strat_replay_sample(const strat_replay* r, uint64_t seed, uint64_t draw_index, int32_t batch,
                        uint16_t* obs, uint32_t* mask, int16_t* action, int8_t* reward, uint8_t* done,
                        void* stream);
/* The same gather for a self-play loop that pushes in place (in-place rings only): issued between
 * two fused steps of `env` on `stream`, it does not separate them - the next strat_rollout_step
 * still overlaps the previous one on the device.  Everything the fused step issued before it
 * pushed is sampled from: in the regular loop (strat_rollout_step into the reserved rows,
 * strat_replay_commit without copies, this call, once per step) the gather runs alongside that step
 * and takes each record as soon as the step has published the record's 32-game batch; after anything
 * else (a copy push, another call on the environment, the first gather) it waits for the whole stream
 * before it.  The fused step after the NEXT gather waits for this one before it reuses ring rows (the
 * ring's spare rows cover exactly that distance), and a gather waits for the one before it before it
 * overwrites the minibatch buffers.  One ring serves one environment this way and one environment
 * feeds one ring (STRAT_BAD_ARG for a ring tied to another environment, STRAT_BAD_STATE for an
 * environment another live ring is tied to; strat_replay_destroy unties); outputs are valid in
 * stream order as usual.  STRAT_BAD_STATE on a plain or empty ring. */
int strat_replay_sample_chained(strat_replay* r, strat_env* env, uint64_t seed, uint64_t draw_index, int32_t batch,
                                uint16_t* obs, uint32_t* mask, int16_t* action, int8_t* reward, uint8_t* done,
                                void* stream);
int strat_replay_state(const strat_replay* r, int64_t* head, int64_t* filled);
/* Rows of the live record at ring position p (0 <= p < filled): `row` in the mask / action /
 * reward / done arrays, `obs_row` in the observation array (both = p for a plain ring). */
int strat_replay_locate(const strat_replay* r, int64_t p, int64_t* row, int64_t* obs_row);

/* ---- board-history ring and historical queries (Table S1 455-480) ---- */
/* The paper's rollout buffer: instead of storing information states and masks, keep the game
 * STATES of the last `length` time steps in a circular, preallocated buffer (128 B per game
 * and step, 72x smaller than a stored transition) and re-materialise any query on demand.
 * Time step t is the state after t state updates since attach (CurrentStep);
 * slot t % length holds, for every game: the device line of the state at t, the action
 * applied at t (GetPlayedActions) and the reward / done byte that action
 * produced (ComputeRewardP10).  Valid queries: cur-length <= t < cur for
 * recorded steps, plus t == cur (the attached environment's live state) for the state
 * queries.  Memory is the caller's (strat_history_bytes), as everywhere else. */
typedef struct strat_history strat_history;
size_t strat_history_bytes(int32_t num_games, int32_t length);
int strat_history_create(void* mem_dev, size_t bytes, int32_t num_games, int32_t length, strat_history** out);
int strat_history_destroy(strat_history* h);
/* A TRACKED ring, for the paper's own information state at past time steps ("reconstruct
 * on-demand past information states"; Table S1, PAPER.md:462 ComputeInfostateTensor(t)): next to the 132 B
 * above it keeps, per game and time step, the 2 KB of trackers the 487 channels are built from
 * (strat_config.infostate) - 46x less than the 97,400 B tensor itself.  Same handle, same calls; 256 B of
 * work counters are cleared on `stream`.  While a tracked ring is attached to an environment with
 * infostate = 1, every recorded step is preceded by one copy kernel (the trackers of the state it starts
 * from), so consecutive fused steps do not overlap; with infostate = 0 nothing more is recorded and
 * strat_history_encode_infostate returns STRAT_BAD_STATE. */
size_t strat_history_bytes_tracked(int32_t num_games, int32_t length);
int strat_history_create_tracked(void* mem_dev, size_t bytes, int32_t num_games, int32_t length, void* stream,
                                 strat_history** out);
/* After attach, every strat_step / strat_rollout_step / strat_step_observe of `env` first records the state it
 * starts from, then the action, reward and done byte, and advances CurrentStep by one (the
 * fused step writes them itself: no copy kernel).  h == NULL detaches.  strat_rollout_uniform
 * refuses to run (STRAT_BAD_STATE) while a history is attached: it keeps the boards on chip
 * and records nothing.  Resets are not time steps. */
int strat_history_attach(strat_env* env, strat_history* h);
int strat_history_current_step(const strat_history* h, int64_t* step);
/* ComputeLegalActionMask(t) / ComputeInfostateTensor(t) / BoardStrs(t): same outputs as the
 * live calls produced (or would have produced) at time step t.  With chase_rule on, the move
 * log of the past state is rebuilt from the actions the ring still holds (up to 63 plies back to
 * the game's last restart, beyond it from the pinned log if there is one): identical to the
 * live mask whenever the ring reaches back as far as the chase did (length >= 63 always does;
 * plies handed over by strat_reset_from_with_plies before the ring's oldest step are not in it). */
int strat_history_legal_mask(const strat_history* h, int64_t t, uint32_t* mask, void* stream);
int strat_history_encode_obs(const strat_history* h, int64_t t, uint16_t* obs, void* stream);
int strat_history_get_boards(const strat_history* h, int64_t t, uint8_t* boards, void* stream);
/* ComputeInfostateTensor(t) in the paper's own 487 channels: what
 * strat_encode_infostate wrote, or would have written, at time step t; layout and alignment as there.
 * Tracked rings only (STRAT_BAD_STATE otherwise, and if the environment keeps no trackers). */
int strat_history_encode_infostate(const strat_history* h, int64_t t, uint16_t* out, void* stream);
/* GetPlayedActions(t), reward(t), done(t): NON-OWNING device pointers into the ring, valid
 * until `length` further steps have been recorded ("non-owning tensor"). */
int strat_history_transition(const strat_history* h, int64_t t, const int16_t** actions, const int8_t** reward,
                             const uint8_t** done);
/* info int32[N][4] = {ActingPlayer(t), GetNumMoves(t), GetNumMovesSinceLastAttack(t),
 * done | reason<<2 of the state at t (non-zero only for a frozen finished game; reason 1 =
 * GetFlagCaptured)}. */
int strat_history_info(const strat_history* h, int64_t t, int32_t* info, void* stream);
/* ComputeTwoSquareRuleApplies(t) uint8[N] (1 iff the two-square rule takes a move away from the
 * acting player), ComputeIsUnknownPiece(t) uint8[N][100] (1 on squares holding an opponent piece
 * whose type the acting player has not seen), GetTerminatedSince(t) int32[N] (steps since the
 * action that ended the game, counted over the steps still in the ring; 0 for a live game)
 * (PAPER.md:467, 469, 470).  Any of the three outputs may be NULL.  ComputePieceTypeOnehot(t)
 * is planes 0-23 of strat_history_encode_obs for the types both players know;
 * the hidden types themselves are in strat_history_get_boards. */
int strat_history_flags(const strat_history* h, int64_t t, uint8_t* two_square_applies, uint8_t* unknown,
                        int32_t* terminated_since, void* stream);
/* Travel back: make the state at time step t the live state of `env` (which need not be the
 * attached one; "efficient capturing of past states", 252-254).  With chase_rule on in
 * both, the move log is restored with it, rebuilt as for strat_history_legal_mask.
 * From a tracked ring (both environments with infostate = 1) the trackers of time step t travel back as
 * well; otherwise they restart from the restored position as after strat_reset_from. */
int strat_history_restore(const strat_history* h, int64_t t, strat_env* env, void* stream);

/* ---- search-shaped batch (BASELINE.json configs[4]) ------------------------------- */
/* out game G = r*samples_per_root + s: root r with the types of the searcher's opponent's
 * unrevealed pieces re-dealt uniformly over their squares among the arrangements that put no
 * Bomb or Flag on a moved piece: each hidden Bomb/Flag draws a free hidden square, redrawing
 * while it is a moved piece's (rejection); the movable types are shuffled over the rest
 * (R22).  More than 4096 draws for one game sets the sticky error of `out` to
 * STRAT_BAD_STATE.  out->num_games must equal roots->num_games * samples_per_root.  If both
 * environments run the chasing rule, each copy inherits its root's move log; so do
 * the games made by strat_search_expand. */
int strat_determinise(const strat_env* roots, int32_t samples_per_root, uint64_t seed, strat_env* out,
                      void* stream);
/* out int32[R][3] = {sum of returns, wins, losses} per root from the searcher's side
 * (root_side uint8[R], 0 red); unfinished games count 0. */
int strat_reduce_returns(const strat_env* games, const uint8_t* root_side, int32_t samples_per_root,
                         int32_t* out, void* stream);

/* ---- one search step without networks (S3.7; R29) -------- */
/* Steps 1-2: root r with L legal actions gets C = max(1, rollouts / L)
 * sampled configurations of the opponent's hidden pieces (strat_determinise's sampler stands
 * in for the belief network, cf. the uniform-belief ablation PAPER.md:277-279) and one game per
 * (configuration c, legal action l): slot r*rollouts + c*L + l of `out` = configuration c with
 * the l-th legal action (ascending) applied - the forced first move.  The min(C*L, rollouts)
 * first slots of a root are used; the rest are frozen finished copies of the root.
 * out->num_games == roots->num_games * rollouts, out->auto_reset == 0, no history attached.
 * Then play the remaining depth-1 plies (strat_rollout_uniform: the uniform policy stands in
 * for the move network) and call strat_search_policy. */
int strat_search_expand(const strat_env* roots, int32_t rollouts, uint64_t seed, strat_env* out, void* stream);
/* Steps 3-4, float32 [R][3600] each, 0 on illegal actions:
 *   qhat(a)   = mean over configurations of the value of the game that started with a; the value
 *               is the game's result from the searcher's side, 0 while it is running (stand-in
 *               for the move network's value head);
 *   rho(a)    = magnet policy: 1 / (pieces that can move * moves of a's piece);
 *   pi_search = [exp(qhat) rho^alpha pi_theta^beta]^(1/(alpha+beta)) normalised over the legal
 *               actions (eq. 8), the maximiser of <qhat,pi> - alpha KL(pi,rho) - beta KL(pi,pi_theta)
 *               (eq. 7).  pi_theta: the caller's prior float32 [R][3600] (e.g. the move network's
 *               policy), or NULL for the uniform distribution over the legal actions.
 * Paper's values: alpha = 0.002, beta = 0.02, 1,000 rollouts of depth 40 (Table S12). */
int strat_search_policy(const strat_env* roots, const strat_env* games, int32_t rollouts, const float* pi_theta,
                        float alpha, float beta, float* qhat, float* rho, float* pi_search, void* stream);
/* The same with the value head's outputs (step 3: "average values q-hat for each legal move
 * according to the value output of the move network at the positions reached by the rollouts"):
 * values float32 [R*rollouts] (device), entry r*rollouts + slot = the value of the position that game
 * reached, from the SEARCHER's side (the player to move at the root).  It counts for the games still
 * running; a game that has ended keeps its result.  values == NULL: strat_search_policy (running games
 * count 0).  qhat is summed per action in slot order in double and rounded once. */
int strat_search_policy_values(const strat_env* roots, const strat_env* games, int32_t rollouts, const float* pi_theta,
                               const float* values, float alpha, float beta, float* qhat, float* rho, float* pi_search,
                               void* stream);

/* ---- legal masks of given positions, for callers that cannot allocate device memory ---- */
/* Everything above works on a workspace the caller allocates.  Some callers have no way to do that:
 * code that is handed nothing but its input and output buffers by the framework it is plugged into
 * (an operator or inference-server plugin, a data-loader stage) and has no access to that framework's
 * allocator; a step in a latency-critical loop, where cudaMalloc / cudaFree would stall the whole
 * device (both synchronise it); a thread that must not touch the allocator because another thread
 * of the process is capturing a stream in the global capture mode, which forbids cudaMalloc
 * process-wide.  For them this one call computes ComputeLegalActionMask (rules
 * PAPER.md:210-212) for up to STRAT_STATIC_MAX_GAMES given positions with no environment, no
 * workspace and no allocation of any kind (no cudaMalloc, cudaFree or allocating library routine,
 * neither here nor in anything it calls): the bit-sliced state lines the mask kernel reads - what
 * strat_reset_from builds in the workspace - go to a fixed array inside the library's device image
 * (STRAT_STATIC_MAX_GAMES x 128 B of lines + 256 B holding the error word = 512.25 KB, held by every
 * GPU that loads libstrat.so until the process exits).
 *
 *   boards  in   uint8[num_games][128] canonical lines (device), as for strat_reset_from
 *   mask    out  uint32[num_games][113] (device): exactly what strat_reset_from + strat_legal_mask
 *                of an environment with this two_square (and chase_rule = 0) write for these boards
 *   status  out  int32[1] (device), or NULL: 0, or STRAT_BAD_STATE if a line gives one side more
 *                than 8 Scouts (what strat_check reports after strat_reset_from); valid in stream order
 *   returns STRAT_TOO_LARGE for num_games > STRAT_STATIC_MAX_GAMES (nothing is launched; split the
 *           batch), STRAT_BAD_ARG for a NULL boards / mask or num_games < 1
 *
 * It runs on the CURRENT device; `stream` must belong to it.  The first call on each device looks up
 * where the array lives on that device (cudaGetSymbolAddress; it may also make the driver load the
 * library's device code): make that first call outside any stream capture, e.g. once at start-up.
 * All calls on one device share the one array, and it keeps what the last call left in it: the call
 * itself clears the error word and overwrites the lines it uses, so the caller clears nothing - but
 * two calls that can run at the same time on one GPU (different streams without an event between
 * them, different host threads or processes sharing a context) race on it and corrupt each other's
 * masks.  Issue them on one stream, or order them with events. */
#define STRAT_STATIC_MAX_GAMES 4096
int strat_legal_mask_static(const uint8_t* boards, int32_t num_games, int32_t two_square, uint32_t* mask,
                            int32_t* status, void* stream);

/* ---- measurement aid ---------------------------------------------------------------- */
/* Streams a constant over dst[0, bytes) with the store instruction the step kernels use for their
 * outputs (16-byte st.global.cs), in pieces of chunk_bytes (a multiple of 16 that divides bytes; a batch
 * of observations is 281,600): the plain-write figure bench.py prints next to its roofline fractions.
 * Persistent CTAs; dynamic = 1: every CTA fetches its next piece from a ticket counter as it finishes
 * one (how the step kernels hand out batches), 0: equal shares by a fixed stride.  On a B200 the two
 * differ by ~17 % (7.2-7.4 against 6.2 TB/s): the SMs do not drain their stores at one rate.  The
 * environment lends its ticket word and SM count; nothing of it is touched.  One probe at a time per
 * environment: two in flight would draw from the same ticket word. */
int strat_probe_write(const strat_env* env, void* dst, size_t bytes, int32_t chunk_bytes, int32_t dynamic, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* STRAT_H_ */
