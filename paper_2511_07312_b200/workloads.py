"""Synthetic workload descriptions and plain board-layout helpers.

This module is shared by the CUDA-path tests, the oracle tests and bench.py.  It holds
NONE of the method's arithmetic (no rules, no RNG, no encoding of observations): only
the five BASELINE.json configurations as data and helpers that place bytes into the
canonical 128-byte line (layout: DESIGN.md "Boundary"; type order PAPER.md:499).
Every random quantity of the method is drawn by Philox inside each implementation from
(seed, game, epoch, ply), so the only shared inputs are these integers.
"""
import numpy as np

LINE = 128
MASK_WORDS = 113
PLANES = 44
OBS_ELEMS = PLANES * 100
ACTIONS = 3600
TRANSITION_BYTES = OBS_ELEMS * 2 + MASK_WORDS * 4 + 2 + 1 + 1  # 9256

EMPTY, SPY, SCOUT, MINER, SERGEANT, LIEUTENANT, CAPTAIN, MAJOR, COLONEL, GENERAL, MARSHAL, FLAG, BOMB = range(13)
LAKE = 15
RED, BLUE = 0, 1
LAKES = (42, 43, 52, 53, 46, 47, 56, 57)
OWNER, MOVED, REVEALED = 0x10, 0x20, 0x40

# BASELINE.json configs[0..4].  `steps` is what the parity tests / bench run.
CONFIGS = [
    dict(name="cfg0_classic_256", variant=0, num_games=256, seed=0, max_plies=0, auto_reset=0, steps=256),
    dict(name="cfg1_barrage_4096", variant=1, num_games=4096, seed=0, max_plies=2000, auto_reset=0, steps=2000),
    dict(name="cfg2_classic_65536", variant=0, num_games=65536, seed=0, max_plies=1000, auto_reset=1, steps=2000),
    dict(name="cfg3_selfplay_262144", variant=0, num_games=262144, seed=0, max_plies=1000, auto_reset=1,
         steps=2000, ring_per_slot=131072, ring_slots=64, sample_batch=4096),
    dict(name="cfg4_search_16x16384", variant=0, num_roots=16, samples_per_root=16384, root_plies=200,
         rollout_plies=64, seed=0),
]


def piece(ptype, owner, moved=False, revealed=False):
    return ptype | (OWNER if owner else 0) | (MOVED if moved else 0) | (REVEALED if revealed else 0)


def action_index(frm, direction, dist):
    """from*36 + dir*9 + (dist-1); dir 0:+row 1:+col 2:-row 3:-col (layout only)."""
    return frm * 36 + direction * 9 + (dist - 1)


def make_line(pieces, ply=0, history=(), battleless=0, epoch=0):
    """Canonical 128-byte line from {cell: byte}; history = [(from,to) most recent first]."""
    L = np.zeros(LINE, np.uint8)
    for c in LAKES:
        L[c] = LAKE
    for c, b in pieces.items():
        assert c not in LAKES and 0 <= c < 100
        L[c] = b
    L[100:116] = 0xFF
    for j, (f, t) in enumerate(history):
        L[100 + 2 * j] = f
        L[101 + 2 * j] = t
    L[116] = ply & 255
    L[117] = ply >> 8
    L[118] = battleless & 255
    L[119] = battleless >> 8
    for k in range(4):
        L[124 + k] = (epoch >> (8 * k)) & 255
    return L


def mask_to_actions(mask_row):
    """Set bits of one packed uint32[113] mask row, ascending (layout only)."""
    bits = np.unpackbits(np.ascontiguousarray(mask_row, dtype="<u4").view(np.uint8), bitorder="little")
    return np.nonzero(bits)[0].tolist()


def board_str(line):
    """ASCII dump of one canonical line (BoardStrs).  Row 9 printed first."""
    sym = ".SsmeLCJOGMFB"  # index = type code; Scout 's', Spy 'S', sErgeant 'e', maJor 'J', cOlonel 'O'
    rows = []
    for r in range(9, -1, -1):
        row = []
        for q in range(10):
            b = int(line[10 * r + q])
            t = b & 15
            if t == LAKE:
                row.append("~~")
            elif t == 0:
                row.append(" .")
            else:
                row.append(("b" if b & OWNER else "r") + sym[t])
        rows.append(" ".join(row))
    return "\n".join(rows)


def capture_at_ply(env_get_boards, env_play_one_ply, num_games, ply):
    """Root positions for the search-shaped batch (BASELINE.json configs[4]: "each reached by
    200 uniform-random plies from a seeded classic setup").  Drives ANY environment exposing
    the two callables (an auto-resetting env playing uniform-random legal actions) and keeps,
    for every game slot, the first line whose ply counter equals `ply` while the game is
    live; a game that ends earlier restarts (next epoch) and is captured in a later epoch.
    Pure bookkeeping: no rule or RNG arithmetic here."""
    roots = np.zeros((num_games, LINE), np.uint8)
    have = np.zeros(num_games, bool)
    for _ in range(100000):
        b = env_get_boards()
        p = b[:, 116].astype(int) | (b[:, 117].astype(int) << 8)
        hit = (~have) & (p == ply) & ((b[:, 120] & 1) == 0)
        roots[hit] = b[hit]
        have |= hit
        if have.all():
            return roots
        env_play_one_ply()
    raise RuntimeError("roots not reached")


def shard_for_rank(cfg, rank, world):
    """Weak-scaling shard of a config for one rank: every rank owns `num_games` independent
    games whose RNG streams are keyed by the global index game_base + local index, so the
    union over ranks equals one world*num_games-game run.  No collective on the data path."""
    assert 0 <= rank < world
    return dict(variant=cfg["variant"], seed=cfg["seed"], max_plies=cfg["max_plies"],
                auto_reset=cfg["auto_reset"], game_base=rank * cfg["num_games"])
