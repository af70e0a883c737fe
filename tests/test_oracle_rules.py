"""Pins for the CPU oracle's rules: RNG, battle table, legal moves, two-square rule.

Each test checks the oracle against something other than itself: published known-answer
vectors, a hand-written table from the rules text, hand-worked positions, closed forms,
symmetries of the board, and a brute-force enumerator written in a different style.
"""
import json
import math
import os

import numpy as np
import pytest

from oracle import orc
from paper_2511_07312_b200 import workloads as W


# ----------------------------------------------------------------------------- RNG
def test_philox_known_answers(golden_dir):
    n = 0
    for line in open(os.path.join(golden_dir, "philox4x32_10_kat.txt")):
        line = line.split("#")[0].split()
        if not line:
            continue
        v = [int(x, 16) for x in line]
        out = orc.philox(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]
        n += 1
    assert n == 3


def test_philox_counter_and_key_sensitivity():
    base = orc.philox([1, 2, 3, 4], [5, 6])
    for i in range(4):
        c = [1, 2, 3, 4]
        c[i] ^= 1
        assert not np.array_equal(orc.philox(c, [5, 6]), base)
    for i in range(2):
        k = [5, 6]
        k[i] ^= 1
        assert not np.array_equal(orc.philox([1, 2, 3, 4], k), base)


# ----------------------------------------------------------------------------- battle
def test_battle_table_matches_rules_text(golden_dir):
    sym = {"W": 1, "L": -1, "T": 0}
    rows = 0
    counts = {1: 0, -1: 0, 0: 0}
    for line in open(os.path.join(golden_dir, "battle_table.txt")):
        line = line.split("#")[0].split()
        if not line:
            continue
        att = int(line[0])
        assert len(line) == 13
        for d, s in enumerate(line[1:], start=1):
            got = orc.battle(att, d)
            assert got == sym[s], (att, d, got, s)
            counts[got] += 1
        rows += 1
    assert rows == 10
    assert counts == {1: 57, -1: 53, 0: 10}


def test_battle_named_special_cases():
    assert orc.battle(W.SPY, W.MARSHAL) == 1      # Spy attacking Marshal wins
    assert orc.battle(W.MARSHAL, W.SPY) == 1      # but the Marshal attacking the Spy wins
    assert orc.battle(W.MINER, W.BOMB) == 1       # Miner defuses Bomb
    for a in range(1, 11):
        if a != W.MINER:
            assert orc.battle(a, W.BOMB) == -1    # every other attacker on a Bomb is lost
        assert orc.battle(a, W.FLAG) == 1         # capturing the Flag
        assert orc.battle(a, a) == 0              # equal ranks both removed


# ----------------------------------------------------------------------------- geometry
def test_board_constants():
    lakes = [c for c in range(100) if orc.is_lake(c)]
    assert sorted(lakes) == sorted(W.LAKES)
    assert 100 - len(lakes) == 92  # PAPER.md:208 "92 occupiable squares"
    # two 2x2 blocks: c5-d6 and g5-h6 (files a..j = cols 0..9, ranks 1..10 = rows 0..9)
    def cell(sq):
        return (int(sq[1:]) - 1) * 10 + (ord(sq[0]) - ord("a"))
    assert sorted(lakes) == sorted(cell(s) for s in ["c5", "d5", "c6", "d6", "g5", "h5", "g6", "h6"])


def test_setup_count_matches_paper():
    # PAPER.md:29 ">10^33 possible piece configurations" per player: 40!/prod(count!)
    ms = orc.multiset(0)
    cnt = np.bincount(ms, minlength=13)
    assert cnt[1:].tolist() == [1, 8, 5, 4, 4, 4, 3, 2, 1, 1, 1, 6]  # Spy..Marshal, Flag, Bomb
    n = math.factorial(40)
    for k in cnt[1:]:
        n //= math.factorial(int(k))
    assert 1.41e33 < n < 1.42e33
    b = orc.multiset(1)
    assert sorted(b[b > 0].tolist()) == sorted([11, 10, 9, 3, 2, 2, 1, 12])
    assert (b == 0).sum() == 32


# ----------------------------------------------------------------------------- positions
def _env_from_line(line, **kw):
    e = orc.Env(1, **kw)
    e.reset_from(line[None, :])
    return e


def _load_positions(golden_dir):
    return json.load(open(os.path.join(golden_dir, "positions.json")))["positions"]


def test_hand_worked_positions(golden_dir):
    for pos in _load_positions(golden_dir):
        pieces = {c: W.piece(t, o) for c, t, o in pos["pieces"]}
        e = _env_from_line(W.make_line(pieces))
        for a in pos["play"]:
            m = e.legal_mask()
            assert a in W.mask_to_actions(m[0]), (pos["name"], a)
            r, d = e.step(np.array([a], np.int16))
            assert e.check() == 0 and d[0] & 1 == 0
        m = e.legal_mask()
        assert W.mask_to_actions(m[0]) == pos["expect"], pos["name"]
        for w, v in pos.get("expect_words", {}).items():
            assert int(m[0, int(w)]) == int(v, 16)
            others = np.delete(m[0], int(w))
            assert not others.any()


def test_two_square_reset_from_history_equals_live_play(golden_dir):
    # the canonical line carries no chain: reset_from must rebuild it from the history
    for pos in _load_positions(golden_dir):
        pieces = {c: W.piece(t, o) for c, t, o in pos["pieces"]}
        e = _env_from_line(W.make_line(pieces))
        for a in pos["play"]:
            e.step(np.array([a], np.int16))
        e2 = orc.Env(1)
        e2.reset_from(e.get_boards())
        assert np.array_equal(e.legal_mask(), e2.legal_mask()), pos["name"]
        assert np.array_equal(e.get_boards(), e2.get_boards())


def test_two_square_off_switch(golden_dir):
    pos = [p for p in _load_positions(golden_dir) if p["name"].startswith("E4a")][0]
    pieces = {c: W.piece(t, o) for c, t, o in pos["pieces"]}
    e = _env_from_line(W.make_line(pieces), two_square=0)
    for a in pos["play"]:
        e.step(np.array([a], np.int16))
    assert W.mask_to_actions(e.legal_mask()[0]) == [1620, 1638, 1647]


def test_two_square_chain_broken_by_other_piece():
    # red shuttles 44<->45 twice, then moves another piece, then may shuttle again
    pieces = {44: W.piece(W.SERGEANT, 0), 20: W.piece(W.MINER, 0), 0: W.piece(W.FLAG, 0),
              95: W.piece(W.SERGEANT, 1), 85: W.piece(W.MINER, 1), 99: W.piece(W.FLAG, 1)}
    e = _env_from_line(W.make_line(pieces))
    A = W.action_index
    seq = [A(44, 1, 1), A(85, 3, 1), A(45, 3, 1), A(84, 3, 1), A(44, 1, 1), A(83, 3, 1),
           A(20, 0, 1), A(82, 3, 1)]  # red's 4th move is the Miner: chain broken
    for a in seq:
        assert a in W.mask_to_actions(e.legal_mask()[0])
        e.step(np.array([a], np.int16))
    acts = W.mask_to_actions(e.legal_mask()[0])
    assert A(45, 3, 1) in acts  # 45->44 legal again


def test_closed_form_ply0_count():
    # At ply 0 of a classic game red's legal moves come only from row 3, columns
    # {0,1,4,5,8,9} (the others face lakes): 0 if Bomb/Flag, Scout 3 (dist 1,2 and the
    # attack at dist 3 on blue's row 6), else 1.
    e = orc.Env(512, seed=11)
    b = e.get_boards()
    m = e.legal_mask()
    for g in range(512):
        exp = 0
        for col in (0, 1, 4, 5, 8, 9):
            t = b[g, 30 + col] & 15
            exp += 0 if t in (W.FLAG, W.BOMB) else (3 if t == W.SCOUT else 1)
        assert len(W.mask_to_actions(m[g])) == exp
        assert e.count_moves(g, 0) == exp


# ----------------------------------------------------------------------------- symmetries
def _mirror_cell(c):
    return (c // 10) * 10 + 9 - (c % 10)


def _mirror_line(line):
    out = line.copy()
    for c in range(100):
        out[_mirror_cell(c)] = line[c]
    for k in range(100, 116):
        if line[k] != 0xFF:
            out[k] = _mirror_cell(int(line[k]))
    return out


def _rot_line(line):
    """Rotate 180 degrees and swap colours and the side to move (ply parity flips)."""
    out = line.copy()
    for c in range(100):
        b = int(line[c])
        t = b & 15
        out[99 - c] = b ^ W.OWNER if 1 <= t <= 12 else b
    for k in range(100, 116):
        if line[k] != 0xFF:
            out[k] = 99 - int(line[k])
    ply = int(line[116]) | (int(line[117]) << 8)
    ply += 1
    out[116], out[117] = ply & 255, ply >> 8
    return out


def _midgame_lines(n, plies, seed, variant=0):
    e = orc.Env(n, variant=variant, seed=seed, max_plies=2000)
    for _ in range(plies):
        e.step(e.sample_uniform(e.legal_mask()))
    return e.get_boards()


@pytest.mark.parametrize("variant,plies", [(0, 60), (0, 301), (1, 40)])
def test_mirror_and_rotation_symmetry(variant, plies):
    lines = _midgame_lines(48, plies, seed=5, variant=variant)
    lines = lines[(lines[:, 120] & 1) == 0]
    assert len(lines) > 8
    n = len(lines)
    e = orc.Env(n, variant=variant)
    e.reset_from(lines)
    base = e.legal_mask()
    e.reset_from(np.stack([_mirror_line(l) for l in lines]))
    mir = e.legal_mask()
    e.reset_from(np.stack([_rot_line(l) for l in lines]))
    rot = e.legal_mask()
    for g in range(n):
        acts = W.mask_to_actions(base[g])
        exp_m = sorted(W.action_index(_mirror_cell(a // 36), {0: 0, 1: 3, 2: 2, 3: 1}[(a % 36) // 9], a % 9 + 1)
                       for a in acts)
        assert W.mask_to_actions(mir[g]) == exp_m
        exp_r = sorted(W.action_index(99 - a // 36, ((a % 36) // 9 + 2) % 4, a % 9 + 1) for a in acts)
        assert W.mask_to_actions(rot[g]) == exp_r


# ----------------------------------------------------------------------------- brute force
def _naive_moves(line):
    """Destination-first enumerator: for every target square look back along the four
    lines for a piece of the side to move that can reach it (a different traversal from
    the oracle's from/dir/dist loops).  Two-square bans are not modelled here."""
    ply = int(line[116]) | (int(line[117]) << 8)
    side = ply & 1
    out = set()
    for to in range(100):
        tb = int(line[to])
        if (tb & 15) == W.LAKE:
            continue
        if 1 <= (tb & 15) <= 12 and ((tb >> 4) & 1) == side:
            continue
        tr, tq = divmod(to, 10)
        for d, (dr, dq) in enumerate([(1, 0), (0, 1), (-1, 0), (0, -1)]):
            # walk backwards from the target against direction d
            for k in range(1, 10):
                r, q = tr - dr * k, tq - dq * k
                if not (0 <= r < 10 and 0 <= q < 10):
                    break
                b = int(line[r * 10 + q])
                if b == 0:
                    continue
                t = b & 15
                if t != W.LAKE and ((b >> 4) & 1) == side and (t == W.SCOUT or (k == 1 and 1 <= t <= 10)):
                    out.add(W.action_index(r * 10 + q, d, k))
                break
    return sorted(out)


@pytest.mark.parametrize("variant,plies", [(0, 0), (0, 150), (0, 600), (1, 80)])
def test_brute_force_enumerator_agrees(variant, plies):
    lines = _midgame_lines(32, plies, seed=9, variant=variant)
    lines = lines[(lines[:, 120] & 1) == 0]
    e = orc.Env(len(lines), variant=variant, two_square=0)
    e.reset_from(lines)
    m = e.legal_mask()
    for g in range(len(lines)):
        assert W.mask_to_actions(m[g]) == _naive_moves(lines[g])
    # with the rule on, the legal set is a subset and differs by at most the banned line
    e2 = orc.Env(len(lines), variant=variant, two_square=1)
    e2.reset_from(lines)
    m2 = e2.legal_mask()
    assert not (m2 & ~m).any()
