"""Pins for the oracle's setup generator, step/terminal logic, encoder, replay ring and
determinisation: closed forms, invariants the rules fix (BASELINE.json north_star: lake
cells never occupied, piece multisets only shrink through battles, a side with no legal
move loses), hand-built endings and statistical checks."""
import os

import numpy as np
import pytest

from oracle import orc
from paper_2511_07312_b200 import workloads as W

ONE = 0x3F80


def _type(b):
    return b & 15


def _counts(line):
    """per (owner, type) piece counts of one line"""
    out = np.zeros((2, 13), int)
    for c in range(100):
        t = int(line[c]) & 15
        if 1 <= t <= 12:
            out[(int(line[c]) >> 4) & 1, t] += 1
    return out


# ----------------------------------------------------------------------------- setup
def test_setup_multiset_homes_and_determinism():
    e = orc.Env(300, seed=3)
    b = e.get_boards()
    ref = np.bincount(orc.multiset(0), minlength=13)
    for g in range(300):
        cnt = _counts(b[g])
        assert (cnt[0] == ref).all() and (cnt[1] == ref).all()
        assert all((b[g, c] & 0x70) == 0 for c in range(40))           # red: no flags set
        assert all((b[g, c] & 0x70) == 0x10 for c in range(60, 100))   # blue: owner bit only
        assert all(b[g, c] == (15 if c in W.LAKES else 0) for c in range(40, 60))
        assert (b[g, 100:116] == 0xFF).all() and not b[g, 116:128].any()
    e2 = orc.Env(300, seed=3)
    assert np.array_equal(b, e2.get_boards())
    e3 = orc.Env(300, seed=4)
    assert not np.array_equal(b, e3.get_boards())
    # keyed by the global game index: a shard starting at game 100 reproduces games 100..
    e4 = orc.Env(50, seed=3, game_base=100)
    assert np.array_equal(e4.get_boards(), b[100:150])


def test_setup_marginals_are_uniform():
    # each type's marginal on every home cell is count/40 (chi-square over 40 cells)
    n = 6000
    b = orc.Env(n, seed=1).get_boards()
    ref = np.bincount(orc.multiset(0), minlength=13)
    for base in (0, 60):
        t = b[:, base:base + 40] & 15
        for typ in range(1, 13):
            obs = (t == typ).sum(axis=0)
            exp = n * ref[typ] / 40.0
            chi2 = ((obs - exp) ** 2 / exp).sum()
            assert chi2 < 80.0, (base, typ, chi2)  # 39 dof: P(chi2 > 80) ~ 1e-4


def test_barrage_setup():
    b = orc.Env(500, variant=1, seed=2).get_boards()
    for g in range(500):
        cnt = _counts(b[g])
        for o in (0, 1):
            assert cnt[o].tolist() == [0, 1, 2, 1, 0, 0, 0, 0, 0, 1, 1, 1, 1]
        assert all(_type(b[g, c]) == 0 or c in W.LAKES for c in range(40, 60))
    occ = ((b[:, :40] & 15) != 0).mean(axis=0)
    assert abs(occ - 0.2).max() < 0.08  # 8 pieces on 40 uniform cells


def test_setup_rejects_immobile_side():
    # R#5: every generated side owns a movable piece that can move or could once the
    # square in front is vacated (depends on own pieces only)
    e = orc.Env(2000, seed=7)
    assert all(e.count_moves(g, 0) > 0 for g in range(2000))


def test_setup_redraw_rate_matches_the_closed_form_and_cases_are_redrawn(golden_dir):
    """R#5: a classic side is immobile at the first attempt iff its six front squares beside the
    lakes hold 6 of its 7 immovable pieces: p = 7*6*5*4*3*2 / (40*39*38*37*36*35) per side."""
    import json
    p = (7 * 6 * 5 * 4 * 3 * 2) / (40 * 39 * 38 * 37 * 36 * 35)
    n = 1_000_000
    hits = orc.find_setup_redraws(0, 0, 0, 0, n)
    lam = 2 * p * n                                       # 3.6 expected; Poisson: P(k > 14) < 1e-5
    assert abs(p - 1.8e-6) < 1e-7 and 0 < len(hits) <= 14, (lam, hits)
    cases = json.load(open(os.path.join(golden_dir, "setup_redraw_cases.json")))
    assert hits == [g for g in cases["epoch0"] if g < n]
    for g in cases["epoch0"]:
        e = orc.Env(1, seed=cases["seed"], game_base=g)
        b = e.get_boards()[0]
        assert e.count_moves(0, 0) + e.count_moves(0, 1) > 0
        front = [30, 31, 34, 35, 38, 39]
        red_stuck = all((b[c] & 15) in (11, 12) for c in front)
        blue_stuck = all((b[99 - c] & 15) in (11, 12) for c in front)
        assert not red_stuck and not blue_stuck          # the setup that was kept can move


# ----------------------------------------------------------------------------- step
def _play(e, n_steps, check=None):
    for _ in range(n_steps):
        before = e.get_boards()
        a = e.sample_uniform(e.legal_mask())
        r, d = e.step(a)
        if check:
            check(before, a, r, d, e.get_boards())
    assert e.check() == 0


def test_rollout_invariants_classic():
    e = orc.Env(96, seed=21, max_plies=700)

    def check(before, a, r, d, after):
        for g in range(len(a)):
            was_done = before[g, 120] & 1
            if was_done:
                assert a[g] == -1 and r[g] == 0 and d[g] == (1 | (before[g, 120] & 0x1C))
                assert np.array_equal(before[g], after[g])
                continue
            assert 0 <= a[g] < 3600
            for c in W.LAKES:
                assert after[g, c] == 15                      # lakes never occupied
            cb, ca = _counts(before[g]), _counts(after[g])
            assert (ca <= cb).all()                            # multisets only shrink
            removed = int((cb - ca).sum())
            f, t = int(after[g, 100]), int(after[g, 101])
            assert f == a[g] // 36
            battle = before[g, t] != 0
            assert removed == (0 if not battle else removed) and removed in (0, 1, 2)
            assert (removed > 0) == battle                     # ... and only through battles
            bl_before = int(before[g, 118]) | (int(before[g, 119]) << 8)
            bl_after = int(after[g, 118]) | (int(after[g, 119]) << 8)
            assert bl_after == (0 if battle else bl_before + 1)
            ply_b = int(before[g, 116]) | (int(before[g, 117]) << 8)
            ply_a = int(after[g, 116]) | (int(after[g, 117]) << 8)
            assert ply_a == ply_b + 1
            assert (d[g] >> 1) & 1 == ply_b & 1                # bit1 = player who acted
            # moved / revealed bits are monotone for surviving, stationary pieces
            for c in range(100):
                if c not in (f, t) and 1 <= (before[g, c] & 15) <= 12:
                    assert after[g, c] == before[g, c]
            # Bombs and Flags never move
            assert (before[g, f] & 15) not in (W.FLAG, W.BOMB)
            for c in range(100):
                if (after[g, c] & 15) in (W.FLAG, W.BOMB):
                    assert not after[g, c] & W.MOVED
            done = d[g] & 1
            assert (after[g, 120] & 1) == done
            reason = (d[g] >> 2) & 7
            flags = [int(ca[o, W.FLAG]) for o in (0, 1)]
            if not done:
                assert r[g] == 0 and reason == 0 and flags == [1, 1]
            else:
                assert (reason == 1) == (sum(flags) == 1)
                if reason in (1, 2):
                    assert r[g] == (1 if (ply_b & 1) == 0 else -1)   # mover wins, reward is red's
                else:
                    assert r[g] == 0
                assert np.int8(after[g, 121]) == r[g]

    _play(e, 700, check)
    b = e.get_boards()
    assert (b[:, 120] & 1).all()  # everything ended by the 700-ply cap
    reasons = np.bincount((b[:, 120] >> 2) & 7, minlength=6)
    assert reasons[4] > 0 and reasons[1] > 0  # both cap draws and flag captures occur


def test_live_game_has_nonzero_mask_and_side_without_moves_loses():
    e = orc.Env(64, variant=1, seed=5, max_plies=2000)
    for _ in range(2000):
        m = e.legal_mask()
        b = e.get_boards()
        live = (b[:, 120] & 1) == 0
        assert (m[live].any(axis=1)).all()
        assert not m[~live].any()
        r, d = e.step(e.sample_uniform(m))
        if not live.any():
            break
    b = e.get_boards()
    assert (b[:, 120] & 1).all()
    for g in range(64):
        reason = (b[g, 120] >> 2) & 7
        if reason == 2:  # the side to move has no legal move and lost
            ply = int(b[g, 116]) | (int(b[g, 117]) << 8)
            stuck = ply & 1
            assert e.count_moves(g, stuck) == 0 and e.count_moves(g, 1 - stuck) > 0
            assert np.int8(b[g, 121]) == (1 if stuck == 1 else -1)


def test_hand_built_endings():
    A = W.action_index
    # (i) flag capture by blue -> red's reward -1, reason 1
    L = W.make_line({50: W.piece(W.FLAG, 0), 60: W.piece(W.MINER, 1), 99: W.piece(W.FLAG, 1),
                     0: W.piece(W.SCOUT, 0)}, ply=1)
    e = orc.Env(1); e.reset_from(L[None])
    r, d = e.step(np.array([A(60, 2, 1)], np.int16))
    assert r[0] == -1 and d[0] == (1 | 2 | (1 << 2))
    # (ii) red captures blue's last movable piece: blue cannot move -> red wins, reason 2
    L = W.make_line({10: W.piece(W.MARSHAL, 0), 0: W.piece(W.FLAG, 0), 20: W.piece(W.SCOUT, 1),
                     99: W.piece(W.FLAG, 1), 98: W.piece(W.BOMB, 1)})
    e = orc.Env(1); e.reset_from(L[None])
    r, d = e.step(np.array([A(10, 0, 1)], np.int16))
    assert r[0] == 1 and d[0] == (1 | 0 | (2 << 2))
    # (iii) equal ranks remove the last movable pieces of both sides -> draw, reason 3
    L = W.make_line({10: W.piece(W.MAJOR, 0), 0: W.piece(W.FLAG, 0), 20: W.piece(W.MAJOR, 1),
                     99: W.piece(W.FLAG, 1)})
    e = orc.Env(1); e.reset_from(L[None])
    r, d = e.step(np.array([A(10, 0, 1)], np.int16))
    assert r[0] == 0 and d[0] == (1 | 0 | (3 << 2))
    b = e.get_boards()[0]
    assert b[10] == 0 and b[20] == 0
    # (iv) attacker lost against a Bomb; Bomb stays, revealed, not moved
    L = W.make_line({10: W.piece(W.GENERAL, 0), 0: W.piece(W.FLAG, 0), 5: W.piece(W.SCOUT, 0),
                     20: W.piece(W.BOMB, 1), 99: W.piece(W.FLAG, 1), 90: W.piece(W.SCOUT, 1)})
    e = orc.Env(1); e.reset_from(L[None])
    r, d = e.step(np.array([A(10, 0, 1)], np.int16))
    b = e.get_boards()[0]
    assert d[0] == 0 and b[10] == 0 and b[20] == W.piece(W.BOMB, 1, moved=False, revealed=True)
    # (v) winner of a battle is revealed and moved; Scout long move reveals it (R#10)
    L = W.make_line({10: W.piece(W.SCOUT, 0), 0: W.piece(W.FLAG, 0), 99: W.piece(W.FLAG, 1),
                     90: W.piece(W.SCOUT, 1)})
    e = orc.Env(1); e.reset_from(L[None])
    e.step(np.array([A(10, 0, 3)], np.int16))
    assert e.get_boards()[0][40] == W.piece(W.SCOUT, 0, moved=True, revealed=True)
    e.step(np.array([A(90, 2, 1)], np.int16))
    assert e.get_boards()[0][80] == W.piece(W.SCOUT, 1, moved=True, revealed=False)
    # (vi) ply cap -> draw reason 4 ; battleless cap -> reason 5
    L = W.make_line({10: W.piece(W.SCOUT, 0), 0: W.piece(W.FLAG, 0), 99: W.piece(W.FLAG, 1),
                     90: W.piece(W.SCOUT, 1)}, ply=9)
    e = orc.Env(1, max_plies=10); e.reset_from(L[None])
    r, d = e.step(np.array([A(90, 2, 1)], np.int16))
    assert r[0] == 0 and d[0] == (1 | 2 | (4 << 2))
    L = W.make_line({10: W.piece(W.SCOUT, 0), 0: W.piece(W.FLAG, 0), 99: W.piece(W.FLAG, 1),
                     90: W.piece(W.SCOUT, 1)}, ply=8, battleless=4)
    e = orc.Env(1, max_battleless=5); e.reset_from(L[None])
    r, d = e.step(np.array([A(10, 0, 1)], np.int16))
    assert r[0] == 0 and d[0] == (1 | 0 | (5 << 2))


def test_illegal_action_sets_sticky_error_and_leaves_game_unchanged():
    e = orc.Env(4, seed=1)
    before = e.get_boards()
    a = e.sample_uniform(e.legal_mask())
    a[2] = 5  # cell 0 moving +row by 6: never legal at ply 0
    r, d = e.step(a)
    assert e.check() == orc.ILLEGAL_ACTION
    after = e.get_boards()
    assert np.array_equal(before[2], after[2]) and r[2] == 0 and d[2] == 0
    assert not np.array_equal(before[0], after[0])
    e.clear_error()
    assert e.check() == 0


def test_auto_reset_restarts_with_next_epoch_and_same_stream():
    e = orc.Env(32, seed=9, max_plies=40, auto_reset=1)
    for _ in range(40):
        r, d = e.step(e.sample_uniform(e.legal_mask()))
    b = e.get_boards()
    ended_now = (d & 1) == 1                  # the cap (or a capture) ended these on step 40 ...
    assert ended_now.sum() >= 24 and ((d >> 2) & 7 == 4).sum() > 0
    assert not (b[:, 120] & 1).any()          # ... and each is already a fresh live game
    assert (b[:, 124] >= 1).all()             # the others ended earlier and restarted then
    assert (b[ended_now, 116] == 0).all() and (b[~ended_now, 116] > 0).all()
    assert (b[ended_now, 100:116] == 0xFF).all()
    # a fresh epoch-1 setup differs from the epoch-0 one but is reproducible
    e2 = orc.Env(32, seed=9, max_plies=40, auto_reset=1)
    for _ in range(40):
        e2.step(e2.sample_uniform(e2.legal_mask()))
    assert np.array_equal(b, e2.get_boards())
    assert not np.array_equal(b[:, :100], orc.Env(32, seed=9).get_boards()[:, :100])


def test_uniform_sampler_is_uniform_and_stream_is_batch_independent():
    e = orc.Env(4096, seed=13)
    m = e.legal_mask()
    a = e.sample_uniform(m)
    for g in range(0, 4096, 97):
        assert a[g] in W.mask_to_actions(m[g])
    # rank of the chosen action among the legal ones, for games with exactly 6 moves
    ranks = []
    for g in range(4096):
        acts = W.mask_to_actions(m[g])
        if len(acts) == 6:
            ranks.append(acts.index(int(a[g])))
    obs = np.bincount(ranks, minlength=6)
    exp = len(ranks) / 6.0
    assert len(ranks) > 300 and ((obs - exp) ** 2 / exp).sum() < 25.0
    # same game, different batch: identical draw
    e2 = orc.Env(10, seed=13, game_base=500)
    assert np.array_equal(e2.sample_uniform(e2.legal_mask()), a[500:510])


# ----------------------------------------------------------------------------- encode
def test_encode_start_position_and_partition():
    e = orc.Env(16, seed=2)
    o = e.encode_obs()
    assert set(np.unique(o)) <= {0, ONE}
    x = (o == ONE).astype(int)
    assert (x[:, :28].sum(axis=1) == 1).all()          # planes 0-27 partition the board
    for g in range(16):
        assert x[g, :12].sum() == 40                   # own pieces, by type
        assert x[g, 25].sum() == 40 and x[g, 24].sum() == 0
        assert x[g, 12:24].sum() == 0
        assert x[g, 26].sum() == 8 and x[g, 27].sum() == 12
        assert x[g, 28:].sum() == 0
        assert x[g, :12].reshape(12, 100)[:, :40].sum() == 40   # red to move: own = rows 0-3
        assert x[g, 25].reshape(100)[60:].sum() == 40
    per_type = x[:, :12].sum(axis=(2, 3))
    assert (per_type == np.array([1, 8, 5, 4, 4, 4, 3, 2, 1, 1, 1, 6])).all()


def test_encode_midgame_planes_and_history():
    e = orc.Env(64, seed=4, max_plies=1000)
    for step in range(150):
        e.step(e.sample_uniform(e.legal_mask()))
    b = e.get_boards()
    o = (e.encode_obs() == ONE).astype(int).reshape(64, 44, 100)
    assert (o[:, :28].sum(axis=1) == 1).all()
    for g in range(64):
        ply = int(b[g, 116]) | (int(b[g, 117]) << 8)
        p = ply & 1
        for c in range(100):
            v = int(b[g, c]); t = v & 15
            if t == 15:
                k = 26
            elif t == 0:
                k = 27
            elif (v >> 4) & 1 == p:
                k = t - 1
            elif v & W.REVEALED:
                k = 11 + t
            else:
                k = 24 if v & W.MOVED else 25
            assert o[g, k, c] == 1
        for j in range(8):
            f, t = int(b[g, 100 + 2 * j]), int(b[g, 101 + 2 * j])
            assert o[g, 28 + 2 * j].sum() == (f != 255) and o[g, 29 + 2 * j].sum() == (t != 255)
            if f != 255:
                assert o[g, 28 + 2 * j, f] == 1 and o[g, 29 + 2 * j, t] == 1
    assert o[:, 12:24].sum() > 0 and o[:, 24].sum() > 0


def test_encode_hand_worked_position():
    """The 44 planes of a six-piece position written out by hand from BASELINE.json configs[0] ("12 own-type
    planes, 12 revealed-opponent-type planes, 2 planes for hidden opponent pieces (moved / unmoved), 1 lake
    plane, 1 empty plane, and from/to planes for the last 8 plies"; order Spy..Marshal, Flag, Bomb: R18),
    blue to move.  Nothing here is computed: a wrong plane index, owner test or history order fails it."""
    pieces = {0: W.piece(W.FLAG, W.RED),                               # opponent, hidden, unmoved   -> plane 25
              14: W.piece(W.SCOUT, W.RED, moved=True, revealed=True),  # opponent, revealed Scout    -> plane 12 + 1
              35: W.piece(W.MAJOR, W.RED, moved=True),                 # opponent, hidden, moved     -> plane 24
              99: W.piece(W.FLAG, W.BLUE),                             # own Flag                    -> plane 10
              64: W.piece(W.MINER, W.BLUE, moved=True),                # own Miner                   -> plane 2
              77: W.piece(W.BOMB, W.BLUE, revealed=True)}              # own Bomb (own: by type only) -> plane 11
    # last plies, most recent first: red 25 -> 35, blue 74 -> 64, red 54 -> 14 (a Scout's long move)
    e = orc.Env(1)
    e.reset_from(W.make_line(pieces, ply=3, history=((25, 35), (74, 64), (54, 14)))[None])
    o = e.encode_obs()[0].reshape(44, 100)
    assert set(np.unique(o)) <= {0, ONE}
    got = {(int(p_), int(c)) for p_, c in zip(*np.nonzero(o)) if p_ not in (26, 27)}
    assert got == {(25, 0), (13, 14), (24, 35), (10, 99), (2, 64), (11, 77),
                   (28, 25), (29, 35), (30, 74), (31, 64), (32, 54), (33, 14)}
    assert sorted(np.nonzero(o[26])[0].tolist()) == [42, 43, 46, 47, 52, 53, 56, 57]          # lakes c5-d6, g5-h6
    assert sorted(np.nonzero(o[27])[0].tolist()) == sorted(set(range(100)) - {42, 43, 46, 47, 52, 53, 56, 57}
                                                           - {0, 14, 35, 99, 64, 77})     # 86 empty squares
    # the same position seen by red (ply 4): own / opponent swap, the history shifts by nothing (it is absolute)
    e.reset_from(W.make_line(pieces, ply=4, history=((25, 35), (74, 64), (54, 14)))[None])
    o = e.encode_obs()[0].reshape(44, 100)
    got = {(int(p_), int(c)) for p_, c in zip(*np.nonzero(o)) if p_ not in (26, 27)}
    assert got == {(10, 0), (1, 14), (6, 35), (25, 99), (24, 64), (23, 77),
                   (28, 25), (29, 35), (30, 74), (31, 64), (32, 54), (33, 14)}


def test_encode_is_an_information_state():
    # re-typing the opponent's unrevealed pieces must not change the observation
    e = orc.Env(8, seed=6, max_plies=1000)
    for _ in range(80):
        e.step(e.sample_uniform(e.legal_mask()))
    b = e.get_boards()
    o = e.encode_obs()
    rng = np.random.default_rng(0)
    b2 = b.copy()
    for g in range(8):
        p = (int(b[g, 116]) | (int(b[g, 117]) << 8)) & 1
        hid = [c for c in range(100) if 1 <= (b[g, c] & 15) <= 12 and ((b[g, c] >> 4) & 1) != p
               and not b[g, c] & W.REVEALED]
        types = [int(b[g, c]) & 15 for c in hid]
        rng.shuffle(types)
        for c, t in zip(hid, types):
            b2[g, c] = (b[g, c] & 0xF0) | t
    e2 = orc.Env(8)
    e2.reset_from(b2)
    assert np.array_equal(o, e2.encode_obs())


# ----------------------------------------------------------------------------- replay
def test_replay_ring_fifo_wraparound_and_uniform_sampling():
    per_slot, slots = 8, 3
    r = orc.Replay(per_slot, slots)
    e = orc.Env(5, seed=3)
    pushed = []
    for step in range(7):  # 35 records into 24 slots: wraps
        obs = e.encode_obs(); m = e.legal_mask(); a = e.sample_uniform(m)
        rew, d = e.step(a)
        r.push(obs, m, a, rew, d)
        for g in range(5):
            pushed.append((obs[g].copy(), m[g].copy(), int(a[g]), int(rew[g]), int(d[g])))
    assert r.filled == 24 and r.head == 35 % 24
    for k, rec in enumerate(pushed):
        if k < len(pushed) - 24:
            continue  # overwritten
        o, m, a, rew, d = r.read(k % 24)
        assert np.array_equal(o, rec[0]) and np.array_equal(m, rec[1]) and (a, rew, d) == rec[2:]
    obs, m, a, rew, d, idx = r.sample(seed=77, draw_index=5, batch=4096)
    assert idx.min() >= 0 and idx.max() < 24
    cnt = np.bincount(idx, minlength=24)
    assert ((cnt - 4096 / 24) ** 2 / (4096 / 24)).sum() < 60.0
    for j in (0, 1, 2, 3, 4, 777, 4095):
        o2, m2, a2, r2, d2 = r.read(int(idx[j]))
        assert np.array_equal(obs[j], o2) and np.array_equal(m[j], m2) and (a[j], rew[j], d[j]) == (a2, r2, d2)
    # element j depends only on (seed, draw_index, j); a different draw_index differs
    *_, idx_small = r.sample(seed=77, draw_index=5, batch=10)
    assert np.array_equal(idx_small, idx[:10])
    *_, idx_other = r.sample(seed=77, draw_index=6, batch=4096)
    assert not np.array_equal(idx_other, idx)
    # before wrap-around only the filled prefix is sampled
    r2 = orc.Replay(8, 3)
    r2.push(obs[:5], m[:5], a[:5], rew[:5], d[:5])
    *_, idx2 = r2.sample(seed=1, draw_index=0, batch=500)
    assert idx2.max() < 5 and len(set(idx2.tolist())) == 5


# ----------------------------------------------------------------------------- determinise
def test_determinise_properties_and_rollout_reduce():
    roots = orc.Env(4, seed=8, max_plies=1000, auto_reset=1)
    for _ in range(120):
        roots.step(roots.sample_uniform(roots.legal_mask()))
    rb = roots.get_boards()
    S = 64
    out = orc.Env(4 * S, seed=8)
    att = orc.determinise(roots, S, seed=99, out=out)
    assert att.min() >= 1
    ob = out.get_boards()
    robs = roots.encode_obs()
    oobs = out.encode_obs()
    differs = 0
    for r in range(4):
        p = (int(rb[r, 116]) | (int(rb[r, 117]) << 8)) & 1
        for s in range(S):
            L = ob[r * S + s]
            assert np.array_equal(L[100:], rb[r, 100:])                   # meta copied
            assert (_counts(L) == _counts(rb[r])).all()                    # multiset preserved
            for c in range(100):
                v0, v1 = int(rb[r, c]), int(L[c])
                assert (v0 & 0xF0) == (v1 & 0xF0)                          # flags kept per cell
                own_or_revealed = not (1 <= (v0 & 15) <= 12) or ((v0 >> 4) & 1) == p or v0 & W.REVEALED
                if own_or_revealed:
                    assert v0 == v1
                elif v1 & W.MOVED:
                    assert (v1 & 15) not in (W.FLAG, W.BOMB)               # the constraint
            assert np.array_equal(oobs[r * S + s], robs[r])                # same information state
            differs += not np.array_equal(L[:100], rb[r, :100])
    assert differs > 3 * S  # almost every sample re-types something
    # determinism and per-game keying
    out2 = orc.Env(4 * S, seed=8)
    orc.determinise(roots, S, seed=99, out=out2)
    assert np.array_equal(ob, out2.get_boards())
    # rollouts + reduction
    side = np.array([(int(rb[r, 116]) | (int(rb[r, 117]) << 8)) & 1 for r in range(4)], np.uint8)
    for _ in range(64):
        out.step(out.sample_uniform(out.legal_mask()))
    red = orc.reduce_returns(out, side, S)
    fb = out.get_boards()
    for r in range(4):
        res = fb[r * S:(r + 1) * S, 121].view(np.int8).astype(int) * (fb[r * S:(r + 1) * S, 120] & 1)
        ret = res * (1 if side[r] == 0 else -1)
        assert red[r].tolist() == [ret.sum(), (ret > 0).sum(), (ret < 0).sum()]


def test_determinise_is_uniform_over_consistent_arrangements():
    # Small hand-built root: blue hides Flag, Bomb, Spy, Scout on 4 squares of which one has
    # moved.  Consistent arrangements: Flag and Bomb on two of the three unmoved squares
    # (3*2 = 6 ordered ways) x 2 orders of {Spy, Scout} on the rest = 12, each with p = 1/12.
    pieces = {0: W.piece(W.FLAG, 0), 11: W.piece(W.MARSHAL, 0),
              88: W.piece(W.FLAG, 1), 89: W.piece(W.BOMB, 1), 78: W.piece(W.SPY, 1),
              68: W.piece(W.SCOUT, 1, moved=True), 99: W.piece(W.MINER, 1, revealed=True)}
    root = orc.Env(1)
    root.reset_from(W.make_line(pieces, ply=10)[None])
    S = 12000
    out = orc.Env(S)
    draws = orc.determinise(root, S, seed=5, out=out)
    b = out.get_boards()
    hid = [68, 78, 88, 89]
    keys = {}
    for s in range(S):
        t = tuple(int(b[s, c]) & 15 for c in hid)
        keys[t] = keys.get(t, 0) + 1
        assert (b[s, 68] & 15) in (W.SPY, W.SCOUT)            # the moved piece is never Bomb/Flag
        assert b[s, 99] == pieces[99] and b[s, 11] == pieces[11]
    assert len(keys) == 12
    exp = S / 12.0
    chi2 = sum((v - exp) ** 2 / exp for v in keys.values())
    assert chi2 < 40.0, chi2  # 11 dof
    assert draws.min() >= 3 and draws.max() < 60


def test_pinned_reset_restarts_from_the_pinned_state():
    """terminated boards restart from a custom non-initial state.  Pin: the restarted
    game IS the pinned line (cells, history, counters), only the epoch keeps counting."""
    o = orc.Env(40, seed=2, max_plies=26, auto_reset=1)
    for _ in range(12):
        o.step(o.sample_uniform(o.legal_mask()))
    pin = o.get_boards()
    o.pin_reset_state(pin)
    seen = 0
    for t in range(40):
        r, d = o.step(o.sample_uniform(o.legal_mask()))
        b = o.get_boards()
        for i in np.nonzero(d & 1)[0]:
            expect = pin[i].copy()
            expect[124:128] = b[i, 124:128]          # epoch of the slot
            assert np.array_equal(b[i], expect)
            assert int(b[i, 124]) >= 1
            seen += 1
    assert seen >= 80  # 14 plies per round: every game restarted at least twice
    o.pin_reset_state(None)
    for t in range(20):
        r, d = o.step(o.sample_uniform(o.legal_mask()))
        b = o.get_boards()
        for i in np.nonzero(d & 1)[0]:
            assert b[i, 116] == 0 and b[i, 117] == 0  # a fresh setup again


def _random_pool(K, seed):
    """K classic setups per side: random permutations of the 40-piece multiset (test input only)."""
    rng = np.random.default_rng(seed)
    base = np.array(orc.multiset(0), np.uint8)
    pool = np.stack([np.stack([rng.permutation(base) for _ in range(K)]) for _ in range(2)])
    for side in range(2):                      # keep every setup mobile: a Scout on a front lane square
        for k in range(K):
            front = 34 if side == 0 else 5     # red's row 3 / blue's row 6 (cell 60+5), files e
            j = int(np.nonzero(pool[side, k] == 2)[0][0])
            pool[side, k, [front, j]] = pool[side, k, [j, front]]
    return pool


def test_setup_pool_deals_pool_entries_uniformly_and_independently():
    """P:234 / R#30: with a pool, every fresh side is one of the pool's setups, chosen uniformly
    and independently for the two sides."""
    K, n = 7, 4000
    pool = _random_pool(K, 1)
    e = orc.Env(n, seed=3, max_plies=4, auto_reset=1)
    e.set_setup_pool(pool)
    e.reset(3)
    counts = np.zeros((2, K), int)
    joint = np.zeros((K, K), int)
    for step in range(13):                     # epoch 0, then the auto-resets of the 4-ply cap (and earlier endings)
        b = e.get_boards()
        fresh = np.nonzero((b[:, 116] == 0) & (b[:, 117] == 0))[0]
        red = b[:, 0:40] & 15
        blue = b[:, 60:100] & 15
        for g in fresh:
            x = int(np.nonzero((pool[0] == red[g]).all(axis=1))[0][0])      # IndexError if the side is no pool entry
            y = int(np.nonzero((pool[1] == blue[g]).all(axis=1))[0][0])
            assert ((b[g, 60:100] >> 4) & 1).all() and not ((b[g, 0:40] >> 4) & 1).any()
            counts[0, x] += 1; counts[1, y] += 1; joint[x, y] += 1
        e.step(e.sample_uniform(e.legal_mask()))
    total = int(joint.sum())
    assert total >= 3 * n
    for side in range(2):
        chi2 = ((counts[side] - total / K) ** 2 / (total / K)).sum()
        assert chi2 < 30, (side, counts[side])                       # 6 dof
    chi2 = ((joint - total / K / K) ** 2 / (total / K / K)).sum()
    assert chi2 < 100, joint                                         # 48 dof: independence of the two sides
    e.set_setup_pool(None)
    e.reset(3)
    plain = orc.Env(n, seed=3)
    assert np.array_equal(e.get_boards(), plain.get_boards())        # uniform permutations again
    bad = pool.copy(); bad[1, 2, 7] = 13
    with pytest.raises(RuntimeError):
        e.set_setup_pool(bad)
    stuck = pool.copy()
    stuck[0, 0] = 0; stuck[0, 0, :8] = [11, 12, 12, 12, 12, 12, 12, 0]  # immovables only: cannot ever move
    with pytest.raises(RuntimeError):
        e.set_setup_pool(stuck)
