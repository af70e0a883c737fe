"""The per-game device logic (csrc/strat_game.cuh: setup, legal mask, both samplers, step with
battle / terminal tests / auto-reset, chasing rule, observation bits) compiled for the HOST
(tests/host_harness.cpp on top of tests/host_shim.h) and compared with the oracle - so that the CPU-only
test run already checks the rules the kernels execute, thread per game.  The kernels themselves
(staging, warp-cooperative paths, overlap) are covered by the `-m gpu` tests."""
import ctypes as C
import json
import os
import subprocess

import numpy as np
import pytest

from chase_scenarios import cage, crowded
from oracle import orc
from paper_2511_07312_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def hh(tmp_path_factory):
    lib = str(tmp_path_factory.mktemp("hh") / "libhh.so")
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-shared", "-fPIC", "-o", lib, os.path.join(HERE, "host_harness.cpp")])
    L = C.CDLL(lib)
    vp = C.c_void_p
    L.hh_reset.argtypes = [C.c_int, C.c_uint64, C.c_uint32, vp]
    L.hh_legal_mask.argtypes = [vp, C.c_int, C.c_int, vp]
    L.hh_pick.argtypes = [vp, C.c_int, C.c_int, C.c_uint32, C.POINTER(C.c_int)]
    L.hh_step.argtypes = [vp, C.c_int, C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp,
                          C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.hh_encode.argtypes = [vp, vp]
    L.hh_track_start.argtypes = [vp, vp]
    L.hh_track_step.argtypes = [vp, vp, C.c_int, C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_int, vp, C.POINTER(C.c_int)]
    return L


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _mask(hh, line, two_square=1, chase=0):
    row = np.zeros(113, np.uint32)
    hh.hh_legal_mask(_p(line), two_square, chase, _p(row))
    return row


@pytest.mark.parametrize("variant,seed", [(0, 0), (1, 9)])
def test_setup_on_host_equals_oracle(hh, variant, seed, golden_dir):
    o = orc.Env(300, variant=variant, seed=seed)
    b = o.get_boards()
    line = np.zeros(128, np.uint8)
    for g in range(300):
        hh.hh_reset(variant, seed, g, _p(line))
        assert np.array_equal(line, b[g]), g
    if variant == 0 and seed == 0:  # the redraw path (R5)
        for g in json.load(open(os.path.join(golden_dir, "setup_redraw_cases.json")))["epoch0"]:
            hh.hh_reset(0, 0, g, _p(line))
            assert np.array_equal(line, orc.Env(1, seed=0, game_base=g).get_boards()[0]), g


@pytest.mark.parametrize("variant,cap,chase", [(0, 120, 0), (1, 400, 0), (0, 150, 1)])
def test_play_on_host_equals_oracle(hh, variant, cap, chase):
    n, seed = 48, 12
    kw = dict(variant=variant, seed=seed, max_plies=cap, auto_reset=1, chase_rule=chase)
    o = orc.Env(n, **kw)
    line_out = np.zeros(128, np.uint8)
    obs = np.zeros(4400, np.uint16)
    rew, done, ill, mf = C.c_int(), C.c_int(), C.c_int(), C.c_int()
    for t in range(260):
        b = o.get_boards()
        om = o.legal_mask()
        oa = o.sample_uniform(om)
        oobs = o.encode_obs().reshape(n, -1) if t % 8 == 0 else None
        for g in range(n):
            line = b[g]
            assert np.array_equal(_mask(hh, line, 1, chase), om[g]), (t, g)
            ply = int(line[116]) | (int(line[117]) << 8)
            epoch = int(line[124]) | (int(line[125]) << 8)
            u = int(orc.philox([g, epoch, ply, 2], [seed, 0])[0])  # the ACTION stream's draw (layout R3)
            a = hh.hh_pick(_p(line), 1, chase, u, C.byref(mf))
            assert a == int(oa[g]) and (chase or mf.value == a), (t, g, a, mf.value, int(oa[g]))
            if oobs is not None:
                hh.hh_encode(_p(line), _p(obs))
                assert np.array_equal(obs, oobs[g]), (t, g)
        orr, od = o.step(oa)
        nb = o.get_boards()
        for g in range(n):
            hh.hh_step(_p(b[g]), variant, seed, g, cap, 1, 1, chase, int(oa[g]), _p(line_out), C.byref(rew), C.byref(done), C.byref(ill))
            assert ill.value == 0 and rew.value == int(orr[g]) and done.value == int(od[g]), (t, g)
            assert np.array_equal(line_out, nb[g]), (t, g)
        if chase:
            o.reset_from(nb)  # the host harness keeps no move log: judge the chase with the line's 8 plies on both sides
    assert (o.get_boards()[:, 124] > 0).any()  # games were re-dealt inside steps (auto-reset path)


def test_chasing_rule_on_host_equals_oracle_on_arbitrary_lines(hh):
    """Random little positions with arbitrary (plausible) histories and chase ages: the XOR-diff
    ban enumeration of the device code against the oracle's candidate-by-candidate memcmp."""
    rng = np.random.default_rng(11)
    n = 3000
    free = [c for c in range(100) if c not in W.LAKES]
    lines = np.zeros((n, 128), np.uint8)
    for i in range(n):
        k = int(rng.integers(4, 14))
        cells = rng.choice(free, k, replace=False)
        pieces = {int(cells[0]): W.piece(W.FLAG, 0), int(cells[1]): W.piece(W.FLAG, 1)}
        for c in cells[2:]:
            pieces[int(c)] = W.piece(int(rng.integers(1, 11)), int(rng.integers(2)), moved=True)
        occ = [int(c) for c in cells[2:]]
        hist = []
        for j in range(8):
            if rng.random() < 0.1:
                hist.append((0xFF, 0xFF))
                continue
            t = occ[int(rng.integers(len(occ)))] if rng.random() < 0.7 else int(free[int(rng.integers(92))])
            cand = [t + d for d in (10, -10, 1, -1)
                    if 0 <= t + d < 100 and abs((t + d) // 10 - t // 10) + abs((t + d) % 10 - t % 10) == 1 and (t + d) not in W.LAKES]
            hist.append((int(cand[int(rng.integers(len(cand)))]), t))
        line = W.make_line(pieces, ply=int(rng.integers(8, 60)), history=hist)
        line[122], line[123] = int(rng.integers(0, 10)), int(rng.integers(0, 10))
        lines[i] = line
    o = orc.Env(n, seed=1, chase_rule=1)
    o.reset_from(lines)
    om = o.legal_mask()
    stripped = lines.copy(); stripped[:, 122:124] = 0
    o0 = orc.Env(n, seed=1)
    o0.reset_from(stripped)
    assert (o0.legal_mask() != om).any(axis=1).sum() > 50  # the rule does ban moves in these positions
    for i in range(n):
        assert np.array_equal(_mask(hh, lines[i], 1, 1), om[i]), i


def test_caged_chases_on_host(hh):
    """Bomb cages (positions recur all the time): masks with the chasing rule, line memory only."""
    rng = np.random.default_rng(3)
    bans = 0
    for game in range(150):
        o = orc.Env(1, chase_rule=1)
        o.reset_from(W.make_line(cage(rng) if game % 5 else crowded(rng))[None, :])
        for ply in range(40):
            b = o.get_boards()
            if b[0, 120] & 1:
                break
            o.reset_from(b)  # line memory (8 plies) on both sides
            om = o.legal_mask()[0]
            assert np.array_equal(_mask(hh, b[0], 1, 1), om), (game, ply)
            bans += int(np.unpackbits((_mask(hh, b[0], 1, 0) ^ om).view(np.uint8)).sum())
            legal = W.mask_to_actions(om)
            if not legal:
                break
            quiet = [a for a in legal if b[0, a // 36 + (a % 9 + 1) * (10, 1, -10, -1)[(a % 36) // 9]] == 0]
            pool = quiet if quiet and rng.random() < 0.9 else legal
            o.step(np.array([pool[rng.integers(len(pool))]], np.int16))
    assert bans > 0


def _channels_from_tracker_block(line, trk):
    """The tracker-derived channels of the 487-channel information state (43-486 except nothing
    else) decoded from a game's tracker block by its documented layout (csrc/strat_game.cuh
    "S2 trackers"): {(channel, square): +1 / -1}.  Test-side restatement of the LAYOUT only."""
    side = (int(line[116]) | (int(line[117]) << 8)) & 1
    ply = int(line[116]) | (int(line[117]) << 8)
    out = {}
    for c in range(100):
        b = int(line[c])
        if (b & 15) in (0, 15):
            continue
        own = ((b >> 4) & 1) == side
        r0, r1, r2, r3 = (int(x) for x in trk[4 * c:4 * c + 4])
        a, p = (43, 251) if own else (76, 303)
        for j in range(22):
            if (r0 >> j) & 1:
                out[(a + j, c)] = 1
        for j in range(11):
            if (r1 >> j) & 1:
                out[(a + 22 + j, c)] = 1
        for j in range(13):
            if (r1 >> (11 + j)) & 1:
                out[(p + j, c)] = 1
            if (r2 >> j) & 1:
                out[(p + 13 + j, c)] = 1
            if (r2 >> (13 + j)) & 1:
                out[(p + 26 + j, c)] = 1
            if (r3 >> j) & 1:
                out[(p + 39 + j, c)] = 1
        out[(355 + ((r0 >> 22) & 127), c)] = 1
    for k in range(int(trk[400])):
        e = int(trk[401 + k])
        start, t, owner, sq, cause = e & 127, (e >> 7) & 15, (e >> 11) & 1, (e >> 12) & 127, (e >> 19) & 7
        j = t - 1 if t <= 10 else 10 if t == 12 else -1
        if j >= 0:
            out[((109 if owner == side else 120) + j, start)] = 1
        if cause:
            out[((131 if owner == side else 191) + 10 * (cause - 1) + t - 1, sq)] = 1
    for j in range(32):
        slot = (ply - 1 - j) & 31
        e = (int(trk[493 + (slot >> 1)]) >> (16 * (slot & 1))) & 0xFFFF
        if e != 0x3FFF:
            out[(455 + j, e >> 7)] = 1
            out[(455 + j, e & 127)] = -1
    return out


@pytest.mark.parametrize("variant,cap", [(0, 160), (1, 300)])
def test_information_state_trackers_on_host_equal_oracle(hh, variant, cap):
    """The per-ply tracker update of the device code (track_ply: threats, evasions, active
    adjacency, protections, captures and causes of death, start squares, move ring) against the
    oracle's 487-channel information state, game by game, every few plies, across auto-resets."""
    n, seed = 24, 5
    kw = dict(variant=variant, seed=seed, max_plies=cap, auto_reset=1, infostate=1)
    o = orc.Env(n, **kw)
    trk = np.zeros((n, 512), np.uint32)
    b = o.get_boards()
    for g in range(n):
        hh.hh_track_start(_p(b[g]), _p(trk[g]))
    line_out = np.zeros(128, np.uint8)
    ill = C.c_int()
    seen = set()
    for t in range(420):
        b = o.get_boards()
        oa = o.sample_uniform(o.legal_mask())
        o.step(oa)
        nb = o.get_boards()
        for g in range(n):
            hh.hh_track_step(_p(b[g]), _p(trk[g]), variant, seed, g, cap, 1, int(oa[g]), _p(line_out), C.byref(ill))
            assert ill.value == 0 and np.array_equal(line_out, nb[g]), (t, g)
        if t % 7 == 6 or t < 12:
            obs = o.encode_infostate().reshape(n, 487, 100)
            for g in range(n):
                want = {}
                ch, sq = np.nonzero(obs[g, 43:])
                for c_, s_ in zip(ch, sq):
                    v = int(obs[g, 43 + c_, s_])
                    want[(int(c_) + 43, int(s_))] = 1 if v == 0x3F80 else -1 if v == 0xBF80 else v
                got = _channels_from_tracker_block(nb[g], trk[g])
                assert got == want, (t, g, sorted(set(got.items()) ^ set(want.items()))[:8])
                seen.update(c_ for c_, _ in got)
    groups = [(43, 54), (54, 65), (65, 76), (109, 131), (131, 251), (251, 264), (264, 277), (277, 290), (290, 303)]
    for lo, hi in groups:  # every channel group was exercised
        assert any(lo <= c_ < hi for c_ in seen), (lo, hi)
    assert (o.get_boards()[:, 124] > 0).any()
