"""Pins of the oracle's 487-channel information state against what the
paper's text fixes: hand-built mini-games whose channels are worked out by hand from the
definitions (threat P:515, evasion P:522, active adjacency P:529, protection P:572, captured
pieces P:551-552, the six causes of death P:556-562, start squares P:606, moves P:610),
channel sums fixed by the piece counts, the information-state property, and channels 12-35
(reading I7) by exhaustive enumeration, by hand and against the empirical
marginals of the determinisation sampler (an independent function of the oracle)."""
import itertools
from fractions import Fraction

import numpy as np

from oracle import orc
from paper_2511_07312_b200 import workloads as W

ONE, MINUS_ONE = 0x3F80, 0xBF80
N, E, S, Wd = 0, 1, 2, 3  # directions: +row, +col, -row, -col


def _env(pieces, ply=0, history=(), battleless=0, **kw):
    e = orc.Env(1, infostate=1, **kw)
    e.reset_from(W.make_line(pieces, ply=ply, history=history, battleless=battleless)[None])
    return e


def _play(e, moves):
    for frm, d, dist in moves:
        r, dn = e.step(np.array([W.action_index(frm, d, dist)], np.int16))
        assert e.check() == 0, (frm, d, dist)
    return e.encode_infostate()[0].reshape(487, 100)


def _nonzero(obs, lo, hi):
    """{(channel, square): value} of the non-zero entries of channels lo..hi-1."""
    ch, sq = np.nonzero(obs[lo:hi])
    return {(int(c) + lo, int(s)): int(obs[c + lo, s]) for c, s in zip(ch, sq)}


def bf16_exact(fr):
    """Round-to-nearest-even bf16 of an exact rational (independent of the oracle's routine)."""
    fr = Fraction(fr)
    if fr == 0:
        return 0
    sign = 0x8000 if fr < 0 else 0
    fr = abs(fr)
    e = 0
    while fr >= 2:
        fr /= 2; e += 1
    while fr < 1:
        fr *= 2; e -= 1
    scaled = fr * 128  # in [128, 256)
    q = int(scaled)
    rem = scaled - q
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and q % 2 == 1):
        q += 1
    if q == 256:
        q, e = 128, e + 1
    return sign | ((e + 127) << 7) | (q - 128)


def test_bf16_of_ratio_known_values_and_exact_rationals():
    known = {(1, 2): 0x3F00, (1, 4): 0x3E80, (1, 3): 0x3EAB, (1, 1): 0x3F80, (3, 8): 0x3EC0, (2, 3): 0x3F2B,
             (100, 4000): 0x3CCD, (0, 7): 0}
    for (a, b), v in known.items():
        assert orc.bf16_of_ratio(a, b) == v, (a, b)
    for a in range(0, 41):
        for b in range(1, 41):
            assert orc.bf16_of_ratio(a, b) == bf16_exact(Fraction(a, b)), (a, b)
    for a, b in [(1, 65535), (999, 1000), (65534, 65535), (37, 1600), (199, 200)]:
        assert orc.bf16_of_ratio(a, b) == bf16_exact(Fraction(a, b))


# ------------------------------------------------------------------ hand-built mini-games
def test_threat_evasion_and_declined_attack():
    """Red Sergeant 24->34 lands next to the hidden blue Captain on 35 (a threat); the Captain
    could take it (it is adjacent and the capture is legal) but steps away to 36 instead: an
    evasion and an active adjacency, both keyed 'hidden' (the Sergeant is unrevealed)."""
    pieces = {0: W.piece(W.FLAG, 0), 99: W.piece(W.FLAG, 1), 24: W.piece(W.SERGEANT, 0), 35: W.piece(W.CAPTAIN, 1)}
    e = _env(pieces)
    obs = _play(e, [(24, N, 1)])
    # blue to move: the Sergeant is the OPPONENT's piece -> channels 76-108; threat of a hidden piece = 86
    assert _nonzero(obs, 43, 109) == {(86, 34): ONE}
    obs = _play(e, [(35, E, 1)])
    # red to move: own Sergeant on 34 has threatened a hidden piece (53); the opponent's Captain on 36 has
    # evaded a hidden piece (97) and has been actively adjacent to a hidden piece (108)
    assert _nonzero(obs, 43, 109) == {(53, 34): ONE, (97, 36): ONE, (108, 36): ONE}
    assert _nonzero(obs, 251, 355) == {}  # no protection took place
    # start squares and the two moves, most recent first
    assert _nonzero(obs, 355, 455) == {(355 + 24, 34): ONE, (355 + 35, 36): ONE, (355 + 0, 0): ONE, (355 + 99, 99): ONE}
    assert _nonzero(obs, 455, 487) == {(455, 36): ONE, (455, 35): MINUS_ONE, (456, 34): ONE, (456, 24): MINUS_ONE}


def test_revealed_types_key_the_threat_channels_and_a_capture_is_no_threat():
    """The same shape with revealed pieces: the keys are the types.  A move that
    captures is a battle, not a threat (reading I1): it sets no threat bit."""
    pieces = {0: W.piece(W.FLAG, 0), 99: W.piece(W.FLAG, 1), 24: W.piece(W.GENERAL, 0, revealed=True),
              35: W.piece(W.MINER, 1, revealed=True), 44: W.piece(W.SCOUT, 1)}
    e = _env(pieces)
    obs = _play(e, [(24, N, 1), (35, E, 1)])
    # own General: threatened a revealed Miner (43+2) and a hidden piece on 44 (53)
    # opponent's Miner: evaded a revealed General (87+8), was actively adjacent to it (98+8);
    # the Scout on 44 was also adjacent to the General and did not take it (98+8 on 44)
    assert _nonzero(obs, 43, 109) == {(45, 34): ONE, (53, 34): ONE, (95, 36): ONE, (106, 36): ONE, (106, 44): ONE}
    obs = _play(e, [(34, N, 1)])  # General takes the Scout on 44: now next to nothing new, and no threat recorded
    # blue to move: own = blue.  The Miner's evasion / adjacency are now "own" channels (54+8, 65+8); the
    # captured Scout's record left the board with it ...
    assert _nonzero(obs, 43, 76) == {(62, 36): ONE, (73, 36): ONE}
    # ... and the General, now on 44, keeps exactly its two earlier threats: the capture added none
    assert _nonzero(obs, 76, 109) == {(78, 44): ONE, (86, 44): ONE}


def test_protection_of_a_piece():
    """Red Major (revealed) 24->34 threatens the revealed blue Miner on 35; blue answers 26->36 with a
    hidden Captain, which becomes adjacent to the Miner: the Captain protected the Miner against
    the Major.  Four records: protector (what it protected, against what) and protected
    (by what, against what)."""
    pieces = {0: W.piece(W.FLAG, 0), 99: W.piece(W.FLAG, 1), 24: W.piece(W.MAJOR, 0, revealed=True),
              35: W.piece(W.MINER, 1, revealed=True), 26: W.piece(W.CAPTAIN, 1)}
    e = _env(pieces)
    obs = _play(e, [(24, N, 1), (26, N, 1)])
    # red to move: blue is the opponent -> 303-354.  Captain on 36: protected a revealed Miner (303+2),
    # against a revealed Major (303+13+6).  Miner on 35: protected by a hidden piece (303+26+12),
    # against a revealed Major (303+39+6).
    assert _nonzero(obs, 251, 355) == {(305, 36): ONE, (322, 36): ONE, (341, 35): ONE, (348, 35): ONE}
    # the Major threatened a revealed Miner (43+2); the Miner declined to take the Major (98+6)
    assert _nonzero(obs, 43, 109) == {(45, 34): ONE, (104, 35): ONE}
    # one ply later the same records read from blue's side: 251-302
    obs = _play(e, [(34, S, 1)])
    assert _nonzero(obs, 251, 355) == {(253, 36): ONE, (270, 36): ONE, (289, 35): ONE, (296, 35): ONE}


def test_protection_of_an_empty_square_and_no_protection_without_adjacency():
    """P:572 'We extend the same terminology to the case in which B is an empty square': red moves to 34;
    blue's Captain 26->36 now shares the empty neighbour 35 with it: protected an empty square (262/314)
    against a hidden piece (276/328).  A reply far away records nothing."""
    pieces = {0: W.piece(W.FLAG, 0), 99: W.piece(W.FLAG, 1), 24: W.piece(W.MAJOR, 0), 26: W.piece(W.CAPTAIN, 1),
              81: W.piece(W.SERGEANT, 1)}
    e = _env(pieces)
    obs = _play(e, [(24, N, 1), (26, N, 1)])
    assert _nonzero(obs, 251, 355) == {(303 + 11, 36): ONE, (303 + 13 + 12, 36): ONE}
    e = _env(pieces)
    obs = _play(e, [(24, N, 1), (81, E, 1)])
    assert _nonzero(obs, 251, 355) == {}
    assert _nonzero(obs, 43, 109) == {}


def test_six_causes_of_death_and_captures_by_start_square():
    """One battle per ply, far apart.  Expected channels by hand; 131-190 own, 191-250
    opponent, offset 10*(cause-1) + type-1; captured 109-119 own / 120-130 opponent by START square."""
    R, B = 0, 1
    pieces = {
        0: W.piece(W.FLAG, R), 99: W.piece(W.FLAG, B),
        10: W.piece(W.SERGEANT, R), 20: W.piece(W.CAPTAIN, B, revealed=True),        # ply 0: cause 1 (red)
        72: W.piece(W.LIEUTENANT, B), 62: W.piece(W.LIEUTENANT, R, revealed=True),   # ply 1: cause 2 (blue), 5 (red)
        14: W.piece(W.MAJOR, R), 24: W.piece(W.COLONEL, B),                          # ply 2: cause 3 (red)
        76: W.piece(W.GENERAL, B), 66: W.piece(W.CAPTAIN, R, revealed=True),         # ply 3: cause 4 (red)
        18: W.piece(W.MARSHAL, R), 28: W.piece(W.SCOUT, B),                          # ply 4: cause 6 (blue)
        79: W.piece(W.MINER, B), 69: W.piece(W.BOMB, R),                             # ply 5: a Bomb is captured
    }
    e = _env(pieces)
    obs = _play(e, [(10, N, 1), (72, S, 1), (14, N, 1), (76, S, 1), (18, N, 1), (79, S, 1)])
    # red to move: own = red
    assert _nonzero(obs, 131, 191) == {(131 + 0 + 3, 20): ONE, (131 + 40 + 4, 62): ONE, (131 + 20 + 6, 24): ONE,
                                       (131 + 30 + 5, 66): ONE}
    assert _nonzero(obs, 191, 251) == {(191 + 10 + 4, 62): ONE, (191 + 50 + 1, 28): ONE}
    assert _nonzero(obs, 109, 120) == {(109 + 3, 10): ONE, (109 + 4, 62): ONE, (109 + 6, 14): ONE, (109 + 5, 66): ONE,
                                       (109 + 10, 69): ONE}
    assert _nonzero(obs, 120, 131) == {(120 + 4, 72): ONE, (120 + 1, 28): ONE}
    # survivors carry their start squares: the blue Captain never moved, the blue Colonel neither, the
    # General went 76->66, the Marshal 18->28, the Miner 79->69
    ss = _nonzero(obs, 355, 455)
    assert ss == {(355 + 0, 0): ONE, (355 + 99, 99): ONE, (355 + 20, 20): ONE, (355 + 24, 24): ONE,
                  (355 + 76, 66): ONE, (355 + 18, 28): ONE, (355 + 79, 69): ONE}
    # a tie against an UNREVEALED piece: attacker cause 3, defender cause 6
    e = _env({0: W.piece(W.FLAG, R), 99: W.piece(W.FLAG, B), 10: W.piece(W.MINER, R), 20: W.piece(W.MINER, B),
              50: W.piece(W.SPY, R), 59: W.piece(W.SPY, B)})
    obs = _play(e, [(10, N, 1)])  # blue to move: own = blue
    assert _nonzero(obs, 131, 251) == {(131 + 50 + 2, 20): ONE, (191 + 20 + 2, 20): ONE}


def test_basic_channels_fractions_and_lake_cells():
    pieces = {0: W.piece(W.FLAG, 0), 99: W.piece(W.FLAG, 1), 24: W.piece(W.MAJOR, 0, moved=True),
              35: W.piece(W.MINER, 1, revealed=True, moved=True), 26: W.piece(W.CAPTAIN, 1)}
    e = _env(pieces, ply=100, battleless=30, max_plies=4000, max_battleless=200)
    obs = e.encode_infostate()[0].reshape(487, 100)  # ply 100: red to move
    assert _nonzero(obs, 0, 12) == {(W.FLAG - 1, 0): ONE, (W.MAJOR - 1, 24): ONE}
    assert _nonzero(obs, 36, 41) == {(36, 0): ONE, (36, 24): ONE, (37, 99): ONE, (37, 26): ONE, (39, 24): ONE, (40, 35): ONE,
                                     **{(38, s): ONE for s in range(100) if s not in pieces and s not in W.LAKES}}
    assert (obs[41] == bf16_exact(Fraction(100, 4000))).all() and (obs[42] == bf16_exact(Fraction(30, 200))).all()
    # P:616 "n moves without a battle was represented as n/100 during training, but n/200 during testing"
    e2 = _env(pieces, ply=100, battleless=30, max_plies=4000, max_battleless=100)
    assert (e2.encode_infostate()[0].reshape(487, 100)[42] == bf16_exact(Fraction(30, 100))).all()
    e3 = _env(pieces, ply=100, battleless=30)  # no caps: the hard ply cap 65535 (R25); k-move rule off -> 0
    o3 = e3.encode_infostate()[0].reshape(487, 100)
    assert (o3[41] == bf16_exact(Fraction(100, 65535))).all() and not o3[42].any()


# ------------------------------------------------------------------ channels 12-35
def _posterior_by_enumeration(hidden):
    """hidden = [(square, type, moved)].  Exact marginals of the uniform distribution over the
    arrangements of the types on the squares with no Bomb/Flag on a moved square."""
    sq = [h[0] for h in hidden]
    types = [h[1] for h in hidden]
    moved = {h[0]: h[2] for h in hidden}
    count, total = {}, 0
    for perm in set(itertools.permutations(types)):
        if any(t in (W.FLAG, W.BOMB) and moved[s] for s, t in zip(sq, perm)):
            continue
        total += 1
        for s, t in zip(sq, perm):
            count[(s, t)] = count.get((s, t), 0) + 1
    return {k: Fraction(v, total) for k, v in count.items()}


def test_type_posterior_by_hand_and_by_exhaustive_enumeration():
    R, B = 0, 1
    # by hand: hidden blue = {Bomb@70, Scout@71 (both unmoved), Miner@55 (moved)}: 4 consistent arrangements;
    # unmoved square: Bomb 1/2, Scout 1/4, Miner 1/4; moved square: Scout 1/2, Miner 1/2.
    pieces = {0: W.piece(W.FLAG, R), 5: W.piece(W.SERGEANT, R), 99: W.piece(W.FLAG, B, revealed=True),
              70: W.piece(W.BOMB, B), 71: W.piece(W.SCOUT, B), 55: W.piece(W.MINER, B, moved=True)}
    obs = _env(pieces).encode_infostate()[0].reshape(487, 100)
    half, quarter = 0x3F00, 0x3E80
    assert _nonzero(obs, 12, 24) == {
        (12 + W.FLAG - 1, 99): ONE,
        (12 + W.BOMB - 1, 70): half, (12 + W.SCOUT - 1, 70): quarter, (12 + W.MINER - 1, 70): quarter,
        (12 + W.BOMB - 1, 71): half, (12 + W.SCOUT - 1, 71): quarter, (12 + W.MINER - 1, 71): quarter,
        (12 + W.SCOUT - 1, 55): half, (12 + W.MINER - 1, 55): half}
    # channels 24-35: red's own two hidden pieces as blue sees them: Flag/Sergeant on two unmoved squares
    assert _nonzero(obs, 24, 36) == {(24 + W.FLAG - 1, 0): half, (24 + W.SERGEANT - 1, 0): half,
                                     (24 + W.FLAG - 1, 5): half, (24 + W.SERGEANT - 1, 5): half}
    # exhaustive enumeration on a larger hand-built case (7 hidden pieces, 3 of them moved)
    hidden = [(60, W.BOMB, False), (61, W.BOMB, False), (62, W.FLAG, False), (63, W.SCOUT, False), (54, W.SCOUT, True),
              (45, W.MARSHAL, True), (44, W.SPY, True)]
    pieces = {0: W.piece(W.FLAG, R), 5: W.piece(W.SERGEANT, R), 80: W.piece(W.COLONEL, B, revealed=True)}
    for s, t, mv in hidden:
        pieces[s] = W.piece(t, B, moved=mv)
    obs = _env(pieces).encode_infostate()[0].reshape(487, 100)
    exact = _posterior_by_enumeration(hidden)
    want = {(12 + t - 1, s): bf16_exact(v) for (s, t), v in exact.items()}
    want[(12 + W.COLONEL - 1, 80)] = ONE
    assert _nonzero(obs, 12, 24) == want


def test_type_posterior_matches_the_determinisation_sampler():
    """Reading I7 = the distribution the search-shaped batch samples from (BASELINE.json configs[4],
    DESIGN.md R22): the channel values equal the marginals of orc.determinise, an independent
    function of the oracle (5-sigma binomial bounds over 20,000 samples per root)."""
    R, S_ = 4, 20000
    src = orc.Env(R, seed=11, max_plies=1000, auto_reset=1, infostate=1)
    for _ in range(150):
        src.step(src.sample_uniform(src.legal_mask()))
    rb = src.get_boards()
    assert not (rb[:, 120] & 1).any()
    obs = src.encode_infostate().reshape(R, 487, 100)
    roots = orc.Env(R, seed=11); roots.reset_from(rb)
    out = orc.Env(R * S_, seed=11)
    orc.determinise(roots, S_, 5, out)
    det = out.get_boards().reshape(R, S_, 128)
    checked = 0
    for r in range(R):
        side = int(rb[r, 116]) & 1
        for s in range(100):
            b = int(rb[r, s])
            if (b & 15) in (0, 15) or ((b >> 4) & 1) == side or (b & W.REVEALED):
                continue
            freq = np.bincount(det[r, :, s] & 15, minlength=13) / S_
            for t in range(1, 13):
                p = float(np.array([obs[r, 12 + t - 1, s]], np.uint16).astype(np.uint32).__lshift__(16).view(np.float32)[0])
                sigma = max((p * (1 - p) / S_) ** 0.5, 1e-4)
                assert abs(freq[t] - p) < 5 * sigma + 2 ** -8 * p, (r, s, t, freq[t], p)
                checked += 1
    assert checked > 600


# ------------------------------------------------------------------ invariants under random play
def _bf16_to_float(a):
    return (a.astype(np.uint32) << 16).view(np.float32)


def test_invariants_under_random_play():
    n = 48
    e = orc.Env(n, seed=4, max_plies=400, auto_reset=1, infostate=1)
    played = [[] for _ in range(n)]
    for t in range(330):
        a = e.sample_uniform(e.legal_mask())
        r, d = e.step(a)
        for g in range(n):
            if d[g] & 1:
                played[g] = []  # auto-reset: the trackers start again
            else:
                played[g].append(int(a[g]))
        if t % 11 != 10:
            continue
        obs = e.encode_infostate().reshape(n, 487, 100)
        boards = e.get_boards()
        for g in range(n):
            o, b = obs[g], boards[g]
            side = int(b[116]) & 1
            cells = b[:100]
            piece = ((cells & 15) >= 1) & ((cells & 15) <= 12)
            mine = piece & (((cells >> 4) & 1) == side)
            theirs = piece & ~mine
            one = (o == ONE)
            # 0-11: the player's pieces by type; 36-40 as defined
            assert np.array_equal(one[0:12].sum(0), mine.astype(int))
            assert np.array_equal(one[36], mine & ((cells & W.REVEALED) == 0)) and np.array_equal(one[37], theirs & ((cells & W.REVEALED) == 0))
            assert np.array_equal(one[39], mine & ((cells & W.MOVED) != 0)) and np.array_equal(one[40], theirs & ((cells & W.MOVED) != 0))
            # 12-23: sums to the opponent-piece indicator on every square, to the type counts over the board
            pr = _bf16_to_float(o[12:24])
            assert np.allclose(pr.sum(0), theirs.astype(float), atol=12 * 2 ** -9)
            for tcode in range(1, 13):
                assert abs(pr[tcode - 1].sum() - int((theirs & ((cells & 15) == tcode)).sum())) < 40 * 2 ** -9 * 2
            pr = _bf16_to_float(o[24:36])
            assert np.allclose(pr.sum(0), mine.astype(float), atol=12 * 2 ** -9)
            # every piece on the board has exactly one start square; a start square is used once
            ss = one[355:455]
            assert np.array_equal(ss.sum(0), piece.astype(int)) and (ss.sum(1) <= 1).all()
            # tracker channels only on squares of the right owner
            for lo, hi, who in ((43, 76, mine), (76, 109, theirs), (251, 303, mine), (303, 355, theirs)):
                assert not (one[lo:hi].any(0) & ~who).any()
            assert not o[275].any() and not o[288].any() and not o[301].any()      # padding channels
            assert not o[275 + 52].any() and not o[288 + 52].any() and not o[301 + 52].any()
            # captured: 80 pieces started; every missing one (the Flags stay) has its start square marked
            assert one[109:131].sum() == 80 - int(piece.sum())
            assert not (one[109:131].any(0) & ss.any(1)).any()  # a captured piece's start square is nobody's now
            # causes of death: at most one per captured movable piece, none for Bombs (reading I6)
            bombs_lost = 12 - int((piece & ((cells & 15) == W.BOMB)).sum())
            assert one[131:251].sum() <= 80 - int(piece.sum()) - bombs_lost
            assert one[131:251].sum() >= 1 or piece.sum() > 70
            # 455-486: the played moves, most recent first
            for j in range(32):
                pl = o[455 + j]
                if j < len(played[g]):
                    a_ = played[g][-1 - j]
                    frm, dd, dist = a_ // 36, (a_ % 36) // 9, a_ % 9 + 1
                    to = frm + dist * (10, 1, -10, -1)[dd]
                    assert {int(s): int(pl[s]) for s in np.nonzero(pl)[0]} == {to: ONE, frm: MINUS_ONE}
                else:
                    assert not pl.any()
            # 41: fraction of the ply cap
            assert (o[41] == bf16_exact(Fraction(int(b[116]) | (int(b[117]) << 8), 400))).all()


def test_information_state_property():
    """The player's information state does not depend on the types of the opponent's unrevealed
    pieces: any consistent re-typing (here: the determinisation sampler's) of the opponent's
    hidden pieces gives the same 487 channels.  The trackers are history, not state, so the
    re-typed positions are compared through their boards only: same multiset, same public bits."""
    R, S_ = 3, 40
    src = orc.Env(R, seed=21, max_plies=1000, auto_reset=1)
    for _ in range(120):
        src.step(src.sample_uniform(src.legal_mask()))
    rb = src.get_boards()
    roots = orc.Env(R, seed=21); roots.reset_from(rb)
    out = orc.Env(R * S_, seed=21)
    orc.determinise(roots, S_, 3, out)
    det = out.get_boards()
    e0 = orc.Env(R, seed=21, infostate=1); e0.reset_from(rb)
    base = e0.encode_infostate().reshape(R, -1)
    e1 = orc.Env(R * S_, seed=21, infostate=1); e1.reset_from(det)
    alt = e1.encode_infostate().reshape(R, S_, -1)
    assert (det.reshape(R, S_, 128)[:, :, :100] != rb[:, None, :100]).any()  # the re-typings do differ
    for r in range(R):
        for s in range(S_):
            assert np.array_equal(alt[r, s], base[r])
