"""Pins of the oracle's continuous-chasing rule (reading R28 in DESIGN.md).

(1) a chase around a 2x2 block worked by hand, (2) the state machine on hand-built plies,
(3) an independent checker written from the paper's definitions that keeps every position of
the game as a snapshot (the oracle instead takes the logged plies back) and is compared with
the oracle's masks over biased random play on crowded little positions."""
import numpy as np

from chase_scenarios import cage as _cage, crowded as _crowded
from oracle import orc
from paper_2511_07312_b200 import workloads as W

CAPTAIN, SERGEANT, SCOUT, MINER, FLAG = W.CAPTAIN, W.SERGEANT, W.SCOUT, W.MINER, W.FLAG


def _env(pieces, chase_rule=1, ply=0):
    o = orc.Env(1, chase_rule=chase_rule, two_square=1)
    o.reset_from(W.make_line(pieces, ply=ply)[None, :])
    return o


def _legal(o):
    return W.mask_to_actions(o.legal_mask()[0])


def _play(o, actions):
    for a in actions:
        assert a in _legal(o), a
        o.step(np.array([a], np.int16))


A = W.action_index
BLOCK = {11: W.piece(CAPTAIN, W.RED), 22: W.piece(SERGEANT, W.BLUE), 9: W.piece(FLAG, W.RED), 99: W.piece(FLAG, W.BLUE)}
# red Captain X chases blue Sergeant Y once around the block {11,12,21,22}
AROUND = [A(11, 1, 1), A(22, 3, 1), A(12, 0, 1), A(21, 2, 1), A(22, 3, 1), A(11, 1, 1), A(21, 2, 1), A(12, 0, 1)]


def test_chase_around_a_block_bans_the_repeating_threat():
    o = _env(BLOCK)
    _play(o, AROUND)
    line = o.get_boards()[0]
    assert (line[122], line[123]) == (8, 0)          # eight positions in red's chase, blue is not chasing
    # X is back on 11, Y on 22.  East (11->12) would recreate the position after the first threat:
    # banned.  North (11->21) is a threat too but returns X to the square it left on red's previous
    # turn: allowed.  South and west threaten nothing.
    assert _legal(o) == [A(11, 0, 1), A(11, 2, 1), A(11, 3, 1)]
    # the same plies without the rule
    o0 = _env(BLOCK, chase_rule=0)
    _play(o0, AROUND)
    assert _legal(o0) == [A(11, 0, 1), A(11, 1, 1), A(11, 2, 1), A(11, 3, 1)]
    assert (o0.get_boards()[0][122], o0.get_boards()[0][123]) == (0, 0)
    # the banned action is rejected by step, too
    before = o.get_boards()
    o.step(np.array([A(11, 1, 1)], np.int16))
    assert o.check() == orc.ILLEGAL_ACTION and np.array_equal(o.get_boards(), before)


def test_chase_around_a_lake_is_caught_after_one_lap():
    """The classic: X chases Y around the lake {42,43,52,53}.  The ring of 12 squares is walked
    once in 24 plies; the 13th threat would recreate the position after the first one."""
    ring = [31, 32, 33, 34, 44, 54, 64, 63, 62, 61, 51, 41]
    pieces = {ring[0]: W.piece(CAPTAIN, W.RED), ring[2]: W.piece(SERGEANT, W.BLUE), 9: W.piece(FLAG, W.RED),
              99: W.piece(FLAG, W.BLUE)}

    def act(a, b):
        d = {10: 0, 1: 1, -10: 2, -1: 3}[b - a]
        return A(a, d, 1)

    for rule in (1, 0):
        o = _env(pieces, chase_rule=rule)
        for k in range(12):
            _play(o, [act(ring[k % 12], ring[(k + 1) % 12])])        # X steps next to Y: threat
            _play(o, [act(ring[(k + 2) % 12], ring[(k + 3) % 12])])  # Y steps on: evade
        line = o.get_boards()[0]
        assert (line[122], line[123]) == ((24, 0) if rule else (0, 0))
        legal = _legal(o)
        again = act(ring[0], ring[1])                                 # X is back on ring[0], Y on ring[2]
        back = act(ring[0], ring[11])                                 # X's return move: no threat here anyway
        assert (again in legal) == (rule == 0) and back in legal
        # a state loaded from its canonical line remembers 8 plies only: the lap is forgotten
        o2 = orc.Env(1, chase_rule=rule)
        o2.reset_from(o.get_boards())
        assert again in _legal(o2)
        # ... unless the plies that led to it are handed over with it ("the continuous chasing
        # rule needs to be tested against the history of board states that leads to the non-initial
        # reset state"): then the lap is remembered across the load
        played = []
        for k in range(12):
            played += [(ring[k % 12], ring[(k + 1) % 12]), (ring[(k + 2) % 12], ring[(k + 3) % 12])]
        plies = np.full((1, 63, 2), 0xFF, np.uint8)
        plies[0, :24] = played[::-1]
        o3 = orc.Env(1, chase_rule=rule)
        o3.reset_from(o.get_boards(), plies)
        assert (again in _legal(o3)) == (rule == 0) and back in _legal(o3)
        assert _legal(o3) == legal
        # taking 23 plies back reaches the position after the first threat (the one `again` would
        # recreate); with 22 known plies it is out of reach
        short = plies.copy(); short[0, 23] = 0xFF
        o4 = orc.Env(1, chase_rule=rule)
        o4.reset_from(o.get_boards(), short)
        assert (again in _legal(o4)) == (rule == 0)
        short[0, 22] = 0xFF
        o4 = orc.Env(1, chase_rule=rule)
        o4.reset_from(o.get_boards(), short)
        assert again in _legal(o4)


def test_chase_memory_survives_pinned_restarts_and_determinised_copies():
    """P:250 / P:252-254: a game pinned to restart from the lake-lap state restarts with the lap in
    its memory; a determinised copy of the state (search) inherits it too."""
    ring = [31, 32, 33, 34, 44, 54, 64, 63, 62, 61, 51, 41]

    def act(a, b):
        return A(a, {10: 0, 1: 1, -10: 2, -1: 3}[b - a], 1)

    pieces = {ring[0]: W.piece(CAPTAIN, W.RED), ring[2]: W.piece(SERGEANT, W.BLUE), 9: W.piece(FLAG, W.RED),
              99: W.piece(FLAG, W.BLUE), 8: W.piece(MINER, W.RED), 98: W.piece(MINER, W.BLUE)}
    o = _env(pieces)
    played = []
    for k in range(12):
        mv = [(ring[k % 12], ring[(k + 1) % 12]), (ring[(k + 2) % 12], ring[(k + 3) % 12])]
        _play(o, [act(*mv[0]), act(*mv[1])])
        played += mv
    lap = o.get_boards()
    plies = np.full((1, 63, 2), 0xFF, np.uint8)
    plies[0, :24] = played[::-1]
    again = act(ring[0], ring[1])
    # pinned: a short game (ply cap) that restarts from the lap state
    p = orc.Env(1, chase_rule=1, max_plies=30, auto_reset=1)
    p.reset_from(lap, plies)
    p.pin_reset_state(lap, plies)
    assert again not in _legal(p)
    for _ in range(6):  # plies 24..29: the cap ends the game, it restarts from the pin
        p.step(p.sample_uniform(p.legal_mask()))
    b = p.get_boards()[0]
    assert b[124] == 1 and (int(b[116]) | (int(b[117]) << 8)) == 24
    assert again not in _legal(p)                      # the restart remembers the lap
    q = orc.Env(1, chase_rule=1, max_plies=30, auto_reset=1)
    q.reset_from(lap, plies)
    q.pin_reset_state(lap)                             # pinned without its history: forgotten at the restart
    for _ in range(6):
        q.step(q.sample_uniform(q.legal_mask()))
    assert again in _legal(q)
    # determinised copies (red is the searcher; blue's hidden pieces are re-dealt): the memory travels
    roots = orc.Env(1, chase_rule=1); roots.reset_from(lap, plies)
    out = orc.Env(8, chase_rule=1)
    orc.determinise(roots, 8, 3, out)
    m = out.legal_mask()
    for k in range(8):
        acts = W.mask_to_actions(m[k])
        assert again not in acts and act(ring[0], ring[11]) in acts


def test_chase_state_machine_on_hand_built_plies():
    o = _env(BLOCK)
    ages = []
    for a in AROUND[:6]:
        _play(o, [a])
        ages.append(tuple(int(x) for x in o.get_boards()[0][122:124]))
    assert ages == [(1, 0), (2, 0), (3, 0), (4, 0), (5, 0), (6, 0)]
    # a ply of the chaser that threatens nothing ends the chase
    _play(o, [A(21, 0, 1)])                      # X 21->31: no blue piece next to 31
    assert tuple(o.get_boards()[0][122:124]) == (0, 0)
    # a threat answered by a move that is no evade ends it as well
    o = _env({**BLOCK, 55: W.piece(MINER, W.BLUE)})
    _play(o, [A(11, 1, 1), A(55, 0, 1)])         # X threatens Y; blue moves another piece
    assert tuple(o.get_boards()[0][122:124]) == (0, 0)
    # an evade that lands next to another red piece is a threat of blue's own
    o = _env({**BLOCK, 31: W.piece(MINER, W.RED)})
    _play(o, [A(11, 1, 1), A(22, 3, 1)])         # Y 22->21 leaves X (on 12) and touches the Miner on 31
    assert tuple(o.get_boards()[0][122:124]) == (2, 1)
    # a battle ends every chase
    _play(o, [A(31, 2, 1)])                      # Miner 31x21
    assert tuple(o.get_boards()[0][122:124]) == (0, 0)
    # moving next to a piece by capturing is a battle, not a threat; a Scout's long move can threaten
    o = _env({40: W.piece(SCOUT, W.RED), 45: W.piece(SERGEANT, W.BLUE), 9: W.piece(FLAG, W.RED), 99: W.piece(FLAG, W.BLUE)})
    _play(o, [A(40, 1, 1)])                      # 40->41: lake on 42 blocks further; nothing adjacent
    assert tuple(o.get_boards()[0][122:124]) == (0, 0)
    o = _env({4: W.piece(SCOUT, W.RED), 45: W.piece(SERGEANT, W.BLUE), 9: W.piece(FLAG, W.RED), 99: W.piece(FLAG, W.BLUE)})
    _play(o, [A(4, 0, 3)])                       # 4->34, now below the Sergeant on... 44? no: 45 is not adjacent
    assert tuple(o.get_boards()[0][122:124]) == (0, 0)
    _play(o, [A(45, 3, 1)])                      # Sergeant 45->44: adjacent to the Scout on 34 -> blue threatens
    assert tuple(o.get_boards()[0][122:124]) == (0, 1)
    _play(o, [A(34, 2, 2)])                      # Scout flees two squares down the file: an evade
    assert tuple(o.get_boards()[0][122:124]) == (0, 2)


# ----------------------------------------------------------------------------- independent checker
def _adj(a, b):
    return abs(a // 10 - b // 10) + abs(a % 10 - b % 10) == 1


class SnapshotChecker:
    """The rule restated with full position snapshots."""

    def __init__(self, cells):
        self.pos = [tuple(int(c) & 0x1F for c in cells)]  # position after k plies
        self.start = [None, None]                          # index of the first chase position per player
        self.last = [None, None]                           # last move per player
        self.last_threat = None                            # (player, square of the threatening piece)

    def threat(self, board, side, f, t):
        if board[t] != 0:
            return False
        for d in (10, -10, 1, -1):
            c = t + d
            if c < 0 or c > 99 or not _adj(c, t) or c == f:
                continue
            b = board[c]
            if 1 <= (b & 15) <= 12 and ((b >> 4) & 1) != side:
                return True
        return False

    def banned(self, side, f, t):
        board = self.pos[-1]
        if self.start[side] is None or not self.threat(board, side, f, t):
            return False
        if self.last[side] == (t, f):
            return False
        r = list(board)
        r[t], r[f] = r[f], 0
        now = len(self.pos) - 1
        lo = max(self.start[side], now - 63)  # the move log remembers 63 plies
        return tuple(r) in self.pos[lo:now]

    def push(self, side, f, t):
        board = self.pos[-1]
        fight = board[t] != 0
        th = self.threat(board, side, f, t)
        q = side ^ 1
        ev = (self.last_threat is not None and self.last_threat[0] == q and not fight
              and _adj(f, self.last_threat[1]) and not _adj(t, self.last_threat[1]))
        if fight:
            self.start = [None, None]
        else:
            if self.start[q] is not None and not ev:
                self.start[q] = None
            if th:
                if self.start[side] is None:
                    self.start[side] = len(self.pos)  # the position this ply creates
            else:
                self.start[side] = None
        self.last_threat = (side, t) if (th and not fight) else None
        self.last[side] = (f, t)


def test_oracle_masks_equal_the_snapshot_checker_on_biased_random_play():
    rng = np.random.default_rng(5)
    bans = chases = 0
    for game in range(1000):
        pieces = _crowded(rng) if game < 60 else _cage(rng)
        o1, o0 = _env(pieces, 1), orc.Env(1, chase_rule=0)
        chk = SnapshotChecker(o1.get_boards()[0][:100])
        for ply in range(120):
            line = o1.get_boards()
            if line[0, 120] & 1:
                break
            side = ply & 1
            stripped = line.copy(); stripped[0, 122:124] = 0
            o0.reset_from(stripped)
            base = _legal(o0)
            got = _legal(o1)
            want = []
            for a in base:
                f, d, k = a // 36, (a % 36) // 9, a % 9 + 1
                t = f + k * (10, 1, -10, -1)[d]
                if chk.banned(side, f, t):
                    bans += 1
                else:
                    want.append(a)
            assert got == want, (game, ply)
            if not got:
                break
            chases += chk.start[side] is not None
            # biased policy: keep chases going (threats for the chaser, anything for the other side)
            board = chk.pos[-1]
            pref = [a for a in got if chk.threat(board, side, a // 36, a // 36 + (a % 9 + 1) * (10, 1, -10, -1)[(a % 36) // 9])]
            pick = pref if (pref and rng.random() < 0.7) else got
            a = int(pick[rng.integers(len(pick))])
            f, d, k = a // 36, (a % 36) // 9, a % 9 + 1
            chk.push(side, f, f + k * (10, 1, -10, -1)[d])
            o1.step(np.array([a], np.int16))
            assert o1.check() == 0
            chk.pos.append(tuple(int(c) & 0x1F for c in o1.get_boards()[0][:100]))
    assert chases > 100 and bans > 20  # the games did produce chases and banned threats
    print("chase plies", chases, "banned moves", bans)


def test_two_square_chain_is_interrupted_by_a_gap_in_a_hand_built_history():
    """R24 / P:212 "three consecutive turns of its owner": red's Sergeant shuttled 44->45->44->45
    on red's last three plies (entries 5, 3, 1) - moving back to 44 is banned.  With the same
    three moves one turn older (entries 7, 5, 3) and red's latest ply unknown (0xFF), nothing
    says the turns were consecutive: no ban."""
    pieces = {45: W.piece(SERGEANT, W.RED, moved=True), 95: W.piece(SERGEANT, W.BLUE, moved=True),
              0: W.piece(FLAG, W.RED), 99: W.piece(FLAG, W.BLUE)}
    blue = (95, 96)
    full = [blue, (44, 45), blue, (45, 44), blue, (44, 45), (0xFF, 0xFF), (0xFF, 0xFF)]
    o = orc.Env(1)
    o.reset_from(W.make_line(pieces, ply=6, history=full)[None, :])
    assert A(45, 3, 1) not in _legal(o) and A(45, 0, 1) in _legal(o)
    gap = [blue, (0xFF, 0xFF), blue, (44, 45), blue, (45, 44), blue, (44, 45)]
    o.reset_from(W.make_line(pieces, ply=8, history=gap)[None, :])
    assert A(45, 3, 1) in _legal(o)
