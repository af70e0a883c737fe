"""Pins of the oracle's network-free search step (S3.7; R29):
structure of the expansion, hand-computed magnet policy, averaging of values, and eq. (8)
checked against the optimisation problem eq. (7) it solves."""
import numpy as np

from oracle import orc
from paper_2511_07312_b200 import workloads as W

A = W.action_index


def _env_from(lines, **kw):
    o = orc.Env(len(lines), **kw)
    o.reset_from(np.stack(lines))
    return o


def _roots(n=3, plies=60, seed=4):
    o = orc.Env(n, seed=seed, max_plies=1000, auto_reset=1)
    for _ in range(plies):
        o.step(o.sample_uniform(o.legal_mask()))
    return o


def test_expand_structure():
    roots = _roots()
    rollouts = 200
    out = orc.Env(roots.n * rollouts, seed=4)
    orc.search_expand(roots, rollouts, 99, out)
    rb, ob = roots.get_boards(), out.get_boards()
    masks = roots.legal_mask()
    for r in range(roots.n):
        legal = W.mask_to_actions(masks[r])
        L = len(legal); C = max(1, rollouts // L); used = min(C * L, rollouts)
        assert L > 1 and used <= rollouts
        blk = ob[r * rollouts:(r + 1) * rollouts]
        # unused slots: the root, frozen
        for s in range(used, rollouts):
            assert blk[s, 120] & 1 and np.array_equal(blk[s, :100], rb[r, :100])
        side = (int(rb[r, 116]) | (int(rb[r, 117]) << 8)) & 1
        for c in range(C):
            base = None
            for l in range(L):
                s = c * L + l
                if s >= used:
                    break
                a = legal[l]
                f, d, k = a // 36, (a % 36) // 9, a % 9 + 1
                t = f + k * (10, 1, -10, -1)[d]
                g = blk[s]
                assert (g[100], g[101]) == (f, t)                      # the forced first move is the l-th legal action
                assert (int(g[116]) | (int(g[117]) << 8)) == (int(rb[r, 116]) | (int(rb[r, 117]) << 8)) + 1
                # enemy pieces away from the move: identical for every action of one configuration ...
                enemy = np.array([(x & 15) if (1 <= (x & 15) <= 12 and ((x >> 4) & 1) != side) else 0 for x in g[:100]])
                enemy[t] = 0; 
                ref = np.array([(x & 15) if (1 <= (x & 15) <= 12 and ((x >> 4) & 1) != side) else 0 for x in rb[r, :100]])
                if base is None:
                    base = (enemy.copy(), t)
                else:
                    e0, t0 = base
                    same = np.ones(100, bool); same[t] = False; same[t0] = False
                    assert np.array_equal(enemy[same], e0[same])
                # ... and a permutation of the root's hidden types (multiset preserved, unless the move captured one)
                assert sorted(enemy[enemy > 0].tolist()) in (sorted(ref[ref > 0].tolist()),) or len(enemy[enemy > 0]) == len(ref[ref > 0]) - 1
        # different configurations do differ somewhere (with overwhelming probability)
        if C >= 2:
            assert not np.array_equal(blk[0, :100], blk[L, :100])


def test_magnet_policy_and_uniform_values_by_hand():
    # red: Sergeant on 44 (lakes on 43 and... 45 is free): moves N, E, S = 3 (west is lake 43);
    #      Miner on 0 with the Flag on 1 beside it: only north = 1 move.
    pieces = {44: W.piece(W.SERGEANT, W.RED), 0: W.piece(W.MINER, W.RED), 1: W.piece(W.FLAG, W.RED),
              99: W.piece(W.FLAG, W.BLUE), 98: W.piece(W.BOMB, W.BLUE), 77: W.piece(W.SERGEANT, W.BLUE)}
    roots = _env_from([W.make_line(pieces)])
    legal = W.mask_to_actions(roots.legal_mask()[0])
    assert legal == [A(0, 0, 1), A(44, 0, 1), A(44, 1, 1), A(44, 2, 1)]
    rollouts = 8
    games = orc.Env(rollouts, seed=0)
    orc.search_expand(roots, rollouts, 1, games)          # nobody has won after one ply: every value is 0
    alpha, beta = 0.002, 0.02
    q, rho, pi = orc.search_policy(roots, games, rollouts, alpha, beta)
    assert not q.any()
    want_rho = {A(0, 0, 1): 1 / 2, A(44, 0, 1): 1 / 6, A(44, 1, 1): 1 / 6, A(44, 2, 1): 1 / 6}
    for a, v in want_rho.items():
        assert abs(rho[0, a] - v) < 1e-7
    assert abs(rho.sum() - 1) < 1e-6 and (rho[0, [a for a in range(3600) if a not in want_rho]] == 0).all()
    # equal values, uniform prior: pi ~ rho^(alpha/(alpha+beta))
    w = np.array([want_rho[a] for a in legal]) ** (alpha / (alpha + beta))
    assert np.allclose(pi[0, legal], w / w.sum(), rtol=1e-6)
    assert abs(pi.sum() - 1) < 1e-6
    # a prior that rules an action out gives it probability 0
    prior = np.zeros((1, 3600), np.float32); prior[0, legal[:3]] = 1 / 3
    _, _, pi2 = orc.search_policy(roots, games, rollouts, alpha, beta, prior)
    assert pi2[0, legal[3]] == 0 and abs(pi2.sum() - 1) < 1e-6


def _games_with_results(root_line, rollouts, results):
    """`rollouts` copies of a line, game s finished with red's result results[s] (None = running)."""
    lines = []
    for s in range(rollouts):
        L = root_line.copy()
        if results[s] is not None:
            L[120] = 1 | (1 << 2); L[121] = np.uint8(np.int8(results[s]).view(np.uint8))
        lines.append(L)
    return _env_from(lines)


def test_values_are_averaged_per_action_from_the_searchers_side():
    pieces = {44: W.piece(W.SERGEANT, W.BLUE), 0: W.piece(W.FLAG, W.RED), 99: W.piece(W.FLAG, W.BLUE),
              10: W.piece(W.BOMB, W.RED)}
    line = W.make_line(pieces, ply=1)                      # blue to move: 3 legal actions, L = 3
    roots = _env_from([line])
    legal = W.mask_to_actions(roots.legal_mask()[0])
    assert len(legal) == 3
    rollouts = 7                                           # C = 2, used = 6, slot 6 unused
    res = [+1, -1, None, -1, -1, 0, +1]                    # red's results; slot = c*3 + l
    games = _games_with_results(line, rollouts, res)
    q, _, pi = orc.search_policy(roots, games, rollouts, 0.5, 0.5)
    # blue's view: action 0: (-1 + 1)/2 = 0; action 1: (1 + 1)/2 = 1; action 2: (0 + 0)/2 = 0
    assert np.allclose(q[0, legal], [0.0, 1.0, 0.0])
    assert pi[0, legal[1]] > pi[0, legal[0]] and abs(pi[0, legal[0]] - pi[0, legal[2]]) < 1e-7


def test_leaf_values_count_for_running_games_only_blue_searcher():
    """q-hat averages the value of the position each rollout reached.  Caller-supplied leaf values
    (from the searcher's side) stand for the games still running; a finished game keeps its result.
    Worked by hand with fractional values, blue searching."""
    pieces = {44: W.piece(W.SERGEANT, W.BLUE), 0: W.piece(W.FLAG, W.RED), 99: W.piece(W.FLAG, W.BLUE),
              10: W.piece(W.BOMB, W.RED)}
    line = W.make_line(pieces, ply=1)                      # blue to move, L = 3
    roots = _env_from([line])
    legal = W.mask_to_actions(roots.legal_mask()[0])
    rollouts = 7                                           # C = 2, used = 6: slots 0..5, slot = c*3 + l
    res = [+1, None, None, None, -1, None, None]           # red's results of the finished games (slots 0 and 4)
    vals = np.array([0.9, 0.25, -0.5, 0.125, 0.75, 0.375, 0.6], np.float32)   # slot 0, 4: ignored (finished); 6: unused
    games = _games_with_results(line, rollouts, res)
    q, _, pi = orc.search_policy(roots, games, rollouts, 0.5, 0.5, values=vals)
    # blue's view.  action 0: slots 0 (finished, red won: -1) and 3 (running: 0.125) -> -0.4375
    #               action 1: slots 1 (0.25) and 4 (finished, blue won: +1)          ->  0.625
    #               action 2: slots 2 (-0.5) and 5 (0.375)                           -> -0.0625
    assert np.array_equal(q[0, legal], np.array([-0.4375, 0.625, -0.0625], np.float32))
    assert pi[0, legal[1]] > pi[0, legal[2]] > pi[0, legal[0]]
    # without values the running games count 0, as before
    q0, _, _ = orc.search_policy(roots, games, rollouts, 0.5, 0.5)
    assert np.array_equal(q0[0, legal], np.array([-0.5, 0.5, 0.0], np.float32))
    # all-zero values change nothing
    qz, _, piz = orc.search_policy(roots, games, rollouts, 0.5, 0.5, values=np.zeros(7, np.float32))
    assert np.array_equal(qz, q0)


def test_eq8_solves_eq7():
    """pi_search of eq. (8) must maximise <q, pi> - alpha KL(pi, rho) - beta KL(pi, pi_theta) over the
    simplex of legal actions (eq. (7)): no perturbed distribution scores higher."""
    rng = np.random.default_rng(0)
    roots = _roots(n=2, plies=80, seed=7)
    rollouts = 300
    games = orc.Env(2 * rollouts, seed=7)
    orc.search_expand(roots, rollouts, 5, games)
    for _ in range(30):
        games.step(games.sample_uniform(games.legal_mask()))
    # give the values some spread: finish a third of the games by hand
    gb = games.get_boards()
    for s in range(0, len(gb), 3):
        gb[s, 120] = 1 | (1 << 2); gb[s, 121] = np.uint8(np.int8(rng.choice([-1, 1])).view(np.uint8))
    games.reset_from(gb)
    masks = roots.legal_mask()
    prior = np.zeros((2, 3600), np.float32)
    for r in range(2):
        legal = W.mask_to_actions(masks[r])
        p = rng.random(len(legal)) + 0.05
        prior[r, legal] = p / p.sum()
    for alpha, beta in ((0.002, 0.02), (0.3, 0.1)):
        q, rho, pi = orc.search_policy(roots, games, rollouts, alpha, beta, prior)
        for r in range(2):
            legal = W.mask_to_actions(masks[r])
            qq, rr, pt, ps = (x[r, legal].astype(np.float64) for x in (q, rho, prior, pi))
            assert abs(ps.sum() - 1) < 1e-5 and qq.std() > 0

            def objective(p):
                nz = p > 0
                return (qq * p).sum() - alpha * (p[nz] * np.log(p[nz] / rr[nz])).sum() - beta * (p[nz] * np.log(p[nz] / pt[nz])).sum()

            # stationarity on the simplex (all p > 0): q - alpha (ln(p/rho) + 1) - beta (ln(p/pi_theta) + 1)
            # takes one value for every action; the outputs are float32, hence the 1e-5
            kkt = qq - alpha * (np.log(ps / rr) + 1) - beta * (np.log(ps / pt) + 1)
            assert (ps > 0).all() and kkt.max() - kkt.min() < 1e-5 * max(1.0, 1 / (alpha + beta)) * 0.1
            best = objective(ps)
            for _ in range(200):
                d = rng.normal(size=len(legal)) * rng.choice([3e-2, 1e-1, 0.5])
                p = np.clip(ps + d * ps, 1e-12, None); p /= p.sum()
                assert objective(p) <= best + 1e-7


def test_degenerate_priors():
    """DESIGN.md R29: a prior of 0 gives probability 0; a prior with its whole mass on one legal action
    gives that action (beta > 0: any other pi has infinite KL); a prior with no mass on any legal
    action of a root says nothing there and that root falls back to "no prior" - no NaN anywhere."""
    pieces = {44: W.piece(W.SERGEANT, W.BLUE), 0: W.piece(W.FLAG, W.RED), 99: W.piece(W.FLAG, W.BLUE),
              10: W.piece(W.BOMB, W.RED)}
    line = W.make_line(pieces, ply=1)
    roots = _env_from([line, line, line])
    legal = W.mask_to_actions(roots.legal_mask()[0])
    rollouts = 6
    games = _env_from(list(_games_with_results(line, rollouts, [+1, -1, 0, -1, -1, 0]).get_boards()) * 3)
    prior = np.zeros((3, 3600), np.float32)
    prior[0, legal[2]] = 1.0                     # root 0: one-hot on a legal action
    prior[1, 5] = 1.0                            # root 1: all mass on an illegal action
    prior[2, legal[0]] = 0.25; prior[2, legal[1]] = 0.75   # root 2: one legal action excluded
    q, rho, pi = orc.search_policy(roots, games, rollouts, 0.3, 0.2, prior)
    _, _, pi_none = orc.search_policy(roots, games, rollouts, 0.3, 0.2)
    assert np.isfinite(pi).all() and np.allclose(pi.sum(axis=1), 1.0, atol=1e-6)
    assert pi[0, legal[2]] == 1.0
    assert np.array_equal(pi[1], pi_none[1])
    assert pi[2, legal[2]] == 0.0 and pi[2, legal[0]] > 0 and pi[2, legal[1]] > 0
    # root 2 by hand: weights exp(q/(a+b)) * rho^(a/(a+b)) * prior^(b/(a+b)), rho equal for one piece
    w = np.exp(q[2, legal[:2]].astype(np.float64) / 0.5) * np.array([0.25, 0.75]) ** (0.2 / 0.5)
    assert np.allclose(pi[2, legal[:2]], w / w.sum(), atol=1e-6)
