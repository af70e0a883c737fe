"""Continuous-chasing rule (R28) on the CUDA path: bit-exact with
the oracle in every kernel that generates or applies moves."""
import numpy as np
import pytest
import torch

from chase_scenarios import cage, crowded
from oracle import orc
from paper_2511_07312_b200 import binding as B
from paper_2511_07312_b200 import workloads as W

pytestmark = pytest.mark.gpu
A = W.action_index


def _np(t):
    return t.detach().cpu().numpy()


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _mask_np(t):
    return _np(t).view(np.uint32)


def test_chase_around_a_block_on_gpu():
    pieces = {11: W.piece(W.CAPTAIN, W.RED), 22: W.piece(W.SERGEANT, W.BLUE), 9: W.piece(W.FLAG, W.RED),
              99: W.piece(W.FLAG, W.BLUE)}
    around = [A(11, 1, 1), A(22, 3, 1), A(12, 0, 1), A(21, 2, 1), A(22, 3, 1), A(11, 1, 1), A(21, 2, 1), A(12, 0, 1)]
    for rule, expect in ((1, [A(11, 0, 1), A(11, 2, 1), A(11, 3, 1)]), (0, [A(11, 0, 1), A(11, 1, 1), A(11, 2, 1), A(11, 3, 1)])):
        g = B.Env(1, chase_rule=rule)
        g.reset_from(_dev(W.make_line(pieces)[None, :]))
        for a in around:
            g.step(_dev(np.array([a], np.int16)))
        assert g.check() == 0
        assert W.mask_to_actions(_mask_np(g.legal_mask())[0]) == expect
        assert tuple(_np(g.get_boards())[0][122:124]) == ((8, 0) if rule else (0, 0))
    g.step(_dev(np.array([A(11, 1, 1)], np.int16)))  # rule off above: legal
    g = B.Env(1, chase_rule=1)
    g.reset_from(_dev(W.make_line(pieces)[None, :]))
    for a in around:
        g.step(_dev(np.array([a], np.int16)))
    g.step(_dev(np.array([A(11, 1, 1)], np.int16)))
    assert g.check() == B.ILLEGAL_ACTION


def _scenario_boards(n, seed):
    rng = np.random.default_rng(seed)
    lines = np.zeros((n, 128), np.uint8)
    for i in range(n):
        lines[i] = W.make_line(cage(rng) if i % 4 else crowded(rng))
    return lines


def test_chase_around_a_lake_on_gpu_every_kernel():
    """One lap (24 plies) around the lake {42,43,52,53}: the 13th threat repeats the position after
    the first one.  The plies are fed through strat_step / strat_step_observe; the ban must then
    show in strat_legal_mask, the fused step's mask, step validation and the on-chip sampler."""
    ring = [31, 32, 33, 34, 44, 54, 64, 63, 62, 61, 51, 41]
    pieces = {ring[0]: W.piece(W.CAPTAIN, W.RED), ring[2]: W.piece(W.SERGEANT, W.BLUE), 9: W.piece(W.FLAG, W.RED),
              99: W.piece(W.FLAG, W.BLUE)}

    def act(a, b):
        return A(a, {10: 0, 1: 1, -10: 2, -1: 3}[b - a], 1)

    n = 64  # the same game 64 times: on-chip sampling over many action streams
    kw = dict(seed=3, chase_rule=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    lines = np.repeat(W.make_line(pieces)[None, :], n, axis=0)
    g.reset_from(_dev(lines)); o.reset_from(lines)
    mask, rew, done, obs = g.new_mask(), g.new_reward(), g.new_done(), g.new_obs()
    for k in range(12):
        for a in (act(ring[k % 12], ring[(k + 1) % 12]), act(ring[(k + 2) % 12], ring[(k + 3) % 12])):
            acts = np.full(n, a, np.int16)
            o.step(acts)
            if k % 2:
                g.step(_dev(acts), rew, done)
            else:
                g.step_observe(_dev(acts), rew, done, mask, obs)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert tuple(o.get_boards()[0][122:124]) == (24, 0)
    om = o.legal_mask()
    again = act(ring[0], ring[1])
    assert again not in W.mask_to_actions(om[0])
    assert np.array_equal(_mask_np(g.legal_mask()), om)
    # fused step: same mask, same sampled actions; on-chip: same resulting boards
    g2 = B.Env(n, **kw)
    g2.reset_from(g.get_boards().clone())  # a loaded state forgets the lap: the move is legal again
    assert again in W.mask_to_actions(_mask_np(g2.legal_mask())[0])
    act_t = g.new_actions()
    oa = o.sample_uniform(om); o.step(oa)
    g.rollout_step(mask, act_t, rew, done, obs)
    assert np.array_equal(_mask_np(mask), om) and np.array_equal(_np(act_t), oa)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert g.check() == 0


def test_onchip_rollout_respects_a_long_chase_ban():
    """Same lap, then ONE on-chip ply for 4,096 copies with different action streams: none may
    play the banned move; the boards equal the oracle's."""
    ring = [31, 32, 33, 34, 44, 54, 64, 63, 62, 61, 51, 41]
    pieces = {ring[0]: W.piece(W.CAPTAIN, W.RED), ring[2]: W.piece(W.SERGEANT, W.BLUE), 9: W.piece(W.FLAG, W.RED),
              99: W.piece(W.FLAG, W.BLUE)}
    n = 4096
    kw = dict(seed=11, chase_rule=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    lines = np.repeat(W.make_line(pieces)[None, :], n, axis=0)
    g.reset_from(_dev(lines)); o.reset_from(lines)
    rew, done = g.new_reward(), g.new_done()
    for k in range(12):
        for f, t in ((ring[k % 12], ring[(k + 1) % 12]), (ring[(k + 2) % 12], ring[(k + 3) % 12])):
            acts = np.full(n, A(f, {10: 0, 1: 1, -10: 2, -1: 3}[t - f], 1), np.int16)
            o.step(acts); g.step(_dev(acts), rew, done)
    g.rollout_uniform(1)
    oa = o.sample_uniform(o.legal_mask()); o.step(oa)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert (oa != A(ring[0], 1, 1)).all() and len(set(oa.tolist())) == 3  # the three other moves of X all occur
    assert g.check() == 0


def _biased_actions(masks, boards, rng):
    """Test-side policy that keeps chases alive: prefer moves to empty squares next to an enemy
    piece (threats), then any non-capturing move, rarely anything.  Layout arithmetic only."""
    out = np.full(len(masks), -1, np.int16)
    for i in range(len(masks)):
        legal = W.mask_to_actions(masks[i])
        if not legal:
            continue
        cells = boards[i, :100]
        side = int(boards[i, 116]) & 1
        quiet, threats = [], []
        for a in legal:
            f, d, k = a // 36, (a % 36) // 9, a % 9 + 1
            t = f + k * (10, 1, -10, -1)[d]
            if cells[t] != 0:
                continue
            quiet.append(a)
            for dd in (10, -10, 1, -1):
                c = t + dd
                if 0 <= c <= 99 and abs(c // 10 - t // 10) + abs(c % 10 - t % 10) == 1 and c != f:
                    b = int(cells[c])
                    if 1 <= (b & 15) <= 12 and ((b >> 4) & 1) != side:
                        threats.append(a)
                        break
        u = rng.random()
        pool = threats if (threats and u < 0.75) else quiet if (quiet and u < 0.97) else legal
        out[i] = pool[rng.integers(len(pool))]
    return out


def test_chase_rule_parity_on_chase_heavy_positions():
    """400 little games (most of them two pieces in a Bomb cage, where positions recur and
    threats get banned all the time), restarted from their pinned position whenever they end.
    A test-side policy keeps the chases going; every fourth ply is played by the fused step and
    every fourth by the on-chip rollout kernel, whose uniform samplers must skip the banned moves."""
    n, steps = 400, 160
    kw = dict(variant=0, seed=77, max_plies=60, auto_reset=1, chase_rule=1)
    rng = np.random.default_rng(1)
    lines = np.zeros((n, 128), np.uint8)
    for i in range(n):
        lines[i] = W.make_line(cage(rng) if i % 8 else crowded(rng))
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    o0 = orc.Env(n, **dict(kw, chase_rule=0))
    g.reset_from(_dev(lines)); o.reset_from(lines)
    g.pin_reset_state(_dev(lines)); o.pin_reset_state(lines)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    banned_seen = banned_at_sampled = 0
    for t in range(steps):
        boards = o.get_boards()
        om = o.legal_mask()
        assert np.array_equal(_mask_np(g.legal_mask(mask)), om), t
        stripped = boards.copy(); stripped[:, 122:124] = 0
        o0.reset_from(stripped)
        nban = int(np.unpackbits((o0.legal_mask() ^ om).view(np.uint8)).sum())
        banned_seen += nban
        kind = t % 4
        if kind in (0, 1):
            a = _biased_actions(om, boards, rng)
            orr, od = o.step(a)
            if kind == 0:
                g.step(_dev(a), rew, done)
            else:
                g.step_observe(_dev(a), rew, done, mask, obs)
                assert np.array_equal(_mask_np(mask), o.legal_mask()), t
        else:
            banned_at_sampled += nban
            oa = o.sample_uniform(om); orr, od = o.step(oa)
            if kind == 2:
                g.rollout_step(mask, act, rew, done, obs)
                assert np.array_equal(_mask_np(mask), om) and np.array_equal(_np(act), oa), t
            else:
                g.rollout_uniform(1)
        if kind != 3:
            assert np.array_equal(_np(rew), orr) and np.array_equal(_np(done), od), t
        assert np.array_equal(_np(g.get_boards()), o.get_boards()), t
    assert banned_seen > 100 and banned_at_sampled > 20, (banned_seen, banned_at_sampled)
    assert g.check() == 0 and o.check() == 0


def test_chase_rule_classic_selfplay_parity_with_auto_reset():
    kw = dict(variant=0, seed=5, max_plies=400, auto_reset=1, chase_rule=1)
    n = 500
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    ages = 0
    for t in range(500):
        om = o.legal_mask(); oa = o.sample_uniform(om); orr, od = o.step(oa)
        g.rollout_step(mask, act, rew, done, obs)
        assert np.array_equal(_np(act), oa) and np.array_equal(_np(rew), orr) and np.array_equal(_np(done), od), t
        if t % 25 == 0 or t == 499:
            assert np.array_equal(_mask_np(mask), om), t
            b = o.get_boards()
            assert np.array_equal(_np(g.get_boards()), b), t
            assert np.array_equal(_np(obs.view(torch.int16)).view(np.uint16), o.encode_obs()), t
            ages += int((b[:, 122:124] >= 2).sum())
    assert ages > 0  # chases of two positions and more did occur
    assert g.check() == 0
