"""The chasing rule's memory across non-initial resets ("the continuous chasing rule
needs to be tested against the history of board states that leads to the non-initial reset state")
on the CUDA path: loads with plies, pinned restarts, determinised copies / search expansion and
the board-history ring (past masks, travel back) against the oracle."""
import numpy as np
import pytest
import torch

from chase_scenarios import cage, crowded
from oracle import orc
from paper_2511_07312_b200 import binding as B
from paper_2511_07312_b200 import workloads as W
from test_gpu_chase import _biased_actions

pytestmark = pytest.mark.gpu
A = W.action_index
RING = [31, 32, 33, 34, 44, 54, 64, 63, 62, 61, 51, 41]  # the 12 squares around the lake {42,43,52,53}


def _np(t):
    return t.detach().cpu().numpy()


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _mask_np(t):
    return _np(t).view(np.uint32)


def _act(a, b):
    return A(a, {10: 0, 1: 1, -10: 2, -1: 3}[b - a], 1)


def _lap(extra=()):
    """The lake lap played on the oracle: (line after 24 plies, the plies most recent first)."""
    pieces = {RING[0]: W.piece(W.CAPTAIN, W.RED), RING[2]: W.piece(W.SERGEANT, W.BLUE), 9: W.piece(W.FLAG, W.RED),
              99: W.piece(W.FLAG, W.BLUE)}
    pieces.update(extra)
    o = orc.Env(1, chase_rule=1)
    o.reset_from(W.make_line(pieces)[None, :])
    played = []
    for k in range(12):
        for f, t in ((RING[k % 12], RING[(k + 1) % 12]), (RING[(k + 2) % 12], RING[(k + 3) % 12])):
            o.step(np.array([_act(f, t)], np.int16))
            played.append((f, t))
    plies = np.full((63, 2), 0xFF, np.uint8)
    plies[:24] = played[::-1]
    return W.make_line(pieces), o.get_boards()[0], plies, played


def test_lap_split_across_a_load_with_plies():
    _, lap, plies, _ = _lap()
    again = _act(RING[0], RING[1])
    n = 4  # all 24 plies, 23, 22, none
    P = np.repeat(plies[None], n, axis=0)
    P[1, 23:] = 0xFF; P[2, 22:] = 0xFF; P[3, :] = 0xFF
    lines = np.repeat(lap[None], n, axis=0)
    for rule in (1, 0):
        g, o = B.Env(n, chase_rule=rule), orc.Env(n, chase_rule=rule)
        g.reset_from(_dev(lines), _dev(P)); o.reset_from(lines, P)
        om = o.legal_mask()
        assert [again in W.mask_to_actions(om[i]) for i in range(n)] == ([False, False, True, True] if rule else [True] * 4)
        assert np.array_equal(_mask_np(g.legal_mask()), om)
        mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
        for _ in range(12):  # played on: the handed-over plies and the new ones form one log
            om = o.legal_mask(); oa = o.sample_uniform(om); o.step(oa)
            g.rollout_step(mask, act, rew, done, obs)
            assert np.array_equal(_mask_np(mask), om) and np.array_equal(_np(act), oa)
        assert np.array_equal(_np(g.get_boards()), o.get_boards())
        assert g.check() == 0
    g = B.Env(n, chase_rule=1)
    g.reset_from(_dev(lines), _dev(P))
    g.step(_dev(np.full(n, again, np.int16)))
    assert g.check() == B.ILLEGAL_ACTION


def test_malformed_plies_end_the_known_plies():
    """A ply with a square >= 100 (or a known `from` with `to` = 0xFF) names no move: it ends the known
    plies exactly like 0xFF,0xFF instead of becoming a log entry that collides with a real one."""
    _, lap, plies, _ = _lap()
    n = 5
    bad = np.repeat(plies[None], n, axis=0)
    bad[0, 20] = (100, 5); bad[1, 20] = (37, 0xFF); bad[2, 20] = (200, 201); bad[3, 0] = (44, 130)   # game 4: intact
    cut = np.repeat(plies[None], n, axis=0)
    cut[0:3, 20:] = 0xFF; cut[3, :] = 0xFF
    lines = np.repeat(lap[None], n, axis=0)
    g, ref, o = B.Env(n, chase_rule=1), B.Env(n, chase_rule=1), orc.Env(n, chase_rule=1)
    g.reset_from(_dev(lines), _dev(bad)); ref.reset_from(_dev(lines), _dev(cut)); o.reset_from(lines, cut)
    assert torch.equal(g.legal_mask(), ref.legal_mask())
    assert np.array_equal(_mask_np(g.legal_mask()), o.legal_mask())
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for _ in range(30):
        om = o.legal_mask(); oa = o.sample_uniform(om); o.step(oa)
        g.rollout_step(mask, act, rew, done, obs)
        assert np.array_equal(_mask_np(mask), om) and np.array_equal(_np(act), oa)
    assert g.check() == 0
    # the same through a pin
    pin = B.Env(n, chase_rule=1, max_plies=30, auto_reset=1, seed=5)
    pin_ref = B.Env(n, chase_rule=1, max_plies=30, auto_reset=1, seed=5)
    pin.pin_reset_state(_dev(lines), _dev(bad)); pin_ref.pin_reset_state(_dev(lines), _dev(cut))
    pin.reset_from(_dev(lines), _dev(bad)); pin_ref.reset_from(_dev(lines), _dev(cut))
    m2 = pin_ref.new_mask()
    for _ in range(20):  # restarts from the pin inside (the ply cap ends every game after 6 plies)
        pin.rollout_step(mask, act, rew, done, obs)
        pin_ref.rollout_step(m2, act, rew, done, obs)
        assert torch.equal(mask, m2)
    assert torch.equal(pin.get_boards(), pin_ref.get_boards())


@pytest.mark.parametrize("with_plies", [True, False])
def test_pinned_restart_remembers_the_plies_of_its_pin(with_plies):
    extra = {8: W.piece(W.MINER, W.RED), 98: W.piece(W.MINER, W.BLUE)}
    _, lap, plies, _ = _lap(extra)
    again = _act(RING[0], RING[1])
    n = 96
    lines, P = np.repeat(lap[None], n, axis=0), np.repeat(plies[None], n, axis=0)
    kw = dict(seed=5, chase_rule=1, max_plies=30, auto_reset=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    g.reset_from(_dev(lines), _dev(P)); o.reset_from(lines, P)
    if with_plies:
        g.pin_reset_state(_dev(lines), _dev(P)); o.pin_reset_state(lines, P)
    else:
        g.pin_reset_state(_dev(lines)); o.pin_reset_state(lines)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    restarts = 0
    for t in range(40):  # the ply cap ends every game after 6 plies
        om = o.legal_mask()
        if t % 6 == 0:
            legal0 = [again in W.mask_to_actions(om[i]) for i in range(n)]
            assert legal0 == [not (with_plies or t == 0)] * n, t
        oa = o.sample_uniform(om); orr, od = o.step(oa)
        restarts += int((od & 1).sum())
        kind = t % 3
        if kind == 0:
            g.rollout_step(mask, act, rew, done, obs)
            assert np.array_equal(_mask_np(mask), om) and np.array_equal(_np(act), oa), t
        elif kind == 1:
            assert np.array_equal(_mask_np(g.legal_mask()), om), t
            g.step(_dev(oa), rew, done)
        else:
            g.step_observe(_dev(oa), rew, done, mask, obs)
            assert np.array_equal(_mask_np(mask), o.legal_mask()), t
        assert np.array_equal(_np(rew), orr) and np.array_equal(_np(done), od), t
        assert np.array_equal(_np(g.get_boards()), o.get_boards()), t
    assert restarts == 6 * n and g.check() == 0
    # the on-chip rollouts restart from the pin as well
    g.rollout_uniform(14)
    for _ in range(14):
        o.step(o.sample_uniform(o.legal_mask()))
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert np.array_equal(_mask_np(g.legal_mask()), o.legal_mask())


def _chase_heavy(n, seed, plies_played, history=None):
    """n little chase-heavy games played for a while with the biased test policy on both sides."""
    rng = np.random.default_rng(seed)
    lines = np.zeros((n, 128), np.uint8)
    for i in range(n):
        lines[i] = W.make_line(cage(rng) if i % 8 else crowded(rng))
    kw = dict(variant=0, seed=seed, max_plies=90, auto_reset=1, chase_rule=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    g.reset_from(_dev(lines)); o.reset_from(lines)
    g.pin_reset_state(_dev(lines)); o.pin_reset_state(lines)
    if history is not None:
        history.attach(g)
    rew, done = g.new_reward(), g.new_done()
    recs = []
    for t in range(plies_played):
        boards, om = o.get_boards(), o.legal_mask()
        a = _biased_actions(om, boards, rng)
        recs.append(dict(boards=boards, mask=om, act=a))
        o.step(a)
        g.step(_dev(a), rew, done)
    return g, o, recs, kw, lines


def _eight_ply_mask(boards):
    o8 = orc.Env(len(boards), chase_rule=1)
    o8.reset_from(boards)
    return o8.legal_mask()


def test_determinised_copies_and_search_expansion_inherit_the_chase_memory():
    R, S = 160, 12
    g, o, _, kw, _ = _chase_heavy(R, 21, 37)
    om = o.legal_mask()
    assert np.array_equal(_mask_np(g.legal_mask()), om)
    long_bans = int(np.unpackbits((_eight_ply_mask(o.get_boards()) ^ om).view(np.uint8)).sum())
    assert long_bans > 0  # some roots carry bans that only the move log explains
    kwo = dict(kw, auto_reset=0)
    go, gg = orc.Env(R * S, **kwo), B.Env(R * S, **kwo)
    orc.determinise(o, S, 99, go); B.determinise(g, S, 99, gg)
    assert np.array_equal(_np(gg.get_boards()), go.get_boards())
    dm = go.legal_mask()
    assert np.array_equal(_mask_np(gg.legal_mask()), dm)
    assert int(np.unpackbits((_eight_ply_mask(go.get_boards()) ^ dm).view(np.uint8)).sum()) > 0
    for _ in range(6):
        go.step(go.sample_uniform(go.legal_mask()))
    gg.rollout_uniform(6)
    assert np.array_equal(_np(gg.get_boards()), go.get_boards())
    # search expansion: configurations x legal actions with the forced first move appended to the inherited log
    rollouts = 40
    eo, eg = orc.Env(R * rollouts, **kwo), B.Env(R * rollouts, **kwo)
    orc.search_expand(o, rollouts, 7, eo); B.search_expand(g, rollouts, 7, eg)
    assert np.array_equal(_np(eg.get_boards()), eo.get_boards())
    assert np.array_equal(_mask_np(eg.legal_mask()), eo.legal_mask())
    for _ in range(5):
        eo.step(eo.sample_uniform(eo.legal_mask()))
    eg.rollout_uniform(5)
    assert np.array_equal(_np(eg.get_boards()), eo.get_boards())
    assert gg.check() == 0 and eg.check() == 0 and g.check() == 0


def test_past_masks_and_travel_back_with_the_chasing_rule():
    """A past mask is the mask that WAS: long chases (> 8 plies) are judged with the plies the ring
    holds.  Then travel back and replay forward."""
    n, length, T = 240, 100, 150
    h = B.History(n, length)
    g, o, recs, kw, lines = _chase_heavy(n, 8, T, history=h)
    long_bans, oldest = 0, T - length
    for t in range(oldest, T):
        pm = _mask_np(h.legal_mask(t))
        # the ring holds t - oldest plies before time step t (the line itself 8): every game whose chases
        # are no older than that gets the mask it had; from oldest + 63 on that is every game
        ages = recs[t]["boards"][:, 122:124].astype(np.int32).max(axis=1)
        sure = np.minimum(ages - 1, 63) <= max(8, t - oldest)
        assert sure.all() or t < oldest + 63
        assert np.array_equal(pm[sure], recs[t]["mask"][sure]), t
        if t % 8 == 0:
            long_bans += int(np.unpackbits((_eight_ply_mask(recs[t]["boards"]) ^ pm).view(np.uint8)).sum())
    assert long_bans > 0
    assert np.array_equal(_mask_np(h.legal_mask(T)), o.legal_mask())  # the live state
    # travel back into a second environment (and into the attached one) and replay the recorded actions
    t0 = T - 36
    g2 = B.Env(n, **kw)
    g2.pin_reset_state(_dev(lines))
    h.restore(t0, g2)
    rew, done = g2.new_reward(), g2.new_done()
    for t in range(t0, T):
        assert np.array_equal(_mask_np(g2.legal_mask()), recs[t]["mask"]), t
        g2.step(_dev(recs[t]["act"]), rew, done)
    assert np.array_equal(_np(g2.get_boards()), o.get_boards())
    assert np.array_equal(_mask_np(g2.legal_mask()), o.legal_mask())
    assert g2.check() == 0 and g.check() == 0


def test_lake_lap_through_the_history_ring():
    start, _, _, played = _lap()
    again, back = _act(RING[0], RING[1]), _act(RING[0], RING[11])
    n = 33
    for length, remembered in ((32, True), (16, False)):
        g = B.Env(n, chase_rule=1)
        g.reset_from(_dev(np.repeat(start[None], n, axis=0)))
        h = B.History(n, length)
        h.attach(g)
        for f, t in played:
            g.step(_dev(np.full(n, _act(f, t), np.int16)))
        live = W.mask_to_actions(_mask_np(g.legal_mask())[0])
        assert again not in live and back in live
        g.step(_dev(np.full(n, back, np.int16)))                          # X steps back,
        g.step(_dev(np.full(n, _act(RING[2], RING[3]), np.int16)))        # Y walks on
        assert h.current_step() == 26
        past = _mask_np(h.legal_mask(24))
        for i in (0, n - 1):
            acts = W.mask_to_actions(past[i])
            assert (again not in acts) == remembered and back in acts
            assert (acts == live) == remembered
        g2 = B.Env(n, chase_rule=1)
        h.restore(24, g2)
        acts = W.mask_to_actions(_mask_np(g2.legal_mask())[n - 1])
        assert (again not in acts) == remembered
        g3 = B.Env(n, chase_rule=0)  # an environment without the rule takes the state and ignores the plies
        h.restore(24, g3)
        assert again in W.mask_to_actions(_mask_np(g3.legal_mask())[0])
        assert g.check() == 0 and g2.check() == 0
