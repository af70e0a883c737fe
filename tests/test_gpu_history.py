"""The board-history ring (Table S1 455-480): a historical query at time
step t must return what the quantity WAS at time t.  The expected values are the CPU oracle's
live outputs, recorded step by step."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_2511_07312_b200 import binding as B

pytestmark = pytest.mark.gpu


def _np(t):
    return t.detach().cpu().numpy()


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _live_record(o):
    """what the oracle says about its current state (time step t), then one uniform ply"""
    b = o.get_boards()
    m = o.legal_mask()
    obs = o.encode_obs()
    a = o.sample_uniform(m)
    r, d = o.step(a)
    ply = b[:, 116].astype(np.int32) | (b[:, 117].astype(np.int32) << 8)
    batl = b[:, 118].astype(np.int32) | (b[:, 119].astype(np.int32) << 8)
    info = np.stack([ply & 1, ply, batl, b[:, 120].astype(np.int32)], axis=1).astype(np.int32)
    return dict(boards=b, mask=m, obs=obs, act=a, rew=r, done=d, info=info)


def _check_time_step(h, t, rec, live=False):
    assert np.array_equal(_np(h.get_boards(t)), rec["boards"]), t
    assert np.array_equal(_np(h.legal_mask(t)).view(np.uint32), rec["mask"]), t
    assert np.array_equal(_np(h.encode_obs(t).view(torch.int16)).view(np.uint16), rec["obs"]), t
    assert np.array_equal(_np(h.info(t)), rec["info"]), t
    if not live:
        a, r, d = h.transition(t)
        assert np.array_equal(_np(a), rec["act"]) and np.array_equal(_np(r), rec["rew"]), t
        assert np.array_equal(_np(d), rec["done"]), t


@pytest.mark.parametrize("variant,n,length,cap", [(0, 300, 16, 45), (1, 77, 5, 300)])
def test_historical_queries_equal_live_oracle_values(variant, n, length, cap):
    kw = dict(variant=variant, seed=11, max_plies=cap, auto_reset=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    h = B.History(n, length)
    h.attach(g)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    recs = []
    for t in range(60):
        recs.append(_live_record(o))
        if t % 4 == 3:  # the separate calls record as well
            g.step(g.sample_uniform(g.legal_mask()), rew, done)
        else:
            g.rollout_step(mask, act, rew, done, obs)
        cur = h.current_step()
        assert cur == t + 1
        if t % 7 == 0 or t == 59:
            for q in range(max(0, cur - length), cur):
                _check_time_step(h, q, recs[q])
    # the live state is time step `cur`
    live = _live_record(o)
    _check_time_step(h, 60, live, live=True)
    # outside the ring
    for bad in (-1, 60 - length - 1, 61):
        with pytest.raises(B.StratError):
            h.legal_mask(bad)
    with pytest.raises(B.StratError):
        h.transition(60)
    with pytest.raises(B.StratError):
        g.rollout_uniform(3)  # on-chip plies would not be recorded
    assert g.check() == 0


def test_history_of_overlapped_fused_steps_and_restore():
    """200 fused steps launched back to back (they overlap on the device) with a 64-step ring;
    then travel back 37 steps into a second environment and replay forward."""
    n, length, steps = 2048 + 40, 64, 200
    kw = dict(variant=0, seed=3, max_plies=120, auto_reset=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    h = B.History(n, length)
    h.attach(g)
    obs = g.new_obs()
    for _ in range(steps):
        g.rollout_step(None, None, None, None, obs)
    recs = {}
    for t in range(steps):
        rec = _live_record(o)
        if t >= steps - length:
            recs[t] = rec
    for t in (steps - length, steps - 37, steps - 1):
        _check_time_step(h, t, recs[t])
    g2 = B.Env(n, **kw)
    h.restore(steps - 37, g2)
    assert np.array_equal(_np(g2.get_boards()), recs[steps - 37]["boards"])
    for t in range(steps - 37, steps):  # the action stream is keyed by (game, epoch, ply): replays exactly
        a, r, d = g2.sample_uniform(g2.legal_mask()), None, None
        assert np.array_equal(_np(a), recs[t]["act"]), t
        r, d = g2.step(a)
        assert np.array_equal(_np(r), recs[t]["rew"]) and np.array_equal(_np(d), recs[t]["done"]), t
    assert torch.equal(g2.get_boards(), g.get_boards())
    h.detach()
    g.rollout_uniform(2)  # allowed again
    assert h.current_step() == steps
    assert g.check() == 0 and g2.check() == 0


INFO_GROUPS = ((43, 109), (109, 131), (131, 251), (251, 355), (455, 487))   # S2 tracker-fed channel groups


def _info487(t):
    return t.view(torch.int16).cpu().numpy().view(np.uint16).reshape(t.shape[0], 487, 100)


@pytest.mark.parametrize("variant,n,length,cap,chase", [(0, 150, 12, 45, 0), (1, 77, 5, 300, 1), (0, 40, 16, 70, 1)])
def test_historical_infostate_487_equals_live_oracle_values(variant, n, length, cap, chase):
    """ComputeInfostateTensor(t) in the paper's own 487 channels from a tracked ring:
    all 48,700 values of every game at every ring position equal what the oracle's live encoder said at that
    time step - across wrap-around, auto-resets, pinned restarts, all three step calls - and travelling back
    (strat_history_restore) brings the trackers along, so that play continues with the same tensors."""
    steps = 64
    kw = dict(variant=variant, seed=13, max_plies=cap, auto_reset=1, infostate=1, chase_rule=chase)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    h = B.History(n, length, tracked=True)
    h.attach(g)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    recs, acts = {}, {}
    seen = np.zeros(len(INFO_GROUPS), bool)
    for t in range(steps):
        if t == 20:   # from here on finished games restart from a pinned mid-game state
            b = o.get_boards()
            g.pin_reset_state(_dev(b)); o.pin_reset_state(b)
        recs[t] = o.encode_infostate().reshape(n, 487, 100).copy()
        seen |= np.array([recs[t][:, a:b].any() for a, b in INFO_GROUPS])
        recs.pop(t - length - 1, None)
        a = o.sample_uniform(o.legal_mask())
        acts[t] = a
        o.step(a)
        if t % 3 == 0:
            g.rollout_step(mask, act, rew, done, obs)
        elif t % 3 == 1:
            g.step(g.sample_uniform(g.legal_mask()), rew, done)
        else:
            g.step_observe(_dev(a), rew, done, mask, obs)
        cur = h.current_step()
        if t % 9 == 0 or t == steps - 1:
            for q in range(max(0, cur - length), cur):
                got = _info487(h.encode_infostate(q))
                assert np.array_equal(got, recs[q]), (t, q, np.argwhere(got != recs[q])[:4].tolist())
    assert seen.all(), seen   # no channel group passed because it was empty
    assert (o.get_boards()[:, 124] > 0).any()   # games restarted inside the window
    # the live state is time step cur
    assert np.array_equal(_info487(h.encode_infostate(steps)), o.encode_infostate().reshape(n, 487, 100))
    assert torch.equal(h.encode_infostate(steps).view(torch.int16), g.encode_infostate().view(torch.int16))
    # travel back: state, move log and trackers of time step q in a second environment, then the same plies again
    q = steps - min(length, 9)
    g2 = B.Env(n, **kw)
    h.restore(q, g2)
    assert np.array_equal(_info487(g2.encode_infostate()), recs[q])
    for t in range(q, steps):
        if (acts[t] < 0).any():
            break
        r2, d2 = g2.step(_dev(acts[t]))
        if (_np(d2) & 1).any():   # a restart would need g's pin in g2: stop comparing there
            break
        if t + 1 < steps:
            assert np.array_equal(_info487(g2.encode_infostate()), recs[t + 1]), t
    # outside the ring / not tracked
    with pytest.raises(B.StratError):
        h.encode_infostate(steps - length - 1)
    plain = B.History(n, length)
    h.detach()
    plain.attach(g)
    g.rollout_step(mask, act, rew, done, obs)
    with pytest.raises(B.StratError, match="bad state"):
        plain.encode_infostate(0)
    assert h.current_step() == steps
    assert np.array_equal(_info487(h.encode_infostate(steps - 1)), recs[steps - 1])   # a detached ring still answers
    assert g.check() == 0 and g2.check() == 0


def test_history_shape_checks():
    assert B.lib().strat_history_bytes(0, 4) == 0 and B.lib().strat_history_bytes(4, 0) == 0
    assert B.lib().strat_history_bytes(65536, 256) == 65536 * 256 * 132 + 65536 * 128  # ring + one scratch move log per game
    g = B.Env(64, seed=1)
    h = B.History(32, 4)
    with pytest.raises(B.StratError):
        h.attach(g)  # game counts differ


def test_two_square_applies_unknown_pieces_terminated_since():
    """The remaining Table S1 queries against plain restatements: the rule
    'applies' iff switching it off changes the oracle's mask; a piece is unknown iff it is the
    opponent's and unrevealed; terminated-since counts the steps since the ending action."""
    n, length, cap = 400, 12, 70
    kw = dict(variant=0, seed=23, max_plies=cap, auto_reset=0)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    o_off = orc.Env(n, **dict(kw, two_square=0))
    h = B.History(n, length)
    h.attach(g)
    obs = g.new_obs()
    recs, ended_at = [], np.full(n, -1)
    applied = 0
    for t in range(cap + 9):
        b = o.get_boards()
        o_off.reset_from(b)
        ts = (o.legal_mask() != o_off.legal_mask()).any(axis=1).astype(np.uint8)
        side = (b[:, 116] & 1)[:, None]
        cells = b[:, :100]
        piece = ((cells & 15) >= 1) & ((cells & 15) <= 12)
        unk = (piece & (((cells >> 4) & 1) != side) & ((cells & 0x40) == 0)).astype(np.uint8)
        finished = (b[:, 120] & 1) == 1
        since = np.where(finished, t - ended_at, 0).astype(np.int32)
        recs.append((ts, unk, since))
        applied += int(ts.sum())
        r, d = o.step(o.sample_uniform(o.legal_mask()))
        newly = ((d & 1) == 1) & (ended_at < 0)
        ended_at[newly] = t
        g.rollout_step(None, None, None, None, obs)
    cur = h.current_step()
    assert cur == cap + 9 and applied > 0 and (ended_at >= 0).all()
    for t in range(cur - length, cur):
        ts, unk, since = h.flags(t)
        e_ts, e_unk, e_since = recs[t]
        assert np.array_equal(_np(ts), e_ts), t
        assert np.array_equal(_np(unk), e_unk), t
        depth = t - (cur - length)                      # steps before t that are still in the ring
        assert np.array_equal(_np(since), np.minimum(e_since, depth)), t
    # the live state: every game is frozen since `cur - ended_at` steps, seen through 12 ring steps
    ts, unk, since = h.flags(cur)
    assert not _np(ts).any() and (_np(since) == np.minimum(cur - ended_at, length)).all()
    assert g.check() == 0
