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


def test_history_shape_checks():
    assert B.lib().strat_history_bytes(0, 4) == 0 and B.lib().strat_history_bytes(4, 0) == 0
    assert B.lib().strat_history_bytes(65536, 256) == 65536 * 256 * 132
    g = B.Env(64, seed=1)
    h = B.History(32, 4)
    with pytest.raises(B.StratError):
        h.attach(g)  # game counts differ
