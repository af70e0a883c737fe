"""Parity of the CUDA path's 487-channel information state (strat_encode_infostate)
with the oracle's: all 48,700 bf16 values of every game bit for bit - the 0/1 and +-1 channels
exactly, and the real-valued ones (type posteriors 12-35, fractions 41-42) too, because both
sides round the same IEEE double quotient once to bf16 (reading I8)."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_2511_07312_b200 import binding as B
from paper_2511_07312_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _info_np(t):
    return t.view(torch.int16).cpu().numpy().view(np.uint16)


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _diff(got, want):
    bad = np.argwhere(got != want)
    return [(int(g), int(c), int(s // 10), int(s % 10)) for g, c, s in bad.reshape(-1, 3)[:6]] if bad.size else []


def _check(g, o, tag):
    got = _info_np(g.encode_infostate()).reshape(g.n, 487, 100)
    want = o.encode_infostate().reshape(o.n, 487, 100)
    assert np.array_equal(got, want), (tag, _diff(got, want))


@pytest.mark.parametrize("variant,n,cap,kbl,fused", [(0, 77, 90, 0, True), (1, 130, 400, 25, True), (0, 64, 120, 40, False)])
def test_infostate_random_play_with_auto_reset(variant, n, cap, kbl, fused):
    kw = dict(variant=variant, seed=6, max_plies=cap, max_battleless=kbl, auto_reset=1, infostate=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    _check(g, o, "start")
    for t in range(300):
        if fused:
            g.rollout_step(mask, act, rew, done, obs)
        else:
            g.step(g.sample_uniform(g.legal_mask()))
        o.step(o.sample_uniform(o.legal_mask()))
        if t % 9 == 8 or t < 6:
            _check(g, o, t)
    assert np.array_equal(g.get_boards().cpu().numpy(), o.get_boards())
    assert (o.get_boards()[:, 124] > 0).any()  # trackers restarted inside steps (auto-reset)
    assert g.check() == 0


def test_infostate_step_observe_and_larger_batch():
    """External actions (strat_step_observe, the data-collection shape) on 3,000 games: the
    trackers are updated by the kExternal variant of the fused kernel."""
    n = 3000
    kw = dict(variant=0, seed=2, max_plies=70, auto_reset=1, infostate=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    mask, rew, done, obs = g.new_mask(), g.new_reward(), g.new_done(), g.new_obs()
    for t in range(100):
        oa = o.sample_uniform(o.legal_mask())
        o.step(oa)
        g.step_observe(_dev(oa), rew, done, mask, obs)
        if t % 33 == 32:
            _check(g, o, t)
    assert g.check() == 0


def test_infostate_hand_built_games():
    """The oracle's hand-worked mini-games (tests/test_oracle_infostate.py) through the CUDA path:
    loaded with strat_reset_from, played with strat_step, every game in one batch."""
    R, Bl = 0, 1
    games = [
        ({0: W.piece(W.FLAG, R), 99: W.piece(W.FLAG, Bl), 24: W.piece(W.SERGEANT, R), 35: W.piece(W.CAPTAIN, Bl)},
         [(24, 0, 1), (35, 1, 1)]),
        ({0: W.piece(W.FLAG, R), 99: W.piece(W.FLAG, Bl), 24: W.piece(W.GENERAL, R, revealed=True),
          35: W.piece(W.MINER, Bl, revealed=True), 44: W.piece(W.SCOUT, Bl)}, [(24, 0, 1), (35, 1, 1), (34, 0, 1)]),
        ({0: W.piece(W.FLAG, R), 99: W.piece(W.FLAG, Bl), 24: W.piece(W.MAJOR, R, revealed=True),
          35: W.piece(W.MINER, Bl, revealed=True), 26: W.piece(W.CAPTAIN, Bl)}, [(24, 0, 1), (26, 0, 1), (34, 2, 1)]),
        ({0: W.piece(W.FLAG, R), 99: W.piece(W.FLAG, Bl), 24: W.piece(W.MAJOR, R), 26: W.piece(W.CAPTAIN, Bl),
          81: W.piece(W.SERGEANT, Bl)}, [(24, 0, 1), (26, 0, 1)]),
        ({0: W.piece(W.FLAG, R), 99: W.piece(W.FLAG, Bl),
          10: W.piece(W.SERGEANT, R), 20: W.piece(W.CAPTAIN, Bl, revealed=True),
          72: W.piece(W.LIEUTENANT, Bl), 62: W.piece(W.LIEUTENANT, R, revealed=True),
          14: W.piece(W.MAJOR, R), 24: W.piece(W.COLONEL, Bl), 76: W.piece(W.GENERAL, Bl), 66: W.piece(W.CAPTAIN, R, revealed=True),
          18: W.piece(W.MARSHAL, R), 28: W.piece(W.SCOUT, Bl), 79: W.piece(W.MINER, Bl), 69: W.piece(W.BOMB, R)},
         [(10, 0, 1), (72, 2, 1), (14, 0, 1), (76, 2, 1), (18, 0, 1), (79, 2, 1)]),
        ({0: W.piece(W.FLAG, R), 99: W.piece(W.FLAG, Bl), 10: W.piece(W.MINER, R), 20: W.piece(W.MINER, Bl),
          50: W.piece(W.SPY, R), 59: W.piece(W.SPY, Bl)}, [(10, 0, 1)]),
        # a Scout's long move reveals it (R10): the key of what it protects with / threatens as changes
        ({0: W.piece(W.FLAG, R), 99: W.piece(W.FLAG, Bl), 24: W.piece(W.MAJOR, R), 35: W.piece(W.MINER, Bl),
          85: W.piece(W.SCOUT, Bl)}, [(24, 0, 1), (85, 2, 4)]),  # 85 -> 45 along column 5, next to the Miner
    ]
    n = len(games)
    lines = np.stack([W.make_line(p) for p, _ in games])
    kw = dict(variant=0, seed=1, max_plies=4000, max_battleless=200, infostate=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    g.reset_from(_dev(lines)); o.reset_from(lines)
    _check(g, o, "loaded")
    for t in range(max(len(m) for _, m in games)):
        # a game whose script is over plays its first legal action
        om = o.legal_mask()
        a = np.array([W.action_index(*m[t]) if t < len(m) else W.mask_to_actions(om[k])[0] for k, (_, m) in enumerate(games)], np.int16)
        o.step(a); g.step(_dev(a))
        assert o.check() == 0 and g.check() == 0
        _check(g, o, t)


def test_infostate_after_loads_restores_and_pinned_restarts():
    """Reading I9: a loaded position is where the trackers start - strat_reset_from, a pinned
    restart, strat_history_restore, strat_determinise into an environment with infostate."""
    n = 96
    kw = dict(variant=0, seed=13, max_plies=60, auto_reset=1, infostate=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for _ in range(45):
        g.rollout_step(mask, act, rew, done, obs); o.step(o.sample_uniform(o.legal_mask()))
    b = o.get_boards()
    g.reset_from(_dev(b)); o.reset_from(b)          # load: histories of the lines become the known moves
    _check(g, o, "reset_from")
    g.pin_reset_state(_dev(b)); o.pin_reset_state(b)  # every game that ends restarts from its pinned line
    for t in range(50):
        g.rollout_step(mask, act, rew, done, obs); o.step(o.sample_uniform(o.legal_mask()))
        if t % 10 == 9:
            _check(g, o, ("pinned", t))
    assert (o.get_boards()[:, 124] > 0).any()
    g.pin_reset_state(None); o.pin_reset_state(None)
    # history restore
    hist = B.History(n, 8)
    hist.attach(g)
    snap = None
    for t in range(6):
        if t == 2:
            snap = o.get_boards()
        g.rollout_step(mask, act, rew, done, obs); o.step(o.sample_uniform(o.legal_mask()))
    hist.restore(2, g); o.reset_from(snap)
    _check(g, o, "restore")
    hist.detach()
    for t in range(12):
        g.rollout_step(mask, act, rew, done, obs); o.step(o.sample_uniform(o.legal_mask()))
    _check(g, o, "after restore")
    # determinise into a tracked environment
    roots_g, roots_o = B.Env(4, seed=13), orc.Env(4, seed=13)
    live = [k for k in range(n) if not (o.get_boards()[k, 120] & 1)][:4]
    rb = o.get_boards()[live]
    roots_g.reset_from(_dev(rb)); roots_o.reset_from(rb)
    out_g = B.Env(4 * 16, seed=13, infostate=1); out_o = orc.Env(4 * 16, seed=13, infostate=1)
    B.determinise(roots_g, 16, 99, out_g); orc.determinise(roots_o, 16, 99, out_o)
    _check(out_g, out_o, "determinise")
    assert g.check() == 0


def test_infostate_into_a_buffer_at_8_mod_16():
    """`out` need only be 8-byte aligned (strat.h).  A game is 97,400 B = 8 mod 16, so big[1:] of a larger
    tensor starts at 8 mod 16 and the games whose first nibble goes out alone are the even ones there."""
    n = 77
    kw = dict(variant=0, seed=4, max_plies=60, auto_reset=1, infostate=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for _ in range(75):
        g.rollout_step(mask, act, rew, done, obs)
        o.step(o.sample_uniform(o.legal_mask()))
    big = torch.full((n + 2, 487, 10, 10), 7.0, dtype=torch.bfloat16, device="cuda")
    out = big[1:n + 1]
    assert out.data_ptr() % 16 == 8 and out.is_contiguous()
    g.encode_infostate(out)
    want = o.encode_infostate().reshape(n, 487, 100)
    got = _info_np(out).reshape(n, 487, 100)
    assert np.array_equal(got, want), _diff(got, want)
    assert torch.equal(out.view(torch.int16), g.encode_infostate().view(torch.int16))   # = the 16-byte aligned call
    assert bool((big[0] == 7.0).all()) and bool((big[n + 1] == 7.0).all())               # neighbours untouched
    assert g.check() == 0


def test_infostate_encodes_in_flight_together_on_two_streams():
    """Two strat_encode_infostate calls of one environment on two streams, more games than the encoder has
    CTAs (games handed out by ticket): each call draws from a work counter of its own, so neither skips
    or repeats a game, and the counters are back at zero for the next round."""
    n = 20000
    g = B.Env(n, variant=0, seed=8, max_plies=40, auto_reset=1, infostate=1)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for _ in range(50):
        g.rollout_step(mask, act, rew, done, obs)
    want = g.encode_infostate().view(torch.int16)
    outs = [g.new_infostate(), g.new_infostate()]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for rnd in range(70):   # more rounds than there are counters: the rotation wraps
        for out, st in zip(outs, streams):
            if rnd % 10 == 0:
                out.fill_(3.0)
            st.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(st):
                g.encode_infostate(out)
        if rnd % 10 == 0:
            torch.cuda.synchronize()
            for out in outs:
                assert torch.equal(out.view(torch.int16), want), rnd
    torch.cuda.synchronize()
    for out in outs:
        assert torch.equal(out.view(torch.int16), want)
    assert g.check() == 0


def test_infostate_argument_errors():
    L, s = B.lib(), B._stream()
    plain = B.Env(40, seed=1)
    out = torch.empty((40, 487, 10, 10), dtype=torch.bfloat16, device="cuda")
    assert L.strat_encode_infostate(plain.h, B._ptr(out), s) == B.BAD_STATE  # no trackers kept
    tracked = B.Env(40, seed=1, infostate=1)
    assert L.strat_encode_infostate(tracked.h, None, s) == B.BAD_ARG
    assert L.strat_rollout_uniform(tracked.h, 4, s) == B.BAD_STATE  # on-chip plies are not tracked
    bad = B.strat_config(10, 0, 0, 0, 0, 0, 1, 0, 0, 0, 2, 0)
    import ctypes as C
    assert L.strat_workspace_bytes(C.byref(bad)) == 0
    assert tracked.check() == 0


def test_infostate_full_size_ticketed_encoder():
    """65,536 games (the bench shape: more games than the encoder has CTAs, so games are handed out by its
    self-resetting ticket counter), trackers kept by overlapped fused steps; four slices of 16 games spread
    over the batch are mirrored by oracle shards keyed by their global game index.  Encoded twice: the
    counter must have cleaned up after the first pass."""
    n, steps = 65536, 45
    kw = dict(variant=0, seed=12, max_plies=30, auto_reset=1, infostate=1)   # 30-ply cap: resets inside the window
    g = B.Env(n, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for _ in range(steps):
        g.rollout_step(mask, act, rew, done, obs)
    first = g.encode_infostate()
    second = g.encode_infostate(g.new_infostate())
    assert torch.equal(first.view(torch.int16), second.view(torch.int16))
    got = first.view(torch.int16)
    for base in (0, 1777, 30001, 65520):
        o = orc.Env(16, game_base=base, **kw)
        for _ in range(steps):
            o.step(o.sample_uniform(o.legal_mask()))
        want = o.encode_infostate().reshape(16, -1)
        have = got[base:base + 16].cpu().numpy().view(np.uint16).reshape(16, -1)
        assert np.array_equal(have, want), base
    # every game was written: channel 38 (empty) + lakes + pieces cover the board, so no row is all zero
    assert bool((got.view(n, -1) != 0).any(dim=1).all())
    assert g.check() == 0
