"""Parity of the CUDA path (through the C ABI) with the CPU oracle: bit-exact boards, masks,
actions, rewards, done bytes and bf16 planes on the same seeded inputs."""
import json
import os

import numpy as np
import pytest
import torch

from oracle import orc
from paper_2511_07312_b200 import binding as B
from paper_2511_07312_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _np(t):
    return t.detach().cpu().numpy()


def _mask_np(t):
    return _np(t).view(np.uint32)


def _obs_np(t):
    return _np(t.view(torch.int16)).view(np.uint16)


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _pair(n, **kw):
    return B.Env(n, **kw), orc.Env(n, **kw)


# ----------------------------------------------------------------------------- reset / lines
@pytest.mark.parametrize("variant,n,seed,base", [(0, 300, 0, 0), (1, 77, 5, 0), (0, 33, 2**40 + 7, 1000)])
def test_reset_matches_oracle(variant, n, seed, base):
    g, o = _pair(n, variant=variant, seed=seed, game_base=base)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    g.reset(seed + 1); o.reset(seed + 1)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert g.check() == 0


def test_reset_from_get_boards_roundtrip_on_oracle_positions():
    o = orc.Env(203, seed=3, max_plies=500, auto_reset=1)
    g = B.Env(203, seed=99)
    for step in range(330):
        o.step(o.sample_uniform(o.legal_mask()))
        if step % 30 == 29:
            b = o.get_boards()
            g.reset_from(_dev(b))
            assert np.array_equal(_np(g.get_boards()), b)


# ----------------------------------------------------------------------------- call by call
@pytest.mark.parametrize("variant,n,plies,cap", [(0, 131, 400, 350), (1, 97, 600, 2000)])
def test_each_call_on_injected_oracle_states(variant, n, plies, cap):
    """The oracle plays; before every ply its state is injected with reset_from and each
    C-ABI call is compared on its own."""
    kw = dict(variant=variant, seed=17, max_plies=cap, auto_reset=0)
    g, o = _pair(n, **kw)
    for t in range(plies):
        b = o.get_boards()
        g.reset_from(_dev(b))
        om = o.legal_mask()
        gm = g.legal_mask()
        assert np.array_equal(_mask_np(gm), om), t
        oa = o.sample_uniform(om)
        ga = g.sample_uniform(gm)
        assert np.array_equal(_np(ga), oa), t
        assert np.array_equal(_obs_np(g.encode_obs()), o.encode_obs().reshape(n, 44, 10, 10)), t
        orr, od = o.step(oa)
        gr, gd = g.step(ga)
        assert np.array_equal(_np(gr), orr) and np.array_equal(_np(gd), od), t
        assert np.array_equal(_np(g.get_boards()), o.get_boards()), t
    assert g.check() == 0
    assert (o.get_boards()[:, 120] & 1).sum() > 0  # some games ended inside the test


def test_hand_worked_positions_on_gpu(golden_dir):
    for pos in json.load(open(os.path.join(golden_dir, "positions.json")))["positions"]:
        pieces = {c: W.piece(t, o) for c, t, o in pos["pieces"]}
        g = B.Env(1)
        g.reset_from(_dev(W.make_line(pieces)[None, :]))
        for a in pos["play"]:
            g.step(_dev(np.array([a], np.int16)))
        assert g.check() == 0
        assert W.mask_to_actions(_mask_np(g.legal_mask())[0]) == pos["expect"], pos["name"]


def test_illegal_action_sets_sticky_error():
    g, o = _pair(40, seed=1)
    a = o.sample_uniform(o.legal_mask())
    a[7] = 5
    a[20] = -1
    before = _np(g.get_boards()).copy()
    r, d = g.step(_dev(a))
    assert g.check() == B.ILLEGAL_ACTION
    after = _np(g.get_boards())
    orr, od = o.step(a)
    assert np.array_equal(after, o.get_boards())
    assert np.array_equal(before[7], after[7]) and np.array_equal(before[20], after[20])
    assert np.array_equal(_np(r), orr) and np.array_equal(_np(d), od)
    g.clear_error()
    assert g.check() == 0


# ----------------------------------------------------------------------------- rollouts (configs 0-2)
def _run_separate(g, o, steps, every=1):
    n = g.n
    for t in range(steps):
        gm = g.legal_mask(); ga = g.sample_uniform(gm); gr, gd = g.step(ga)
        om = o.legal_mask(); oa = o.sample_uniform(om); orr, od = o.step(oa)
        assert np.array_equal(_np(ga), oa), t
        assert np.array_equal(_np(gr), orr) and np.array_equal(_np(gd), od), t
        if t % every == 0 or t == steps - 1:
            assert np.array_equal(_mask_np(gm), om), t
            assert np.array_equal(_np(g.get_boards()), o.get_boards()), t
            assert np.array_equal(_obs_np(g.encode_obs()), o.encode_obs().reshape(n, 44, 10, 10)), t
    assert g.check() == 0 and o.check() == 0


def test_config0_classic_256_games_256_plies():
    c = W.CONFIGS[0]
    g, o = _pair(c["num_games"], variant=c["variant"], seed=c["seed"], max_plies=c["max_plies"],
                 auto_reset=c["auto_reset"])
    _run_separate(g, o, c["steps"])


def _run_fused(g, o, steps, every=1, lo=0):
    """fused rollout_step of the big env g vs oracle o that mirrors games lo..lo+o.n"""
    n, k = g.n, o.n
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for t in range(steps):
        om = o.legal_mask(); oa = o.sample_uniform(om); orr, od = o.step(oa)
        g.rollout_step(mask, act, rew, done, obs)
        s = slice(lo, lo + k)
        assert np.array_equal(_np(act[s]), oa), t
        assert np.array_equal(_np(rew[s]), orr) and np.array_equal(_np(done[s]), od), t
        if t % every == 0 or t == steps - 1:
            assert np.array_equal(_mask_np(mask[s]), om), t
            assert np.array_equal(_obs_np(obs[s]), o.encode_obs().reshape(k, 44, 10, 10)), t
            assert np.array_equal(_np(g.get_boards()[s]), o.get_boards()), t
    assert g.check() == 0


def test_fused_step_small_with_auto_reset_and_ragged_tail():
    kw = dict(variant=0, seed=4, max_plies=90, auto_reset=1)
    g, o = _pair(1000, **kw)  # 1000 = 31 full batches + a tail of 8; every game resets 3 times
    _run_fused(g, o, 300, every=7)
    assert (o.get_boards()[:, 124] >= 3).all()


def test_fused_step_barrage_with_frequent_auto_resets():
    kw = dict(variant=1, seed=14, max_plies=25, auto_reset=1)  # the cooperative reset deals 8 pieces + 32 empties
    g, o = _pair(650, **kw)
    _run_fused(g, o, 160, every=9)
    assert (o.get_boards()[:, 124] >= 5).all()


def test_k_move_rule_and_ply_cap_draws():
    """The k-move rule (draw after k plies without a battle; 100 in training, 200 in
    evaluation) and the maximum game length, in the fused step and in strat_step."""
    kw = dict(variant=0, seed=6, max_plies=300, max_battleless=40, auto_reset=1)
    g, o = B.Env(400, **kw), orc.Env(400, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    reasons = np.zeros(8, int)
    for t in range(330):
        oa = o.sample_uniform(o.legal_mask()); orr, od = o.step(oa)
        if t % 2:
            g.step(_dev(oa), rew, done)
        else:
            g.rollout_step(mask, act, rew, done, obs)
        assert np.array_equal(_np(rew), orr) and np.array_equal(_np(done), od), t
        reasons += np.bincount((od[(od & 1) == 1] >> 2) & 7, minlength=8)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert reasons[5] > 0 and reasons[1] + reasons[2] + reasons[4] > 0  # battleless draws and other endings occurred
    assert g.check() == 0


def test_two_square_rule_switched_off():
    kw = dict(variant=0, seed=2, max_plies=200, auto_reset=1, two_square=0)
    g, o = _pair(300, **kw)
    _run_fused(g, o, 220, every=11)
    o_on = orc.Env(300, **dict(kw, two_square=1))
    diff = 0
    for _ in range(30):  # the switch matters: from the same states the rule-on masks differ sometimes
        b = o.get_boards(); o_on.reset_from(b)
        diff += int((o_on.legal_mask() != o.legal_mask()).any(axis=1).sum())
        o.step(o.sample_uniform(o.legal_mask()))
    assert diff > 0


def test_fused_step_null_outputs():
    g1 = B.Env(500, seed=6, max_plies=80, auto_reset=1)
    g2 = B.Env(500, seed=6, max_plies=80, auto_reset=1)
    obs1, obs2 = g1.new_obs(), g2.new_obs()
    mask, act, rew, done = g1.new_mask(), g1.new_actions(), g1.new_reward(), g1.new_done()
    for _ in range(100):
        g1.rollout_step(mask, act, rew, done, obs1)
        g2.rollout_step(None, None, None, None, obs2)
    assert torch.equal(obs1.view(torch.int16), obs2.view(torch.int16))
    assert torch.equal(g1.get_boards(), g2.get_boards())


def test_fused_steps_back_to_back_overlap_equals_synchronised_run():
    """Consecutive fused steps overlap on the device (programmatic dependent launch, ordered
    per batch by version flags).  400 launches with no host sync in between, at the bench's
    size, must leave exactly what a run synchronised after every launch leaves, and what the
    oracle computes for sampled game ranges."""
    c = W.CONFIGS[2]
    kw = dict(variant=0, seed=c["seed"], max_plies=150, auto_reset=1)  # cap 150: every game resets at least twice
    n, steps = c["num_games"], 400
    g1, g2 = B.Env(n, **kw), B.Env(n, **kw)
    outs1 = (g1.new_mask(), g1.new_actions(), g1.new_reward(), g1.new_done(), g1.new_obs())
    outs2 = (g2.new_mask(), g2.new_actions(), g2.new_reward(), g2.new_done(), g2.new_obs())
    for _ in range(steps):
        g1.rollout_step(*outs1)
    for _ in range(steps):
        g2.rollout_step(*outs2)
        torch.cuda.synchronize()
    assert torch.equal(g1.get_boards(), g2.get_boards())
    for a, b in zip(outs1, outs2):
        assert torch.equal(a.view(torch.uint8), b.view(torch.uint8))
    ranges = [0, 40000 // 32 * 32 + 8, n - 32]
    for lo in ranges:
        o = orc.Env(32, game_base=lo, **kw)
        for _ in range(steps):
            om = o.legal_mask(); oa = o.sample_uniform(om); orr, od = o.step(oa)
        s = slice(lo, lo + 32)
        assert np.array_equal(_mask_np(outs1[0][s]), om) and np.array_equal(_np(outs1[1][s]), oa)
        assert np.array_equal(_np(outs1[2][s]), orr) and np.array_equal(_np(outs1[3][s]), od)
        assert np.array_equal(_obs_np(outs1[4][s]), o.encode_obs().reshape(32, 44, 10, 10))
        assert np.array_equal(_np(g1.get_boards()[s]), o.get_boards())
    assert g1.check() == 0 and g2.check() == 0


@pytest.mark.parametrize("variant,n,cap", [(0, 1000, 70), (1, 333, 2000)])
def test_step_observe_equals_step_mask_encode_and_oracle(variant, n, cap):
    """strat_step_observe (external actions -> step -> mask + obs of the new state, one kernel)
    against the oracle's step / legal_mask / encode_obs, with auto-reset and a ragged tail."""
    kw = dict(variant=variant, seed=9, max_plies=cap, auto_reset=1)
    g, o = _pair(n, **kw)
    mask, rew, done, obs = g.new_mask(), g.new_reward(), g.new_done(), g.new_obs()
    om = o.legal_mask()
    for t in range(200):
        oa = o.sample_uniform(om)
        orr, od = o.step(oa)
        om = o.legal_mask()
        g.step_observe(_dev(oa), rew, done, mask, obs)
        assert np.array_equal(_np(rew), orr) and np.array_equal(_np(done), od), t
        assert np.array_equal(_mask_np(mask), om), t
        if t % 9 == 0 or t == 199:
            assert np.array_equal(_obs_np(obs), o.encode_obs().reshape(n, 44, 10, 10)), t
            assert np.array_equal(_np(g.get_boards()), o.get_boards()), t
    assert g.check() == 0
    # an illegal action: sticky error, that game unchanged, the others advance
    oa = o.sample_uniform(om)
    bad = oa.copy(); bad[3] = 3599
    before = _np(g.get_boards())[3].copy()
    g.step_observe(_dev(bad), rew, done, None, obs)
    assert g.check() == B.ILLEGAL_ACTION
    after = _np(g.get_boards())
    assert np.array_equal(after[3], before)
    o.step(bad)
    assert np.array_equal(after, o.get_boards())


def test_pinned_reset_state_matches_oracle():
    """Reset Behaviour and Support for Search: finished games restart from
    their pinned non-initial state, in every state-advancing kernel; unpinning brings fresh
    setups back."""
    kw = dict(variant=0, seed=13, max_plies=55, auto_reset=1)
    n = 500
    g, o = _pair(n, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for _ in range(30):
        g.rollout_step(mask, act, rew, done, obs)
        o.step(o.sample_uniform(o.legal_mask()))
    pin = o.get_boards()
    assert np.array_equal(_np(g.get_boards()), pin)
    g.pin_reset_state(_dev(pin)); o.pin_reset_state(pin)
    for t in range(90):  # every game hits the 55-ply cap at least three times
        oa = o.sample_uniform(o.legal_mask()); orr, od = o.step(oa)
        if t % 3 == 0:
            g.rollout_step(mask, act, rew, done, obs)
            assert np.array_equal(_np(act), oa), t
        elif t % 3 == 1:
            g.step(_dev(oa), rew, done)
        else:
            g.step_observe(_dev(oa), rew, done, mask, obs)
        assert np.array_equal(_np(rew), orr) and np.array_equal(_np(done), od), t
    b = o.get_boards()
    assert np.array_equal(_np(g.get_boards()), b)
    ply = b[:, 116].astype(int) | (b[:, 117].astype(int) << 8)
    pin_ply = pin[:, 116].astype(int) | (pin[:, 117].astype(int) << 8)
    assert (ply >= pin_ply).all() and (b[:, 124] >= 2).all()  # restarted from the pin, epochs count up
    g.rollout_uniform(40)
    for _ in range(40):
        o.step(o.sample_uniform(o.legal_mask()))
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    g.pin_reset_state(None); o.pin_reset_state(None)
    for _ in range(40):
        g.rollout_step(mask, act, rew, done, obs)
        o.step(o.sample_uniform(o.legal_mask()))
    b = o.get_boards()
    assert np.array_equal(_np(g.get_boards()), b)
    assert ((b[:, 116].astype(int) | (b[:, 117].astype(int) << 8)) < 30).any()  # fresh games again
    assert g.check() == 0


def test_fused_steps_of_two_environments_chained_through_a_buffer():
    """Environment B replays, with strat_step_observe, the actions environment A's fused step has
    just written - 300 times with no host sync.  The two launches belong to different environments
    (no version flags relate them) and exchange a buffer, so they share one chain record
    (strat_share_chain): B waits for A's grid, and A's next step waits for B's (which is still
    reading the actions A is about to overwrite): stream order has to hold."""
    kw = dict(variant=0, seed=31, max_plies=120, auto_reset=1)
    n = 65536
    a, b = B.Env(n, **kw), B.Env(n, **kw)
    a.share_chain(b)
    mask_a, act, rew_a, done_a, obs_a = a.new_mask(), a.new_actions(), a.new_reward(), a.new_done(), a.new_obs()
    mask_b, rew_b, done_b, obs_b = b.new_mask(), b.new_reward(), b.new_done(), b.new_obs()
    for _ in range(300):
        a.rollout_step(mask_a, act, rew_a, done_a, obs_a)
        b.step_observe(act, rew_b, done_b, mask_b, obs_b)
    assert b.check() == 0  # B never saw a stale (illegal) action
    assert torch.equal(a.get_boards(), b.get_boards())
    assert torch.equal(obs_a.view(torch.int16), obs_b.view(torch.int16))
    assert torch.equal(rew_a, rew_b) and torch.equal(done_a, done_b)


def test_shards_keyed_by_global_game_index_equal_the_unsharded_run():
    """Multi-GPU sharding on the CUDA path: two environments that own games
    [0, n) and [n, 2n) through `game_base` produce exactly the two halves of one 2n-game
    environment - every RNG draw is keyed by the global game index, no collective is needed."""
    n = 3000  # not a multiple of 32: the shards' batches do not line up with the big run's
    kw = dict(variant=0, seed=17, max_plies=50, auto_reset=1)
    whole = B.Env(2 * n, **kw)
    parts = [B.Env(n, game_base=0, **kw), B.Env(n, game_base=n, **kw)]
    outs_w = (whole.new_mask(), whole.new_actions(), whole.new_reward(), whole.new_done(), whole.new_obs())
    outs_p = [(p.new_mask(), p.new_actions(), p.new_reward(), p.new_done(), p.new_obs()) for p in parts]
    for _ in range(120):
        whole.rollout_step(*outs_w)
        for p, o in zip(parts, outs_p):
            p.rollout_step(*o)
    for k in range(2):
        s = slice(k * n, (k + 1) * n)
        assert torch.equal(whole.get_boards()[s], parts[k].get_boards())
        for a, b in zip(outs_w, outs_p[k]):
            assert torch.equal(a[s].view(torch.uint8), b.view(torch.uint8))
    assert whole.check() == 0


def test_host_buffer_entry_points_match_oracle():
    """The e2e calls bench.py times: strat_step_host (pinned host actions in; reward, done, next
    mask, next obs out) and strat_rollout_step_host (all five outputs to host buffers)."""
    n = 777
    kw = dict(variant=0, seed=19, max_plies=45, auto_reset=1)
    g, o = _pair(n, **kw)
    scratch = g.host_scratch()
    h_act = torch.empty(n, dtype=torch.int16).pin_memory()
    h_rew = torch.empty(n, dtype=torch.int8).pin_memory()
    h_done = torch.empty(n, dtype=torch.uint8).pin_memory()
    h_mask = torch.empty((n, 113), dtype=torch.int32).pin_memory()
    h_obs = torch.empty((n, 4400), dtype=torch.bfloat16).pin_memory()
    om = o.legal_mask()
    for t in range(70):
        if t % 2 == 0:
            oa = o.sample_uniform(om); orr, od = o.step(oa)
            h_act.copy_(torch.from_numpy(oa))
            g.step_host(scratch, h_act, h_rew, h_done, h_mask, h_obs)
            om = o.legal_mask()
            assert np.array_equal(h_mask.numpy().view(np.uint32), om), t       # mask of the NEW state
        else:
            oa = o.sample_uniform(om); orr, od = o.step(oa)
            g.rollout_step_host(scratch, h_mask, h_act, h_rew, h_done, h_obs)
            assert np.array_equal(h_mask.numpy().view(np.uint32), om), t       # mask the action was drawn from
            assert np.array_equal(h_act.numpy(), oa), t
            om = o.legal_mask()
        assert np.array_equal(h_rew.numpy(), orr) and np.array_equal(h_done.numpy(), od), t
        assert np.array_equal(h_obs.view(torch.int16).numpy().view(np.uint16), o.encode_obs().reshape(n, -1)), t
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert g.check() == 0


def test_fused_step_interleaved_with_other_calls():
    """A fused step after any other state-changing call (and vice versa) sees that call's result."""
    kw = dict(variant=0, seed=21, max_plies=60, auto_reset=1)
    g, o = _pair(700, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for t in range(120):
        if t % 3 == 2:  # separate calls
            gm = g.legal_mask(); ga = g.sample_uniform(gm); g.step(ga)
        elif t % 10 == 5:  # state round trip through the canonical lines
            g.reset_from(g.get_boards().clone())
            g.rollout_step(mask, act, rew, done, obs)
        else:
            g.rollout_step(mask, act, rew, done, obs)
        o.step(o.sample_uniform(o.legal_mask()))
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    g.rollout_step(mask, act, rew, done, obs)
    o.step(o.sample_uniform(o.legal_mask()))
    assert np.array_equal(_obs_np(obs), o.encode_obs().reshape(700, 44, 10, 10))
    g.reset(5); o.reset(5)
    g.rollout_step(mask, act, rew, done, obs)
    o.step(o.sample_uniform(o.legal_mask()))
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert g.check() == 0


# configs 1 and 2 at full size, ALL games mirrored: tests/test_gpu_allgames.py


# ----------------------------------------------------------------------------- replay ring (config 3 shape)
def test_replay_ring_push_commit_sample_match_oracle():
    n, per_slot, slots = 96, 64, 6  # capacity 384 = 4 pushes of 96
    kw = dict(variant=0, seed=8, max_plies=60, auto_reset=1)
    g, o = _pair(n, **kw)
    ring, oring = B.Replay(per_slot, slots), orc.Replay(per_slot, slots)
    obs = g.encode_obs()
    batch = 512
    s_obs = torch.empty((batch, 44, 10, 10), dtype=torch.bfloat16, device="cuda")
    s_mask = torch.empty((batch, 113), dtype=torch.int32, device="cuda")
    s_act = torch.empty(batch, dtype=torch.int16, device="cuda")
    s_rew = torch.empty(batch, dtype=torch.int8, device="cuda")
    s_done = torch.empty(batch, dtype=torch.uint8, device="cuda")
    for t in range(11):  # wraps the ring twice
        oobs = o.encode_obs(); om = o.legal_mask(); oa = o.sample_uniform(om); orr, od = o.step(oa)
        oring.push(oobs, om, oa, orr, od)
        gm = g.legal_mask(); ga = g.sample_uniform(gm); gr, gd = g.step(ga)
        ring.push(obs, gm, ga, gr, gd)
        obs = g.encode_obs()
        assert ring.state() == (oring.head, oring.filled)
        ring.sample(1234, t, batch, s_obs, s_mask, s_act, s_rew, s_done)
        eo, em, ea, er, ed, idx = oring.sample(1234, t, batch)
        assert np.array_equal(_obs_np(s_obs), eo) and np.array_equal(_mask_np(s_mask), em), t
        assert np.array_equal(_np(s_act), ea) and np.array_equal(_np(s_rew), er) and np.array_equal(_np(s_done), ed), t
    vo, vm, va, vr, vd = ring.views()
    for p in range(ring.capacity):
        eo, em, ea, er, ed = oring.read(p)
        assert np.array_equal(_np(vo[p]).view(np.uint16), eo.reshape(-1))
        assert np.array_equal(_np(vm[p]).view(np.uint32), em)
        assert (int(va[p]), int(vr[p]), int(vd[p])) == (ea, er, ed)


@pytest.mark.parametrize("rows_in_place,chained", [(False, False), (True, False), (True, True)])
def test_replay_in_place_push_equals_oracle_ring_records_and_samples(rows_in_place, chained):
    """Self-play loop of config 3 with the fused step writing mask_t (and optionally action_t,
    reward_t, done_t) and obs_{t+1} straight into the ring rows.  After every push, wrapped or
    not, every sampled (obs, mask, action, reward, done) record equals the oracle ring's, and at
    the end every live ring position holds the oracle's record: what is written ahead never lands
    in a live record (the ring's spare rows)."""
    n = 64
    kw = dict(variant=0, seed=3, max_plies=50, auto_reset=1)
    g, o = _pair(n, **kw)
    ring, oring = B.Replay(32, 8, block=n), orc.Replay(32, 8)  # capacity 256 = 4 blocks of 64
    act, rew, done = g.new_actions(), g.new_reward(), g.new_done()
    batch = 700
    s_obs = torch.empty((batch, 44, 10, 10), dtype=torch.bfloat16, device="cuda")
    s_mask = torch.empty((batch, 113), dtype=torch.int32, device="cuda")
    s_act = torch.empty(batch, dtype=torch.int16, device="cuda")
    s_rew = torch.empty(batch, dtype=torch.int8, device="cuda")
    s_done = torch.empty(batch, dtype=torch.uint8, device="cuda")
    o_ptr, _ = ring.reserve(n, 0)
    B._chk(B.lib().strat_encode_obs(g.h, o_ptr, B._stream()), "encode")  # obs_0 in place
    for t in range(11):  # wraps the ring twice
        oobs = o.encode_obs(); om = o.legal_mask(); oa = o.sample_uniform(om); orr, od = o.step(oa)
        oring.push(oobs, om, oa, orr, od)
        _, m_ptr = ring.reserve(n, 0)        # mask_t -> the rows being completed
        o_next, _ = ring.reserve(n, 1)       # obs_{t+1} -> the rows of the next block
        if rows_in_place:
            a_ptr, r_ptr, d_ptr = ring.reserve_rows(n)
            g.rollout_step_ptrs(m_ptr, a_ptr, r_ptr, d_ptr, o_next)
            ring.commit_in_place(n)
        else:
            g.rollout_step_raw(m_ptr, act, rew, done, o_next)
            ring.commit(act, rew, done)
        assert ring.state() == (oring.head, oring.filled)
        if chained:  # the gather does not separate consecutive fused steps (strat_replay_sample_chained)
            ring.sample_chained(g, 77, t, batch, s_obs, s_mask, s_act, s_rew, s_done)
        else:
            ring.sample(77, t, batch, s_obs, s_mask, s_act, s_rew, s_done)
        eo, em, ea, er, ed, idx = oring.sample(77, t, batch)
        assert np.array_equal(_obs_np(s_obs), eo) and np.array_equal(_mask_np(s_mask), em), t
        assert np.array_equal(_np(s_act), ea) and np.array_equal(_np(s_rew), er) and np.array_equal(_np(s_done), ed), t
    vo, vm, va, vr, vd = ring.views()
    for p in range(ring.capacity):
        row, orow = ring.locate(p)
        eo, em, ea, er, ed = oring.read(p)
        assert np.array_equal(_np(vo[orow]).view(np.uint16), eo.reshape(-1)), p
        assert np.array_equal(_np(vm[row]).view(np.uint32), em), p
        assert (int(va[row]), int(vr[row]), int(vd[row])) == (ea, er, ed), p
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    # a plain ring has no spare rows: writing ahead would tear live records, so it is refused
    with pytest.raises(B.StratError):
        B.Replay(32, 8).reserve(n, 1)


def test_chained_gathers_back_to_back_equal_a_synchronised_run():
    """60 self-play steps of 65,536 games with in-place pushes into a ring that wraps every second
    step and a 2,048-record gather per step, issued back to back with no host synchronisation:
    fused steps overlap each other THROUGH the chained gathers.  Every gathered minibatch, the ring
    and the boards equal those of a run that synchronises after every call and uses the plain
    gather."""
    n, bs, steps = 65536, 2048, 60
    kw = dict(variant=0, seed=5, max_plies=90, auto_reset=1)
    outs = []
    for chained in (True, False):
        g = B.Env(n, **kw)
        ring = B.Replay(n, 2, block=n)  # capacity = 2 blocks
        so = torch.empty((steps, bs, 4400), dtype=torch.int16, device="cuda")
        sm = torch.empty((steps, bs, 113), dtype=torch.int32, device="cuda")
        sa = torch.empty((steps, bs), dtype=torch.int16, device="cuda")
        sr = torch.empty((steps, bs), dtype=torch.int8, device="cuda")
        sd = torch.empty((steps, bs), dtype=torch.uint8, device="cuda")
        o_ptr, _ = ring.reserve(n, 0)
        B._chk(B.lib().strat_encode_obs(g.h, o_ptr, B._stream()), "encode")
        for t in range(steps):
            _, m_ptr = ring.reserve(n, 0)
            o_next, _ = ring.reserve(n, 1)
            a_ptr, r_ptr, d_ptr = ring.reserve_rows(n)
            g.rollout_step_ptrs(m_ptr, a_ptr, r_ptr, d_ptr, o_next)
            ring.commit_in_place(n)
            if chained:
                ring.sample_chained(g, 9, t, bs, so[t], sm[t], sa[t], sr[t], sd[t])
            else:
                ring.sample(9, t, bs, so[t], sm[t], sa[t], sr[t], sd[t])
                torch.cuda.synchronize()
        torch.cuda.synchronize()
        assert g.check() == 0
        live = [ring.locate(p) for p in (0, n)]
        v = ring.views()
        rows = [torch.cat([x[r:r + n] for r, _ in live]) for x in v[1:]] + [torch.cat([v[0][o:o + n] for _, o in live])]
        outs.append((so, sm, sa, sr, sd, g.get_boards().clone(), rows))
        del g, ring
    a, b = outs
    for x, y in zip(a[:6], b[:6]):
        assert torch.equal(x, y)
    for x, y in zip(a[6], b[6]):
        assert torch.equal(x, y)


def test_chained_gathers_in_an_irregular_loop_equal_a_synchronised_run():
    """The chained gather takes a record as soon as its producer has published the record's batch only in
    the regular loop (fused step, commit, gather); anything else - another call on the environment before
    the gather, two steps between two gathers, a copy push - must make it wait for the stream instead.
    Issued back to back without host synchronisation; compared with a synchronised run of plain gathers."""
    n, bs, steps = 8192, 1500, 40
    kw = dict(variant=0, seed=8, max_plies=70, auto_reset=1)
    outs = []
    for chained in (True, False):
        g = B.Env(n, **kw)
        ring = B.Replay(n, 3, block=n)
        so = torch.empty((steps, bs, 4400), dtype=torch.int16, device="cuda")
        sm = torch.empty((steps, bs, 113), dtype=torch.int32, device="cuda")
        sa = torch.empty((steps, bs), dtype=torch.int16, device="cuda")
        sr = torch.empty((steps, bs), dtype=torch.int8, device="cuda")
        sd = torch.empty((steps, bs), dtype=torch.uint8, device="cuda")
        act, rew, done = g.new_actions(), g.new_reward(), g.new_done()
        boards = []
        o_ptr, _ = ring.reserve(n, 0)
        B._chk(B.lib().strat_encode_obs(g.h, o_ptr, B._stream()), "encode")

        def push_in_place():
            _, m_ptr = ring.reserve(n, 0)
            o_next, _ = ring.reserve(n, 1)
            a_ptr, r_ptr, d_ptr = ring.reserve_rows(n)
            g.rollout_step_ptrs(m_ptr, a_ptr, r_ptr, d_ptr, o_next)
            ring.commit_in_place(n)

        for t in range(steps):
            push_in_place()
            if t % 7 == 3:
                push_in_place()                                   # two steps between two gathers
            if t % 5 == 2:
                boards.append(g.get_boards())                     # another call on the environment (device tensor, no sync)
            if t % 11 == 6:                                       # a push with copied small arrays
                _, m_ptr = ring.reserve(n, 0)
                o_next, _ = ring.reserve(n, 1)
                g.rollout_step_raw(m_ptr, act, rew, done, o_next)
                ring.commit(act, rew, done)
            if chained:
                ring.sample_chained(g, 9, t, bs, so[t], sm[t], sa[t], sr[t], sd[t])
            else:
                ring.sample(9, t, bs, so[t], sm[t], sa[t], sr[t], sd[t])
                torch.cuda.synchronize()
        torch.cuda.synchronize()
        assert g.check() == 0
        outs.append((so, sm, sa, sr, sd, g.get_boards().clone(), torch.stack(boards)))
        del g, ring
    for x, y in zip(*outs):
        assert torch.equal(x, y)


def test_config3_full_size_ring_zero_copy_and_sample():
    """BASELINE.json configs[3] at full size in the launch sequence bench.py times: 262,144
    games, 64 x 131,072-record ring (77.6 GB + spare rows), in-place push + 4,096-sample gather
    per step.  The oracle mirrors three 32-game ranges here; 34 steps wrap the ring (capacity =
    32 blocks).  (All games, row by row, on a ring that wraps sooner: tests/test_gpu_allgames.py.)"""
    c = W.CONFIGS[3]
    n, bs = c["num_games"], c["sample_batch"]
    kw = dict(variant=0, seed=c["seed"], max_plies=c["max_plies"], auto_reset=1)
    free, _ = torch.cuda.mem_get_info()
    if free < 95e9:
        pytest.skip("needs ~85 GB of free device memory")
    g = B.Env(n, **kw)
    ring = B.Replay(c["ring_per_slot"], c["ring_slots"], block=n)
    cap = ring.capacity
    ranges = [0, 131072 + 64, n - 32]
    os_ = [orc.Env(32, game_base=lo, **kw) for lo in ranges]
    act, rew, done = g.new_actions(), g.new_reward(), g.new_done()
    s_obs = torch.empty((bs, 44, 10, 10), dtype=torch.bfloat16, device="cuda")
    s_mask = torch.empty((bs, 113), dtype=torch.int32, device="cuda")
    s_act = torch.empty(bs, dtype=torch.int16, device="cuda")
    s_rew = torch.empty(bs, dtype=torch.int8, device="cuda")
    s_done = torch.empty(bs, dtype=torch.uint8, device="cuda")
    o_ptr, _ = ring.reserve(n, 0)
    B._chk(B.lib().strat_encode_obs(g.h, o_ptr, B._stream()), "encode")
    vo, vm, va, vr, vd = ring.views()
    steps, expect = 34, {}
    for t in range(steps):
        for oo, lo in zip(os_, ranges):
            oobs = oo.encode_obs(); om = oo.legal_mask(); oa = oo.sample_uniform(om); orr, od = oo.step(oa)
            expect[(t, lo)] = (oobs.reshape(32, -1).copy(), om.copy(), oa.copy(), orr.copy(), od.copy())
        _, m_ptr = ring.reserve(n, 0)
        o_next, _ = ring.reserve(n, 1)
        a_ptr, r_ptr, d_ptr = ring.reserve_rows(n)
        g.rollout_step_ptrs(m_ptr, a_ptr, r_ptr, d_ptr, o_next)
        ring.commit_in_place(n)
        ring.sample(c["seed"], t, bs, s_obs, s_mask, s_act, s_rew, s_done)
        head, filled = ring.state()
        assert head == ((t + 1) * n) % cap and filled == min((t + 1) * n, cap)
        idx = torch.from_numpy(orc.sample_indices(c["seed"], t, bs, filled)).cuda()
        # ring position -> rows: blocks are contiguous, so locate() of each block start suffices
        blk = torch.div(idx, n, rounding_mode="floor")
        row0 = torch.tensor([ring.locate(k * n) if k * n < filled else (0, 0) for k in range(cap // n)], device="cuda")
        row, orow = row0[blk, 0] + idx - blk * n, row0[blk, 1] + idx - blk * n
        assert torch.equal(s_act, va[row]) and torch.equal(s_rew, vr[row]) and torch.equal(s_done, vd[row])
        assert torch.equal(s_mask, vm[row])
        assert torch.equal(s_obs.view(torch.int16).view(bs, -1), vo[orow])
    for t in range(steps - cap // n, steps):  # the blocks still in the ring: every one is whole
        row, orow = ring.locate((t * n) % cap)
        for lo in ranges:
            eo, em, ea, er, ed = expect[(t, lo)]
            s, so = slice(row + lo, row + lo + 32), slice(orow + lo, orow + lo + 32)
            assert np.array_equal(_np(vo[so]).view(np.uint16), eo), (t, lo)
            assert np.array_equal(_np(vm[s]).view(np.uint32), em), (t, lo)
            assert np.array_equal(_np(va[s]), ea) and np.array_equal(_np(vr[s]), er) and np.array_equal(_np(vd[s]), ed)
    b = _np(g.get_boards())
    for oo, lo in zip(os_, ranges):
        assert np.array_equal(b[lo:lo + 32], oo.get_boards())
    assert g.check() == 0


def test_config4_full_size_determinise_rollout_reduce():
    """BASELINE.json configs[4] at full size: 16 oracle-made roots x 16,384 determinisations,
    64-ply on-chip rollouts, per-root reduction.  Determinised boards are compared for all
    262,144 games; rollouts on three 64-game ranges; the reduction against the oracle's own
    reduction of the same final boards."""
    c = W.CONFIGS[4]
    R, S, plies = c["num_roots"], c["samples_per_root"], c["rollout_plies"]
    src = orc.Env(R, seed=c["seed"], max_plies=1000, auto_reset=1)
    rb = W.capture_at_ply(src.get_boards, lambda: src.step(src.sample_uniform(src.legal_mask())), R, c["root_plies"])
    side = ((rb[:, 116].astype(np.int64) | (rb[:, 117].astype(np.int64) << 8)) & 1).astype(np.uint8)
    roots_o = orc.Env(R, seed=c["seed"]); roots_o.reset_from(rb)
    roots_g = B.Env(R, seed=c["seed"]); roots_g.reset_from(_dev(rb))
    out_o = orc.Env(R * S, seed=c["seed"])
    out_g = B.Env(R * S, seed=c["seed"], max_plies=0, auto_reset=0)
    orc.determinise(roots_o, S, 777, out_o)
    B.determinise(roots_g, S, 777, out_g)
    det = out_o.get_boards()
    assert np.array_equal(_np(out_g.get_boards()), det)
    out_g.rollout_uniform(plies)
    fin = _np(out_g.get_boards())
    for lo in (0, 5 * S + 4000, R * S - 64):
        o = orc.Env(64, seed=c["seed"], game_base=lo)
        o.reset_from(det[lo:lo + 64])
        for _ in range(plies):
            o.step(o.sample_uniform(o.legal_mask()))
        assert np.array_equal(fin[lo:lo + 64], o.get_boards()), lo
    out_o.reset_from(fin)
    assert np.array_equal(_np(B.reduce_returns(out_g, _dev(side), S)), orc.reduce_returns(out_o, side, S))
    # properties at full size: plies advance by <= 64, only finished games stop early
    ply = fin[:, 116].astype(int) | (fin[:, 117].astype(int) << 8)
    donef = (fin[:, 120] & 1) == 1
    assert (ply[~donef] == c["root_plies"] + plies).all() and (ply[donef] <= c["root_plies"] + plies).all()
    assert out_g.check() == 0 and roots_g.check() == 0


# ----------------------------------------------------------------------------- search-shaped batch (config 4 shape)
def test_determinise_rollout_reduce_match_oracle():
    R, S, plies = 4, 96, 64
    src = orc.Env(R, seed=0, max_plies=1000, auto_reset=1)
    rb = W.capture_at_ply(src.get_boards, lambda: src.step(src.sample_uniform(src.legal_mask())), R, 200)
    assert ((rb[:, 116].astype(int) | (rb[:, 117].astype(int) << 8)) == 200).all()
    roots_o = orc.Env(R, seed=0)
    roots_o.reset_from(rb)
    side = np.array([(int(rb[r, 116]) | (int(rb[r, 117]) << 8)) & 1 for r in range(R)], np.uint8)
    roots_g = B.Env(R, seed=0)
    roots_g.reset_from(_dev(rb))
    out_o = orc.Env(R * S, seed=0)
    out_g = B.Env(R * S, seed=0)
    orc.determinise(roots_o, S, 4242, out_o)
    B.determinise(roots_g, S, 4242, out_g)
    assert np.array_equal(_np(out_g.get_boards()), out_o.get_boards())
    for _ in range(plies):
        out_o.step(out_o.sample_uniform(out_o.legal_mask()))
    out_g.rollout_uniform(plies)
    assert np.array_equal(_np(out_g.get_boards()), out_o.get_boards())
    red_o = orc.reduce_returns(out_o, side, S)
    red_g = B.reduce_returns(out_g, _dev(side), S)
    assert np.array_equal(_np(red_g), red_o)
    assert out_g.check() == 0


def test_rollout_uniform_equals_repeated_calls_with_auto_reset():
    kw = dict(variant=0, seed=12, max_plies=70, auto_reset=1)
    g1, g2 = B.Env(333, **kw), B.Env(333, **kw)
    g1.rollout_uniform(150)
    for _ in range(150):
        g2.step(g2.sample_uniform(g2.legal_mask()))
    assert torch.equal(g1.get_boards(), g2.get_boards())
