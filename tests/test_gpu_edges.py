"""Edge cases of the C ABI on the GPU: tiny and ragged batches, empty inputs, degenerate
positions, argument errors."""
import ctypes as C

import numpy as np
import pytest
import torch

from oracle import orc
from paper_2511_07312_b200 import binding as B
from paper_2511_07312_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _np(t):
    return t.detach().cpu().numpy()


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("n", [1, 31, 32, 33, 65])
def test_tiny_and_ragged_batches_every_call(n):
    kw = dict(variant=0, seed=n, max_plies=35, auto_reset=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for t in range(80):
        om = o.legal_mask(); oa = o.sample_uniform(om); orr, od = o.step(oa)
        if t % 3 == 0:
            g.rollout_step(mask, act, rew, done, obs)
        elif t % 3 == 1:
            g.legal_mask(mask); g.sample_uniform(mask, act); g.step(act, rew, done); g.encode_obs(obs)
        else:
            g.legal_mask(mask); g.sample_uniform(mask, act); g.step_observe(act, rew, done, None, obs)
            g_mask_now = _np(mask).view(np.uint32)
            assert np.array_equal(g_mask_now, om), t
        assert np.array_equal(_np(act), oa) and np.array_equal(_np(rew), orr) and np.array_equal(_np(done), od), t
        assert np.array_equal(_np(obs.view(torch.int16)).view(np.uint16), o.encode_obs()), t
        assert np.array_equal(_np(g.get_boards()), o.get_boards()), t
    g.rollout_uniform(0)  # zero plies: a no-op
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert g.check() == 0


def test_degenerate_positions():
    # (a) flags only: the side to move has no legal move and neither has the other -> the mask is
    #     empty, the sampler returns -1, the fused step leaves the (live, stuck) game as it is
    flags = {0: W.piece(W.FLAG, W.RED), 99: W.piece(W.FLAG, W.BLUE)}
    # (b) one move available, and it captures the Flag
    mate = {88: W.piece(W.MINER, W.RED), 0: W.piece(W.FLAG, W.RED), 98: W.piece(W.FLAG, W.BLUE),
            78: W.piece(W.BOMB, W.BLUE), 87: W.piece(W.BOMB, W.BLUE), 89: W.piece(W.BOMB, W.RED)}
    # (c) a Scout with the whole file open: nine distances
    scout = {5: W.piece(W.SCOUT, W.RED), 0: W.piece(W.FLAG, W.RED), 99: W.piece(W.FLAG, W.BLUE)}
    lines = np.stack([W.make_line(flags), W.make_line(mate), W.make_line(scout)])
    g, o = B.Env(3, seed=1), orc.Env(3, seed=1)
    g.reset_from(_dev(lines)); o.reset_from(lines)
    gm = _np(g.legal_mask()).view(np.uint32)
    assert np.array_equal(gm, o.legal_mask())
    assert W.mask_to_actions(gm[0]) == []
    assert W.action_index(5, 0, 9) in W.mask_to_actions(gm[2]) and len(W.mask_to_actions(gm[2])) == 9 + 4 + 4
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    g.rollout_step(mask, act, rew, done, obs)
    oa = o.sample_uniform(o.legal_mask()); orr, od = o.step(oa)
    assert np.array_equal(_np(act), oa) and int(_np(act)[0]) == -1
    assert np.array_equal(_np(rew), orr) and np.array_equal(_np(done), od)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert g.check() == o.check() == B.ILLEGAL_ACTION  # the stuck live game had no action to take
    g.clear_error(); o.clear_error()
    g.rollout_uniform(3)
    for _ in range(3):
        o.step(o.sample_uniform(o.legal_mask()))
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    assert g.check() == o.check() == B.ILLEGAL_ACTION


def test_argument_errors_and_empty_inputs():
    L = B.lib()
    g = B.Env(40, seed=1)
    s = B._stream()
    assert L.strat_legal_mask(g.h, None, s) == B.BAD_ARG
    assert L.strat_step(g.h, None, None, None, s) == B.BAD_ARG
    assert L.strat_rollout_step(g.h, None, None, None, None, None, s) == B.BAD_ARG  # obs is mandatory
    assert L.strat_rollout_uniform(g.h, -1, s) == B.BAD_ARG
    assert L.strat_reset_from(g.h, None, s) == B.BAD_ARG
    bad = B.strat_config(10, 2, 0, 0, 0, 0, 1, 0, 0, 0)  # unknown variant
    assert L.strat_workspace_bytes(C.byref(bad)) == 0
    bad = B.strat_config(10, 0, 0, 0, 0, 0, 1, 0, 7, 0)  # chase_rule must be 0 or 1
    assert L.strat_workspace_bytes(C.byref(bad)) == 0
    ring = B.Replay(8, 2)
    obs, mask = g.encode_obs(), g.legal_mask()
    act = g.sample_uniform(mask); rew, done = g.step(act)
    so = torch.empty((4, 44, 10, 10), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(B.StratError):  # nothing pushed yet
        ring.sample(0, 0, 4, so, None, None, None, None)
    assert L.strat_replay_push(ring.h, B._ptr(obs), B._ptr(mask), B._ptr(act), B._ptr(rew), B._ptr(done), 0, s) == 0
    assert ring.state() == (0, 0)  # an empty push changes nothing
    assert L.strat_replay_push(ring.h, B._ptr(obs), B._ptr(mask), B._ptr(act), B._ptr(rew), B._ptr(done), 17, s) == B.BAD_ARG  # > capacity
    assert L.strat_replay_push(ring.h, B._ptr(obs), B._ptr(mask), B._ptr(act), B._ptr(rew), B._ptr(done), 16, s) == 0
    assert ring.state() == (0, 16)
    ring.sample(0, 0, 0, so, None, None, None, None)  # an empty batch is fine
    with pytest.raises(B.StratError):
        ring.reserve(5, 0)  # blocks must tile the ring
    # the fused step refuses CUDA-graph capture (its launch counter lives on the host)
    cap_stream = torch.cuda.Stream()
    obs40, graph = g.new_obs(), torch.cuda.CUDAGraph()
    with torch.cuda.stream(cap_stream):
        graph.capture_begin()
        rc = L.strat_rollout_step(g.h, None, None, None, None, B._ptr(obs40), B._stream())
        graph.capture_end()
    assert rc == B.BAD_STATE
    torch.cuda.synchronize()
    h = B.History(40, 1)  # a one-step ring
    h.attach(g)
    g.step(g.sample_uniform(g.legal_mask()))
    g.step(g.sample_uniform(g.legal_mask()))
    assert h.current_step() == 2
    h.legal_mask(1); h.legal_mask(2)
    with pytest.raises(B.StratError):
        h.legal_mask(0)  # overwritten
    assert g.check() == 0


def test_one_chained_ring_per_environment_and_groups_grow_one_by_one():
    """strat_replay_sample_chained: the environment's fused steps wait for the gathers of ONE ring, so a second
    live ring is refused instead of silently taking the first one's place.  strat_share_chain(a, b): b joins
    a's group only while b shares its ordering with nobody else."""
    n = 64
    g = B.Env(n, seed=2, max_plies=50, auto_reset=1)
    r1, r2 = B.Replay(32, 8, block=n), B.Replay(32, 8, block=n)
    act, rew, done = g.new_actions(), g.new_reward(), g.new_done()
    bs = 16
    so = torch.empty((bs, 44, 10, 10), dtype=torch.bfloat16, device="cuda")
    sm = torch.empty((bs, 113), dtype=torch.int32, device="cuda")
    sa = torch.empty(bs, dtype=torch.int16, device="cuda")
    sr = torch.empty(bs, dtype=torch.int8, device="cuda")
    sd = torch.empty(bs, dtype=torch.uint8, device="cuda")
    for ring in (r1, r2):
        o_ptr, m_ptr = ring.reserve(n, 0)
        g.rollout_step_raw(m_ptr, act, rew, done, o_ptr)
        ring.commit(act, rew, done)
    r1.sample_chained(g, 1, 0, bs, so, sm, sa, sr, sd)
    with pytest.raises(B.StratError, match="bad state"):
        r2.sample_chained(g, 1, 0, bs, so, sm, sa, sr, sd)
    r1.sample_chained(g, 1, 1, bs, so, sm, sa, sr, sd)   # the first ring goes on
    torch.cuda.synchronize()
    del r1                                               # strat_replay_destroy unties the environment
    r2.sample_chained(g, 1, 0, bs, so, sm, sa, sr, sd)
    torch.cuda.synchronize()
    assert g.check() == 0
    a, b, c, d = (B.Env(8, seed=k) for k in range(4))
    a.share_chain(b)
    a.share_chain(b)                                     # already one group: nothing to do
    a.share_chain(c)                                     # a lone environment joins
    d.share_chain(d)
    with pytest.raises(B.StratError, match="bad state"):
        d.share_chain(b)                                 # b shares with a and c: they would be left behind
    b.share_chain(d)                                     # the other way round d joins the group


def test_sample_uniform_is_uniform_over_the_legal_set():
    """Chi-square of the sampled rank r = position of the action inside its mask, over many
    seeds on one position (the closed form: every legal action has probability 1/n)."""
    line = W.make_line({44: W.piece(W.SCOUT, W.RED), 0: W.piece(W.FLAG, W.RED), 99: W.piece(W.FLAG, W.BLUE),
                        15: W.piece(W.CAPTAIN, W.RED)})
    n = 20000
    g = B.Env(n, seed=123)
    g.reset_from(_dev(np.repeat(line[None, :], n, axis=0)))
    mask = g.legal_mask()
    legal = W.mask_to_actions(_np(mask).view(np.uint32)[0])
    a = _np(g.sample_uniform(mask)).astype(int)
    counts = np.array([(a == x).sum() for x in legal])
    assert counts.sum() == n
    expect = n / len(legal)
    chi2 = ((counts - expect) ** 2 / expect).sum()
    assert chi2 < 3 * len(legal) + 30, (chi2, len(legal))


def test_random_hand_built_boards_all_calls():
    """2,000 arbitrary positions (any number of pieces of any type anywhere, random moved /
    revealed bits, either side to move): mask, observation, sampled action, step, terminal
    verdicts and the resulting lines against the oracle; then three more plies."""
    rng = np.random.default_rng(42)
    n = 2000
    lines = np.zeros((n, 128), np.uint8)
    free = [c for c in range(100) if c not in W.LAKES]
    for i in range(n):
        k = int(rng.integers(2, 60))
        cells = rng.choice(free, k, replace=False)
        pieces = {}
        for j, c in enumerate(cells):
            if j < 2:
                t, owner = W.FLAG, j  # one Flag each
            else:
                t, owner = int(rng.integers(1, 13)), int(rng.integers(2))
                if t == W.FLAG:
                    t = W.BOMB
            immobile = t in (W.FLAG, W.BOMB)
            pieces[int(c)] = W.piece(t, owner, moved=bool(rng.integers(2)) and not immobile, revealed=bool(rng.integers(2)))
        lines[i] = W.make_line(pieces, ply=int(rng.integers(0, 50)), battleless=int(rng.integers(0, 30)))
    kw = dict(variant=0, seed=9, max_plies=52, auto_reset=0)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    g.reset_from(_dev(lines)); o.reset_from(lines)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for t in range(4):
        om = o.legal_mask(); oobs = o.encode_obs(); oa = o.sample_uniform(om)
        assert np.array_equal(_np(g.legal_mask(mask)).view(np.uint32), om), t
        assert np.array_equal(_np(g.encode_obs(obs).view(torch.int16)).view(np.uint16), oobs), t
        assert np.array_equal(_np(g.sample_uniform(mask, act)), oa), t
        live_stuck = (oa < 0) & ((o.get_boards()[:, 120] & 1) == 0)
        orr, od = o.step(oa)
        g.step(act, rew, done)
        assert np.array_equal(_np(rew), orr) and np.array_equal(_np(done), od), t
        assert np.array_equal(_np(g.get_boards()), o.get_boards()), t
        assert g.check() == o.check() == (B.ILLEGAL_ACTION if live_stuck.any() else 0)
        g.clear_error(); o.clear_error()
    reasons = np.bincount((o.get_boards()[:, 120] >> 2) & 7, minlength=6)
    assert reasons[1] > 0 and reasons[2] > 0 and reasons[4] > 0  # flag captures, no-move wins, ply caps all occurred


def test_setup_redraw_cases_on_gpu(golden_dir):
    """Setups that are immobile at the first attempt (R5; found by the oracle, tests/golden/
    setup_redraw_cases.json): the thread-per-game reset (k_reset, epoch 0) and the warp-cooperative
    auto-reset's fallback inside the fused step and strat_step (epoch 1) redraw like the oracle."""
    import json
    import os
    cases = json.load(open(os.path.join(golden_dir, "setup_redraw_cases.json")))
    for gidx in cases["epoch0"]:
        kw = dict(variant=0, seed=cases["seed"], game_base=gidx - 5)
        g, o = B.Env(40, **kw), orc.Env(40, **kw)
        assert np.array_equal(_np(g.get_boards()), o.get_boards()), gidx
    for k, gidx in enumerate(cases["epoch1"]):
        kw = dict(variant=0, seed=cases["seed"], game_base=gidx - 7, max_plies=3, auto_reset=1)
        g, o = B.Env(40, **kw), orc.Env(40, **kw)
        mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
        for t in range(7):  # the 3-ply cap ends every game at t = 2: epoch 1 is set up inside that step
            oa = o.sample_uniform(o.legal_mask()); o.step(oa)
            if k % 2 == 0:
                g.rollout_step(mask, act, rew, done, obs)
            else:
                g.step(_dev(oa), rew, done)
            b = o.get_boards()
            assert np.array_equal(_np(g.get_boards()), b), (gidx, t)
        assert (b[:, 124] >= 2).all()
        assert g.check() == 0


def test_large_batch_beyond_4_gib_of_observations():
    """600,011 games: 5.3 GB of observations per step (byte offsets above 2^32), a ragged last
    batch; the oracle mirrors the first and the last games."""
    n = 600011
    free, _ = torch.cuda.mem_get_info()
    if free < 12e9:
        pytest.skip("needs ~8 GB of free device memory")
    kw = dict(variant=0, seed=2, max_plies=6, auto_reset=1)
    g = B.Env(n, **kw)
    lo = n - 43
    o_first, o_last = orc.Env(32, **kw), orc.Env(43, game_base=lo, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for t in range(8):  # every game is reset once (6-ply cap)
        g.rollout_step(mask, act, rew, done, obs)
        for oo, s in ((o_first, slice(0, 32)), (o_last, slice(lo, n))):
            om = oo.legal_mask(); oa = oo.sample_uniform(om); orr, od = oo.step(oa)
            assert np.array_equal(_np(act[s]), oa) and np.array_equal(_np(rew[s]), orr) and np.array_equal(_np(done[s]), od), t
            assert np.array_equal(_np(mask[s]).view(np.uint32), om), t
            assert np.array_equal(_np(obs[s].view(torch.int16)).view(np.uint16), oo.encode_obs()), t
    b = g.get_boards()
    assert np.array_equal(_np(b[lo:]), o_last.get_boards()) and np.array_equal(_np(b[:32]), o_first.get_boards())
    x = obs.view(torch.int16)[:, :28].reshape(n, 28, 100)
    assert bool(((x != 0).sum(dim=1) == 1).all())  # planes 0-27 partition the board for every game
    assert g.check() == 0


def test_setup_pool_matches_oracle_in_every_reset_path():
    """Customised initial boards (R30): strat_reset, the cooperative auto-reset of the
    fused step and of strat_step, and the on-chip rollout's reset all deal the oracle's pool entries."""
    from test_oracle_game import _random_pool
    K, n = 11, 700
    pool = _random_pool(K, 5)
    kw = dict(variant=0, seed=8, max_plies=9, auto_reset=1)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    g.set_setup_pool(_dev(pool)); o.set_setup_pool(pool)
    g.reset(8); o.reset(8)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for t in range(40):
        oa = o.sample_uniform(o.legal_mask()); o.step(oa)
        if t % 3 == 0:
            g.rollout_step(mask, act, rew, done, obs)
        elif t % 3 == 1:
            g.step(_dev(oa), rew, done)
        else:
            g.rollout_uniform(1)
        assert np.array_equal(_np(g.get_boards()), o.get_boards()), t
    assert (o.get_boards()[:, 124] >= 4).all() and g.check() == 0
    g.set_setup_pool(None); o.set_setup_pool(None)
    for t in range(12):
        o.step(o.sample_uniform(o.legal_mask())); g.rollout_step(mask, act, rew, done, obs)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    bad = pool.copy(); bad[0, 3, 0] = 14
    g.set_setup_pool(_dev(bad))
    assert g.check() == B.BAD_ARG


def test_hand_built_lines_with_arbitrary_histories():
    """DESIGN.md R24: a hand-built line may carry any history.  3,000 random positions whose eight
    history entries are random straight moves (or absent): the two-square ban derived from them,
    the mask, the observation's history planes and one step must agree with the oracle."""
    rng = np.random.default_rng(7)
    n = 3000
    lines = np.zeros((n, 128), np.uint8)
    free = [c for c in range(100) if c not in W.LAKES]
    for i in range(n):
        k = int(rng.integers(4, 40))
        cells = rng.choice(free, k, replace=False)
        pieces = {int(cells[0]): W.piece(W.FLAG, 0), int(cells[1]): W.piece(W.FLAG, 1)}
        for c in cells[2:]:
            t = int(rng.integers(1, 11)) if rng.random() < 0.8 else W.BOMB
            pieces[int(c)] = W.piece(t, int(rng.integers(2)), moved=bool(rng.integers(2)) and t != W.BOMB,
                                     revealed=bool(rng.integers(2)))
        hist = []
        movers = [int(c) for c in cells[2:]]
        # shuttles of one piece along a line make two-square bans likely; the rest is noise
        a = movers[int(rng.integers(len(movers)))]
        r, q = divmod(a, 10)
        line_cells = [10 * r + x for x in range(10)] if rng.random() < 0.5 else [10 * y + q for y in range(10)]
        for j in range(8):
            u = rng.random()
            if u < 0.15:
                hist.append((0xFF, 0xFF))
            elif u < 0.75 and j % 2 == 1:   # entries 1, 3, 5 = the side to move's own last plies
                f = a if j == 1 else hist[j - 2][0] if hist[j - 2][0] != 0xFF else a
                t = int(line_cells[int(rng.integers(10))])
                hist.append((t, f))         # moved t -> f, so the chain ends on the piece's square
            else:
                f = int(rng.integers(100)); t = int(rng.integers(100))
                hist.append((f, t))
        lines[i] = W.make_line(pieces, ply=int(rng.integers(8, 60)), history=hist)
    kw = dict(variant=0, seed=1, max_plies=200, auto_reset=0)
    g, o = B.Env(n, **kw), orc.Env(n, **kw)
    g.reset_from(_dev(lines)); o.reset_from(lines)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())
    om = o.legal_mask()
    gm = _np(g.legal_mask()).view(np.uint32)
    bad = np.nonzero((gm != om).any(axis=1))[0]
    assert len(bad) == 0, (len(bad), bad[:5])
    assert np.array_equal(_np(g.encode_obs().view(torch.int16)).view(np.uint16), o.encode_obs())
    o_off = orc.Env(n, **dict(kw, two_square=0)); o_off.reset_from(lines)
    assert (o_off.legal_mask() != om).any()    # the two-square rule did bite somewhere
    oa = o.sample_uniform(om)
    orr, od = o.step(oa)
    gr, gd = g.step(_dev(oa))
    assert np.array_equal(_np(gr), orr) and np.array_equal(_np(gd), od)
    assert np.array_equal(_np(g.get_boards()), o.get_boards())


def test_more_than_eight_scouts_a_side_are_refused():
    """The mask-free sampler of the on-chip rollouts lists at most 8 Scouts per side (no variant has more):
    a loaded or pinned line, or a pool setup, with more is refused instead of silently dropping moves."""
    pieces = {0: W.piece(W.FLAG, W.RED), 99: W.piece(W.FLAG, W.BLUE), 90: W.piece(W.MINER, W.BLUE)}
    for k in range(9):
        pieces[10 + k] = W.piece(W.SCOUT, W.RED)
    nine = W.make_line(pieces)
    del pieces[18]
    eight = W.make_line(pieces)
    g = B.Env(2, seed=1)
    g.reset_from(torch.from_numpy(np.stack([eight, eight])).cuda())
    assert g.check() == 0
    g.reset_from(torch.from_numpy(np.stack([eight, nine])).cuda())
    assert g.check() == B.BAD_STATE
    g.clear_error()
    g.reset_from(torch.from_numpy(np.stack([eight, eight])).cuda())
    g.pin_reset_state(torch.from_numpy(np.stack([nine, eight])).cuda())
    assert g.check() == B.BAD_STATE
    g.clear_error(); g.pin_reset_state(None)
    pool = np.zeros((2, 1, 40), np.uint8)
    pool[:, 0, 0] = W.FLAG
    pool[:, 0, 1:10] = W.SCOUT                       # nine Scouts
    g.set_setup_pool(torch.from_numpy(pool).cuda())
    assert g.check() == B.BAD_ARG
    g.clear_error()
    pool[:, 0, 9] = W.MINER
    g.set_setup_pool(torch.from_numpy(pool).cuda())
    assert g.check() == 0


def test_probe_write_fills_the_buffer_and_checks_its_arguments():
    g = B.Env(64, seed=1)
    for dyn in (True, False):
        buf = torch.zeros(5000 * 1600, dtype=torch.uint8, device="cuda")
        g.probe_write(buf, 1600, dyn)            # more pieces than CTAs: every piece, by ticket and by stride
        assert bool((buf.view(torch.int16) == 0x3F80).all())
        small = torch.zeros(3 * 32, dtype=torch.uint8, device="cuda")
        g.probe_write(small, 32, dyn)            # fewer pieces than CTAs
        assert bool((small.view(torch.int16) == 0x3F80).all())
    L = B.lib()
    buf = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    assert L.strat_probe_write(g.h, B._ptr(buf), 4096, 24, 1, B._stream()) == B.BAD_ARG    # not a multiple of 16
    assert L.strat_probe_write(g.h, B._ptr(buf), 4096, 4000 // 16 * 16, 1, B._stream()) == B.BAD_ARG  # does not divide
    assert L.strat_probe_write(g.h, B._ptr(buf), 0, 16, 1, B._stream()) == B.OK
    assert g.check() == 0
    # the ticket word cleans up after itself: a second environment-sized use right after works too
    g.probe_write(buf, 16, True); g.probe_write(buf, 16, True)
    assert bool((buf.view(torch.int16) == 0x3F80).all())
