"""ALL-GAMES parity of the CUDA path with the oracle at the full sizes of BASELINE.json
configs 1-3 (SURVEY.md section 8d "Checked"): every game of the batch is mirrored by the CPU
oracle, sharded over the host's cores (tests/oracle_shards.py: test plumbing).  Actions,
rewards, done bytes and boards are compared on every step, masks and observations on a
schedule; for config 3 every ring row of a wrapping ring is compared.  The comparisons run on
the device (the oracle's arrays are uploaded), so a step costs one H2D copy."""
import numpy as np
import pytest
import torch

from oracle import orc
from oracle_shards import ShardedOracle, host_cores
from paper_2511_07312_b200 import binding as B
from paper_2511_07312_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _up(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.view(dtype)


def _same(dev, host, view=None):
    d = dev if view is None else dev.view(view)
    return torch.equal(d.reshape(-1), _up(host).view(d.dtype).reshape(-1))


def _first_bad(dev, host):
    d = dev.reshape(dev.shape[0], -1)
    h = _up(host).view(d.dtype).reshape(d.shape[0], -1)
    bad = (d != h).any(dim=1).nonzero()
    return int(bad[0]) if bad.numel() else -1


def test_config1_barrage_all_4096_games_to_termination():
    c = W.CONFIGS[1]
    n = c["num_games"]
    kw = dict(variant=1, seed=c["seed"], max_plies=c["max_plies"], auto_reset=0)
    print("host cores for the sharded oracle:", host_cores())
    g = B.Env(n, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    with ShardedOracle(n, **kw) as o:
        for t in range(c["steps"]):
            sched = t % 8 == 0 or t == c["steps"] - 1
            g.rollout_step(mask, act, rew, done, obs)
            o.step(want_mask=sched, want_obs_after=sched, want_boards=True)
            assert _same(act, o.act) and _same(rew, o.rew) and _same(done, o.done), (t, _first_bad(act, o.act))
            assert _same(g.get_boards(), o.boards), (t, _first_bad(g.get_boards(), o.boards))
            if sched:
                assert _same(mask, o.mask), (t, _first_bad(mask, o.mask))
                assert _same(obs.view(torch.int16), o.obs), (t, _first_bad(obs.view(torch.int16), o.obs))
        b = o.boards.copy()
    assert (b[:, 120] & 1).all()  # 2000-ply cap: every game is over
    reasons = np.bincount((b[:, 120] >> 2) & 7, minlength=6)
    print("config 1 termination reasons (flag, no-move win, no-move draw, ply cap, battleless):", reasons[1:].tolist())
    assert reasons[0] == 0 and reasons[1] > 0 and reasons.sum() == n
    assert not g.legal_mask().any()  # frozen games: zero mask
    assert g.check() == 0


@pytest.mark.parametrize("cap,steps", [(48, 72), (1000, 64)])
def test_config2_all_65536_games(cap, steps):
    """Config 2's launch shape (65,536 games, auto-reset).  cap = 48 forces the reset burst (every
    game still running hits the ply cap on the same step) inside the window; cap = 1000 is the
    configuration bench.py times."""
    c = W.CONFIGS[2]
    n = c["num_games"]
    kw = dict(variant=0, seed=c["seed"], max_plies=cap, auto_reset=1)
    print("host cores for the sharded oracle:", host_cores())
    g = B.Env(n, **kw)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    resets = 0
    with ShardedOracle(n, **kw) as o:
        for t in range(steps):
            sched = t % 8 == 0 or t == steps - 1 or t in (cap - 1, cap)
            g.rollout_step(mask, act, rew, done, obs)
            o.step(want_mask=sched, want_obs_after=sched, want_boards=True)
            assert _same(act, o.act) and _same(rew, o.rew) and _same(done, o.done), (t, _first_bad(act, o.act))
            assert _same(g.get_boards(), o.boards), (t, _first_bad(g.get_boards(), o.boards))
            if sched:
                assert _same(mask, o.mask), (t, _first_bad(mask, o.mask))
                assert _same(obs.view(torch.int16), o.obs), (t, _first_bad(obs.view(torch.int16), o.obs))
            resets += int((o.done & 1).sum())
    if cap < steps:
        assert resets > n // 2  # the burst happened
    assert g.check() == 0


def test_config3_all_262144_games_wrapping_ring_row_by_row():
    """Config 3's launch sequence (262,144 games, in-place push of all five arrays, 4,096-sample
    gather per step) on a ring of 2 blocks so that it wraps inside the window: after every push
    the block just completed is compared row by row, for ALL games, with the oracle's transition
    (obs_t, mask_t, action_t, reward_t, done_t), and the gathered minibatch with the oracle's
    indices applied to the oracle's records; at the end every live ring position is re-checked."""
    c = W.CONFIGS[3]
    n, bs = c["num_games"], c["sample_batch"]
    kw = dict(variant=0, seed=c["seed"], max_plies=c["max_plies"], auto_reset=1)
    free, _ = torch.cuda.mem_get_info()
    if free < 30e9:
        pytest.skip("needs ~25 GB of free device memory")
    print("host cores for the sharded oracle:", host_cores())
    g = B.Env(n, **kw)
    per_slot, slots = c["ring_per_slot"], 4  # capacity 524,288 = 2 blocks of 262,144
    ring = B.Replay(per_slot, slots, block=n)
    cap = ring.capacity
    s_obs = torch.empty((bs, 4400), dtype=torch.int16, device="cuda")
    s_mask = torch.empty((bs, 113), dtype=torch.int32, device="cuda")
    s_act = torch.empty(bs, dtype=torch.int16, device="cuda")
    s_rew = torch.empty(bs, dtype=torch.int8, device="cuda")
    s_done = torch.empty(bs, dtype=torch.uint8, device="cuda")
    o_ptr, _ = ring.reserve(n, 0)
    B._chk(B.lib().strat_encode_obs(g.h, o_ptr, B._stream()), "encode")
    vo, vm, va, vr, vd = ring.views()
    steps = 5
    keep = {}  # oracle records of the blocks that are still live at the end
    with ShardedOracle(n, with_obs=False, with_obs_before=True, **kw) as o:
        for t in range(steps):
            _, m_ptr = ring.reserve(n, 0)
            o_next, _ = ring.reserve(n, 1)
            a_ptr, r_ptr, d_ptr = ring.reserve_rows(n)
            g.rollout_step_ptrs(m_ptr, a_ptr, r_ptr, d_ptr, o_next)
            ring.commit_in_place(n)
            ring.sample_chained(g, c["seed"], t, bs, s_obs, s_mask, s_act, s_rew, s_done)  # as bench.py --workload cfg3
            o.step(want_mask=True, want_obs_before=True, want_boards=(t == steps - 1))
            head, filled = ring.state()
            assert head == ((t + 1) * n) % cap and filled == min((t + 1) * n, cap)
            rec = tuple(_up(x) for x in (o.obs_before, o.mask, o.act, o.rew, o.done))
            keep[t] = rec
            keep.pop(t - cap // n, None)
            # the block just completed, every row
            row, orow = ring.locate((t * n) % cap)
            assert torch.equal(vo[orow:orow + n], rec[0].view(torch.int16)), t
            assert torch.equal(vm[row:row + n], rec[1].view(torch.int32)), t
            assert torch.equal(va[row:row + n], rec[2]) and torch.equal(vr[row:row + n], rec[3]), t
            assert torch.equal(vd[row:row + n], rec[4]), t
            # the minibatch: the oracle's indices into the oracle's records
            idx = torch.from_numpy(orc.sample_indices(c["seed"], t, bs, filled)).cuda()
            blk = torch.div(idx, n, rounding_mode="floor")  # ring position -> block of the ring, game
            gi = idx - blk * n
            for k in keep:
                sel = blk == (k % (cap // n))
                if not sel.any():
                    continue
                e = keep[k]
                assert torch.equal(s_obs[sel], e[0].view(torch.int16)[gi[sel]]), (t, k)
                assert torch.equal(s_mask[sel], e[1].view(torch.int32)[gi[sel]]), (t, k)
                assert torch.equal(s_act[sel], e[2][gi[sel]]) and torch.equal(s_rew[sel], e[3][gi[sel]]), (t, k)
                assert torch.equal(s_done[sel], e[4][gi[sel]]), (t, k)
        assert _same(g.get_boards(), o.boards)
    for k, e in keep.items():  # every live position, after the wrap
        row, orow = ring.locate((k * n) % cap)
        assert torch.equal(vo[orow:orow + n], e[0].view(torch.int16)), k
        assert torch.equal(vm[row:row + n], e[1].view(torch.int32)), k
        assert torch.equal(va[row:row + n], e[2]) and torch.equal(vr[row:row + n], e[3]) and torch.equal(vd[row:row + n], e[4]), k
    assert g.check() == 0
