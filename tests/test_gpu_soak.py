"""Soak of the overlapped fused step: thousands of back-to-back launches (programmatic dependent launch,
per-batch version flags, ticket ring wrapping) with the board-history ring attached, then the mirrored
games must stand exactly where the oracle leaves them.  A lost update, a batch processed twice or a
launch running ahead of its predecessor's state would show up in some game."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_2511_07312_b200 import binding as B

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("chase,steps", [(0, 9000), (1, 3000)])
def test_soak_overlapped_fused_steps_with_history(chase, steps):
    n, mirrored, cap = 65536, 48, 150          # cap 150: ~60 auto-resets per game, every batch sees many
    kw = dict(variant=0, seed=11, max_plies=cap, auto_reset=1, chase_rule=chase)
    g = B.Env(n, **kw)
    h = B.History(n, 64)
    h.attach(g)
    mask, act, rew, done, obs = g.new_mask(), g.new_actions(), g.new_reward(), g.new_done(), g.new_obs()
    for _ in range(steps):                      # > 8,192 launches in the first case: the ticket ring wraps
        g.rollout_step(mask, act, rew, done, obs)
    torch.cuda.synchronize()
    assert g.check() == 0 and h.current_step() == steps
    o = orc.Env(mirrored, **kw)                 # global game indices 0..47 = the first games of the batch
    last = None
    for _ in range(steps):
        m = o.legal_mask()
        a = o.sample_uniform(m)
        last = (m, a) + o.step(a)
    gb = g.get_boards().cpu().numpy()
    assert np.array_equal(gb[:mirrored], o.get_boards())
    assert np.array_equal(mask.cpu().numpy().view(np.uint32)[:mirrored], last[0])
    assert np.array_equal(act.cpu().numpy()[:mirrored], last[1])
    assert np.array_equal(rew.cpu().numpy()[:mirrored], last[2]) and np.array_equal(done.cpu().numpy()[:mirrored], last[3])
    assert np.array_equal(obs.view(torch.int16).cpu().numpy().view(np.uint16)[:mirrored], o.encode_obs())
    # every game of the batch went through the same number of plies as a whole: epochs advanced everywhere
    epoch = gb[:, 124:128].copy().view(np.uint32)[:, 0]
    assert epoch.min() >= steps // cap - 1 and np.array_equal(epoch[:mirrored], o.get_boards()[:, 124:128].copy().view(np.uint32)[:, 0])
