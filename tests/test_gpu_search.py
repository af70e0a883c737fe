"""The network-free search step (S3.7) on the CUDA path against the oracle:
expansion bit-exact; values exact; rho and pi_search within the float32 tolerance derived in
DESIGN.md (logits up to ~50 in float32 -> relative 1e-5; asserted at 1e-4)."""
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


def _roots(R, ply, seed):
    src = orc.Env(R, seed=seed, max_plies=1000, auto_reset=1)
    return W.capture_at_ply(src.get_boards, lambda: src.step(src.sample_uniform(src.legal_mask())), R, ply)


@pytest.mark.parametrize("R,ply,rollouts,depth,chase", [(6, 120, 1000, 40, 0), (5, 60, 37, 10, 0), (4, 200, 1000, 40, 1)])
def test_search_step_matches_oracle(R, ply, rollouts, depth, chase):
    rb = _roots(R, ply, seed=3)
    kw = dict(seed=3, chase_rule=chase)
    ro, rg = orc.Env(R, **kw), B.Env(R, **kw)
    ro.reset_from(rb); rg.reset_from(_dev(rb))
    go, gg = orc.Env(R * rollouts, **kw), B.Env(R * rollouts, **kw)
    orc.search_expand(ro, rollouts, 2024, go)
    B.search_expand(rg, rollouts, 2024, gg)
    assert np.array_equal(_np(gg.get_boards()), go.get_boards())
    for _ in range(depth - 1):
        go.step(go.sample_uniform(go.legal_mask()))
    gg.rollout_uniform(depth - 1)
    assert np.array_equal(_np(gg.get_boards()), go.get_boards())
    rng = np.random.default_rng(1)
    masks = ro.legal_mask()
    prior = np.zeros((R, 3600), np.float32)
    for r in range(R):
        legal = W.mask_to_actions(masks[r])
        p = rng.random(len(legal)) + 0.05
        prior[r, legal] = p / p.sum()
    for alpha, beta, pt in ((0.002, 0.02, None), (0.002, 0.02, prior), (0.5, 0.25, prior)):
        eq, er, ep = orc.search_policy(ro, go, rollouts, alpha, beta, pt)
        q, rho, pi = B.search_policy(rg, gg, rollouts, alpha, beta, None if pt is None else _dev(pt))
        q, rho, pi = _np(q), _np(rho), _np(pi)
        assert np.allclose(q, eq, rtol=1e-6, atol=0) and np.allclose(rho, er, rtol=1e-6, atol=0)
        assert np.array_equal(pi == 0, ep == 0) or np.allclose(pi, ep, rtol=1e-4, atol=1e-30)
        assert np.allclose(pi, ep, rtol=1e-4, atol=1e-12)
        assert np.allclose(pi.sum(axis=1), 1, atol=1e-5)
        assert depth < 40 or (q != 0).any()  # deep rollouts from late positions: some did finish
    # leaf values for the games still running: qhat to 1e-6, the policy as above
    vals = (rng.random(R * rollouts, dtype=np.float32) * 2 - 1).astype(np.float32)
    running = (go.get_boards()[:, 120] & 1) == 0
    assert running.any() and (~running).any() or depth < 40
    for alpha, beta, pt in ((0.002, 0.02, None), (0.5, 0.25, prior)):
        eq, er, ep = orc.search_policy(ro, go, rollouts, alpha, beta, pt, values=vals)
        q, rho, pi = B.search_policy(rg, gg, rollouts, alpha, beta, None if pt is None else _dev(pt), values=_dev(vals))
        q, rho, pi = _np(q), _np(rho), _np(pi)
        assert np.allclose(q, eq, rtol=1e-6, atol=1e-7) and np.allclose(rho, er, rtol=1e-6, atol=0)
        assert np.allclose(pi, ep, rtol=1e-4, atol=1e-12)
        assert np.allclose(pi.sum(axis=1), 1, atol=1e-5)
        assert (q != _np(B.search_policy(rg, gg, rollouts, alpha, beta, None if pt is None else _dev(pt))[0])).any()
    assert gg.check() == 0 and rg.check() == 0


def test_search_argument_errors():
    roots = B.Env(2, seed=1)
    out = B.Env(2 * 10, seed=1, auto_reset=1)
    with pytest.raises(B.StratError):
        B.search_expand(roots, 10, 0, out)  # the rollout games must not auto-reset
    out = B.Env(2 * 10 + 1, seed=1)
    with pytest.raises(B.StratError):
        B.search_expand(roots, 10, 0, out)  # size mismatch


def test_degenerate_priors_match_oracle():
    """One-hot priors, a prior excluding a legal action, and priors with no mass on any legal action
    (the root then falls back to "no prior", R29): finite, and equal to the oracle."""
    R, rollouts = 6, 300
    rb = _roots(R, 90, seed=5)
    ro, rg = orc.Env(R, seed=5), B.Env(R, seed=5)
    ro.reset_from(rb); rg.reset_from(_dev(rb))
    go, gg = orc.Env(R * rollouts, seed=5), B.Env(R * rollouts, seed=5)
    orc.search_expand(ro, rollouts, 11, go); B.search_expand(rg, rollouts, 11, gg)
    for _ in range(30):
        go.step(go.sample_uniform(go.legal_mask()))
    gg.rollout_uniform(30)
    masks = ro.legal_mask()
    prior = np.zeros((R, 3600), np.float32)
    legal = [W.mask_to_actions(masks[r]) for r in range(R)]
    prior[0, legal[0][1]] = 1.0                                   # one-hot on a legal action
    illegal = sorted(set(range(3600)) - set(legal[1]))
    prior[1, illegal[:7]] = 1.0 / 7                               # all mass on illegal actions
    prior[2, legal[2][1:]] = 1.0 / (len(legal[2]) - 1)            # first legal action excluded
    # root 3: all zeros; roots 4, 5: ordinary priors
    prior[4, legal[4]] = 1.0 / len(legal[4]); prior[5, legal[5]] = np.linspace(1, 2, len(legal[5]))
    eq, er, ep = orc.search_policy(ro, go, rollouts, 0.002, 0.02, prior)
    q, rho, pi = (_np(x) for x in B.search_policy(rg, gg, rollouts, 0.002, 0.02, _dev(prior)))
    assert np.isfinite(pi).all() and np.isfinite(ep).all()
    assert np.allclose(q, eq, rtol=1e-6, atol=0) and np.allclose(rho, er, rtol=1e-6, atol=0)
    assert np.allclose(pi, ep, rtol=1e-4, atol=1e-12)
    assert pi[0, legal[0][1]] == 1.0 and pi[2, legal[2][0]] == 0.0
    _, _, pn = (_np(x) for x in B.search_policy(rg, gg, rollouts, 0.002, 0.02, None))
    assert np.array_equal(pi[1], pn[1]) and np.array_equal(pi[3], pn[3])
