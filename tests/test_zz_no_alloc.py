"""strat_legal_mask_static: the legal-mask query for callers that cannot allocate device memory.

Who that is: code that only ever receives its input and output buffers from the framework it runs
inside (an operator / server plugin, a data-loader stage) and cannot reach that framework's
allocator; a latency-critical loop that cannot take the device-wide stall of cudaMalloc / cudaFree;
a thread of a process in which another thread is capturing a stream in the global capture mode
(cudaMalloc is forbidden process-wide meanwhile).  For them the library keeps the scratch of this one
call (the bit-sliced state lines + the error word) in a fixed array of its own device image, 512.25 KB
for at most B.STATIC_MAX_GAMES positions, and allocates nothing.

The test compares the call with the path that already exists and is itself checked against the oracle
(Env.reset_from + Env.legal_mask on a caller-allocated workspace), bit for bit - the tolerance of every
mask test here - on two calls in a row that share the array: the second follows the first on the stream
with no synchronisation in between, uses fewer games than the first (so stale lines of the first call
sit right behind its own) and comes after a call that raised the error word (which must be cleared).

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not
hide the tests of the main path.  It passes alone in a fresh process (then its first call is the one
that looks up the array's address) and after all the other tests.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2511_07312_b200 import binding as B
from paper_2511_07312_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _positions(n, seed, plies, variant=0):
    """n mid-game positions (canonical lines, device) produced by the existing path."""
    g = B.Env(n, variant=variant, seed=seed, max_plies=400, auto_reset=1)
    g.rollout_uniform(plies)
    b = g.get_boards()
    assert g.check() == 0
    return b


def _existing_path(boards, two_square):
    ref = B.Env(boards.shape[0], two_square=two_square)
    ref.reset_from(boards)
    m = ref.legal_mask()
    return m, ref.check()


def test_static_scratch_masks_equal_the_workspace_path_on_two_calls_in_a_row():
    nmax = B.STATIC_MAX_GAMES
    first = _positions(nmax, seed=11, plies=57)                 # the maximum size: 128 batches of 32 games
    second = _positions(1237, seed=12, plies=140, variant=1)    # 38 batches and a ragged tail of 21, Barrage
    # a line the import refuses: nine red Scouts (no variant has more than eight)
    bad = second.clone()
    pieces = {c: W.piece(2, 0) for c in range(9)}
    pieces[99] = W.piece(11, 1)
    bad[5] = torch.from_numpy(np.ascontiguousarray(W.make_line(pieces))).cuda()

    # every buffer is the caller's, allocated before the calls
    m_bad = torch.full((1237, B.MASK_WORDS), -1, dtype=torch.int32, device="cuda")
    m1 = torch.full((nmax, B.MASK_WORDS), -1, dtype=torch.int32, device="cuda")
    m2 = torch.full((1237, B.MASK_WORDS), -1, dtype=torch.int32, device="cuda")
    st = torch.full((3,), 77, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()

    B.legal_mask_static(bad, m_bad, two_square=1, status=st[0:1])   # raises the error word in the shared array
    B.legal_mask_static(first, m1, two_square=1, status=st[1:2])    # call 1: full size, error word must be clean again
    B.legal_mask_static(second, m2, two_square=0, status=st[2:3])   # call 2: right behind it, smaller, other rule switch
    torch.cuda.synchronize()

    assert st.cpu().tolist() == [B.BAD_STATE, 0, 0]
    for boards, ts, got in ((first, 1, m1), (second, 0, m2)):
        want, err = _existing_path(boards, ts)
        assert err == 0
        assert torch.equal(got, want)
        assert int((want != 0).any(dim=1).sum()) > boards.shape[0] // 2   # real masks, not all-zero rows
    # the refused line is reported the way the workspace path reports it; the other games are unaffected
    want_bad, err_bad = _existing_path(bad, 1)
    assert err_bad == B.BAD_STATE
    keep = torch.ones(1237, dtype=torch.bool, device="cuda")
    keep[5] = False
    assert torch.equal(m_bad[keep], want_bad[keep])

    # the two-square switch matters somewhere in these positions (the argument is not ignored)
    m2_ts = torch.empty_like(m2)
    B.legal_mask_static(second, m2_ts, two_square=1)
    assert torch.equal(m2_ts, _existing_path(second, 1)[0])


def test_static_scratch_refuses_more_games_than_it_holds():
    n = B.STATIC_MAX_GAMES + 1
    boards = torch.zeros((n, B.LINE), dtype=torch.uint8, device="cuda")
    mask = torch.full((n, B.MASK_WORDS), -1, dtype=torch.int32, device="cuda")
    with pytest.raises(B.StratError, match="more games than the built-in scratch holds"):
        B.legal_mask_static(boards, mask)
    torch.cuda.synchronize()
    assert bool((mask == -1).all())  # nothing was launched
    L = B.lib()
    vp = C.c_void_p
    assert L.strat_legal_mask_static(vp(boards.data_ptr()), 0, 1, vp(mask.data_ptr()), vp(0), vp(0)) == B.BAD_ARG
    assert L.strat_legal_mask_static(vp(0), 8, 1, vp(mask.data_ptr()), vp(0), vp(0)) == B.BAD_ARG
    assert L.strat_legal_mask_static(vp(boards.data_ptr()), 8, 1, vp(0), vp(0), vp(0)) == B.BAD_ARG
