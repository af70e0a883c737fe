"""ctypes wrapper of the CPU oracle (TEST INFRASTRUCTURE ONLY; see __init__.py).

Argument marshalling only; every rule lives in stratego_oracle.cpp.
"""
import ctypes as C

import numpy as np

from .build import ensure_built

LINE = 128
MASK_WORDS = 113
PLANES = 44
OBS = PLANES * 100
INFO_PLANES = 487

OK, BAD_ARG, BAD_STATE, ILLEGAL_ACTION = 0, -1, -2, -4


class Config(C.Structure):
    _fields_ = [
        ("num_games", C.c_int32),
        ("variant", C.c_int32),
        ("seed", C.c_uint64),
        ("max_plies", C.c_int32),
        ("max_battleless", C.c_int32),
        ("auto_reset", C.c_int32),
        ("two_square", C.c_int32),
        ("device", C.c_int32),
        ("chase_rule", C.c_int32),
        ("game_base", C.c_uint64),
        ("infostate", C.c_int32),
        ("reserved", C.c_int32),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(ensure_built())
        vp = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(Config), C.POINTER(vp)]
        L.orc_destroy.argtypes = [vp]
        L.orc_reset.argtypes = [vp, C.c_uint64]
        L.orc_reset_from.argtypes = [vp, vp]
        L.orc_get_boards.argtypes = [vp, vp]
        L.orc_pin_reset_state.argtypes = [vp, vp]
        L.orc_reset_from_with_plies.argtypes = [vp, vp, vp]
        L.orc_pin_reset_state_with_plies.argtypes = [vp, vp, vp]
        L.orc_set_setup_pool.argtypes = [vp, vp, C.c_int32]
        L.orc_legal_mask.argtypes = [vp, vp]
        L.orc_sample_uniform.argtypes = [vp, vp, vp]
        L.orc_step.argtypes = [vp, vp, vp, vp]
        L.orc_encode_obs.argtypes = [vp, vp]
        L.orc_encode_infostate.argtypes = [vp, vp]
        L.orc_bf16_of_ratio.argtypes = [C.c_int64, C.c_int64]
        L.orc_bf16_of_ratio.restype = C.c_uint16
        L.orc_check.argtypes = [vp]
        L.orc_clear_error.argtypes = [vp]
        L.orc_replay_create.argtypes = [C.c_int32, C.c_int32, C.POINTER(vp)]
        L.orc_replay_destroy.argtypes = [vp]
        L.orc_replay_push.argtypes = [vp, vp, vp, vp, vp, vp, C.c_int32]
        L.orc_replay_sample.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_int32, vp, vp, vp, vp, vp, vp]
        L.orc_replay_read.argtypes = [vp, C.c_int64, vp, vp, vp, vp, vp]
        L.orc_replay_head.argtypes = [vp]
        L.orc_replay_head.restype = C.c_int64
        L.orc_replay_filled.argtypes = [vp]
        L.orc_replay_filled.restype = C.c_int64
        L.orc_sample_indices.argtypes = [C.c_uint64, C.c_uint64, C.c_int32, C.c_int64, vp]
        L.orc_search_expand.argtypes = [vp, C.c_int32, C.c_uint64, vp]
        L.orc_search_policy.argtypes = [vp, vp, C.c_int32, vp, C.c_double, C.c_double, vp, vp, vp]
        L.orc_search_policy_values.argtypes = [vp, vp, C.c_int32, vp, vp, C.c_double, C.c_double, vp, vp, vp]
        L.orc_determinise.argtypes = [vp, C.c_int32, C.c_uint64, vp, vp]
        L.orc_reduce_returns.argtypes = [vp, vp, C.c_int32, vp]
        L.orc_find_setup_redraws.argtypes = [C.POINTER(Config), C.c_uint32, C.c_uint32, C.c_uint32, vp, C.c_int]
        L.orc_philox.argtypes = [vp, vp, vp]
        L.orc_philox.restype = None
        L.orc_battle.argtypes = [C.c_int, C.c_int]
        L.orc_is_lake.argtypes = [C.c_int]
        L.orc_multiset.argtypes = [C.c_int, vp]
        L.orc_multiset.restype = None
        L.orc_chain.argtypes = [vp, C.c_int, C.c_int, vp]
        L.orc_count_moves.argtypes = [vp, C.c_int, C.c_int]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError("oracle %s failed: %d" % (what, rc))


class Env:
    def __init__(self, num_games, variant=0, seed=0, max_plies=0, max_battleless=0,
                 auto_reset=0, two_square=1, game_base=0, chase_rule=0, infostate=0):
        self.cfg = Config(num_games, variant, seed, max_plies, max_battleless, auto_reset,
                          two_square, 0, chase_rule, game_base, infostate, 0)
        self.n = num_games
        self.h = C.c_void_p()
        _chk(lib().orc_create(C.byref(self.cfg), C.byref(self.h)), "create")

    def __del__(self):
        if getattr(self, "h", None) and self.h.value:
            if _lib is not None:  # module globals may be gone at interpreter shutdown
                _lib.orc_destroy(self.h)
            self.h = None

    def reset(self, seed):
        _chk(lib().orc_reset(self.h, seed), "reset")

    def reset_from(self, boards, plies=None):
        """plies uint8[N][63][2]: the plies that led to each state, most recent first."""
        b = np.ascontiguousarray(boards, dtype=np.uint8)
        assert b.shape == (self.n, LINE)
        if plies is None:
            _chk(lib().orc_reset_from(self.h, _p(b)), "reset_from")
            return
        pl = np.ascontiguousarray(plies, dtype=np.uint8)
        assert pl.shape == (self.n, 63, 2)
        _chk(lib().orc_reset_from_with_plies(self.h, _p(b), _p(pl)), "reset_from_with_plies")

    def set_setup_pool(self, pool):
        """pool uint8[2][K][40] (red setups, blue setups), or None for uniform permutations."""
        if pool is None:
            _chk(lib().orc_set_setup_pool(self.h, None, 0), "set_setup_pool")
            return
        p = np.ascontiguousarray(pool, dtype=np.uint8)
        assert p.ndim == 3 and p.shape[0] == 2 and p.shape[2] == 40
        _chk(lib().orc_set_setup_pool(self.h, _p(p), p.shape[1]), "set_setup_pool")

    def pin_reset_state(self, boards, plies=None):
        """boards uint8[N][128], or None to unpin."""
        if boards is None:
            _chk(lib().orc_pin_reset_state(self.h, None), "pin_reset_state")
            return
        b = np.ascontiguousarray(boards, dtype=np.uint8)
        assert b.shape == (self.n, LINE)
        if plies is not None:
            pl = np.ascontiguousarray(plies, dtype=np.uint8)
            assert pl.shape == (self.n, 63, 2)
            _chk(lib().orc_pin_reset_state_with_plies(self.h, _p(b), _p(pl)), "pin_reset_state_with_plies")
            return
        _chk(lib().orc_pin_reset_state(self.h, _p(b)), "pin_reset_state")

    def get_boards(self):
        b = np.zeros((self.n, LINE), np.uint8)
        _chk(lib().orc_get_boards(self.h, _p(b)), "get_boards")
        return b

    def legal_mask(self):
        m = np.zeros((self.n, MASK_WORDS), np.uint32)
        _chk(lib().orc_legal_mask(self.h, _p(m)), "legal_mask")
        return m

    def sample_uniform(self, mask):
        m = np.ascontiguousarray(mask, dtype=np.uint32)
        a = np.zeros(self.n, np.int16)
        _chk(lib().orc_sample_uniform(self.h, _p(m), _p(a)), "sample_uniform")
        return a

    def step(self, actions):
        a = np.ascontiguousarray(actions, dtype=np.int16)
        r = np.zeros(self.n, np.int8)
        d = np.zeros(self.n, np.uint8)
        _chk(lib().orc_step(self.h, _p(a), _p(r), _p(d)), "step")
        return r, d

    def encode_obs(self):
        o = np.zeros((self.n, PLANES, 10, 10), np.uint16)
        _chk(lib().orc_encode_obs(self.h, _p(o)), "encode_obs")
        return o

    def encode_infostate(self):
        """The paper's 487-channel information state as bf16 bit patterns."""
        o = np.zeros((self.n, INFO_PLANES, 10, 10), np.uint16)
        _chk(lib().orc_encode_infostate(self.h, _p(o)), "encode_infostate")
        return o

    def check(self):
        return lib().orc_check(self.h)

    def clear_error(self):
        lib().orc_clear_error(self.h)

    def chain(self, gi, side):
        pos = np.zeros(4, np.int32)
        n = lib().orc_chain(self.h, gi, side, _p(pos))
        return [int(x) for x in pos[:n]]

    def count_moves(self, gi, side):
        return lib().orc_count_moves(self.h, gi, side)


class Replay:
    def __init__(self, per_slot, slots):
        self.h = C.c_void_p()
        self.capacity = per_slot * slots
        _chk(lib().orc_replay_create(per_slot, slots, C.byref(self.h)), "replay_create")

    def __del__(self):
        if getattr(self, "h", None) and self.h.value:
            if _lib is not None:
                _lib.orc_replay_destroy(self.h)
            self.h = None

    def push(self, obs, mask, action, reward, done):
        n = len(action)
        obs = np.ascontiguousarray(obs, np.uint16)
        mask = np.ascontiguousarray(mask, np.uint32)
        action = np.ascontiguousarray(action, np.int16)
        reward = np.ascontiguousarray(reward, np.int8)
        done = np.ascontiguousarray(done, np.uint8)
        _chk(lib().orc_replay_push(self.h, _p(obs), _p(mask), _p(action), _p(reward), _p(done), n), "replay_push")

    def sample(self, seed, draw_index, batch):
        obs = np.zeros((batch, PLANES, 10, 10), np.uint16)
        mask = np.zeros((batch, MASK_WORDS), np.uint32)
        action = np.zeros(batch, np.int16)
        reward = np.zeros(batch, np.int8)
        done = np.zeros(batch, np.uint8)
        idx = np.zeros(batch, np.int64)
        _chk(lib().orc_replay_sample(self.h, seed, draw_index, batch, _p(obs), _p(mask), _p(action),
                                     _p(reward), _p(done), _p(idx)), "replay_sample")
        return obs, mask, action, reward, done, idx

    def read(self, p):
        obs = np.zeros((PLANES, 10, 10), np.uint16)
        mask = np.zeros(MASK_WORDS, np.uint32)
        a = np.zeros(1, np.int16)
        r = np.zeros(1, np.int8)
        d = np.zeros(1, np.uint8)
        _chk(lib().orc_replay_read(self.h, p, _p(obs), _p(mask), _p(a), _p(r), _p(d)), "replay_read")
        return obs, mask, int(a[0]), int(r[0]), int(d[0])

    @property
    def head(self):
        return lib().orc_replay_head(self.h)

    @property
    def filled(self):
        return lib().orc_replay_filled(self.h)


def sample_indices(seed, draw_index, batch, filled):
    idx = np.zeros(batch, np.int64)
    _chk(lib().orc_sample_indices(seed, draw_index, batch, filled, _p(idx)),
         "sample_indices")
    return idx


def determinise(roots: Env, samples_per_root: int, seed: int, out: Env):
    att = np.zeros(out.n, np.int32)
    _chk(lib().orc_determinise(roots.h, samples_per_root, seed, out.h, _p(att)), "determinise")
    return att


def search_expand(roots: Env, rollouts: int, seed: int, out: Env):
    _chk(lib().orc_search_expand(roots.h, rollouts, seed, out.h), "search_expand")


def search_policy(roots: Env, games: Env, rollouts: int, alpha: float, beta: float, pi_theta=None, values=None):
    """-> (qhat, rho, pi_search), float32 [R, 3600] each (computed in double).  values: float32 [R*rollouts]
    leaf values from the searcher's side for the games still running, or None."""
    R = roots.n
    q, rho, pi = (np.zeros((R, 3600), np.float32) for _ in range(3))
    prior = None if pi_theta is None else np.ascontiguousarray(pi_theta, np.float32)
    if values is None:
        _chk(lib().orc_search_policy(roots.h, games.h, rollouts, None if prior is None else _p(prior), alpha, beta,
                                     _p(q), _p(rho), _p(pi)), "search_policy")
        return q, rho, pi
    vals = np.ascontiguousarray(values, np.float32)
    assert vals.shape == (R * rollouts,)
    _chk(lib().orc_search_policy_values(roots.h, games.h, rollouts, None if prior is None else _p(prior), _p(vals), alpha, beta,
                                        _p(q), _p(rho), _p(pi)), "search_policy_values")
    return q, rho, pi


def reduce_returns(games: Env, root_side, samples_per_root: int):
    rs = np.ascontiguousarray(root_side, np.uint8)
    out = np.zeros((games.n // samples_per_root, 3), np.int32)
    _chk(lib().orc_reduce_returns(games.h, _p(rs), samples_per_root, _p(out)), "reduce_returns")
    return out


def find_setup_redraws(variant, seed, epoch, start, count, max_out=64):
    """Global game indices in [start, start+count) whose setup at `epoch` needs a redraw (R#5)."""
    cfg = Config(1, variant, seed, 0, 0, 0, 1, 0, 0, 0, 0, 0)
    out = np.zeros(max_out, np.uint32)
    n = lib().orc_find_setup_redraws(C.byref(cfg), epoch, start, count, _p(out), max_out)
    assert n >= 0
    return out[:n].tolist()


def bf16_of_ratio(num, den):
    return int(lib().orc_bf16_of_ratio(num, den))


def philox(ctr, key):
    c = np.asarray(ctr, np.uint32)
    k = np.asarray(key, np.uint32)
    o = np.zeros(4, np.uint32)
    lib().orc_philox(_p(c), _p(k), _p(o))
    return o


def battle(att, deff):
    return lib().orc_battle(att, deff)


def is_lake(c):
    return bool(lib().orc_is_lake(c))


def multiset(variant):
    out = np.zeros(40, np.int32)
    lib().orc_multiset(variant, _p(out))
    return out
