"""Thin Python binding of libstrat.so (include/strat.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the
library's CUDA kernels.  There is no CPU fallback: loading fails loudly if the library
cannot be built/loaded, and every call fails if CUDA is unavailable.
"""
import ctypes as C

import torch

from .build import ensure_built

LINE = 128
MASK_WORDS = 113
OBS_ELEMS = 4400
INFO_PLANES = 487
OK, BAD_ARG, BAD_STATE, CUDA_ERROR, ILLEGAL_ACTION, TOO_LARGE = 0, -1, -2, -3, -4, -5
STATIC_MAX_GAMES = 4096  # STRAT_STATIC_MAX_GAMES

EXPORTS = [
    "strat_error_string", "strat_workspace_bytes", "strat_create", "strat_destroy", "strat_reset",
    "strat_reset_from", "strat_reset_from_with_plies", "strat_get_boards", "strat_pin_reset_state", "strat_pin_reset_state_with_plies", "strat_set_setup_pool", "strat_legal_mask", "strat_sample_uniform", "strat_step",
    "strat_encode_obs", "strat_encode_infostate", "strat_rollout_step", "strat_step_observe", "strat_host_scratch_bytes", "strat_rollout_step_host",
    "strat_step_host", "strat_rollout_uniform", "strat_check", "strat_clear_error", "strat_replay_bytes", "strat_replay_layout",
    "strat_replay_create", "strat_replay_destroy", "strat_replay_bytes_in_place", "strat_replay_create_in_place",
    "strat_replay_locate", "strat_share_chain", "strat_replay_sample_chained", "strat_replay_push", "strat_replay_reserve",
    "strat_replay_reserve_rows",
    "strat_replay_commit", "strat_replay_sample", "strat_replay_state", "strat_determinise",
    "strat_reduce_returns", "strat_probe_write", "strat_legal_mask_static", "strat_history_bytes", "strat_history_create", "strat_history_destroy",
    "strat_history_bytes_tracked", "strat_history_create_tracked", "strat_history_encode_infostate",
    "strat_history_attach", "strat_history_current_step", "strat_history_legal_mask", "strat_history_encode_obs",
    "strat_history_get_boards", "strat_history_transition", "strat_history_info", "strat_history_restore",
    "strat_history_flags",
    "strat_search_expand", "strat_search_policy", "strat_search_policy_values",
]


class strat_config(C.Structure):
    _fields_ = [
        ("num_games", C.c_int32), ("variant", C.c_int32), ("seed", C.c_uint64),
        ("max_plies", C.c_int32), ("max_battleless", C.c_int32), ("auto_reset", C.c_int32),
        ("two_square", C.c_int32), ("device", C.c_int32), ("chase_rule", C.c_int32),
        ("game_base", C.c_uint64), ("infostate", C.c_int32), ("reserved", C.c_int32),
    ]


_lib = None


def lib():
    """Load (building if stale) the C-ABI library.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        L = C.CDLL(ensure_built())
        vp, i32, u64, sz = C.c_void_p, C.c_int32, C.c_uint64, C.c_size_t
        L.strat_error_string.restype = C.c_char_p
        L.strat_error_string.argtypes = [C.c_int]
        L.strat_workspace_bytes.restype = sz
        L.strat_workspace_bytes.argtypes = [C.POINTER(strat_config)]
        L.strat_create.argtypes = [C.POINTER(strat_config), vp, sz, vp, C.POINTER(vp)]
        L.strat_destroy.argtypes = [vp]
        L.strat_reset.argtypes = [vp, u64, vp]
        L.strat_reset_from.argtypes = [vp, vp, vp]
        L.strat_get_boards.argtypes = [vp, vp, vp]
        L.strat_pin_reset_state.argtypes = [vp, vp, vp, vp]
        L.strat_reset_from_with_plies.argtypes = [vp, vp, vp, vp]
        L.strat_pin_reset_state_with_plies.argtypes = [vp, vp, vp, vp, vp, vp]
        L.strat_set_setup_pool.argtypes = [vp, vp, i32, vp]
        L.strat_legal_mask.argtypes = [vp, vp, vp]
        L.strat_sample_uniform.argtypes = [vp, vp, vp, vp]
        L.strat_step.argtypes = [vp, vp, vp, vp, vp]
        L.strat_encode_obs.argtypes = [vp, vp, vp]
        L.strat_encode_infostate.argtypes = [vp, vp, vp]
        L.strat_probe_write.argtypes = [vp, vp, sz, i32, i32, vp]
        L.strat_legal_mask_static.argtypes = [vp, i32, i32, vp, vp, vp]
        L.strat_rollout_step.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.strat_step_observe.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.strat_host_scratch_bytes.restype = sz
        L.strat_host_scratch_bytes.argtypes = [C.POINTER(strat_config)]
        L.strat_rollout_step_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
        L.strat_step_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
        L.strat_rollout_uniform.argtypes = [vp, i32, vp]
        L.strat_check.argtypes = [vp]
        L.strat_clear_error.argtypes = [vp, vp]
        L.strat_replay_bytes.restype = sz
        L.strat_replay_bytes.argtypes = [i32, i32]
        L.strat_replay_layout.argtypes = [i32, i32, i32, C.POINTER(sz)]
        L.strat_replay_bytes_in_place.restype = sz
        L.strat_replay_bytes_in_place.argtypes = [i32, i32, i32]
        L.strat_replay_create_in_place.argtypes = [vp, sz, i32, i32, i32, C.POINTER(vp)]
        L.strat_replay_locate.argtypes = [vp, C.c_int64, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.strat_share_chain.argtypes = [vp, vp]
        L.strat_replay_create.argtypes = [vp, sz, i32, i32, C.POINTER(vp)]
        L.strat_replay_destroy.argtypes = [vp]
        L.strat_replay_push.argtypes = [vp, vp, vp, vp, vp, vp, i32, vp]
        L.strat_replay_reserve.argtypes = [vp, i32, i32, C.POINTER(vp), C.POINTER(vp)]
        L.strat_replay_reserve_rows.argtypes = [vp, i32, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.strat_replay_commit.argtypes = [vp, vp, vp, vp, i32, vp]
        L.strat_replay_sample.argtypes = [vp, u64, u64, i32, vp, vp, vp, vp, vp, vp]
        L.strat_replay_sample_chained.argtypes = [vp, vp, u64, u64, i32, vp, vp, vp, vp, vp, vp]
        L.strat_replay_state.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.strat_determinise.argtypes = [vp, i32, u64, vp, vp]
        L.strat_reduce_returns.argtypes = [vp, vp, i32, vp, vp]
        L.strat_search_expand.argtypes = [vp, i32, u64, vp, vp]
        L.strat_search_policy.argtypes = [vp, vp, i32, vp, C.c_float, C.c_float, vp, vp, vp, vp]
        L.strat_search_policy_values.argtypes = [vp, vp, i32, vp, vp, C.c_float, C.c_float, vp, vp, vp, vp]
        i64 = C.c_int64
        L.strat_history_bytes.restype = sz
        L.strat_history_bytes.argtypes = [i32, i32]
        L.strat_history_create.argtypes = [vp, sz, i32, i32, C.POINTER(vp)]
        L.strat_history_destroy.argtypes = [vp]
        L.strat_history_bytes_tracked.restype = sz
        L.strat_history_bytes_tracked.argtypes = [i32, i32]
        L.strat_history_create_tracked.argtypes = [vp, sz, i32, i32, vp, C.POINTER(vp)]
        L.strat_history_encode_infostate.argtypes = [vp, i64, vp, vp]
        L.strat_history_attach.argtypes = [vp, vp]
        L.strat_history_current_step.argtypes = [vp, C.POINTER(i64)]
        L.strat_history_legal_mask.argtypes = [vp, i64, vp, vp]
        L.strat_history_encode_obs.argtypes = [vp, i64, vp, vp]
        L.strat_history_get_boards.argtypes = [vp, i64, vp, vp]
        L.strat_history_transition.argtypes = [vp, i64, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.strat_history_info.argtypes = [vp, i64, vp, vp]
        L.strat_history_restore.argtypes = [vp, i64, vp, vp]
        L.strat_history_flags.argtypes = [vp, i64, vp, vp, vp, vp]
        _lib = L
    return _lib


class StratError(RuntimeError):
    pass


def _chk(rc, what):
    if rc != 0:
        raise StratError("%s: %s (%d)" % (what, lib().strat_error_string(rc).decode(), rc))


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t, dtype=None):
    if t is None:
        return C.c_void_p(0)
    assert t.is_cuda and t.is_contiguous(), "device, contiguous tensors only"
    if dtype is not None:
        assert t.dtype == dtype, (t.dtype, dtype)
    return C.c_void_p(t.data_ptr())


def _require_cuda():
    if not torch.cuda.is_available():
        raise StratError("CUDA device required: this library has no CPU path")


class Env:
    """N parallel games bound to a caller-owned (torch) workspace."""

    def __init__(self, num_games, variant=0, seed=0, max_plies=0, max_battleless=0, auto_reset=0,
                 two_square=1, device=0, game_base=0, chase_rule=0, infostate=0):
        _require_cuda()
        self.cfg = strat_config(num_games, variant, seed, max_plies, max_battleless, auto_reset,
                                two_square, device, chase_rule, game_base, infostate, 0)
        self.n = num_games
        self.device = torch.device("cuda", device)
        nbytes = lib().strat_workspace_bytes(C.byref(self.cfg))
        if nbytes == 0:
            raise StratError("bad configuration")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.h = C.c_void_p()
        with torch.cuda.device(self.device):
            _chk(lib().strat_create(C.byref(self.cfg), _ptr(self.workspace), nbytes, _stream(), C.byref(self.h)),
                 "strat_create")

    def __del__(self):
        if getattr(self, "h", None) is not None and self.h.value:
            if _lib is not None:  # module globals may be gone at interpreter shutdown
                _lib.strat_destroy(self.h)
            self.h = None

    # -- allocation helpers (plumbing)
    def new_mask(self):
        return torch.empty((self.n, MASK_WORDS), dtype=torch.int32, device=self.device)

    def new_obs(self):
        return torch.empty((self.n, 44, 10, 10), dtype=torch.bfloat16, device=self.device)

    def new_actions(self):
        return torch.empty(self.n, dtype=torch.int16, device=self.device)

    def new_reward(self):
        return torch.empty(self.n, dtype=torch.int8, device=self.device)

    def new_done(self):
        return torch.empty(self.n, dtype=torch.uint8, device=self.device)

    # -- the C-ABI calls, same names
    def reset(self, seed):
        _chk(lib().strat_reset(self.h, seed, _stream()), "strat_reset")

    def reset_from(self, boards, plies=None):
        """plies uint8[N][63][2] on the device: the plies that led to each state, most recent first."""
        assert boards.shape == (self.n, LINE)
        if plies is None:
            _chk(lib().strat_reset_from(self.h, _ptr(boards, torch.uint8), _stream()), "strat_reset_from")
            return
        assert plies.shape == (self.n, 63, 2)
        _chk(lib().strat_reset_from_with_plies(self.h, _ptr(boards, torch.uint8), _ptr(plies, torch.uint8), _stream()),
             "strat_reset_from_with_plies")

    def set_setup_pool(self, pool):
        """pool uint8[2][K][40] on the device (red setups, blue setups), or None for uniform permutations."""
        if pool is None:
            _chk(lib().strat_set_setup_pool(self.h, None, 0, _stream()), "strat_set_setup_pool")
            self._pool = None
            return
        assert pool.dim() == 3 and pool.shape[0] == 2 and pool.shape[2] == 40
        _chk(lib().strat_set_setup_pool(self.h, _ptr(pool, torch.uint8), pool.shape[1], _stream()), "strat_set_setup_pool")
        self._pool = pool  # the library reads it until replaced

    def pin_reset_state(self, boards, plies=None):
        """boards uint8[N][128] on the device, or None to unpin; plies as in reset_from."""
        if boards is None:
            _chk(lib().strat_pin_reset_state(self.h, None, None, _stream()), "strat_pin_reset_state")
            self._pin = None
            return
        assert boards.shape == (self.n, LINE)
        pin = torch.empty((self.n, LINE), dtype=torch.uint8, device=self.device)
        if plies is not None:
            assert plies.shape == (self.n, 63, 2)
            logs = torch.empty((self.n, 128), dtype=torch.uint8, device=self.device)
            _chk(lib().strat_pin_reset_state_with_plies(self.h, _ptr(pin), _ptr(logs), _ptr(boards, torch.uint8),
                                                        _ptr(plies, torch.uint8), _stream()), "strat_pin_reset_state_with_plies")
            self._pin = (pin, logs)
            return
        _chk(lib().strat_pin_reset_state(self.h, _ptr(pin), _ptr(boards, torch.uint8), _stream()), "strat_pin_reset_state")
        self._pin = pin  # the library reads it until unpinned

    def get_boards(self, out=None):
        out = out if out is not None else torch.empty((self.n, LINE), dtype=torch.uint8, device=self.device)
        _chk(lib().strat_get_boards(self.h, _ptr(out, torch.uint8), _stream()), "strat_get_boards")
        return out

    def legal_mask(self, out=None):
        out = out if out is not None else self.new_mask()
        _chk(lib().strat_legal_mask(self.h, _ptr(out, torch.int32), _stream()), "strat_legal_mask")
        return out

    def sample_uniform(self, mask, out=None):
        out = out if out is not None else self.new_actions()
        _chk(lib().strat_sample_uniform(self.h, _ptr(mask, torch.int32), _ptr(out, torch.int16), _stream()),
             "strat_sample_uniform")
        return out

    def step(self, actions, reward=None, done=None):
        reward = reward if reward is not None else self.new_reward()
        done = done if done is not None else self.new_done()
        _chk(lib().strat_step(self.h, _ptr(actions, torch.int16), _ptr(reward, torch.int8),
                              _ptr(done, torch.uint8), _stream()), "strat_step")
        return reward, done

    def encode_obs(self, out=None):
        out = out if out is not None else self.new_obs()
        _chk(lib().strat_encode_obs(self.h, _ptr(out, torch.bfloat16), _stream()), "strat_encode_obs")
        return out

    def new_infostate(self):
        return torch.empty((self.n, INFO_PLANES, 10, 10), dtype=torch.bfloat16, device=self.device)

    def encode_infostate(self, out=None):
        """The paper's 487-channel information state (needs infostate=1)."""
        out = out if out is not None else self.new_infostate()
        _chk(lib().strat_encode_infostate(self.h, _ptr(out, torch.bfloat16), _stream()), "strat_encode_infostate")
        return out

    def rollout_step(self, mask, actions, reward, done, obs):
        _chk(lib().strat_rollout_step(self.h, _ptr(mask), _ptr(actions), _ptr(reward), _ptr(done), _ptr(obs),
                                      _stream()), "strat_rollout_step")

    def step_observe(self, actions, reward, done, mask, obs):
        _chk(lib().strat_step_observe(self.h, _ptr(actions, torch.int16), _ptr(reward, torch.int8),
                                      _ptr(done, torch.uint8), _ptr(mask), _ptr(obs), _stream()), "strat_step_observe")

    def rollout_step_ptrs(self, mask_ptr, act_ptr, rew_ptr, done_ptr, obs_ptr):
        """rollout_step with raw device addresses for all five outputs (the replay ring's rows)."""
        _chk(lib().strat_rollout_step(self.h, C.c_void_p(mask_ptr), C.c_void_p(act_ptr), C.c_void_p(rew_ptr),
                                      C.c_void_p(done_ptr), C.c_void_p(obs_ptr), _stream()), "strat_rollout_step")

    def rollout_step_raw(self, mask_ptr, actions, reward, done, obs_ptr):
        """rollout_step with raw device addresses for mask/obs (e.g. replay_reserve's)."""
        _chk(lib().strat_rollout_step(self.h, C.c_void_p(mask_ptr), _ptr(actions), _ptr(reward), _ptr(done),
                                      C.c_void_p(obs_ptr), _stream()), "strat_rollout_step")

    def host_scratch(self):
        return torch.empty(lib().strat_host_scratch_bytes(C.byref(self.cfg)), dtype=torch.uint8, device=self.device)

    def rollout_step_host(self, scratch, mask_h, actions_h, reward_h, done_h, obs_h):
        for t in (mask_h, actions_h, reward_h, done_h, obs_h):
            assert not t.is_cuda and t.is_contiguous()
        _chk(lib().strat_rollout_step_host(self.h, _ptr(scratch), C.c_void_p(mask_h.data_ptr()),
                                           C.c_void_p(actions_h.data_ptr()), C.c_void_p(reward_h.data_ptr()),
                                           C.c_void_p(done_h.data_ptr()), C.c_void_p(obs_h.data_ptr()), _stream()),
             "strat_rollout_step_host")

    def step_host(self, scratch, actions_h, reward_h, done_h, mask_h, obs_h):
        for t in (actions_h, reward_h, done_h, mask_h, obs_h):
            assert not t.is_cuda and t.is_contiguous()
        _chk(lib().strat_step_host(self.h, _ptr(scratch), C.c_void_p(actions_h.data_ptr()),
                                   C.c_void_p(reward_h.data_ptr()), C.c_void_p(done_h.data_ptr()),
                                   C.c_void_p(mask_h.data_ptr()), C.c_void_p(obs_h.data_ptr()), _stream()),
             "strat_step_host")

    def rollout_uniform(self, plies):
        _chk(lib().strat_rollout_uniform(self.h, plies, _stream()), "strat_rollout_uniform")

    def share_chain(self, other):
        _chk(lib().strat_share_chain(self.h, other.h), "strat_share_chain")

    def probe_write(self, dst, chunk_bytes: int, dynamic: bool):
        """Measurement aid: stream a constant over the uint8 tensor dst (see strat_probe_write)."""
        _chk(lib().strat_probe_write(self.h, _ptr(dst, torch.uint8), dst.numel(), chunk_bytes, 1 if dynamic else 0, _stream()),
             "strat_probe_write")

    def check(self):
        return lib().strat_check(self.h)

    def clear_error(self):
        _chk(lib().strat_clear_error(self.h, _stream()), "strat_clear_error")


class Replay:
    """Device replay ring in a caller-owned (torch) buffer."""

    def __init__(self, per_slot, slots, device=0, block=0):
        """block = 0: plain ring (copying push); block = records per in-place push (spare rows)."""
        _require_cuda()
        self.device = torch.device("cuda", device)
        self.per_slot, self.slots, self.capacity, self.block = per_slot, slots, per_slot * slots, block
        self.rows, self.obs_rows = self.capacity + block, self.capacity + 2 * block
        nbytes = lib().strat_replay_bytes_in_place(per_slot, slots, block)
        if nbytes == 0:
            raise StratError("bad ring shape")
        self.mem = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        off = (C.c_size_t * 5)()
        _chk(lib().strat_replay_layout(per_slot, slots, block, off), "strat_replay_layout")
        self.offsets = list(off)
        self.h = C.c_void_p()
        if block:
            _chk(lib().strat_replay_create_in_place(_ptr(self.mem), nbytes, per_slot, slots, block, C.byref(self.h)),
                 "strat_replay_create_in_place")
        else:
            _chk(lib().strat_replay_create(_ptr(self.mem), nbytes, per_slot, slots, C.byref(self.h)), "strat_replay_create")

    def __del__(self):
        if getattr(self, "h", None) is not None and self.h.value:
            if _lib is not None:  # module globals may be gone at interpreter shutdown
                _lib.strat_replay_destroy(self.h)
            self.h = None

    def push(self, obs, mask, action, reward, done):
        n = action.numel()
        _chk(lib().strat_replay_push(self.h, _ptr(obs), _ptr(mask), _ptr(action, torch.int16),
                                     _ptr(reward, torch.int8), _ptr(done, torch.uint8), n, _stream()),
             "strat_replay_push")

    def reserve(self, n, ahead=0):
        obs, mask = C.c_void_p(), C.c_void_p()
        _chk(lib().strat_replay_reserve(self.h, n, ahead, C.byref(obs), C.byref(mask)), "strat_replay_reserve")
        return obs.value, mask.value

    def reserve_rows(self, n):
        a, r, d = C.c_void_p(), C.c_void_p(), C.c_void_p()
        _chk(lib().strat_replay_reserve_rows(self.h, n, C.byref(a), C.byref(r), C.byref(d)), "strat_replay_reserve_rows")
        return a.value, r.value, d.value

    def commit_in_place(self, n):
        _chk(lib().strat_replay_commit(self.h, None, None, None, n, _stream()), "strat_replay_commit")

    def commit(self, action, reward, done):
        _chk(lib().strat_replay_commit(self.h, _ptr(action, torch.int16), _ptr(reward, torch.int8),
                                       _ptr(done, torch.uint8), action.numel(), _stream()), "strat_replay_commit")

    def sample(self, seed, draw_index, batch, obs, mask, action, reward, done):
        _chk(lib().strat_replay_sample(self.h, seed, draw_index, batch, _ptr(obs), _ptr(mask), _ptr(action),
                                       _ptr(reward), _ptr(done), _stream()), "strat_replay_sample")

    def sample_chained(self, env, seed, draw_index, batch, obs, mask, action, reward, done):
        """Gather between two fused steps of `env` without separating them (in-place rings)."""
        _chk(lib().strat_replay_sample_chained(self.h, env.h, seed, draw_index, batch, _ptr(obs), _ptr(mask), _ptr(action),
                                               _ptr(reward), _ptr(done), _stream()), "strat_replay_sample_chained")
        self._env = env

    def state(self):
        h, f = C.c_int64(), C.c_int64()
        _chk(lib().strat_replay_state(self.h, C.byref(h), C.byref(f)), "strat_replay_state")
        return h.value, f.value

    def locate(self, p):
        """(row, obs_row) of the live record at ring position p."""
        r, o = C.c_int64(), C.c_int64()
        _chk(lib().strat_replay_locate(self.h, p, C.byref(r), C.byref(o)), "strat_replay_locate")
        return r.value, o.value

    # typed views of the ring arrays by physical row (tests); see locate()
    def views(self):
        Rn, Ro = self.rows, self.obs_rows
        o = self.offsets
        obs = self.mem[o[0]:o[0] + Ro * OBS_ELEMS * 2].view(torch.int16).view(Ro, OBS_ELEMS)
        mask = self.mem[o[1]:o[1] + Rn * MASK_WORDS * 4].view(torch.int32).view(Rn, MASK_WORDS)
        act = self.mem[o[2]:o[2] + Rn * 2].view(torch.int16)
        rew = self.mem[o[3]:o[3] + Rn].view(torch.int8)
        done = self.mem[o[4]:o[4] + Rn]
        return obs, mask, act, rew, done


class History:
    """Board-history ring (the paper's rollout buffer) in a caller-owned (torch) buffer."""

    def __init__(self, num_games, length, device=0, tracked=False):
        """tracked: also keep the S2 trackers per time step (strat_history_create_tracked), for encode_infostate(t)."""
        _require_cuda()
        self.device = torch.device("cuda", device)
        self.n, self.length = num_games, length
        nbytes = (lib().strat_history_bytes_tracked if tracked else lib().strat_history_bytes)(num_games, length)
        if nbytes == 0:
            raise StratError("bad history shape")
        self.mem = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.h = C.c_void_p()
        self.env = None
        if tracked:
            with torch.cuda.device(self.device):
                _chk(lib().strat_history_create_tracked(_ptr(self.mem), nbytes, num_games, length, _stream(), C.byref(self.h)),
                     "strat_history_create_tracked")
        else:
            _chk(lib().strat_history_create(_ptr(self.mem), nbytes, num_games, length, C.byref(self.h)),
                 "strat_history_create")

    def __del__(self):
        if getattr(self, "h", None) is not None and self.h.value:
            if _lib is not None:  # module globals may be gone at interpreter shutdown
                _lib.strat_history_destroy(self.h)
            self.h = None

    def attach(self, env):
        _chk(lib().strat_history_attach(env.h, self.h), "strat_history_attach")
        self.env = env  # keeps the environment alive as long as the ring refers to it

    def detach(self):
        if self.env is not None:
            _chk(lib().strat_history_attach(self.env.h, None), "strat_history_attach")
            self.env = None

    def current_step(self):
        s = C.c_int64()
        _chk(lib().strat_history_current_step(self.h, C.byref(s)), "strat_history_current_step")
        return s.value

    def legal_mask(self, t, out=None):
        out = out if out is not None else torch.empty((self.n, MASK_WORDS), dtype=torch.int32, device=self.device)
        _chk(lib().strat_history_legal_mask(self.h, t, _ptr(out, torch.int32), _stream()), "strat_history_legal_mask")
        return out

    def encode_obs(self, t, out=None):
        out = out if out is not None else torch.empty((self.n, 44, 10, 10), dtype=torch.bfloat16, device=self.device)
        _chk(lib().strat_history_encode_obs(self.h, t, _ptr(out, torch.bfloat16), _stream()), "strat_history_encode_obs")
        return out

    def encode_infostate(self, t, out=None):
        """The paper's 487-channel information state of time step t (tracked rings)."""
        out = out if out is not None else torch.empty((self.n, INFO_PLANES, 10, 10), dtype=torch.bfloat16, device=self.device)
        _chk(lib().strat_history_encode_infostate(self.h, t, _ptr(out, torch.bfloat16), _stream()),
             "strat_history_encode_infostate")
        return out

    def get_boards(self, t, out=None):
        out = out if out is not None else torch.empty((self.n, LINE), dtype=torch.uint8, device=self.device)
        _chk(lib().strat_history_get_boards(self.h, t, _ptr(out, torch.uint8), _stream()), "strat_history_get_boards")
        return out

    def transition(self, t):
        """Non-owning views (actions int16[N], reward int8[N], done uint8[N]) of time step t."""
        a, r, d = C.c_void_p(), C.c_void_p(), C.c_void_p()
        _chk(lib().strat_history_transition(self.h, t, C.byref(a), C.byref(r), C.byref(d)), "strat_history_transition")
        base = self.mem.data_ptr()

        def view(p, nbytes, dtype):
            return self.mem[p.value - base:p.value - base + nbytes].view(dtype)

        return view(a, 2 * self.n, torch.int16), view(r, self.n, torch.int8), view(d, self.n, torch.uint8)

    def info(self, t, out=None):
        out = out if out is not None else torch.empty((self.n, 4), dtype=torch.int32, device=self.device)
        _chk(lib().strat_history_info(self.h, t, _ptr(out, torch.int32), _stream()), "strat_history_info")
        return out

    def flags(self, t):
        """-> (two_square_applies uint8[N], unknown uint8[N,100], terminated_since int32[N])"""
        ts = torch.empty(self.n, dtype=torch.uint8, device=self.device)
        unk = torch.empty((self.n, 100), dtype=torch.uint8, device=self.device)
        since = torch.empty(self.n, dtype=torch.int32, device=self.device)
        _chk(lib().strat_history_flags(self.h, t, _ptr(ts), _ptr(unk), _ptr(since), _stream()), "strat_history_flags")
        return ts, unk, since

    def restore(self, t, env):
        _chk(lib().strat_history_restore(self.h, t, env.h, _stream()), "strat_history_restore")


def legal_mask_static(boards, mask, two_square=1, status=None):
    """strat_legal_mask_static: legal masks of the given canonical lines without an environment or a
    workspace, for callers that cannot allocate device memory (a plugin that only gets its input and
    output buffers, a loop that cannot afford cudaMalloc's device-wide stall, a process in which
    another thread is capturing a stream in the global mode).  The library's scratch for this call is
    a fixed 512.25 KB array inside its device image, so at most STATIC_MAX_GAMES positions per call
    (StratError "more games than the built-in scratch holds" beyond that).  Nothing is allocated
    here either: the caller passes every buffer, all on the current device -
      boards  uint8[n][128]   in
      mask    int32[n][113]   out, the same bits as Env.reset_from + Env.legal_mask
      status  int32[1]        out, optional: 0, or BAD_STATE for a line with too many Scouts.
    Calls share that one array: keep them on one stream (or order them with events); calls that
    overlap on the GPU corrupt each other.  Make the first call on a device outside stream capture."""
    _require_cuda()
    n = boards.shape[0]
    assert boards.shape == (n, LINE) and mask.shape == (n, MASK_WORDS)
    assert status is None or status.numel() == 1
    _chk(lib().strat_legal_mask_static(_ptr(boards, torch.uint8), n, 1 if two_square else 0, _ptr(mask, torch.int32),
                                       _ptr(status, torch.int32), _stream()), "strat_legal_mask_static")
    return mask


def determinise(roots: Env, samples_per_root: int, seed: int, out: Env):
    _chk(lib().strat_determinise(roots.h, samples_per_root, seed, out.h, _stream()), "strat_determinise")


def search_expand(roots: Env, rollouts: int, seed: int, out: Env):
    _chk(lib().strat_search_expand(roots.h, rollouts, seed, out.h, _stream()), "strat_search_expand")


def search_policy(roots: Env, games: Env, rollouts: int, alpha: float, beta: float, pi_theta=None, out=None, values=None):
    """-> (qhat, rho, pi_search): float32 [R, 3600] device tensors.  values: float32 [R*rollouts] leaf values
    from the searcher's side for the games still running (strat_search_policy_values), or None."""
    if out is None:
        out = tuple(torch.empty((roots.n, 3600), dtype=torch.float32, device=roots.device) for _ in range(3))
    q, rho, pi = out
    if values is not None:
        assert values.numel() == roots.n * rollouts
        _chk(lib().strat_search_policy_values(roots.h, games.h, rollouts,
                                              _ptr(pi_theta, torch.float32) if pi_theta is not None else None,
                                              _ptr(values, torch.float32), alpha, beta, _ptr(q, torch.float32),
                                              _ptr(rho, torch.float32), _ptr(pi, torch.float32), _stream()),
             "strat_search_policy_values")
        return q, rho, pi
    _chk(lib().strat_search_policy(roots.h, games.h, rollouts, _ptr(pi_theta, torch.float32) if pi_theta is not None else None,
                                   alpha, beta, _ptr(q, torch.float32), _ptr(rho, torch.float32), _ptr(pi, torch.float32),
                                   _stream()), "strat_search_policy")
    return q, rho, pi


def reduce_returns(games: Env, root_side, samples_per_root: int, out=None):
    R = games.n // samples_per_root
    out = out if out is not None else torch.empty((R, 3), dtype=torch.int32, device=games.device)
    _chk(lib().strat_reduce_returns(games.h, _ptr(root_side, torch.uint8), samples_per_root,
                                    _ptr(out, torch.int32), _stream()), "strat_reduce_returns")
    return out
