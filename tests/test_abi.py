"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every
symbol include/strat.h declares (no compute calls are made without a GPU)."""
import ctypes as C
import os
import re

from paper_2511_07312_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "strat.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(strat_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = _declared_functions()
    assert len(names) >= 25
    L = C.CDLL(build.ensure_built())
    for n in names:
        assert hasattr(L, n), "libstrat.so does not export %s" % n
    assert sorted(binding.EXPORTS) == names  # the binding marshals exactly the declared calls


def test_host_only_entry_points():
    L = binding.lib()
    cfg = binding.strat_config(65536, 0, 0, 1000, 0, 1, 1, 0, 0, 0, 0, 0)
    ws = L.strat_workspace_bytes(C.byref(cfg))  # lines + error block + ticket ring + 2 flags per 32-game batch + 64 spare counters
    assert ws == 65536 * 128 + 256 + (8192 + 2 * 2048 + 64) * 4
    chase = binding.strat_config(65536, 0, 0, 1000, 0, 1, 1, 0, 1, 0, 0, 0)  # + a 64-ply move log per game
    assert L.strat_workspace_bytes(C.byref(chase)) == ws + 65536 * 128
    info = binding.strat_config(65536, 0, 0, 1000, 0, 1, 1, 0, 0, 0, 1, 0)  # + 2 KB of S2 trackers per game
    assert L.strat_workspace_bytes(C.byref(info)) == ws + 65536 * 2048
    bad = binding.strat_config(0, 0, 0, 0, 0, 0, 1, 0, 0, 0, 0, 0)
    assert L.strat_workspace_bytes(C.byref(bad)) == 0
    assert L.strat_error_string(-4) == b"illegal action for a live game"
    off = (C.c_size_t * 5)()
    assert L.strat_replay_layout(131072, 64, 0, off) == 0
    cap = 131072 * 64
    assert list(off)[:2] == [0, cap * 8800]
    assert L.strat_replay_bytes(131072, 64) >= cap * 9256
    assert L.strat_replay_bytes(0, 1) == 0
    # an in-place ring for pushes of 262,144 records: one spare block of rows, two of observations
    blk = 262144
    assert L.strat_replay_layout(131072, 64, blk, off) == 0
    assert list(off)[:3] == [0, (cap + 2 * blk) * 8800, (cap + 2 * blk) * 8800 + (cap + blk) * 452]
    assert L.strat_replay_bytes_in_place(131072, 64, blk) >= cap * 9256 + blk * (2 * 8800 + 456)
    assert L.strat_replay_bytes_in_place(131072, 64, 3) == 0  # the block must divide the capacity
    # RNG counters carry a 32-bit global game index
    over = binding.strat_config(65536, 0, 0, 1000, 0, 1, 1, 0, 0, (1 << 32) - 65535, 0, 0)
    assert L.strat_workspace_bytes(C.byref(over)) == 0
    edge = binding.strat_config(65536, 0, 0, 1000, 0, 1, 1, 0, 0, (1 << 32) - 65536, 0, 0)
    assert L.strat_workspace_bytes(C.byref(edge)) == ws
    # sizes of the per-step outputs the e2e entry point stages
    n = 1000
    cfg = binding.strat_config(n, 0, 0, 0, 0, 0, 1, 0, 0, 0, 0, 0)
    assert L.strat_host_scratch_bytes(C.byref(cfg)) >= n * 9256


def test_config_struct_matches_header():
    text = open(os.path.join(ROOT, "include", "strat.h")).read()
    body = re.search(r"typedef struct strat_config \{(.*?)\} strat_config;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"(u?int\d+_t)\s+(\w+);", body)
    ctype = {"int32_t": C.c_int32, "uint64_t": C.c_uint64}
    assert [(n, ctype[t]) for t, n in fields] == list(binding.strat_config._fields_)
    assert C.sizeof(binding.strat_config) == 56
