"""Sanitizer tier (SURVEY.md section 4 T3 / section 5 "race detection, sanitizers") for the code that runs
on the host: the CPU oracle (oracle/stratego_oracle.cpp) and the per-game rule code of the kernels compiled
for the host (tests/host_harness.cpp on csrc/strat_game.cuh) are built once with AddressSanitizer and
UndefinedBehaviorSanitizer and driven through setups, random play to termination with auto-reset, the
chasing rule, both encoders, determinisation and the search step.  Any out-of-bounds access, use of an
uninitialised shift, signed overflow or misaligned access aborts the child process.  (compute-sanitizer
for the kernels themselves needs the GPU box.)"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SAN = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g", "-O1"]

DRIVER = r"""
import ctypes as C, sys
import numpy as np
san_orc, san_hh = sys.argv[1], sys.argv[2]
import oracle.build as ob
ob.ensure_built = lambda force=False: san_orc          # the sanitised build instead of oracle/liborc.so
from oracle import orc
from paper_2511_07312_b200 import workloads as W

hh = C.CDLL(san_hh)
vp = C.c_void_p
hh.hh_reset.argtypes = [C.c_int, C.c_uint64, C.c_uint32, vp]
hh.hh_legal_mask.argtypes = [vp, C.c_int, C.c_int, vp]
hh.hh_step.argtypes = [vp, C.c_int, C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp,
                       C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
hh.hh_encode.argtypes = [vp, vp]
p = lambda a: a.ctypes.data_as(vp)

for variant, cap, chase in ((0, 90, 1), (1, 400, 0)):
    n, seed = 24, 5
    o = orc.Env(n, variant=variant, seed=seed, max_plies=cap, max_battleless=60, auto_reset=1, chase_rule=chase, infostate=1)
    line, out, row = np.zeros(128, np.uint8), np.zeros(128, np.uint8), np.zeros(113, np.uint32)
    planes = np.zeros(4400, np.uint16)
    rew, done, ill = C.c_int(), C.c_int(), C.c_int()
    for g in range(n):
        hh.hh_reset(variant, seed, g, p(line))
        assert np.array_equal(line, o.get_boards()[g])
    for t in range(260):
        b = o.get_boards()
        m = o.legal_mask(); a = o.sample_uniform(m)
        if t % 20 == 0:
            o.encode_obs(); o.encode_infostate()
        for g in range(0, n, 5):   # the kernels' rule code on the same positions (chasing rule judged on the line's 8 plies)
            hh.hh_legal_mask(p(b[g]), 1, 0, p(row))
            hh.hh_encode(p(b[g]), p(planes))
            if not chase:
                assert np.array_equal(row, m[g])
                hh.hh_step(p(b[g]), variant, seed, g, cap, 1, 1, 0, int(a[g]), p(out), C.byref(rew), C.byref(done), C.byref(ill))
        o.step(a)
    assert (o.get_boards()[:, 124] > 0).any()

# search-shaped calls: determinise, expand, rollouts, reduce, eq. (8) with and without leaf values
roots = orc.Env(3, seed=4, max_plies=1000, auto_reset=1, chase_rule=1)
for _ in range(70):
    roots.step(roots.sample_uniform(roots.legal_mask()))
det = orc.Env(3 * 8, seed=4, chase_rule=1)
orc.determinise(roots, 8, 9, det)
for _ in range(20):
    det.step(det.sample_uniform(det.legal_mask()))
orc.reduce_returns(det, np.zeros(3, np.uint8), 8)
games = orc.Env(3 * 50, seed=4, chase_rule=1)
orc.search_expand(roots, 50, 11, games)
for _ in range(15):
    games.step(games.sample_uniform(games.legal_mask()))
orc.search_policy(roots, games, 50, 0.002, 0.02)
orc.search_policy(roots, games, 50, 0.002, 0.02, values=np.linspace(-1, 1, 150).astype(np.float32))
# replay ring: push, wrap, sample
ring = orc.Replay(16, 4)
e = orc.Env(24, seed=1, max_plies=40, auto_reset=1)
for _ in range(5):
    obs, m = e.encode_obs(), e.legal_mask(); a = e.sample_uniform(m); r, d = e.step(a)
    ring.push(obs, m, a, r, d)
ring.sample(3, 0, 32)
print("sanitised run ok")
"""


def test_oracle_and_host_compiled_rule_code_under_asan_and_ubsan(tmp_path):
    san_orc, san_hh = str(tmp_path / "liborc_san.so"), str(tmp_path / "libhh_san.so")
    subprocess.check_call(["g++", *SAN, "-std=c++17", "-fPIC", "-shared", os.path.join(ROOT, "oracle", "stratego_oracle.cpp"),
                           "-o", san_orc])
    subprocess.check_call(["g++", *SAN, "-std=c++17", "-fPIC", "-shared", os.path.join(HERE, "host_harness.cpp"), "-o", san_hh])
    asan = subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=97",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1:exitcode=98", PYTHONPATH=ROOT + os.pathsep + HERE)
    out = subprocess.run([sys.executable, "-c", DRIVER, san_orc, san_hh], capture_output=True, text=True, env=env,
                         cwd=ROOT, timeout=900)
    assert out.returncode == 0, (out.returncode, out.stdout[-1500:], out.stderr[-4000:])
    assert "sanitised run ok" in out.stdout
    assert "runtime error" not in out.stderr and "AddressSanitizer" not in out.stderr, out.stderr[-4000:]
