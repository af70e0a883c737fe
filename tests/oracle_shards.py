"""Test plumbing only: the CPU oracle sharded over host processes for ALL-GAMES parity checks.

One worker process per host core, each owning a contiguous range of games as its own
`orc.Env(game_base=lo)` (every RNG draw of the method is keyed by the global game index, so
the union of the shards is the unsharded run: tests/test_sharding.py).  The workers write
their outputs into shared-memory arrays the test compares with the CUDA path's.  Nothing here
computes anything of the method; the product never imports this.
"""
import multiprocessing as mp
import os
from multiprocessing import shared_memory

import numpy as np

LINE, MASK_WORDS, OBS = 128, 113, 4400


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def _attach(specs):
    out, keep = {}, []
    for name, (shm_name, shape, dtype) in specs.items():
        shm = shared_memory.SharedMemory(name=shm_name)
        keep.append(shm)
        out[name] = np.ndarray(shape, dtype=dtype, buffer=shm.buf)
    return out, keep


def _worker(conn, lo, hi, kw, specs):
    import sys
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    from oracle import orc
    arr, keep = _attach(specs)
    e = orc.Env(hi - lo, game_base=lo, **kw)
    s = slice(lo, hi)
    try:
        while True:
            cmd = conn.recv()
            if cmd[0] == "step":
                _, want_mask, want_obs_before, want_obs_after, want_boards = cmd
                if want_obs_before:
                    arr["obs_before"][s] = e.encode_obs().reshape(hi - lo, OBS)
                m = e.legal_mask()
                a = e.sample_uniform(m)
                r, d = e.step(a)
                arr["act"][s] = a
                arr["rew"][s] = r
                arr["done"][s] = d
                if want_mask:
                    arr["mask"][s] = m
                if want_obs_after:
                    arr["obs"][s] = e.encode_obs().reshape(hi - lo, OBS)
                if want_boards:
                    arr["boards"][s] = e.get_boards()
                conn.send(e.check())
            elif cmd[0] == "boards":
                arr["boards"][s] = e.get_boards()
                conn.send(0)
            elif cmd[0] == "quit":
                break
    finally:
        for shm in keep:
            shm.close()


class ShardedOracle:
    """N games of one configuration over `procs` oracle processes.  After step(...) the arrays
    act / rew / done (and mask / obs / obs_before / boards when asked for) hold all N games."""

    def __init__(self, n, procs=None, with_obs=True, with_obs_before=False, **kw):
        self.n = n
        self.procs = max(1, min(procs or host_cores(), (n + 31) // 32))
        shapes = {"act": ((n,), np.int16), "rew": ((n,), np.int8), "done": ((n,), np.uint8),
                  "mask": ((n, MASK_WORDS), np.uint32), "boards": ((n, LINE), np.uint8)}
        if with_obs:
            shapes["obs"] = ((n, OBS), np.uint16)
        if with_obs_before:
            shapes["obs_before"] = ((n, OBS), np.uint16)
        self._shm, specs = [], {}
        for name, (shape, dtype) in shapes.items():
            nbytes = int(np.prod(shape)) * np.dtype(dtype).itemsize
            shm = shared_memory.SharedMemory(create=True, size=max(nbytes, 1))
            self._shm.append(shm)
            specs[name] = (shm.name, shape, dtype)
            setattr(self, name, np.ndarray(shape, dtype=dtype, buffer=shm.buf))
        ctx = mp.get_context("spawn")  # the parent holds a CUDA context: never fork it
        per = -(-n // self.procs)
        per = -(-per // 32) * 32
        self._workers = []
        for lo in range(0, n, per):
            hi = min(n, lo + per)
            parent, child = ctx.Pipe()
            p = ctx.Process(target=_worker, args=(child, lo, hi, kw, specs), daemon=True)
            p.start()
            self._workers.append((p, parent))

    def step(self, want_mask=False, want_obs_before=False, want_obs_after=False, want_boards=False):
        for _, c in self._workers:
            c.send(("step", want_mask, want_obs_before, want_obs_after, want_boards))
        errs = [c.recv() for _, c in self._workers]
        assert not any(errs), errs

    def get_boards(self):
        for _, c in self._workers:
            c.send(("boards",))
        for _, c in self._workers:
            c.recv()
        return self.boards

    def close(self):
        for p, c in self._workers:
            try:
                c.send(("quit",))
            except Exception:
                pass
        for p, _ in self._workers:
            p.join(timeout=10)
            if p.is_alive():
                p.kill()  # the exact process this object started
        self._workers = []
        for name in ("act", "rew", "done", "mask", "boards", "obs", "obs_before"):
            if hasattr(self, name):
                delattr(self, name)
        for shm in self._shm:
            shm.close()
            shm.unlink()
        self._shm = []

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
