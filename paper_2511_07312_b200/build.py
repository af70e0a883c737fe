"""Compile libstrat.so for sm_100a with nvcc (in-tree; no JIT cache)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = [os.path.join(CSRC, "strat.cu")]
DEPS = SOURCES + [os.path.join(CSRC, h) for h in ("strat_game.cuh", "strat_io.cuh", "strat_kernels.cuh",
                                                  "strat_fused.cuh", "strat_search.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "strat.h")]
LIB = os.path.join(HERE, "libstrat.so")
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def nvcc():
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.sep not in p or os.path.exists(p)):
            return p
    raise RuntimeError("nvcc not found")


def ensure_built(force: bool = False, verbose: bool = False) -> str:
    stale = not os.path.exists(LIB) or any(os.path.getmtime(LIB) < os.path.getmtime(d) for d in DEPS)
    if force or stale:
        tmp = LIB + ".tmp.%d" % os.getpid()
        out = subprocess.run([nvcc(), *NVCC_FLAGS, *SOURCES, "-o", tmp], capture_output=True, text=True)
        if out.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + out.stdout + out.stderr)
        if verbose:
            print(out.stdout + out.stderr)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(ensure_built(force=True, verbose=True))
