"""Build libleyline.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_01065_b200.build [--force]

The shared library sits next to this file so that it travels with the source snapshot; it is git-ignored.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libleyline.so")
SOURCES = ["plan.cpp", "splice.cu", "cdc.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler",
              "-fPIC,-Wall,-Wextra,-fvisibility=hidden", "-Xptxas", "-v", "--shared", "-cudart", "static"]


STAMP = LIB + ".flags"      # the nvcc flags the library in place was built with (git-ignored, travels with the .so)


def _extra() -> list:
    return os.environ.get("LEYLINE_NVCC_EXTRA", "").split()      # e.g. -DNAME=value for an experiment build


def _flag_string() -> str:
    return " ".join([*NVCC_FLAGS, *_extra()])


def built_with() -> str:
    """The flag string of the library in place ("" if it was never stamped): bench.py records its -D knobs."""
    try:
        with open(STAMP) as f:
            return f.read()
    except OSError:
        return ""


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    # an experiment build (LEYLINE_NVCC_EXTRA=-D...) must not be picked up silently by a later default run, nor the
    # other way round: the library is rebuilt whenever the flags asked for differ from the flags it was built with
    if built_with() != _flag_string():
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, f) for f in os.listdir(INCLUDE)] + [__file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or _stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, *NVCC_FLAGS, *_extra(), "-I", INCLUDE, "-I", CSRC, "-o", LIB + ".tmp",
           *[os.path.join(CSRC, s) for s in SOURCES]]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed building libleyline.so")
    if verbose:
        sys.stderr.write(r.stdout + r.stderr)
    os.replace(LIB + ".tmp", LIB)
    with open(STAMP, "w") as f:
        f.write(_flag_string())
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
