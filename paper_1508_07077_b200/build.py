"""In-tree build of the CUDA library: nvcc -> paper_1508_07077_b200/libhpmc_b200.so (sm_100a only).

Flags that are part of the method's definition: --fmad=false (no contraction; an FMA only
where fmaf() is written), IEEE division and square root, no flush-to-zero; host code with -ffp-contract=off.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "hpmc_lib.cu")
DEPS = [os.path.join(HERE, "csrc", f) for f in ("hpmc_lib.cu", "move.cuh", "moveq.cuh", "cells.cuh", "geometry.cuh", "philox.cuh", "alu_peak.cuh")]
DEPS.append(os.path.join(os.path.dirname(HERE), "include", "hpmc.h"))
SO = os.path.join(HERE, "libhpmc_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "--fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
    "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math", "-shared",
]


def stale(so: str = SO) -> bool:
    if not os.path.exists(so):
        return True
    t = os.path.getmtime(so)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False, defines: tuple = (), out: str | None = None) -> str:
    """Compile the library if a source is newer than it.  `defines` + `out`: another build of the same sources under
    another file name (a test build with e.g. HPMC_WAIT_LIMIT_NS=1000, loaded through HPMC_LIBRARY_PATH); the default
    build takes no defines."""
    so = SO if out is None else out
    assert out is not None or not defines, "the default library is built without -D overrides"
    if force or stale(so):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = so + ".tmp%d" % os.getpid()
        cmd = [nvcc] + NVCC_FLAGS + ["-D" + d for d in defines] + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp, SRC]
        subprocess.run(cmd, check=True)
        os.replace(tmp, so)
    return so


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
