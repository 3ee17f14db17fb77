"""Build libsph_b200.so (hand-written CUDA for sm_100a) in-tree with nvcc.

`python -m paper_2403_11156_b200.build` or `build()`; the library is rebuilt when any source
under csrc/ or include/sph.h is newer than the .so.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
LIB = os.path.join(_HERE, "libsph_b200.so")
SOURCES = [os.path.join(_HERE, "csrc", "sph_api.cu")]
DEPS = glob.glob(os.path.join(_HERE, "csrc", "*.cu*")) + [os.path.join(_ROOT, "include", "sph.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "--expt-extended-lambda", "--expt-relaxed-constexpr",
    "-Xcompiler", "-fPIC", "-shared",
    "-Xptxas", "-v",
]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc] + NVCC_FLAGS + os.environ.get("SPH_NVCC_EXTRA", "").split() + ["-o", LIB] + SOURCES
        res = subprocess.run(cmd, capture_output=True, text=True)
        log = os.path.join(_HERE, "csrc", "build.log")
        with open(log, "w") as f:
            f.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed building libsph_b200.so (see %s)" % log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
