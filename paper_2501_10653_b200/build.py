"""nvcc build of libiqa_tiles.so for sm_100a (in-tree, next to this file).

    python -m paper_2501_10653_b200.build [--force]

The library is plain CUDA runtime code behind a C ABI (include/iqa_tiles.h); it does not
link against torch.  nvcc cross-compiles without a GPU, so this also runs in CI boxes.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
SOURCES = [os.path.join(CSRC, "iqa_tiles.cu")]
HEADERS = [os.path.join(CSRC, "iqa_kernels.cuh"), os.path.join(CSRC, "iqa_aggregate.cuh"), os.path.join(CSRC, "iqa_generic_vec.cuh"),
           os.path.join(CSRC, "iqa_any.cuh"), os.path.join(CSRC, "iqa_tma.cuh"), os.path.join(CSRC, "iqa_candidates.cuh"),
           os.path.join(_ROOT, "include", "iqa_tiles.h")]
LIB = os.path.join(_HERE, "libiqa_tiles.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "--cudart", "shared"]


class NoCompiler(RuntimeError):
    """nvcc is not installed (as opposed to: nvcc ran and the sources did not compile)."""


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise NoCompiler("nvcc not found: libiqa_tiles.so cannot be built (there is no CPU fallback)")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the library if it is missing or older than its sources. Returns its path."""
    if not force and not is_stale():
        return LIB
    cmd = [_nvcc(), *NVCC_FLAGS, "-o", LIB, *SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
