"""In-tree build of libcorr.so (nvcc, sm_100a only).  `python -m paper_0906_1887_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcorr.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def _sources():
    out = [os.path.join(INCLUDE, "corr.h")]
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in _sources())


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/corr_lib.cu (which includes every kernel) into libcorr.so beside this file."""
    if not force and not stale():
        return LIB
    nvcc = os.environ.get("NVCC") or "nvcc"
    tmp = f"{LIB}.{os.getpid()}.tmp"
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp, os.path.join(CSRC, "corr_lib.cu")]
    try:
        subprocess.check_call(cmd)
    except FileNotFoundError as e:
        raise RuntimeError("nvcc not found: libcorr.so cannot be built (there is no CPU fallback)") from e
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
