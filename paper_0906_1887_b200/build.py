"""In-tree build of libcorr.so (nvcc, sm_100a only) and of its diagnostics twin libcorr_diag.so.
`python -m paper_0906_1887_b200.build [--force] [-v] [--diag]`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcorr.so")
# the same sources with -DCORR_DIAG: adds the entry points of include/corr_diag.h (peak probes, engine
# switches) and the probe-instrumented kernel instantiations, which the product library does not carry
LIB_DIAG = os.path.join(HERE, "libcorr_diag.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def _sources():
    out = [os.path.join(INCLUDE, "corr.h"), os.path.join(INCLUDE, "corr_diag.h")]
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def stale(diag: bool = False) -> bool:
    lib = LIB_DIAG if diag else LIB
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(s) > t for s in _sources())


def build(force: bool = False, verbose: bool = False, diag: bool = False) -> str:
    """Compile csrc/corr_lib.cu (which includes every kernel) into libcorr.so (or libcorr_diag.so) beside this file."""
    lib = LIB_DIAG if diag else LIB
    if not force and not stale(diag):
        return lib
    nvcc = os.environ.get("NVCC") or "nvcc"
    tmp = f"{lib}.{os.getpid()}.tmp"
    cmd = [nvcc] + NVCC_FLAGS + (["-DCORR_DIAG"] if diag else []) + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp, os.path.join(CSRC, "corr_lib.cu")]
    try:
        subprocess.check_call(cmd)
    except FileNotFoundError as e:
        raise RuntimeError("nvcc not found: the library cannot be built (there is no CPU fallback)") from e
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, diag="--diag" in sys.argv))
