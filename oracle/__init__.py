"""oracle -- CPU oracle for the X-engine (ctypes binding over xcorr_oracle.c).

TEST INFRASTRUCTURE: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package.  The product package never does (tests/test_abi_cpu.py::test_product_and_oracle_are_independent checks).

All arithmetic is in ``xcorr_oracle.c`` (read its header for the passages it
follows: PAPER.md:47, :53, :84, :107, :115).  This file only marshals numpy
arrays.  Parity status: every function below is pinned by
``tests/test_oracle_pins.py`` (P1-P9, P11-P12 for the 4-bit mode, P14 for the int64 accumulation, tests/golden/) or, for the F-stage
(``fstage_oracle.c``), ``tests/test_oracle_fstage_pins.py`` (F1-F7); none is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "xcorr_oracle.c")
_SRC_F = os.path.join(_HERE, "fstage_oracle.c")  # F-stage (unpack + DFT), SURVEY 8(f) row 3
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


class OracleOverflow(ArithmeticError):
    """A sum does not fit int32 (oracle refuses rather than wrap)."""


def build(force: bool = False) -> str:
    """gcc -O2, no fused multiply-add contraction (Im V_ii must be exactly 0 in float64)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_F)):
        tmp = f"{_LIB}.{os.getpid()}.tmp"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
             "-o", tmp, _SRC, _SRC_F, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        L, I, P = ctypes.c_long, ctypes.c_int, ctypes.c_void_p
        _lib.oracle_xengine_ci8.argtypes = [P, L, L, L, L, L, P, I]
        _lib.oracle_xengine_cf32.argtypes = [P, L, L, L, L, L, P, I]
        _lib.oracle_xengine_ci4.argtypes = [P, L, L, L, L, L, P, I]
        _lib.oracle_unpack_ci4.argtypes = [ctypes.c_ubyte, ctypes.POINTER(I), ctypes.POINTER(I)]
        _lib.oracle_unpack_ci4.restype = None
        _lib.oracle_readout_i32.argtypes = [P, L, ctypes.c_double, P]
        _lib.oracle_readout_f64.argtypes = [P, L, ctypes.c_double, P]
        _lib.oracle_readout_i32.restype = _lib.oracle_readout_f64.restype = None
        _lib.oracle_xengine_ci8_wide.argtypes = [P, L, L, L, L, L, P, I]
        _lib.oracle_readout_i64.argtypes = [P, L, ctypes.c_double, P]
        _lib.oracle_readout_i64.restype = None
        _lib.oracle_full_matrix_ci8.argtypes = [P, L, L, L, L, P]
        _lib.oracle_full_matrix_cf32.argtypes = [P, L, L, L, L, P]
        _lib.oracle_one_visibility_ci8.argtypes = [P, L, L, L, L, L, L, P]
        _lib.oracle_one_visibility_cf32.argtypes = [P, L, L, L, L, L, L, P]
        _lib.oracle_fstage_ci8.argtypes = [P, L, L, L, P, I]
        _lib.oracle_fstage_ci4.argtypes = [P, L, L, L, P, I]
        _lib.oracle_xengine_cf64.argtypes = [P, L, L, L, P, I]
    return _lib


def _check_cube(x, dtype):
    x = np.ascontiguousarray(x)
    if x.dtype != dtype or x.ndim != 4 or x.shape[3] != 2:
        raise ValueError(f"expected [T][C][N][2] {dtype}, got {x.dtype} {x.shape}")
    return x, x.shape[0], x.shape[1], x.shape[2]


def host_threads() -> int:
    return max(1, len(os.sched_getaffinity(0)))


def xengine_ci8(x, c_begin=0, c_end=None, threads=1):
    """x: int8 [T][C][N][2] -> int32 [c_end-c_begin][N(N+1)/2][2] (raw sums, i>=j row-major)."""
    x, T, C, N = _check_cube(x, np.int8)
    c_end = C if c_end is None else c_end
    vis = np.empty((c_end - c_begin, N * (N + 1) // 2, 2), dtype=np.int32)
    rc = _load().oracle_xengine_ci8(x.ctypes.data, T, C, N, c_begin, c_end, vis.ctypes.data, threads)
    if rc == -2:
        raise OracleOverflow("visibility does not fit int32")
    if rc != 0:
        raise MemoryError("oracle allocation failed")
    return vis


def xengine_ci8_wide(x, c_begin=0, c_end=None, threads=1):
    """x: int8 [T][C][N][2], any T -> int64 [c_end-c_begin][N(N+1)/2][2]: the sums of a long accumulation
    (PAPER.md:84, :125), never refused for overflow."""
    x, T, C, N = _check_cube(x, np.int8)
    c_end = C if c_end is None else c_end
    vis = np.empty((c_end - c_begin, N * (N + 1) // 2, 2), dtype=np.int64)
    rc = _load().oracle_xengine_ci8_wide(x.ctypes.data, T, C, N, c_begin, c_end, vis.ctypes.data, threads)
    if rc != 0:
        raise MemoryError("oracle allocation failed")
    return vis


def unpack_ci4(byte):
    """(re, im) of one packed 4+4-bit sample (reading R18: low nibble Re, high nibble Im, two's complement)."""
    re, im = ctypes.c_int(), ctypes.c_int()
    _load().oracle_unpack_ci4(int(byte) & 255, ctypes.byref(re), ctypes.byref(im))
    return re.value, im.value


def xengine_ci4(x, c_begin=0, c_end=None, threads=1):
    """x: uint8 [T][C][N] packed 4+4-bit samples -> int32 [c_end-c_begin][N(N+1)/2][2]."""
    x = np.ascontiguousarray(x)
    if x.dtype != np.uint8 or x.ndim != 3:
        raise ValueError(f"expected [T][C][N] uint8, got {x.dtype} {x.shape}")
    T, C, N = x.shape
    c_end = C if c_end is None else c_end
    vis = np.empty((c_end - c_begin, N * (N + 1) // 2, 2), dtype=np.int32)
    rc = _load().oracle_xengine_ci4(x.ctypes.data, T, C, N, c_begin, c_end, vis.ctypes.data, threads)
    if rc != 0:
        raise MemoryError("oracle allocation failed")
    return vis


def readout(vis, count):
    """Time-averaged visibilities: raw sums / number of accumulated samples -> float64."""
    vis = np.ascontiguousarray(vis)
    out = np.empty(vis.shape, dtype=np.float64)
    if vis.dtype == np.int32:
        _load().oracle_readout_i32(vis.ctypes.data, vis.size, float(count), out.ctypes.data)
    elif vis.dtype == np.int64:
        _load().oracle_readout_i64(vis.ctypes.data, vis.size, float(count), out.ctypes.data)
    elif vis.dtype == np.float64:
        _load().oracle_readout_f64(vis.ctypes.data, vis.size, float(count), out.ctypes.data)
    else:
        raise ValueError("readout expects int32, int64 or float64 sums")
    return out


def xengine_cf32(x, c_begin=0, c_end=None, threads=1):
    """x: float32 [T][C][N][2] -> float64 [c_end-c_begin][N(N+1)/2][2]."""
    x, T, C, N = _check_cube(x, np.float32)
    c_end = C if c_end is None else c_end
    vis = np.empty((c_end - c_begin, N * (N + 1) // 2, 2), dtype=np.float64)
    rc = _load().oracle_xengine_cf32(x.ctypes.data, T, C, N, c_begin, c_end, vis.ctypes.data, threads)
    if rc != 0:
        raise MemoryError("oracle allocation failed")
    return vis


def full_matrix_ci8(x, c):
    """Full N x N matrix of channel c: int64 [N][N][2]."""
    x, T, C, N = _check_cube(x, np.int8)
    full = np.empty((N, N, 2), dtype=np.int64)
    _load().oracle_full_matrix_ci8(x.ctypes.data, T, C, N, c, full.ctypes.data)
    return full


def full_matrix_cf32(x, c):
    x, T, C, N = _check_cube(x, np.float32)
    full = np.empty((N, N, 2), dtype=np.float64)
    _load().oracle_full_matrix_cf32(x.ctypes.data, T, C, N, c, full.ctypes.data)
    return full


def one_visibility_ci8(x, c, i, j):
    """(re, im) of V[c][(i,j)] as python ints."""
    x, T, C, N = _check_cube(x, np.int8)
    out = np.empty(2, dtype=np.int64)
    _load().oracle_one_visibility_ci8(x.ctypes.data, T, C, N, c, i, j, out.ctypes.data)
    return int(out[0]), int(out[1])


def one_visibility_cf32(x, c, i, j):
    x, T, C, N = _check_cube(x, np.float32)
    out = np.empty(2, dtype=np.float64)
    _load().oracle_one_visibility_cf32(x.ctypes.data, T, C, N, c, i, j, out.ctypes.data)
    return float(out[0]), float(out[1])


# --------------------------------------------------------------------------- F-stage (fstage_oracle.c)

def fstage_ci8(x, threads=1):
    """x: [B][N_C][N_I][2] int8 raw voltages -> [B][N_C][N_I][2] float64 spectra, the plain O(N^2) DFT with
    exp(-2 pi i k n / N), unnormalised (readings R19-R21)."""
    x = np.ascontiguousarray(x)
    assert x.dtype == np.int8 and x.ndim == 4 and x.shape[3] == 2, x.shape
    B, N, I, _ = x.shape
    out = np.empty((B, N, I, 2), dtype=np.float64)
    rc = _load().oracle_fstage_ci8(x.ctypes.data, B, N, I, out.ctypes.data, int(threads))
    assert rc == 0
    return out


def fstage_ci4(x, threads=1):
    """x: [B][N_C][N_I] uint8 (low nibble Re, high nibble Im, 4-bit two's complement: the paper's 1-byte mode,
    PAPER.md:164) -> [B][N_C][N_I][2] float64 spectra."""
    x = np.ascontiguousarray(x)
    assert x.dtype == np.uint8 and x.ndim == 3, (x.dtype, x.shape)
    B, N, I = x.shape
    out = np.empty((B, N, I, 2), dtype=np.float64)
    rc = _load().oracle_fstage_ci4(x.ctypes.data, B, N, I, out.ctypes.data, int(threads))
    assert rc == 0
    return out


def xengine_cf64(x, threads=1):
    """x: [T][C][N][2] float64 spectra -> [C][N(N+1)/2][2] float64 (the X-engine definition in float64)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    assert x.ndim == 4 and x.shape[3] == 2, x.shape
    T, C, N, _ = x.shape
    vis = np.empty((C, N * (N + 1) // 2, 2), dtype=np.float64)
    rc = _load().oracle_xengine_cf64(x.ctypes.data, T, C, N, vis.ctypes.data, int(threads))
    assert rc == 0
    return vis
