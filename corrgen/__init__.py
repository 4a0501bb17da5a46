"""corrgen -- seeded synthetic voltage generators and the workload table.

Shared by the oracle's tests, the CUDA parity tests and ``bench.py``.  It makes
INPUTS only: none of the correlator's arithmetic lives here (see gen.c header).

Two implementations of the same counter-based recipe:

* ``gen.c`` (gcc, OpenMP) -- fills gigabyte cubes in seconds; used everywhere.
* ``*_numpy`` mirrors below -- vectorised numpy restatement used by the tests
  to pin the C generator (same hash, same Box-Muller, same rounding).

Workloads ``CONFIGS`` are BASELINE.json's five configs (seed k-1 for config k);
they stand in for the MWA-32T recordings the paper timed (PAPER.md:164-166,
:178): those recordings are not available and are not needed.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libcorrgen.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile gen.c -> libcorrgen.so (gcc -O2 -fopenmp) if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = f"{_LIB}.{os.getpid()}.tmp"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
             "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        L, D, U, I = ctypes.c_long, ctypes.c_double, ctypes.c_uint64, ctypes.c_int
        P = ctypes.c_void_p
        _lib.corrgen_gauss_i8.argtypes = [P, L, L, L, L, U, D, D, D, I]
        _lib.corrgen_uniform_i8.argtypes = [P, L, L, L, L, U, I, I]
        _lib.corrgen_gauss_f32.argtypes = [P, L, L, L, L, U, D, D, I]
        for f in (_lib.corrgen_gauss_i8, _lib.corrgen_uniform_i8, _lib.corrgen_gauss_f32):
            f.restype = None
    return _lib


def default_threads() -> int:
    return max(1, len(os.sched_getaffinity(0)))


# --------------------------------------------------------------------------- C generators

def gauss_i8(T, C, N, seed, sigma, clip, tone_amp=0.0, t_begin=0, t_end=None, out=None, threads=None):
    """int8 cube [t_end-t_begin][C][N][2] of clip(rint(sigma*g + tone))."""
    t_end = T if t_end is None else t_end
    if out is None:
        out = np.empty((t_end - t_begin, C, N, 2), dtype=np.int8)
    assert out.dtype == np.int8 and out.flags.c_contiguous and out.size == (t_end - t_begin) * C * N * 2
    _load().corrgen_gauss_i8(out.ctypes.data, t_begin, t_end, C, N, seed, float(sigma), float(clip),
                             float(tone_amp), threads or default_threads())
    return out


def uniform_i8(T, C, N, seed, clip, t_begin=0, t_end=None, out=None, threads=None):
    t_end = T if t_end is None else t_end
    if out is None:
        out = np.empty((t_end - t_begin, C, N, 2), dtype=np.int8)
    assert out.dtype == np.int8 and out.flags.c_contiguous and out.size == (t_end - t_begin) * C * N * 2
    _load().corrgen_uniform_i8(out.ctypes.data, t_begin, t_end, C, N, seed, int(clip),
                               threads or default_threads())
    return out


def gauss_f32(T, C, N, seed, sigma, tone_amp=0.0, t_begin=0, t_end=None, out=None, threads=None):
    t_end = T if t_end is None else t_end
    if out is None:
        out = np.empty((t_end - t_begin, C, N, 2), dtype=np.float32)
    assert out.dtype == np.float32 and out.flags.c_contiguous and out.size == (t_end - t_begin) * C * N * 2
    _load().corrgen_gauss_f32(out.ctypes.data, t_begin, t_end, C, N, seed, float(sigma),
                              float(tone_amp), threads or default_threads())
    return out


# --------------------------------------------------------------------------- numpy mirrors

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
TONE_SALT = 0x746F6E655F706869


def mix64_numpy(x):
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = x + np.uint64(0x9E3779B97F4A7C15)
        x = (x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return x ^ (x >> np.uint64(31))


def _unit_open(h):
    return ((h >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def _hashes(T, C, N, seed, t_begin, t_end):
    key = mix64_numpy(np.uint64(seed))
    t = np.arange(t_begin, t_end, dtype=np.uint64)[:, None, None]
    c = np.arange(C, dtype=np.uint64)[None, :, None]
    i = np.arange(N, dtype=np.uint64)[None, None, :]
    e = (t * np.uint64(C) + c) * np.uint64(N) + i
    h1 = mix64_numpy(key ^ (np.uint64(2) * e))
    h2 = mix64_numpy(key ^ (np.uint64(2) * e + np.uint64(1)))
    return h1, h2


def tone_phase_numpy(C, N, seed):
    """phi[c][i] in [0, 2 pi)."""
    key = mix64_numpy(np.uint64(seed) ^ np.uint64(TONE_SALT))
    idx = np.arange(C * N, dtype=np.uint64).reshape(C, N)
    return 2.0 * np.pi * _unit_open(mix64_numpy(key ^ idx))


def tone_omega(C):
    """w_c in rad/sample."""
    return 2.0 * np.pi * ((np.arange(C) % 16) + 1) / 64.0


def _gauss_numpy(T, C, N, seed, sigma, tone_amp, t_begin, t_end):
    h1, h2 = _hashes(T, C, N, seed, t_begin, t_end)
    r = np.sqrt(-2.0 * np.log(_unit_open(h1)))
    a = 2.0 * np.pi * _unit_open(h2)
    re, im = sigma * (r * np.cos(a)), sigma * (r * np.sin(a))
    if tone_amp != 0.0:
        t = np.arange(t_begin, t_end, dtype=np.float64)[:, None, None]
        ph = tone_omega(C)[None, :, None] * t + tone_phase_numpy(C, N, seed)[None, :, :]
        re = re + tone_amp * np.cos(ph)
        im = im + tone_amp * np.sin(ph)
    return re, im


def gauss_i8_numpy(T, C, N, seed, sigma, clip, tone_amp=0.0, t_begin=0, t_end=None):
    t_end = T if t_end is None else t_end
    re, im = _gauss_numpy(T, C, N, seed, sigma, tone_amp, t_begin, t_end)
    out = np.empty((t_end - t_begin, C, N, 2), dtype=np.int8)
    out[..., 0] = np.clip(np.rint(re), -clip, clip)
    out[..., 1] = np.clip(np.rint(im), -clip, clip)
    return out


def uniform_i8_numpy(T, C, N, seed, clip, t_begin=0, t_end=None):
    t_end = T if t_end is None else t_end
    h1, h2 = _hashes(T, C, N, seed, t_begin, t_end)
    span = np.uint64(2 * clip + 1)
    out = np.empty((t_end - t_begin, C, N, 2), dtype=np.int8)
    out[..., 0] = ((h1 >> np.uint64(32)) % span).astype(np.int64) - clip
    out[..., 1] = ((h2 >> np.uint64(32)) % span).astype(np.int64) - clip
    return out


def gauss_f32_numpy(T, C, N, seed, sigma, tone_amp=0.0, t_begin=0, t_end=None):
    t_end = T if t_end is None else t_end
    re, im = _gauss_numpy(T, C, N, seed, sigma, tone_amp, t_begin, t_end)
    out = np.empty((t_end - t_begin, C, N, 2), dtype=np.float32)
    out[..., 0] = re
    out[..., 1] = im
    return out


def pack_ci4(x):
    """int8 cube [T][C][N][2] with values in [-8, 7] -> uint8 [T][C][N], one byte per complex sample:
    low nibble = Re, high nibble = Im, two's complement (the paper's "1-byte mode").
    Input generation only: no method arithmetic."""
    x = np.asarray(x)
    if x.dtype != np.int8 or x.shape[-1] != 2 or x.min() < -8 or x.max() > 7:
        raise ValueError("pack_ci4 needs int8 [...][2] with values in [-8, 7]")
    u = x.view(np.uint8)
    return ((u[..., 0] & 15) | ((u[..., 1] & 15) << 4)).astype(np.uint8)


# --------------------------------------------------------------------------- workloads

@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config.  dtype: 'ci8' or 'cf32'."""
    name: str
    n_inputs: int
    n_chan: int
    n_time: int
    dtype: str
    seed: int
    kind: str            # 'gauss' | 'uniform'
    sigma: float = 0.0
    clip: int = 0
    tone_amp: float = 0.0
    n_integrations: int = 1

    @property
    def n_baselines(self) -> int:
        return self.n_inputs * (self.n_inputs + 1) // 2

    @property
    def cmacs(self) -> int:
        """Useful complex MACs per integration: T*C*N(N+1)/2."""
        return self.n_time * self.n_chan * self.n_baselines

    @property
    def in_bytes(self) -> int:
        return self.n_time * self.n_chan * self.n_inputs * (2 if self.dtype == "ci8" else 8)

    @property
    def vis_bytes(self) -> int:
        return self.n_chan * self.n_baselines * 8

    def generate(self, integration: int = 0, t_begin: int = 0, t_end=None, out=None, threads=None):
        """Input cube [T][C][N][2] (int8 or float32) for one integration."""
        T, C, N = self.n_time, self.n_chan, self.n_inputs
        # distinct data per integration: fold the integration index into the seed
        seed = self.seed + 1000003 * integration
        if self.dtype == "ci8":
            if self.kind == "uniform":
                return uniform_i8(T, C, N, seed, self.clip, t_begin, t_end, out, threads)
            return gauss_i8(T, C, N, seed, self.sigma, self.clip, self.tone_amp, t_begin, t_end, out, threads)
        return gauss_f32(T, C, N, seed, self.sigma, self.tone_amp, t_begin, t_end, out, threads)


CONFIGS = {
    # BASELINE.json configs[0..4]; sigma for c5 is 1/sqrt(2) per component = CN(0,1)
    "c1": Workload("c1", 32, 128, 1000, "ci8", seed=0, kind="gauss", sigma=3.0, clip=7),
    "c2": Workload("c2", 64, 768, 10000, "ci8", seed=1, kind="gauss", sigma=3.0, clip=7, tone_amp=2.0),
    "c3": Workload("c3", 256, 512, 4000, "ci8", seed=2, kind="uniform", clip=127),
    "c4": Workload("c4", 1024, 128, 1000, "ci8", seed=3, kind="gauss", sigma=16.0, clip=127),
    "c5": Workload("c5", 64, 1536, 500, "cf32", seed=4, kind="gauss", sigma=2.0 ** -0.5, tone_amp=0.5,
                   n_integrations=20),
}


def scaled(w: Workload, **kw) -> Workload:
    """Same recipe, different shape (parity-test sizes)."""
    d = dict(w.__dict__)
    d.update(kw)
    return Workload(**d)
