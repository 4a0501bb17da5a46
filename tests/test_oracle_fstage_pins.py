"""Pins of the F-stage oracle (oracle/fstage_oracle.c: unpack + plain DFT).

The oracle is the O(N^2) definition in float64.  It is pinned by things other than itself:
F1 a library routine (numpy.fft.fft) on random int8 blocks; F2 the closed form of a shifted impulse (pins the
SIGN of the exponent, reading R19); F3 exact integer tones at N = 4 (x[n] = i^(k0 n)); F4 Parseval; F5 layout:
blocks and inputs are independent and stay in place; F6 a hand-worked 4-point example (tests/golden/);
F7 the float64 X-engine restatement used for the F -> X chain against numpy X X^H and the cf32 oracle.
"""
from __future__ import annotations

import os

import numpy as np

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _c(a):
    return a[..., 0] + 1j * a[..., 1]


def _rand(B, N, I, seed, lo=-16, hi=16):
    return np.random.default_rng(seed).integers(lo, hi, size=(B, N, I, 2)).astype(np.int8)


def test_f1_numpy_fft_library_routine():
    for (B, N, I) in [(3, 128, 5), (2, 16, 3), (1, 12, 2), (2, 7, 1)]:   # incl. non-powers of two: it is a DFT
        x = _rand(B, N, I, seed=B * 1000 + N)
        ref = np.fft.fft(_c(x).astype(np.complex128), axis=1)
        got = _c(oracle.fstage_ci8(x))
        assert np.max(np.abs(got - ref)) <= 1e-9 * np.sqrt(N) * 16 * N


def test_f2_shifted_impulse_closed_form_and_sign():
    N = 128
    for n0, amp in [(0, 5 + 0j), (1, 3 - 2j), (37, -7 + 1j)]:
        x = np.zeros((1, N, 1, 2), np.int8)
        x[0, n0, 0] = (int(amp.real), int(amp.imag))
        got = _c(oracle.fstage_ci8(x))[0, :, 0]
        k = np.arange(N)
        want = amp * np.exp(-2j * np.pi * k * n0 / N)
        assert np.max(np.abs(got - want)) < 1e-12 * 16
    # sign of the exponent: a unit impulse at n = 1 gives X_1 = exp(-2 pi i / N), negative imaginary part
    x = np.zeros((1, N, 1, 2), np.int8)
    x[0, 1, 0, 0] = 1
    X1 = _c(oracle.fstage_ci8(x))[0, 1, 0]
    assert X1.imag < 0 and abs(X1 - np.exp(-2j * np.pi / N)) < 1e-15


def test_f3_exact_integer_tones():
    # x[n] = i^(k0 n) is the tone exp(+2 pi i k0 n / 4) in exact integers: X[k0] = 4, all other channels 0
    pw = [(1, 0), (0, 1), (-1, 0), (0, -1)]
    for k0 in range(4):
        x = np.zeros((1, 4, 1, 2), np.int8)
        for n in range(4):
            x[0, n, 0] = pw[(k0 * n) % 4]
        got = _c(oracle.fstage_ci8(x))[0, :, 0]
        want = np.zeros(4, complex)
        want[k0] = 4
        assert np.max(np.abs(got - want)) < 1e-14


def test_f4_parseval():
    x = _rand(4, 128, 6, seed=7)
    X = _c(oracle.fstage_ci8(x))
    e_t = np.sum(np.abs(_c(x).astype(np.complex128)) ** 2, axis=1)
    e_f = np.sum(np.abs(X) ** 2, axis=1)
    assert np.allclose(e_f, 128 * e_t, rtol=1e-12)


def test_f5_blocks_and_inputs_independent_and_in_place():
    x = _rand(5, 32, 4, seed=11)
    X = oracle.fstage_ci8(x)
    pb, pi = np.array([3, 0, 4, 1, 2]), np.array([2, 3, 0, 1])
    Xp = oracle.fstage_ci8(np.ascontiguousarray(x[pb][:, :, pi]))
    assert np.array_equal(Xp, X[pb][:, :, pi])
    # threads only spread blocks: same numbers
    assert np.array_equal(oracle.fstage_ci8(x, threads=3), X)
    # linearity in exact integers: F(x + y) = F(x) + F(y) up to float64 rounding
    y = _rand(5, 32, 4, seed=12)
    s = (x.astype(np.int16) + y).astype(np.int8)
    assert np.allclose(oracle.fstage_ci8(s), X + oracle.fstage_ci8(y), atol=1e-10)


def test_f6_golden_worked_example():
    sec, rows = None, {"input": [], "output": []}
    for line in open(os.path.join(GOLDEN, "f6_dft_worked_example.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("["):
            sec = line[1:].split()[0]
            continue
        rows[sec].append([int(v) for v in line.split()])
    x = np.zeros((1, 4, 1, 2), np.int8)
    for n, re, im in rows["input"]:
        x[0, n, 0] = (re, im)
    got = oracle.fstage_ci8(x)[0, :, 0]
    want = np.array([[re, im] for _, re, im in rows["output"]], dtype=np.float64)
    assert np.max(np.abs(got - want)) < 1e-14


def test_f7_float64_xengine_restatement():
    rng = np.random.default_rng(5)
    x = rng.standard_normal((9, 3, 6, 2))
    vis = _c(oracle.xengine_cf64(x, threads=2))
    ii, jj = np.tril_indices(6)
    for c in range(3):
        X = _c(x[:, c]).T                      # [N][T]
        full = X @ X.conj().T                  # textbook Hermitian rank-T update
        assert np.allclose(vis[c], full[ii, jj], rtol=1e-13, atol=1e-13)
    # same numbers as the cf32 oracle when the input is representable in float32
    x32 = x.astype(np.float32)
    assert np.array_equal(oracle.xengine_cf64(x32.astype(np.float64)), oracle.xengine_cf32(x32))


def test_f8_one_byte_mode_matches_int8_routine_and_byte_table():
    """The packed (4+4-bit) F-stage oracle against (a) the int8 routine on data unpacked by numpy with the hand-written
    table of tests/golden/p11_ci4_unpack.txt semantics (low nibble Re, high nibble Im, two's complement) and (b) numpy.fft."""
    rng = np.random.default_rng(3)
    xb = rng.integers(0, 256, size=(3, 16, 5), dtype=np.uint8)          # every byte value can occur
    lo, hi = (xb & 15).astype(np.int16), (xb >> 4).astype(np.int16)
    re = np.where(lo >= 8, lo - 16, lo).astype(np.int8)
    im = np.where(hi >= 8, hi - 16, hi).astype(np.int8)
    x8 = np.stack([re, im], axis=-1)
    got = oracle.fstage_ci4(xb, threads=2)
    assert np.array_equal(got, oracle.fstage_ci8(x8))
    assert np.max(np.abs(_c(got) - np.fft.fft(_c(x8).astype(np.complex128), axis=1))) < 1e-11
    # single bytes: 0x7F = 7 - 1i... written out: low nibble F = -1 (Re), high nibble 7 = +7 (Im)
    one = np.zeros((1, 4, 1), np.uint8)
    one[0, 0, 0] = 0x7F
    X = _c(oracle.fstage_ci4(one))[0, :, 0]
    assert np.allclose(X, (-1 + 7j) * np.ones(4))
