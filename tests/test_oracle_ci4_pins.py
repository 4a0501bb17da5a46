"""Pins of the 4-bit ("1-byte mode") oracle: P11 hand-written unpack table, P12 closed forms and
agreement with the already pinned int8 oracle on independently unpacked data."""
from __future__ import annotations

import os

import numpy as np

import corrgen
import oracle

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "p11_ci4_unpack.txt")


def test_p11_unpack_table():
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    assert len(rows) == 15
    for hx, re, im in rows:
        assert oracle.unpack_ci4(int(hx, 16)) == (int(re), int(im)), hx
    # every byte value: nibbles are independent, range is [-8, 7], and the map is a bijection
    seen = {oracle.unpack_ci4(b) for b in range(256)}
    assert len(seen) == 256 and all(-8 <= r <= 7 and -8 <= i <= 7 for r, i in seen)
    for b in range(256):
        re, im = oracle.unpack_ci4(b)
        assert (re & 15) == (b & 15) and (im & 15) == (b >> 4)   # two's complement, low nibble = Re


def test_p12_constant_input_closed_form():
    """x_i(t) = x_i constant: V_ij = T x_i conj(x_j) (pin P2 in the packed mode)."""
    T, C, N = 37, 2, 6
    vals = [(7, -8), (-8, 7), (1, 0), (0, -1), (-3, 5), (4, 4)]
    x = np.zeros((T, C, N), np.uint8)
    for i, (re, im) in enumerate(vals):
        x[:, :, i] = (re & 15) | ((im & 15) << 4)
    vis = oracle.xengine_ci4(x)
    b = 0
    for i in range(N):
        for j in range(i + 1):
            z = T * complex(*vals[i]) * complex(*vals[j]).conjugate()
            assert tuple(vis[0, b]) == (int(z.real), int(z.imag)) and tuple(vis[1, b]) == tuple(vis[0, b])
            b += 1


def test_p12_matches_the_int8_oracle_on_unpacked_data():
    """The packed oracle on pack(x) equals the (pinned) int8 oracle on x; the unpacking used here is numpy's
    own sign extension of the two nibbles, written independently of the oracle's C."""
    rng = np.random.default_rng(12)
    x = rng.integers(-8, 8, size=(45, 3, 20, 2), dtype=np.int8)
    p = corrgen.pack_ci4(x)
    lo = (p & 15).astype(np.int16); hi = (p >> 4).astype(np.int16)
    back = np.stack([np.where(lo > 7, lo - 16, lo), np.where(hi > 7, hi - 16, hi)], axis=-1).astype(np.int8)
    assert np.array_equal(back, x)
    assert np.array_equal(oracle.xengine_ci4(p, threads=2), oracle.xengine_ci8(x))
    assert np.array_equal(oracle.xengine_ci4(p, 1, 3), oracle.xengine_ci8(x, 1, 3))


def test_p13_readout_is_the_time_average():
    """sums divided by the update count.  Constant input x_i: the average is x_i conj(x_j) exactly;
    and accumulating two batches equals one long integration (pin P4), so count = T1 + T2."""
    T1, T2, N = 40, 24, 4
    vals = np.array([[3, -2], [1, 1], [-7, 0], [0, 5]], np.int8)
    x = np.broadcast_to(vals, (T1 + T2, 1, N, 2)).copy()
    total = oracle.xengine_ci8(x[:T1]).astype(np.int64) + oracle.xengine_ci8(x[T1:]).astype(np.int64)
    assert np.array_equal(total, oracle.xengine_ci8(x))
    avg = oracle.readout(oracle.xengine_ci8(x), T1 + T2)
    b = 0
    for i in range(N):
        for j in range(i + 1):
            z = complex(*vals[i].tolist()) * complex(*vals[j].tolist()).conjugate()
            assert avg[0, b, 0] == z.real and avg[0, b, 1] == z.imag
            b += 1
    f = oracle.readout(np.array([[[1.5, -3.0]]]), 4)
    assert f[0, 0, 0] == 0.375 and f[0, 0, 1] == -0.75
