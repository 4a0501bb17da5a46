"""Pins for the CPU oracle (CPU only).  Each pin checks the oracle against
something other than itself: a hand-worked fixture, a closed form, an invariant
of the definition, a brute-force pure-Python restatement, or numpy's Hermitian
product.  SURVEY.md 8(c) P1-P9; the paper passages are cited per test.
"""
import os

import numpy as np
import pytest

import corrgen
import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def tri_index(i, j):
    """Row-major lower-triangle index, re-derived here (reading R2), not imported."""
    assert i >= j
    return i * (i + 1) // 2 + j


def rand_ci8(T, C, N, seed, lo=-128, hi=127):
    rng = np.random.default_rng(seed)
    return rng.integers(lo, hi + 1, size=(T, C, N, 2), dtype=np.int8)


def rand_cf32(T, C, N, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((T, C, N, 2)).astype(np.float32)


def as_complex(x):
    return x[..., 0].astype(np.float64) + 1j * x[..., 1].astype(np.float64)


# ----------------------------------------------------------------------------- golden

def _read_sections(path):
    sections, cur = {}, None
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("["):
            cur = sections.setdefault(line.split()[0].strip("[]"), [])
            continue
        cur.append([int(v) for v in line.split()])
    return sections


def test_p5_hand_worked_example():
    """PAPER.md:53, :107 + readings R1/R2; fixture worked by hand."""
    s = _read_sections(os.path.join(GOLDEN, "p5_worked_example.txt"))
    x = np.zeros((2, 1, 2, 2), dtype=np.int8)
    for t, c, i, re, im in s["input"]:
        x[t, c, i] = (re, im)
    vis = oracle.xengine_ci8(x)
    for c, b, re, im in s["visibility"]:
        assert tuple(vis[c, b]) == (re, im)
    # float path on the same numbers
    visf = oracle.xengine_cf32(x.astype(np.float32))
    for c, b, re, im in s["visibility"]:
        assert tuple(visf[c, b]) == (float(re), float(im))


def test_product_counts():
    """N_I(N_I+1)/2 products including autos."""
    for line in open(os.path.join(GOLDEN, "counts.txt")):
        if line.startswith("#") or not line.strip():
            continue
        n, nb = map(int, line.split())
        if n > 64:
            assert corrgen.CONFIGS["c3" if n == 256 else "c4"].n_baselines == nb
            continue
        vis = oracle.xengine_ci8(np.ones((1, 1, n, 2), dtype=np.int8))
        assert vis.shape == (1, nb, 2)


def test_conjugation_side_and_sign():
    """Reading R1: x_i = i, x_j = 1 (i > j) gives V_ij = +i; swapped gives -i."""
    x = np.zeros((1, 1, 2, 2), dtype=np.int8)
    x[0, 0, 1] = (0, 1)   # higher index: imaginary unit
    x[0, 0, 0] = (1, 0)
    assert tuple(oracle.xengine_ci8(x)[0, tri_index(1, 0)]) == (0, 1)
    x[0, 0, 1] = (1, 0)
    x[0, 0, 0] = (0, 1)
    assert tuple(oracle.xengine_ci8(x)[0, tri_index(1, 0)]) == (0, -1)


# ----------------------------------------------------------------------------- P1

@pytest.mark.parametrize("N", [1, 2, 5, 32])
def test_p1_full_matrix_vs_packed(N):
    """Fig. 2: autos on the diagonal, redundant halves; PAPER.md:47 count."""
    T, C = 9, 3
    x = rand_ci8(T, C, N, seed=N)
    vis = oracle.xengine_ci8(x)
    assert vis.shape == (C, N * (N + 1) // 2, 2)
    for c in range(C):
        full = oracle.full_matrix_ci8(x, c)
        # Hermitian: V_ji = conj(V_ij); autos real and non-negative
        assert np.array_equal(full[..., 0], full[..., 0].T)
        assert np.array_equal(full[..., 1], -full[..., 1].T)
        assert np.all(np.diagonal(full[..., 1]) == 0)
        assert np.all(np.diagonal(full[..., 0]) >= 0)
        seen = 0
        for i in range(N):
            for j in range(i + 1):
                assert tuple(vis[c, tri_index(i, j)]) == tuple(full[i, j])
                seen += 1
        assert seen == vis.shape[1]


def test_p1_full_matrix_float():
    T, C, N = 17, 2, 6
    x = rand_cf32(T, C, N, seed=3)
    vis = oracle.xengine_cf32(x)
    for c in range(C):
        full = oracle.full_matrix_cf32(x, c)
        for i in range(N):
            assert full[i, i, 1] == 0.0 and full[i, i, 0] >= 0.0
            for j in range(i + 1):
                np.testing.assert_allclose(vis[c, tri_index(i, j)], full[i, j], rtol=0, atol=1e-12)
                np.testing.assert_allclose(full[j, i], full[i, j] * [1, -1], rtol=0, atol=1e-12)
    # autos: imaginary part exactly zero (needs -ffp-contract=off)
    for i in range(N):
        assert np.all(vis[:, tri_index(i, i), 1] == 0.0)


# ----------------------------------------------------------------------------- P2

def test_p2_constant_input_closed_form():
    """x_i(t) = x_i  =>  V_ij = T x_i conj(x_j)."""
    T, C, N = 37, 2, 7
    x0 = rand_ci8(1, C, N, seed=5, lo=-11, hi=11)
    x = np.repeat(x0, T, axis=0)
    vis = oracle.xengine_ci8(x)
    z = as_complex(x0[0])
    for c in range(C):
        for i in range(N):
            for j in range(i + 1):
                want = T * z[c, i] * np.conj(z[c, j])
                assert tuple(vis[c, tri_index(i, j)]) == (int(want.real), int(want.imag))
    visf = oracle.xengine_cf32(x.astype(np.float32))
    np.testing.assert_array_equal(visf, vis.astype(np.float64))


def test_max_magnitude_constant():
    """All samples -128-128i: V_ij = T * 2 * 128^2 real; T = 65535 still fits int32."""
    T = 65535
    x = np.full((T, 1, 2, 2), -128, dtype=np.int8)
    vis = oracle.xengine_ci8(x)
    assert np.all(vis[0, :, 0] == T * 2 * 128 * 128) and np.all(vis[0, :, 1] == 0)
    assert T * 2 * 128 * 128 < 2 ** 31
    with pytest.raises(oracle.OracleOverflow):
        oracle.xengine_ci8(np.full((65536, 1, 1, 2), -128, dtype=np.int8))


# ----------------------------------------------------------------------------- P3

def test_p3_single_nonzero_input():
    T, C, N, k = 21, 2, 6, 3
    x = np.zeros((T, C, N, 2), dtype=np.int8)
    x[:, :, k] = rand_ci8(T, C, 1, seed=8)[:, :, 0]
    vis = oracle.xengine_ci8(x)
    power = (x[:, :, k].astype(np.int64) ** 2).sum(axis=(0, 2))
    for c in range(C):
        for i in range(N):
            for j in range(i + 1):
                want = (power[c], 0) if (i == k and j == k) else (0, 0)
                assert tuple(vis[c, tri_index(i, j)]) == want


# ----------------------------------------------------------------------------- P4

def test_p4_linearity_over_split_integrations():
    """Accumulation is a plain sum over time."""
    T1, T2, C, N = 13, 29, 3, 8
    x = rand_ci8(T1 + T2, C, N, seed=11)
    whole = oracle.xengine_ci8(x).astype(np.int64)
    parts = oracle.xengine_ci8(x[:T1]).astype(np.int64) + oracle.xengine_ci8(x[T1:]).astype(np.int64)
    assert np.array_equal(whole, parts)
    xf = rand_cf32(T1 + T2, C, N, seed=12)
    np.testing.assert_allclose(oracle.xengine_cf32(xf),
                               oracle.xengine_cf32(xf[:T1]) + oracle.xengine_cf32(xf[T1:]),
                               rtol=0, atol=1e-10)


# ----------------------------------------------------------------------------- P6

def test_p6_orthogonal_sequences():
    """x_i(t) = i^(k_i t mod 4): V_ij = T if k_i == k_j (mod 4) else 0.
    Catches Re/Im cross-term sign errors that a constant input cannot."""
    T, N = 16, 8
    units = [(1, 0), (0, 1), (-1, 0), (0, -1)]
    ks = [0, 1, 2, 3, 1, 3, 0, 2]
    x = np.zeros((T, 1, N, 2), dtype=np.int8)
    for t in range(T):
        for i, k in enumerate(ks):
            x[t, 0, i] = units[(k * t) % 4]
    vis = oracle.xengine_ci8(x)
    for i in range(N):
        for j in range(i + 1):
            want = (T, 0) if ks[i] % 4 == ks[j] % 4 else (0, 0)
            assert tuple(vis[0, tri_index(i, j)]) == want


# ----------------------------------------------------------------------------- P7

@pytest.mark.parametrize("T,C,N", [(1, 1, 1), (33, 2, 9), (64, 3, 32)])
def test_p7_hermitian_rank_k_update(T, C, N):
    """Per channel V = X X^H with X the N x T sample matrix (textbook restatement
    of PAPER.md:107); lower triangle extracted here, not in the oracle."""
    x = rand_ci8(T, C, N, seed=T + N)
    vis = oracle.xengine_ci8(x)
    xr, xi = x[..., 0].astype(np.int64), x[..., 1].astype(np.int64)
    il, jl = np.tril_indices(N)      # row-major lower triangle order
    for c in range(C):
        Xr, Xi = xr[:, c, :].T, xi[:, c, :].T          # [N][T]
        re = Xr @ Xr.T + Xi @ Xi.T
        im = Xi @ Xr.T - Xr @ Xi.T
        assert np.array_equal(vis[c, :, 0], re[il, jl])
        assert np.array_equal(vis[c, :, 1], im[il, jl])
    xf = rand_cf32(T, C, N, seed=T)
    visf = oracle.xengine_cf32(xf)
    z = as_complex(xf)
    for c in range(C):
        X = z[:, c, :].T
        V = X @ X.conj().T
        np.testing.assert_allclose(visf[c, :, 0], V.real[il, jl], rtol=1e-12, atol=1e-12)
        np.testing.assert_allclose(visf[c, :, 1], V.imag[il, jl], rtol=1e-12, atol=1e-12)


def test_brute_force_pure_python():
    """Tiny case with python ints and python complex arithmetic, term by term."""
    T, C, N = 5, 2, 4
    x = rand_ci8(T, C, N, seed=21)
    vis = oracle.xengine_ci8(x)
    for c in range(C):
        b = 0
        for i in range(N):
            for j in range(i + 1):
                acc = 0j
                for t in range(T):
                    xi = complex(int(x[t, c, i, 0]), int(x[t, c, i, 1]))
                    xj = complex(int(x[t, c, j, 0]), int(x[t, c, j, 1]))
                    acc += xi * xj.conjugate()
                assert (int(acc.real), int(acc.imag)) == tuple(vis[c, b])
                b += 1


# ----------------------------------------------------------------------------- P8

def test_p8_channel_independence():
    """'The products are formed independently for each frequency channel'."""
    T, C, N = 11, 6, 5
    x = rand_ci8(T, C, N, seed=31)
    perm = np.array([3, 0, 5, 1, 4, 2])
    assert np.array_equal(oracle.xengine_ci8(x[:, perm]), oracle.xengine_ci8(x)[perm])
    # channel sub-range == slice of the whole
    assert np.array_equal(oracle.xengine_ci8(x, 2, 5), oracle.xengine_ci8(x)[2:5])
    # OpenMP over channels changes nothing
    assert np.array_equal(oracle.xengine_ci8(x, threads=4), oracle.xengine_ci8(x))
    xf = rand_cf32(T, C, N, seed=32)
    assert np.array_equal(oracle.xengine_cf32(xf, threads=4), oracle.xengine_cf32(xf))


# ----------------------------------------------------------------------------- P9

def test_p9_phase_rotation_covariance():
    """Multiply input k by the imaginary unit ((a,b)->(-b,a), exact): V_kj -> i V_kj (j<k),
    V_ik -> -i V_ik (i>k), everything else unchanged."""
    T, C, N, k = 19, 2, 6, 2
    x = rand_ci8(T, C, N, seed=41, lo=-100, hi=100)
    y = x.copy()
    y[:, :, k, 0] = -x[:, :, k, 1]
    y[:, :, k, 1] = x[:, :, k, 0]
    v, w = oracle.xengine_ci8(x), oracle.xengine_ci8(y)
    for i in range(N):
        for j in range(i + 1):
            re, im = v[:, tri_index(i, j), 0], v[:, tri_index(i, j), 1]
            got = w[:, tri_index(i, j)]
            if i == k and j < k:       # i * (re + i im) = -im + i re
                want = np.stack([-im, re], axis=-1)
            elif j == k and i > k:     # -i * (re + i im) = im - i re
                want = np.stack([im, -re], axis=-1)
            else:
                want = np.stack([re, im], axis=-1)
            assert np.array_equal(got, want)


# ----------------------------------------------------------------------------- sampled routine

def test_one_visibility_matches_packed():
    T, C, N = 23, 3, 7
    x = rand_ci8(T, C, N, seed=51)
    vis = oracle.xengine_ci8(x)
    xf = rand_cf32(T, C, N, seed=52)
    visf = oracle.xengine_cf32(xf)
    for c in range(C):
        for i in range(N):
            for j in range(i + 1):
                assert oracle.one_visibility_ci8(x, c, i, j) == tuple(vis[c, tri_index(i, j)])
                assert oracle.one_visibility_cf32(xf, c, i, j) == tuple(visf[c, tri_index(i, j)])


# ----------------------------------------------------------------------------- P10 (statistical)

def test_p10_tone_phase_statistics():
    """Common tone: arg V_ij ~ phi_i - phi_j (generator sanity, statistical)."""
    w = corrgen.scaled(corrgen.CONFIGS["c2"], n_chan=2, n_time=4096, n_inputs=4)
    x = w.generate()
    vis = oracle.xengine_ci8(x)
    phi = corrgen.tone_phase_numpy(w.n_chan, w.n_inputs, w.seed)
    for c in range(w.n_chan):
        for i in range(w.n_inputs):
            for j in range(i):
                v = complex(*vis[c, tri_index(i, j)])
                d = np.angle(v * np.exp(-1j * (phi[c, i] - phi[c, j])))
                assert abs(d) < 0.15


# ----------------------------------------------------------------------------- P14: int64 accumulation
# (PAPER.md:84 "after a specified time, usually a few seconds"; :125, :166: batches are ADDED to the accumulators)

def test_p14_wide_closed_form_beyond_int32():
    """Constant full-scale input for T = 70000 samples: V_ij = T x_i conj(x_j) = 70000 * 2 * 127^2 = 2.26e9 > 2^31 - 1.
    The int32 routine must refuse it, the int64 routine must give the closed form exactly."""
    T = 70000
    x = np.empty((T, 1, 2, 2), np.int8)
    x[:, 0, 0] = (127, -127)
    x[:, 0, 1] = (-128, 127)
    with pytest.raises(oracle.OracleOverflow):
        oracle.xengine_ci8(x)
    v = oracle.xengine_ci8_wide(x)
    assert v.dtype == np.int64
    z = [127 - 127j, -128 + 127j]
    want = {(0, 0): T * z[0] * np.conj(z[0]), (1, 0): T * z[1] * np.conj(z[0]), (1, 1): T * z[1] * np.conj(z[1])}
    for (i, j), w in want.items():
        assert v[0, tri_index(i, j), 0] == int(round(w.real)) and v[0, tri_index(i, j), 1] == int(round(w.imag)), (i, j)
    assert v[0, tri_index(0, 0), 0] > 2**31 - 1


def test_p14_wide_equals_int32_routine_and_sums_of_batches():
    """Where the sums fit, the int64 routine equals the (pinned) int32 routine; and it is the sum of the batches'
    int32 results -- what an accumulating correlator adds up (linearity, P4)."""
    x = rand_ci8(90, 3, 6, 21)
    wide = oracle.xengine_ci8_wide(x, threads=2)
    assert np.array_equal(wide, oracle.xengine_ci8(x).astype(np.int64))
    parts = sum(oracle.xengine_ci8(x[a:b]).astype(np.int64) for a, b in ((0, 17), (17, 60), (60, 90)))
    assert np.array_equal(wide, parts)
    sub = oracle.xengine_ci8_wide(x, 1, 3)
    assert np.array_equal(sub, wide[1:3])


def test_p14_wide_against_numpy_hermitian_product():
    x = rand_ci8(40, 2, 5, 22)
    wide = oracle.xengine_ci8_wide(x)
    z = as_complex(x)
    for c in range(2):
        X = z[:, c, :].T                                   # [N][T]
        V = X @ X.conj().T
        for i in range(5):
            for j in range(i + 1):
                assert wide[c, tri_index(i, j), 0] == int(round(V[i, j].real))
                assert wide[c, tri_index(i, j), 1] == int(round(V[i, j].imag))


def test_p14_readout_of_int64_sums():
    v = np.array([[[2**40 + 4, -(2**35)]]], dtype=np.int64)
    out = oracle.readout(v, 4)
    assert out[0, 0, 0] == 2.0**38 + 1.0 and out[0, 0, 1] == -(2.0**33)
