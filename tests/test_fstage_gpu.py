"""GPU parity of the F-stage (corr_fstage_*) against the float64 DFT oracle, and of the
F -> X chain (raw voltages -> spectra -> visibilities) against the same chain in float64.

Tolerance: |X_gpu - X_ref| <= 1e-5 * ||x[b][:][i]||_2 per channel -- an FP32 transform of
length 128 has a worst-case error of ~ log2(128) * 2^-24 * sqrt(128) * ||x||_2 = 4.7e-6 ||x||_2, typically 3e-7.
Raw voltages: seeded 5-bit Gaussian samples, the recipe of DESIGN.md section 4.
"""
from __future__ import annotations

import numpy as np
import pytest

import corrgen
import oracle
from parity_util import f32_tolerance_check

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pkg():
    import paper_0906_1887_b200 as p
    p.lib()
    return p


def raw_voltages(B, I, seed, tone=None):
    """[B][128][I][2] int8: clip(rint(4 g), -16, 15), optionally plus a tone exp(2 pi i k0 n / 128) of amplitude 6."""
    x = corrgen.gauss_i8(B, 128, I, seed, 4.0, 15.0).astype(np.float64)
    if tone is not None:
        n = np.arange(128)[None, :, None]
        ph = 2 * np.pi * tone * n / 128 + 0.3 * np.arange(I)[None, None, :]
        x[..., 0] += 6 * np.cos(ph)
        x[..., 1] += 6 * np.sin(ph)
    return np.clip(np.rint(x), -16, 15).astype(np.int8)


def check_spectra(got, x):
    ref = oracle.fstage_ci8(x, threads=oracle.host_threads())
    norm = np.sqrt(np.sum(x.astype(np.float64) ** 2, axis=(1, 3)))[:, None, :]      # ||x[b][:][i]||_2
    err = np.hypot(got[..., 0] - ref[..., 0], got[..., 1] - ref[..., 1])
    zero = norm == 0
    assert np.all(err[np.broadcast_to(zero, err.shape)] == 0)
    worst = float(np.max(np.where(zero, 0.0, err / np.where(zero, 1.0, norm))))
    assert worst <= 1e-5, f"F-stage out of tolerance: {worst:.3e}"
    return worst


@pytest.mark.parametrize("B,I", [(1, 32), (3, 64), (7, 96), (40, 64), (2, 256)])
def test_fstage_matches_dft_oracle(pkg, B, I):
    x = raw_voltages(B, I, seed=100 + B, tone=5 if B % 2 else None)
    f = pkg.corr_fstage_create(I, 128, B)
    spec = torch.full((B, 128, I, 2), float("nan"), dtype=torch.float32, device="cuda")  # poison
    pkg.corr_fstage_run(f, torch.from_numpy(x).cuda(), spec)
    torch.cuda.synchronize()
    worst = check_spectra(spec.cpu().numpy().astype(np.float64), x)
    assert worst < 2e-6       # typical FP32 error is far below the tolerance
    pkg.corr_fstage_destroy(f)


def test_fstage_special_inputs(pkg):
    I, B = 32, 3
    x = np.zeros((B, 128, I, 2), np.int8)
    x[0, 0, :, 0] = 7                       # impulse at n = 0 -> flat spectrum 7 + 0i, exactly
    x[1, :, :, 0] = -16                     # constant -> 128 * (-16) in channel 0, zero elsewhere
    x[2, 1, 3] = (1, 0)                     # impulse at n = 1 on input 3 -> exp(-2 pi i k / 128)
    f = pkg.corr_fstage_create(I, 128, B)
    spec = pkg.corr_fstage_run(f, torch.from_numpy(x).cuda()).cpu().numpy()
    assert np.all(spec[0, :, :, 0] == 7) and np.all(spec[0, :, :, 1] == 0)
    assert np.all(spec[1, 0, :, 0] == -2048) and np.all(spec[1, 1:] == 0) and np.all(spec[1, 0, :, 1] == 0)
    k = np.arange(128)
    assert np.max(np.abs(spec[2, :, 3, 0] - np.cos(2 * np.pi * k / 128))) < 3e-7
    assert np.max(np.abs(spec[2, :, 3, 1] + np.sin(2 * np.pi * k / 128))) < 3e-7   # forward sign (R19)
    assert np.all(spec[2, :, 4] == 0)
    check_spectra(spec.astype(np.float64), x)
    pkg.corr_fstage_destroy(f)


def test_fx_chain_matches_float64_chain(pkg):
    """raw [T][bands][128][I] -> F -> [T][bands * 128][I] -> X (cf32) vs oracle DFT -> oracle X in float64."""
    T, bands, I = 24, 2, 64
    x = raw_voltages(T * bands, I, seed=9, tone=17)
    f = pkg.corr_fstage_create(I, 128, T * bands)
    spec = pkg.corr_fstage_run(f, torch.from_numpy(x).cuda())
    h = pkg.corr_create(I, bands * 128, T, "cf32")
    vis = pkg.corr_xengine(h, spec.view(T, bands * 128, I, 2)).cpu().numpy()
    ref_spec = oracle.fstage_ci8(x, threads=oracle.host_threads()).reshape(T, bands * 128, I, 2)
    ref = oracle.xengine_cf64(ref_spec, threads=oracle.host_threads())
    # the chain's error is the X-engine's (1e-5 scale) plus the F-stage's relative 3e-7 twice: same tolerance x2
    f32_tolerance_check(vis, ref, I, rel=2e-5)
    pkg.corr_destroy(h)
    pkg.corr_fstage_destroy(f)


def test_fstage_full_size_sampled(pkg):
    """The batch bench.py times (one c5 integration: 500 spectra x 12 bands x 64 inputs); sampled blocks."""
    B, I = 6000, 64
    x = raw_voltages(B, I, seed=4)
    f = pkg.corr_fstage_create(I, 128, B)
    spec = pkg.corr_fstage_run(f, torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    pick = np.array([0, 1, 147, 148, 2999, 5998, 5999])
    check_spectra(spec[pick].cpu().numpy().astype(np.float64), x[pick])
    # Parseval on every block (holds at any size): sum_k |X|^2 = 128 sum_n |x|^2
    e_f = (spec.double() ** 2).sum(dim=(1, 3)).cpu().numpy()
    e_t = 128.0 * (x.astype(np.float64) ** 2).sum(axis=(1, 3))
    assert np.allclose(e_f, e_t, rtol=2e-6)
    pkg.corr_fstage_destroy(f)


def test_stream_run_fx_matches_float64_chain(pkg):
    """corr_stream_run_fx: pinned raw voltages -> H2D (double-buffered) -> F -> X, three integrations."""
    T, bands, I, n_int = 10, 1, 32, 3
    raws = [raw_voltages(T * bands, I, seed=20 + k, tone=3 + k) for k in range(n_int)]
    f = pkg.corr_fstage_create(I, 128, T * bands)
    h = pkg.corr_create(I, bands * 128, T, "cf32")
    pinned = [torch.from_numpy(r).pin_memory() for r in raws]
    d_vis, stats = h.stream_run(pinned, fstage=f)
    torch.cuda.synchronize()
    assert stats["device_s"] > 0 and stats["kernel_s"] > 0
    out = d_vis.cpu().numpy()
    for k in range(n_int):
        ref_spec = oracle.fstage_ci8(raws[k], threads=oracle.host_threads()).reshape(T, bands * 128, I, 2)
        f32_tolerance_check(out[k], oracle.xengine_cf64(ref_spec, threads=oracle.host_threads()), I, rel=2e-5)
    # a handle of another shape is refused
    h2 = pkg.corr_create(I, 128, T + 1, "cf32")
    with pytest.raises(pkg.CorrError):
        h2.stream_run([torch.from_numpy(raws[0]).pin_memory()], fstage=f)
    pkg.corr_destroy(h2)
    pkg.corr_destroy(h)
    pkg.corr_fstage_destroy(f)


def raw_voltages_4bit(B, I, seed):
    """4+4-bit samples: clip(rint(2.5 g), -8, 7), as int8 pairs and packed one byte per sample."""
    x = corrgen.gauss_i8(B, 128, I, seed, 2.5, 7.0)
    x[0, :3, 0] = [(-8, 7), (7, -8), (-1, -1)]          # the corners of the 4-bit range
    x = np.clip(x, -8, 7).astype(np.int8)
    return x, corrgen.pack_ci4(x)


@pytest.mark.parametrize("B,I", [(2, 32), (9, 64), (33, 96)])
def test_fstage_one_byte_mode(pkg, B, I):
    """corr_fstage_set_input(CORR_CI4): packed raw voltages give the spectra of the oracle's packed routine -- and
    bit-identical spectra to the int8 mode on the same samples (the unpack is exact in both)."""
    x8, xb = raw_voltages_4bit(B, I, seed=60 + B)
    f = pkg.corr_fstage_create(I, 128, B)
    s8 = pkg.corr_fstage_run(f, torch.from_numpy(x8).cuda()).cpu().numpy()
    f.set_input("ci4")
    assert f.in_bytes == B * 128 * I
    spec = torch.full((B, 128, I, 2), float("nan"), dtype=torch.float32, device="cuda")
    pkg.corr_fstage_run(f, torch.from_numpy(xb).cuda(), spec)
    s4 = spec.cpu().numpy()
    assert np.array_equal(s4, s8)
    ref = oracle.fstage_ci4(xb, threads=oracle.host_threads())
    norm = np.sqrt(np.sum(x8.astype(np.float64) ** 2, axis=(1, 3)))[:, None, :]
    err = np.hypot(s4[..., 0] - ref[..., 0], s4[..., 1] - ref[..., 1])
    assert np.max(err / norm) <= 1e-5
    with pytest.raises(ValueError):
        pkg.corr_fstage_run(f, torch.from_numpy(x8).cuda())       # wrong size for the packed mode
    pkg.corr_fstage_destroy(f)


def test_stream_run_fx_one_byte_mode(pkg):
    T, I, n_int = 12, 64, 2
    pairs = [raw_voltages_4bit(T, I, seed=80 + k) for k in range(n_int)]
    f = pkg.corr_fstage_create(I, 128, T)
    f.set_input("ci4")
    h = pkg.corr_create(I, 128, T, "cf32")
    d_vis, _ = h.stream_run([torch.from_numpy(xb).pin_memory() for _, xb in pairs], fstage=f)
    out = d_vis.cpu().numpy()
    for k, (_, xb) in enumerate(pairs):
        ref_spec = oracle.fstage_ci4(xb, threads=oracle.host_threads())
        f32_tolerance_check(out[k], oracle.xengine_cf64(ref_spec, threads=oracle.host_threads()), I, rel=2e-5)
    pkg.corr_destroy(h)
    pkg.corr_fstage_destroy(f)
