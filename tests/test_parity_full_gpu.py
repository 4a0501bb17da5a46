"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times: the whole
output is produced by one corr_xengine call; the oracle recomputes sampled channels (all baselines of
each sampled channel: channels are independent) plus sampled single visibilities."""
from __future__ import annotations

import numpy as np
import pytest

import corrgen
import oracle
from parity_util import f32_tolerance_check

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

SAMPLED_CHANNELS = {"c1": None, "c2": [0, 1, 383, 766, 767], "c3": [0, 255, 511], "c4": [0, 127]}


@pytest.mark.parametrize("key", ["c1", "c2", "c3", "c4"])
def test_ci8_full_config_bit_exact(key):
    import paper_0906_1887_b200 as pkg
    w = corrgen.CONFIGS[key]
    x = w.generate()
    h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, "ci8")
    vis = h.empty_vis()
    vis.fill_(-0x55555555)
    pkg.corr_xengine(h, torch.from_numpy(x).cuda(), vis)
    torch.cuda.synchronize()
    out = vis.cpu().numpy()
    pkg.corr_destroy(h)
    threads = oracle.host_threads()
    chans = SAMPLED_CHANNELS[key]
    if chans is None:
        assert np.array_equal(out, oracle.xengine_ci8(x, threads=threads))
    else:
        for c in chans:
            assert np.array_equal(out[c:c + 1], oracle.xengine_ci8(x, c, c + 1, threads=1)), f"channel {c}"
        rng = np.random.default_rng(11)
        for _ in range(64):  # single visibilities anywhere in the cube
            c = int(rng.integers(w.n_chan)); i = int(rng.integers(w.n_inputs)); j = int(rng.integers(i + 1))
            re, im = oracle.one_visibility_ci8(x, c, i, j)
            assert tuple(out[c, i * (i + 1) // 2 + j]) == (re, im), (c, i, j)
    # properties that hold at any size: nothing left unwritten, autos real and non-negative
    assert not (out == -0x55555555).any()
    ii = np.arange(w.n_inputs)
    autos = out[:, ii * (ii + 1) // 2 + ii]
    assert (autos[..., 1] == 0).all() and (autos[..., 0] >= 0).all()


def test_cf32_full_config_within_tolerance():
    """One integration of c5 (N_I=64, 1536 channels, T=500), sampled channels vs the float64 oracle."""
    import paper_0906_1887_b200 as pkg
    w = corrgen.CONFIGS["c5"]
    x = w.generate()
    h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, "cf32")
    vis = h.empty_vis()
    vis.fill_(float("nan"))
    pkg.corr_xengine(h, torch.from_numpy(x).cuda(), vis)
    torch.cuda.synchronize()
    out = vis.cpu().numpy()
    pkg.corr_destroy(h)
    assert not np.isnan(out).any()
    for c in (0, 1, 700, 1535):
        f32_tolerance_check(out[c:c + 1], oracle.xengine_cf32(x, c, c + 1, threads=1), w.n_inputs)
