"""GPU parity of the 4-bit packed input mode (the paper's "1-byte mode"):
bit-exact against the packed CPU oracle."""
from __future__ import annotations

import numpy as np
import pytest

import corrgen
import oracle

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def run_ci4(x_packed):
    import paper_0906_1887_b200 as pkg
    T, C, N = x_packed.shape
    h = pkg.corr_create(N, C, T, "ci4")
    assert h.in_bytes == T * C * N
    vis = h.empty_vis()
    vis.fill_(-0x55555555)
    pkg.corr_xengine(h, torch.from_numpy(x_packed).cuda(), vis)
    torch.cuda.synchronize()
    out = vis.cpu().numpy()
    pkg.corr_destroy(h)
    return out


SHAPES = [(64, 3, 100), (64, 5, 1), (64, 2, 31), (64, 2, 33), (64, 1, 257), (64, 200, 40), (32, 4, 100), (32, 3, 70),
          (32, 301, 33), (96, 2, 64), (128, 2, 300), (256, 2, 130), (320, 1, 64), (1024, 1, 96),
          # > 64 MB with more panel groups than SMs: the mixed whole / sliced plan (every item reduce-adds in this kernel)
          (64, 1300, 900)]


@pytest.mark.parametrize("N,C,T", SHAPES)
def test_ci4_bit_exact(N, C, T):
    w = corrgen.scaled(corrgen.CONFIGS["c2"], n_inputs=N, n_chan=C, n_time=T)   # clip +-7 fits 4 bits
    p = corrgen.pack_ci4(w.generate())
    assert np.array_equal(run_ci4(p), oracle.xengine_ci4(p, threads=oracle.host_threads()))


def test_ci4_every_byte_value():
    """All 256 byte values appear (including -8 nibbles, which the clipped recipes never produce)."""
    rng = np.random.default_rng(3)
    p = rng.integers(0, 256, size=(200, 3, 64), dtype=np.uint8)
    assert np.array_equal(run_ci4(p), oracle.xengine_ci4(p))


def test_ci4_full_c2_sampled():
    """c2 in 1-byte mode at full size (491 MB of input): sampled channels vs the oracle."""
    w = corrgen.CONFIGS["c2"]
    p = corrgen.pack_ci4(w.generate())
    out = run_ci4(p)
    assert not (out == -0x55555555).any()
    for c in (0, 383, 767):
        assert np.array_equal(out[c:c + 1], oracle.xengine_ci4(p, c, c + 1)), f"channel {c}"
