"""GPU parity of SURVEY 8(f) row 2: accumulate mode and read-out normalisation
(PAPER.md:84).  Accumulating batches equals one long integration (oracle pin P4), so the expected result
is the oracle on the concatenated input."""
from __future__ import annotations

import numpy as np
import pytest

import corrgen
import oracle
from parity_util import f32_tolerance_check

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.mark.parametrize("dtype,key,N,C,T", [("ci8", "c2", 64, 5, 100), ("ci8", "c1", 32, 6, 70), ("ci8", "c4", 256, 2, 90),
                                             ("ci8", "c4", 512, 2, 64), ("ci4", "c2", 64, 5, 100), ("cf32", "c5", 64, 3, 50)])
def test_accumulate_then_normalize(dtype, key, N, C, T):
    import paper_0906_1887_b200 as pkg
    w = corrgen.scaled(corrgen.CONFIGS[key], n_inputs=N, n_chan=C, n_time=T)
    xs = [w.generate(integration=k) for k in range(3)]
    h = pkg.corr_create(N, C, T, dtype)
    h.set_accumulate(True)
    vis = h.empty_vis()
    vis.zero_()
    for x in xs:
        d_in = torch.from_numpy(corrgen.pack_ci4(x) if dtype == "ci4" else x).cuda()
        pkg.corr_xengine(h, d_in, vis)
    avg = h.normalize(vis, 3 * T)
    torch.cuda.synchronize()
    out, avg = vis.cpu().numpy(), avg.cpu().numpy()
    pkg.corr_destroy(h)
    long_x = np.concatenate(xs, axis=0)
    if dtype == "cf32":
        ref = oracle.xengine_cf32(long_x)
        f32_tolerance_check(out, ref, N)
    else:
        ref = oracle.xengine_ci8(long_x)
        assert np.array_equal(out, ref)
    want = oracle.readout(ref, 3 * T)
    scale = np.maximum(np.abs(want), 1e-30)
    assert np.all(np.abs(avg - want) <= 2e-6 * scale + 1e-6 * np.abs(want).max())


def test_accumulate_off_overwrites_again():
    import paper_0906_1887_b200 as pkg
    w = corrgen.scaled(corrgen.CONFIGS["c2"], n_chan=4, n_time=80)
    x = w.generate()
    h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, "ci8")
    vis = h.empty_vis()
    vis.fill_(12345)
    h.set_accumulate(True)
    h.set_accumulate(False)
    pkg.corr_xengine(h, torch.from_numpy(x).cuda(), vis)
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy(), oracle.xengine_ci8(x))
    pkg.corr_destroy(h)
