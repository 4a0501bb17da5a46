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


def oracle_unpacked(packed):
    """uint8 [T][C][N] packed 4+4-bit samples -> int8 [T][C][N][2] through the oracle's own unpack table (pin P11)."""
    table = np.array([oracle.unpack_ci4(b) for b in range(256)], dtype=np.int8)
    return table[packed]


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


def test_accumulate_refuses_the_batch_that_could_overflow_int32():
    """Full-scale constant batches up to the bound stay bit-exact; the next batch is refused with CORR_EUNSUPPORTED and
    adds nothing (reading R6: exact iff count * T * 2 * 128^2 < 2^31).  T = 16384: 2^31 / (T * 2^15) = 4 batches
    would reach 2^31 exactly, so 3 are admitted."""
    import paper_0906_1887_b200 as pkg
    N, C, T = 32, 2, 16384
    x = np.full((T, C, N, 2), -128, np.int8)
    x[:, :, 1::2, 1] = 127
    h = pkg.corr_create(N, C, T, "ci8")
    h.set_accumulate(True)
    vis = h.empty_vis().zero_()
    d_in = torch.from_numpy(x).cuda()
    admitted = 0
    for k in range(6):
        try:
            pkg.corr_xengine(h, d_in, vis)
            admitted += 1
        except pkg.CorrError as e:
            assert e.status == pkg.CORR_EUNSUPPORTED and "overflow" in str(e)
    torch.cuda.synchronize()
    assert admitted == 3 and h.accumulate_count == 3
    want = 3 * oracle.xengine_ci8_wide(x)
    assert np.abs(want).max() < 2**31 and want.max() == 3 * T * 2 * 128 * 128
    assert np.array_equal(vis.cpu().numpy().astype(np.int64), want)
    # a new accumulation starts with corr_set_accumulate: the counter is reset
    h.set_accumulate(True)
    assert h.accumulate_count == 0
    vis.zero_()
    pkg.corr_xengine(h, d_in, vis)
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy().astype(np.int64), oracle.xengine_ci8_wide(x))
    pkg.corr_destroy(h)


@pytest.mark.parametrize("dtype,N,C,T,batches", [("ci8", 32, 2, 16384, 9), ("ci8", 256, 1, 300, 3), ("ci4", 64, 3, 200, 4)])
def test_accumulate_wide_is_exact_beyond_int32(dtype, N, C, T, batches):
    """corr_accumulate_wide: int64 accumulators, any number of batches.  9 full-scale batches of T = 16384 sum to
    9 * 2^29 > 2^31: exact against the int64 oracle on the concatenated input; read-out against the oracle's."""
    import paper_0906_1887_b200 as pkg
    if T == 16384:
        xs = []
        for k in range(batches):
            x = np.full((T, C, N, 2), 127 if k % 2 else -128, np.int8)
            x[:, :, k % N, 0] = 5 * k
            xs.append(x)
    else:
        w = corrgen.scaled(corrgen.CONFIGS["c3" if dtype == "ci8" else "c2"], n_inputs=N, n_chan=C, n_time=T)
        xs = [w.generate(integration=k) for k in range(batches)]
    h = pkg.corr_create(N, C, T, dtype)
    acc = h.empty_acc()
    for x in xs:
        h.accumulate_wide(torch.from_numpy(corrgen.pack_ci4(x) if dtype == "ci4" else x).cuda(), acc)
    avg = h.normalize_wide(acc, batches * T)
    torch.cuda.synchronize()
    got = acc.cpu().numpy()
    long_x = np.concatenate(xs, axis=0)
    if dtype == "ci4":
        # the 4-bit mode keeps bits 0..3 of each component: the int8 samples the packed bytes stand for
        long_x = np.ascontiguousarray(oracle_unpacked(corrgen.pack_ci4(long_x)))
    want = oracle.xengine_ci8_wide(long_x, threads=oracle.host_threads())
    assert got.dtype == np.int64 and np.array_equal(got, want)
    if T == 16384:
        assert np.abs(want).max() > 2**31
    ref_avg = oracle.readout(want, batches * T)
    assert np.all(np.abs(avg.cpu().numpy() - ref_avg) <= 2e-7 * np.abs(ref_avg) + 1e-30)
    pkg.corr_destroy(h)


def test_accumulate_wide_float_into_double():
    import paper_0906_1887_b200 as pkg
    N, C, T = 64, 3, 80
    w = corrgen.scaled(corrgen.CONFIGS["c5"], n_inputs=N, n_chan=C, n_time=T)
    xs = [w.generate(integration=k) for k in range(4)]
    h = pkg.corr_create(N, C, T, "cf32")
    acc = h.empty_acc()
    for x in xs:
        h.accumulate_wide(torch.from_numpy(x).cuda(), acc)
    torch.cuda.synchronize()
    assert acc.dtype == torch.float64
    f32_tolerance_check(acc.cpu().numpy(), oracle.xengine_cf32(np.concatenate(xs, axis=0)), N)
    pkg.corr_destroy(h)


@pytest.mark.parametrize("plan,accumulate", [(256 * 4 + 3, False), (256 * 4 + 3, True), (256 * 1 + 1, True)])
def test_captured_graph_with_sliced_and_accumulating_calls(plan, accumulate):
    """Programmatic dependent launches under capture next to memset nodes (time-sliced plan) and in accumulate mode:
    consecutive calls into the SAME d_vis, graph replayed twice, bit-exact."""
    import paper_0906_1887_b200 as pkg
    w = corrgen.scaled(corrgen.CONFIGS["c1"], n_chan=24, n_time=600)
    xs = [w.generate(integration=k) for k in range(3)]
    refs = [oracle.xengine_ci8(x, threads=oracle.host_threads()).astype(np.int64) for x in xs]
    h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, "ci8")
    h.set_option(pkg.CORR_OPT_DIAG_PLAN, plan)
    d = [torch.from_numpy(x).cuda() for x in xs]
    vis = h.empty_vis()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        pkg.corr_xengine(h, d[0], vis, s)   # warm-up outside the capture
        torch.cuda.synchronize()
        if accumulate:
            h.set_accumulate(True)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            if accumulate:
                vis.zero_()
            for k in range(3):
                pkg.corr_xengine(h, d[k], vis, s)
        for _ in range(2):
            vis.fill_(-0x55555555)
            g.replay()
            torch.cuda.synchronize()
            want = (refs[0] + refs[1] + refs[2]) if accumulate else refs[2]
            assert np.array_equal(vis.cpu().numpy().astype(np.int64), want)
    del g
    pkg.corr_destroy(h)
