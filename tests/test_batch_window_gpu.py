"""GPU parity of the round-2 entry points, each against the CPU oracle:

* corr_xengine_batch  -- n integrations in one launch: every d_vis[k] bit-exact, poison-filled;
* corr_set_chan_window -- a handle correlates a channel window of the full [T][C][N] cube in place:
  the windows of a 2-rank (and 3-rank) split, run one after the other on one GPU, concatenate to the oracle's cube;
* handles with different shared-memory footprints alive side by side (the per-function attribute is set once).
"""
from __future__ import annotations

import numpy as np
import pytest

import corrgen
import oracle
from parity_util import f32_tolerance_check

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

POISON = -0x55555555


@pytest.fixture(scope="module")
def pkg():
    import paper_0906_1887_b200 as p
    p.lib()
    return p


def _threads():
    return oracle.host_threads()


# (N, C, T, n): diag plans (N <= 64, incl. the two-channels-per-panel mode and an odd channel count), slab plans
# (128 <= N < 512), one batch larger than the 64 integrations a launch takes, ragged K tails
BATCH_SHAPES = [(32, 16, 100, 5), (32, 7, 33, 3), (64, 9, 130, 4), (64, 3, 64, 70), (128, 2, 96, 3), (256, 1, 70, 2),
                (32, 128, 257, 6)]


@pytest.mark.parametrize("N,C,T,n", BATCH_SHAPES)
def test_batch_every_output_bit_exact(pkg, N, C, T, n):
    w = corrgen.scaled(corrgen.CONFIGS["c1"], n_inputs=N, n_chan=C, n_time=T)
    xs = [w.generate(integration=k) for k in range(n)]
    h = pkg.corr_create(N, C, T, "ci8")
    d_in = [torch.from_numpy(x).cuda() for x in xs]
    d_vis = [h.empty_vis() for _ in range(n)]
    for v in d_vis:
        v.fill_(POISON)
    pkg.corr_xengine_batch(h, d_in, d_vis)
    torch.cuda.synchronize()
    for k in range(n):
        assert np.array_equal(d_vis[k].cpu().numpy(), oracle.xengine_ci8(xs[k], threads=_threads())), f"integration {k}"
    pkg.corr_destroy(h)


@pytest.mark.parametrize("plan", ["4,1", "2,1", "1,1", "4,2", "2,3"])
def test_batch_forced_diag_plans(pkg, plan):
    """Every panel-group width, and time slices (reduce-add into zeroed outputs), inside a batched launch."""
    g, sl = (int(v) for v in plan.split(","))
    N, C, T, n = 32, 22, 400, 4
    w = corrgen.scaled(corrgen.CONFIGS["c1"], n_inputs=N, n_chan=C, n_time=T)
    xs = [w.generate(integration=k) for k in range(n)]
    h = pkg.corr_create(N, C, T, "ci8")
    h.set_option(pkg.CORR_OPT_DIAG_PLAN, 256 * g + sl)
    d_vis = [h.empty_vis().fill_(POISON) for _ in range(n)]
    pkg.corr_xengine_batch(h, [torch.from_numpy(x).cuda() for x in xs], d_vis)
    torch.cuda.synchronize()
    for k in range(n):
        assert np.array_equal(d_vis[k].cpu().numpy(), oracle.xengine_ci8(xs[k], threads=_threads())), f"integration {k}"
    pkg.corr_destroy(h)


@pytest.mark.parametrize("dtype,N,C,T", [("ci8", 512, 2, 70), ("ci4", 64, 5, 100), ("cf32", 64, 4, 50)])
def test_batch_falls_back_to_single_calls(pkg, dtype, N, C, T):
    """CTA-pair plans, the 4-bit mode and the float path run n ordinary calls: same results."""
    key = {"ci8": "c4", "ci4": "c2", "cf32": "c5"}[dtype]
    w = corrgen.scaled(corrgen.CONFIGS[key], n_inputs=N, n_chan=C, n_time=T)
    xs = [w.generate(integration=k) for k in range(3)]
    h = pkg.corr_create(N, C, T, dtype)
    d_in = [torch.from_numpy(corrgen.pack_ci4(x) if dtype == "ci4" else x).cuda() for x in xs]
    d_vis = pkg.corr_xengine_batch(h, d_in)
    torch.cuda.synchronize()
    for k, x in enumerate(xs):
        out = d_vis[k].cpu().numpy()
        if dtype == "cf32":
            f32_tolerance_check(out, oracle.xengine_cf32(x, threads=_threads()), N)
        elif dtype == "ci4":
            assert np.array_equal(out, oracle.xengine_ci4(corrgen.pack_ci4(x), threads=_threads()))
        else:
            assert np.array_equal(out, oracle.xengine_ci8(x, threads=_threads()))
    pkg.corr_destroy(h)


def test_batch_argument_errors(pkg):
    import ctypes
    L = pkg.lib()
    h = pkg.corr_create(32, 4, 50, "ci8")
    x = torch.zeros(h.in_bytes, dtype=torch.int8, device="cuda")
    v = h.empty_vis()
    ok_in = (ctypes.c_void_p * 2)(x.data_ptr(), x.data_ptr())
    ok_out = (ctypes.c_void_p * 2)(v.data_ptr(), v.data_ptr())
    bad_in = (ctypes.c_void_p * 2)(x.data_ptr(), None)
    mis_in = (ctypes.c_void_p * 2)(x.data_ptr(), x.data_ptr() + 4)
    assert L.corr_xengine_batch(h._h, ok_in, ok_out, 0, None) == pkg.CORR_EINVAL
    assert L.corr_xengine_batch(h._h, None, ok_out, 2, None) == pkg.CORR_EINVAL
    assert L.corr_xengine_batch(h._h, bad_in, ok_out, 2, None) == pkg.CORR_EINVAL
    assert L.corr_xengine_batch(h._h, mis_in, ok_out, 2, None) == pkg.CORR_EINVAL
    assert b"corr_xengine_batch" in L.corr_last_error()
    pkg.corr_destroy(h)


# ------------------------------------------------------------------------------------------------ channel windows

def _shards(n_chan, world):
    out = []
    for rank in range(world):
        base, extra = divmod(n_chan, world)
        c0 = rank * base + min(rank, extra)
        out.append((c0, c0 + base + (1 if rank < extra else 0)))
    return out


@pytest.mark.parametrize("dtype,key,N,C,T,world,turn", [
    ("ci8", "c2", 64, 11, 130, 2, False), ("ci8", "c1", 32, 13, 100, 2, False), ("ci8", "c1", 32, 12, 100, 3, False),
    ("ci8", "c4", 256, 5, 70, 2, False), ("ci8", "c4", 512, 3, 70, 2, False), ("ci8", "c3", 256, 3, 2100, 2, False),
    ("ci8", "c2", 64, 10, 90, 2, True), ("ci8", "c1", 32, 12, 90, 2, True),
    ("ci4", "c2", 64, 7, 100, 2, False), ("ci4", "c2", 256, 3, 64, 2, False),
    ("cf32", "c5", 64, 17, 60, 2, False), ("cf32", "c5", 128, 5, 40, 3, False)])
def test_channel_sharded_run_equals_the_oracle_cube(pkg, dtype, key, N, C, T, world, turn):
    """The `world` ranks of a channel-sharded run (each a handle on ITS window of the one seeded cube, read in place),
    executed back to back on one GPU: the concatenation of their outputs is the oracle's whole cube."""
    w = corrgen.scaled(corrgen.CONFIGS[key], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    xin = corrgen.pack_ci4(x) if dtype == "ci4" else x
    d_in = torch.from_numpy(xin).cuda()
    nb = N * (N + 1) // 2
    full = torch.empty((C, nb, 2), dtype=torch.float32 if dtype == "cf32" else torch.int32, device="cuda")
    full.fill_(float("nan") if dtype == "cf32" else POISON)
    for c0, c1 in _shards(C, world):
        h = pkg.corr_create(N, c1 - c0, T, dtype)
        h.set_chan_window(C, c0)
        assert h.in_bytes == d_in.numel() * d_in.element_size()
        if turn:
            h.set_turn(pkg.CORR_TURN_STANDALONE)
        pkg.corr_xengine(h, d_in, full[c0:c1])
        torch.cuda.synchronize()
        pkg.corr_destroy(h)
    out = full.cpu().numpy()
    if dtype == "cf32":
        f32_tolerance_check(out, oracle.xengine_cf32(x, threads=_threads()), N)
    elif dtype == "ci4":
        assert np.array_equal(out, oracle.xengine_ci4(xin, threads=_threads()))
    else:
        assert np.array_equal(out, oracle.xengine_ci8(x, threads=_threads()))


def test_chan_window_errors_and_reset(pkg):
    h = pkg.corr_create(64, 4, 50, "ci8")
    for total, c0 in [(3, 0), (6, 3), (8, -1), (0, 0)]:
        with pytest.raises(pkg.CorrError) as e:
            h.set_chan_window(total, c0)
        assert e.value.status == pkg.CORR_EINVAL
    w = corrgen.scaled(corrgen.CONFIGS["c2"], n_chan=4, n_time=50)
    x = w.generate()
    h.set_chan_window(9, 2)
    h.set_chan_window(4, 0)   # back to the default
    out = pkg.corr_xengine(h, torch.from_numpy(x).cuda()).cpu().numpy()
    assert np.array_equal(out, oracle.xengine_ci8(x))
    pkg.corr_destroy(h)


def test_windowed_batch(pkg):
    """Window and batch together: n integrations of a channel window in one launch."""
    N, C, T, n = 32, 20, 120, 3
    w = corrgen.scaled(corrgen.CONFIGS["c1"], n_inputs=N, n_chan=C, n_time=T)
    xs = [w.generate(integration=k) for k in range(n)]
    h = pkg.corr_create(N, 8, T, "ci8")
    h.set_chan_window(C, 6)
    d_vis = [h.empty_vis().fill_(POISON) for _ in range(n)]
    pkg.corr_xengine_batch(h, [torch.from_numpy(x).cuda() for x in xs], d_vis)
    torch.cuda.synchronize()
    for k in range(n):
        assert np.array_equal(d_vis[k].cpu().numpy(), oracle.xengine_ci8(xs[k], 6, 14, threads=_threads()))
    pkg.corr_destroy(h)


# ------------------------------------------------------------------------------------------------ several handles

def test_handles_with_different_footprints_alive_together(pkg):
    """A CI8 handle (N_I = 256: 227 KB of dynamic shared memory) and a CI4 handle (N_I = 256: a smaller ring) are
    created one after the other and then used alternately: the function attribute must not shrink under the first."""
    N, C, T = 256, 2, 90
    w = corrgen.scaled(corrgen.CONFIGS["c4"], n_inputs=N, n_chan=C, n_time=T)
    x8 = w.generate()
    w4 = corrgen.scaled(corrgen.CONFIGS["c2"], n_inputs=N, n_chan=C, n_time=T)
    x4 = corrgen.pack_ci4(w4.generate())
    ref8, ref4 = oracle.xengine_ci8(x8, threads=_threads()), oracle.xengine_ci4(x4, threads=_threads())
    h8 = pkg.corr_create(N, C, T, "ci8")
    h4 = pkg.corr_create(N, C, T, "ci4")
    h64 = pkg.corr_create(64, 3, 40, "ci8")
    d8, d4 = torch.from_numpy(x8).cuda(), torch.from_numpy(x4).cuda()
    for _ in range(2):
        v8 = h8.empty_vis().fill_(POISON)
        v4 = h4.empty_vis().fill_(POISON)
        pkg.corr_xengine(h8, d8, v8)
        pkg.corr_xengine(h4, d4, v4)
        torch.cuda.synchronize()
        assert np.array_equal(v8.cpu().numpy(), ref8)
        assert np.array_equal(v4.cpu().numpy(), ref4)
    for h in (h8, h4, h64):
        pkg.corr_destroy(h)


def test_ci4_wide_rows_keep_a_deep_ring(pkg):
    """CI4 at N_I = 256 and 512 (slab plans): bit-exact, several stages, ragged T."""
    for N, C, T in [(256, 2, 300), (512, 1, 130), (192, 2, 257)]:
        w = corrgen.scaled(corrgen.CONFIGS["c2"], n_inputs=N, n_chan=C, n_time=T)
        x4 = corrgen.pack_ci4(w.generate())
        h = pkg.corr_create(N, C, T, "ci4")
        v = h.empty_vis().fill_(POISON)
        pkg.corr_xengine(h, torch.from_numpy(x4).cuda(), v)
        torch.cuda.synchronize()
        assert np.array_equal(v.cpu().numpy(), oracle.xengine_ci4(x4, threads=_threads())), (N, C, T)
        pkg.corr_destroy(h)


def test_batch_of_one_and_replanning_between_sizes(pkg):
    """n = 1 is an ordinary call; a handle re-plans when the batch size changes (3 -> 64 -> 3) and stays usable for
    single calls in between; options set after the first use re-plan as well."""
    N, C, T = 32, 10, 90
    w = corrgen.scaled(corrgen.CONFIGS["c1"], n_inputs=N, n_chan=C, n_time=T)
    xs = [w.generate(integration=k) for k in range(64)]
    refs = [oracle.xengine_ci8(x, threads=_threads()) for x in xs[:4]] + [None] * 60
    d_in = [torch.from_numpy(x).cuda() for x in xs]
    h = pkg.corr_create(N, C, T, "ci8")
    for n in (1, 3, 64, 3):
        outs = [h.empty_vis().fill_(POISON) for _ in range(n)]
        pkg.corr_xengine_batch(h, d_in[:n], outs)
        torch.cuda.synchronize()
        for k in range(min(n, 4)):
            assert np.array_equal(outs[k].cpu().numpy(), refs[k]), (n, k)
        if n == 64:
            k = 63
            assert np.array_equal(outs[k].cpu().numpy(), oracle.xengine_ci8(xs[k], threads=_threads()))
        single = pkg.corr_xengine(h, d_in[2])
        torch.cuda.synchronize()
        assert np.array_equal(single.cpu().numpy(), refs[2])
    h.set_option(pkg.CORR_OPT_DIAG_PLAN, 256 * 2 + 2)
    outs = pkg.corr_xengine_batch(h, d_in[:3])
    torch.cuda.synchronize()
    for k in range(3):
        assert np.array_equal(outs[k].cpu().numpy(), refs[k])
    pkg.corr_destroy(h)


def test_window_with_accumulate_and_wide_accumulators(pkg):
    """A channel-window handle in accumulate mode and with corr_accumulate_wide: batches of the window add up."""
    N, C, T = 64, 9, 70
    w = corrgen.scaled(corrgen.CONFIGS["c2"], n_inputs=N, n_chan=C, n_time=T)
    xs = [w.generate(integration=k) for k in range(3)]
    want = oracle.xengine_ci8_wide(np.concatenate(xs, axis=0), 2, 7, threads=_threads())
    h = pkg.corr_create(N, 5, T, "ci8")
    h.set_chan_window(C, 2)
    h.set_accumulate(True)
    vis = h.empty_vis().zero_()
    acc = h.empty_acc()
    for x in xs:
        d = torch.from_numpy(x).cuda()
        pkg.corr_xengine(h, d, vis)
        h.accumulate_wide(d, acc)
    torch.cuda.synchronize()
    assert h.accumulate_count == 3
    assert np.array_equal(vis.cpu().numpy().astype(np.int64), want)
    assert np.array_equal(acc.cpu().numpy(), want)
    pkg.corr_destroy(h)
