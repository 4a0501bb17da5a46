"""Host-side planning and argument checks of the library, observed through corr_plan_info (include/corr.h):
which kernel and schedule a handle will launch, that forced plans are honoured wherever they are documented to apply,
that a channel window's plan does not depend on the order of the set-up calls, and that corr_xengine_batch refuses
batches whose buffers overlap.  Every case that launches also checks the result against the CPU oracle."""
from __future__ import annotations

import ctypes

import numpy as np
import pytest

import corrgen
import oracle

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pkg():
    import paper_0906_1887_b200 as p
    p.lib()
    return p


def _x(N, C, T, seed=0):
    return corrgen.uniform_i8(T, C, N, seed, 127)


@pytest.mark.parametrize("dtype,N,C,T,kernel,kid", [
    ("ci8", 32, 128, 1000, "xengine_i8_kernel", 0), ("ci8", 64, 768, 10000, "xengine_i8_kernel", 0),
    ("ci8", 192, 4, 500, "xengine_i8_kernel", 0), ("ci8", 256, 512, 4000, "xengine_i8_pair_kernel", 1),
    ("ci8", 1024, 128, 1000, "xengine_i8_pair_kernel", 2), ("ci8", 256, 8, 1000, "xengine_i8_pair_kernel", 2),
    ("ci8", 512, 8, 1500, "xengine_i8_pair_kernel", 1), ("ci4", 64, 768, 10000, "xengine_i4_kernel", 3),
    ("cf32", 64, 1536, 500, "xengine_f32_n64_kernel", 5), ("cf32", 96, 8, 100, "xengine_f32_kernel", 4)])
def test_plan_info_names_the_kernel_of_the_paper_shaped_configs(pkg, dtype, N, C, T, kernel, kid):
    h = pkg.corr_create(N, C, T, dtype)
    p = h.plan_info()
    assert (p["kernel"], p["kernel_id"]) == (kernel, kid), p
    assert p["grid"] >= 1 and p["slices"] >= 1
    if dtype != "cf32":
        assert p["stages"] >= 2 and 0 < p["smem"] <= 227 * 1024
        assert p["grid"] <= 148 + 4  # one CTA (or CTA pair) per SM at most
    pkg.corr_destroy(h)


@pytest.mark.parametrize("N,T,kid", [
    (256, 1024, 2), (256, 1152, 2), (256, 1153, 0), (384, 1100, 2), (512, 1152, 2), (512, 1153, 1),   # 4 / 6 / 8 panels: to T = 1152
    (320, 1000, 0), (288, 500, 0), (448, 1000, 0), (416, 300, 0),                                     # 5 / 7 panels: slabs
    (576, 1024, 2), (576, 1100, 1), (1024, 1000, 2), (1024, 1100, 1)])                                # >= 9 panels: to T = 1024
def test_resident_plan_is_taken_where_it_was_measured_to_pay(pkg, N, T, kid):
    """DESIGN.md section 11 (round 3): thresholds of the resident-A plan, and CORR_OPT_RESIDENT = 2 / 0 around them."""
    h = pkg.corr_create(N, 3, T, "ci8")
    assert h.plan_info()["kernel_id"] == kid, h.plan_info()
    h.set_option(pkg.CORR_OPT_RESIDENT, 2)
    assert h.plan_info()["kernel_id"] == (2 if T <= 1152 else kid)
    h.set_option(pkg.CORR_OPT_RESIDENT, 0)
    assert h.plan_info()["kernel_id"] != 2
    pkg.corr_destroy(h)


@pytest.mark.parametrize("N,C,T", [(320, 2, 1100), (448, 1, 1152), (1024, 1, 1130), (256, 2, 1025)])
def test_forced_resident_plan_is_bit_exact(pkg, N, C, T):
    h = pkg.corr_create(N, C, T, "ci8")
    h.set_option(pkg.CORR_OPT_RESIDENT, 2)
    assert h.plan_info()["resident"]
    x = _x(N, C, T, seed=N + T)
    vis = h.empty_vis()
    vis.fill_(-0x55555555)
    pkg.corr_xengine(h, torch.from_numpy(x).cuda(), vis)
    torch.cuda.synchronize()
    assert np.array_equal(vis.cpu().numpy(), oracle.xengine_ci8(x, threads=oracle.host_threads()))
    pkg.corr_destroy(h)


def test_plan_info_argument_errors(pkg):
    L = pkg.lib()
    h = pkg.corr_create(32, 4, 50, "ci8")
    info = (ctypes.c_int * 8)()
    assert L.corr_plan_info(None, info, None, 0) == pkg.CORR_EINVAL
    assert L.corr_plan_info(h._h, None, None, 0) == pkg.CORR_EINVAL
    assert L.corr_plan_info(h._h, info, None, 0) == pkg.CORR_OK      # the name is optional
    pkg.corr_destroy(h)


@pytest.mark.parametrize("N,C,T", [(32, 22, 400), (64, 40, 300), (64, 768, 3000)])   # <= 64 MB twice, > 64 MB once
@pytest.mark.parametrize("g", [1, 2, 4])
def test_forced_group_width_is_honoured_for_every_input_size(pkg, N, C, T, g):
    """CORR_OPT_DIAG_PLAN with slices = 0 forces only the group width -- also for inputs <= 64 MB."""
    h = pkg.corr_create(N, C, T, "ci8")
    h.set_option(pkg.CORR_OPT_DIAG_PLAN, 256 * g)
    assert h.plan_info()["gsize"] == g
    x = _x(N, C, T, seed=g)
    vis = pkg.corr_xengine(h, torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    want = oracle.xengine_ci8(x[:, :6], threads=oracle.host_threads())
    assert np.array_equal(vis.cpu().numpy()[:6], want)
    h.set_option(pkg.CORR_OPT_DIAG_PLAN, 0)
    auto = h.plan_info()["gsize"]
    assert auto in (1, 2, 4)
    pkg.corr_destroy(h)


@pytest.mark.parametrize("g", [1, 2, 4])
def test_forced_group_width_reaches_the_batched_launch(pkg, g):
    N, C, T, n = 32, 22, 200, 3
    h = pkg.corr_create(N, C, T, "ci8")
    h.set_option(pkg.CORR_OPT_DIAG_PLAN, 256 * g)
    xs = [_x(N, C, T, seed=10 + k) for k in range(n)]
    out = pkg.corr_xengine_batch(h, [torch.from_numpy(x).cuda() for x in xs])
    torch.cuda.synchronize()
    for k in range(n):
        assert np.array_equal(out[k].cpu().numpy(), oracle.xengine_ci8(xs[k], threads=oracle.host_threads()))
    pkg.corr_destroy(h)


def test_window_plan_does_not_depend_on_call_order(pkg):
    """A 4-channel window (4 MB of work) of a cube far above the planner's 64 MB threshold: the plan must be the small
    window's whether an option is set before or after corr_set_chan_window (the re-plan used to see the cube)."""
    N, Cw, T, Ctot = 64, 4, 8192, 96                       # window 4 * 8192 * 128 B = 4 MB; cube 100 MB
    a = pkg.corr_create(N, Cw, T, "ci8")
    before = a.plan_info()
    a.set_chan_window(Ctot, 40)
    assert a.plan_info() == before
    a.set_option(pkg.CORR_OPT_MIX, 1)                      # a no-op value: forces a re-plan after the window was set
    assert a.plan_info() == before
    b = pkg.corr_create(N, Cw, T, "ci8")
    b.set_option(pkg.CORR_OPT_MIX, 1)
    b.set_chan_window(Ctot, 40)
    assert b.plan_info() == before
    # and the windowed result is the oracle's for those channels
    x = corrgen.gauss_i8(T, Ctot, N, 3, 3.0, 7)
    vis = pkg.corr_xengine(a, torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    want = oracle.xengine_ci8(np.ascontiguousarray(x[:, 40:44]), threads=oracle.host_threads())
    assert np.array_equal(vis.cpu().numpy(), want)
    pkg.corr_destroy(a)
    pkg.corr_destroy(b)


def test_batch_rejects_overlapping_buffers(pkg):
    L = pkg.lib()
    N, C, T = 32, 4, 50
    h = pkg.corr_create(N, C, T, "ci8")
    x0 = torch.from_numpy(_x(N, C, T, 1)).cuda()
    x1 = torch.from_numpy(_x(N, C, T, 2)).cuda()
    v0, v1 = h.empty_vis(), h.empty_vis()
    big = torch.zeros(2 * h.vis_bytes, dtype=torch.int8, device="cuda")
    arr = lambda *t: (ctypes.c_void_p * len(t))(*[p if isinstance(p, int) else p.data_ptr() for p in t])
    v0.fill_(7)
    v1.fill_(7)
    # the same output twice; an output that is another entry's input; two outputs that overlap by half
    assert L.corr_xengine_batch(h._h, arr(x0, x1), arr(v0, v0), 2, None) == pkg.CORR_EINVAL
    assert b"overlaps" in L.corr_last_error()
    xin = torch.zeros(max(h.in_bytes, h.vis_bytes), dtype=torch.int8, device="cuda")
    assert L.corr_xengine_batch(h._h, arr(x0, xin), arr(xin, v1), 2, None) == pkg.CORR_EINVAL
    assert L.corr_xengine_batch(h._h, arr(x0, x1), arr(big, big.data_ptr() + h.vis_bytes // 2 // 16 * 16), 2, None) == pkg.CORR_EINVAL
    torch.cuda.synchronize()
    assert bool((v0 == 7).all()) and bool((v1 == 7).all())     # nothing was enqueued
    # one input for two outputs is fine (inputs are only read) ...
    assert L.corr_xengine_batch(h._h, arr(x0, x0), arr(v0, v1), 2, None) == pkg.CORR_OK
    torch.cuda.synchronize()
    assert torch.equal(v0, v1)
    # ... and in accumulate mode (call by call, stream-ordered) several entries may add into one output
    h.set_accumulate(True)
    acc = h.empty_vis()
    acc.zero_()
    assert L.corr_xengine_batch(h._h, arr(x0, x1), arr(acc, acc), 2, None) == pkg.CORR_OK
    torch.cuda.synchronize()
    want = oracle.xengine_ci8(x0.cpu().numpy()) + oracle.xengine_ci8(x1.cpu().numpy())
    assert np.array_equal(acc.cpu().numpy(), want)
    assert L.corr_xengine_batch(h._h, arr(x0, acc), arr(acc, v1), 2, None) == pkg.CORR_EINVAL   # output == an input: never
    pkg.corr_destroy(h)
