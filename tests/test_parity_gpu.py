"""GPU parity: the CUDA X-engine (through the C ABI binding) vs the CPU oracle, element by element.

int8 path: bit-exact.  float32 path: |delta| <= 1e-5 sqrt(|V_ii V_jj|) against the float64 oracle
(north_star).  Inputs are the seeded synthetic recipes of DESIGN.md.
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


def _threads():
    return oracle.host_threads()


def run_ci8(pkg, x, turn=None, options=()):
    T, C, N, _ = x.shape
    h = pkg.corr_create(N, C, T, "ci8")
    for key, value in options:
        h.set_option(key, value)
    if turn is not None:
        h.set_turn(turn)
    d_in = torch.from_numpy(x).cuda()
    vis = h.empty_vis()
    vis.fill_(-0x55555555)  # poison: every element must be overwritten
    pkg.corr_xengine(h, d_in, vis)
    torch.cuda.synchronize()
    out = vis.cpu().numpy()
    pkg.corr_destroy(h)
    return out


def run_cf32(pkg, x, options=()):
    T, C, N, _ = x.shape
    h = pkg.corr_create(N, C, T, "cf32")
    for key, value in options:
        h.set_option(key, value)
    d_in = torch.from_numpy(x).cuda()
    vis = h.empty_vis()
    vis.fill_(float("nan"))
    pkg.corr_xengine(h, d_in, vis)
    torch.cuda.synchronize()
    out = vis.cpu().numpy()
    pkg.corr_destroy(h)
    return out


# (N, C, T): several tiles + ragged tails; T in {1,31,32,33} pins K zero-padding (reading R11);
# N=32 exercises the two-channels-per-panel mode incl. odd C; N=96/320/640 multi-panel, separate-A
# and multi-segment items; N=1024 the c4 tile schedule (CTA pairs, cta_group::2).
CI8_SHAPES = [(64, 3, 100), (64, 5, 1), (64, 2, 31), (64, 2, 32), (64, 2, 33), (64, 1, 257), (64, 200, 40),
              (32, 4, 100), (32, 3, 70), (32, 1, 64), (32, 301, 33), (96, 2, 64), (128, 2, 300),
              (256, 2, 130), (320, 1, 64), (640, 1, 40), (1024, 1, 96),
              # CTA-pair kernel (N_I >= 512): even / odd panel counts, several stages, ragged T, many channels
              (512, 3, 200), (576, 2, 70), (512, 40, 33), (2048, 1, 64),
              # long integrations (T >= 2048): 512-wide pair tiles from N_I = 256 up, mixed with 256-wide ones
              (256, 3, 2100), (320, 1, 2050), (512, 1, 2081),
              # resident-A plans (N_I >= 512, T <= 1024): full-length A region, ragged last sub-stage, odd panel count
              (512, 2, 1000), (640, 3, 1024), (576, 5, 129), (1024, 2, 300),
              # CTA pairs without the resident plan: 1152 < T < 2048
              (512, 1, 1200),
              # round 3: resident plan up to T = 1152 (9 sub-stages, 3-stage ring) for 4 / 6 / 8 panels per channel, ragged last
              # sub-stage; 5 / 7 panels (N_I = 320, 448) back on single-CTA slabs; 9 panels streaming above T = 1024
              (256, 3, 1100), (384, 2, 1152), (512, 2, 1150), (320, 2, 1000), (448, 2, 700), (576, 1, 1100),
              # the largest N_I the ABI admits (528 schedule kinds per channel)
              (4096, 1, 40)]


@pytest.mark.parametrize("N,C,T", CI8_SHAPES)
def test_ci8_gauss_bit_exact(pkg, N, C, T):
    w = corrgen.scaled(corrgen.CONFIGS["c2"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    assert np.array_equal(run_ci8(pkg, x), oracle.xengine_ci8(x, threads=_threads()))


@pytest.mark.parametrize("N,C,T", [(64, 3, 100), (256, 2, 130), (32, 4, 100)])
def test_ci8_uniform_full_range_bit_exact(pkg, N, C, T):
    w = corrgen.scaled(corrgen.CONFIGS["c3"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    assert np.array_equal(run_ci8(pkg, x), oracle.xengine_ci8(x, threads=_threads()))


@pytest.mark.parametrize("N,C,T", [(512, 2, 100), (256, 2, 2100), (1024, 1, 64)])
def test_ci8_single_cta_slabs_when_pairs_are_disabled(pkg, N, C, T):
    """corr_set_option(CORR_OPT_PAIRS, 0) (the A/B knob of DESIGN.md section 7) selects the single-CTA slab schedule."""
    w = corrgen.scaled(corrgen.CONFIGS["c4"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    assert np.array_equal(run_ci8(pkg, x, options=[(pkg.CORR_OPT_PAIRS, 0)]), oracle.xengine_ci8(x, threads=_threads()))


@pytest.mark.parametrize("N,C,T", [(512, 3, 200), (576, 2, 70), (1024, 1, 96), (512, 2, 1000)])
def test_ci8_pair_tiles_without_the_resident_plan(pkg, N, C, T):
    """corr_set_option(CORR_OPT_RESIDENT, 0): N_I >= 512, T <= 1024 on the streaming 256 x 256 pair tiles."""
    w = corrgen.scaled(corrgen.CONFIGS["c4"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    assert np.array_equal(run_ci8(pkg, x, options=[(pkg.CORR_OPT_RESIDENT, 0)]), oracle.xengine_ci8(x, threads=_threads()))


@pytest.mark.parametrize("N,C,T", [(256, 2, 2100), (384, 1, 2081)])
def test_ci8_wide_pair_tiles_without_collector_reuse(pkg, N, C, T):
    w = corrgen.scaled(corrgen.CONFIGS["c4"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    assert np.array_equal(run_ci8(pkg, x, options=[(pkg.CORR_OPT_COLLECT, 0)]), oracle.xengine_ci8(x, threads=_threads()))


@pytest.mark.parametrize("N,C,T", [(512, 1, 2081), (640, 1, 1030)])
def test_ci8_wide_pair_tiles_forced_for_many_panels(pkg, N, C, T):
    """CORR_OPT_WIDE = 2: 512-wide tiles also from N_I = 512 up and for short integrations (by default 256-wide there)."""
    w = corrgen.scaled(corrgen.CONFIGS["c4"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    assert np.array_equal(run_ci8(pkg, x, options=[(pkg.CORR_OPT_WIDE, 2)]), oracle.xengine_ci8(x, threads=_threads()))


@pytest.mark.parametrize("N,C,T", [(256, 2, 2100), (512, 1, 2081)])
def test_ci8_pair_tiles_without_the_wide_ones(pkg, N, C, T):
    w = corrgen.scaled(corrgen.CONFIGS["c4"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    assert np.array_equal(run_ci8(pkg, x, options=[(pkg.CORR_OPT_WIDE, 0)]), oracle.xengine_ci8(x, threads=_threads()))


def test_ci8_zero_input(pkg):
    x = np.zeros((40, 3, 64, 2), np.int8)
    assert not run_ci8(pkg, x).any()


@pytest.mark.parametrize("val", [-128, 127])
def test_ci8_extreme_constant_longest_integration(pkg, val):
    """T = 65535 with every component at +-full scale: the largest sums the ABI admits (reading R6)."""
    x = np.full((65535, 2, 32, 2), val, np.int8)
    out = run_ci8(pkg, x)
    assert np.array_equal(out, oracle.xengine_ci8(x, threads=_threads()))
    assert out[..., 0].max() == 65535 * 2 * val * val


@pytest.mark.parametrize("N,C,T", [(64, 6, 100), (32, 4, 70), (256, 2, 64), (96, 2, 40), (512, 2, 70), (256, 1, 2100)])
def test_ci8_standalone_corner_turn_path(pkg, N, C, T):
    w = corrgen.scaled(corrgen.CONFIGS["c4"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    assert np.array_equal(run_ci8(pkg, x, turn=pkg.CORR_TURN_STANDALONE), oracle.xengine_ci8(x, threads=_threads()))


@pytest.mark.parametrize("dtype,N,C,T", [("ci8", 64, 7, 100), ("ci8", 32, 6, 33), ("ci8", 1024, 3, 20),
                                         ("cf32", 64, 5, 50), ("cf32", 32, 3, 17)])
def test_corner_turn_is_the_permutation(pkg, dtype, N, C, T):
    """[T][C][N] -> [C][T][N] (channel pairs for N_I = 32 int8): pure byte permutation, bit-exact."""
    rng = np.random.default_rng(5)
    if dtype == "ci8":
        x = rng.integers(-128, 128, size=(T, C, N, 2), dtype=np.int8)
    else:
        x = rng.standard_normal((T, C, N, 2)).astype(np.float32)
    h = pkg.corr_create(N, C, T, dtype)
    out = h.corner_turn(torch.from_numpy(x).cuda()).cpu().numpy()
    pkg.corr_destroy(h)
    if dtype == "ci8" and N == 32:
        want = x.reshape(T, C // 2, 2 * N, 2).transpose(1, 0, 2, 3)
    else:
        want = x.transpose(1, 0, 2, 3)
    assert np.array_equal(out.reshape(want.shape), want)


CF32_SHAPES = [(64, 3, 50), (64, 2, 500), (64, 40, 17), (32, 3, 33), (96, 2, 20), (128, 2, 40), (192, 1, 30),
               # the generic kernel's many-block rows and diagonals: corr_create admits CF32 up to N_I = 4096
               (256, 2, 40), (512, 1, 30), (1024, 1, 20), (2048, 1, 4)]


@pytest.mark.parametrize("N,C,T", CF32_SHAPES)
def test_cf32_within_tolerance(pkg, N, C, T):
    w = corrgen.scaled(corrgen.CONFIGS["c5"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    f32_tolerance_check(run_cf32(pkg, x), oracle.xengine_cf32(x, threads=_threads()), N)


def test_cf32_single_nonzero_input_exact_zeros(pkg):
    """Only input k non-zero: every other visibility is exactly 0 (oracle pin P3 on the GPU)."""
    x = np.zeros((30, 2, 64, 2), np.float32)
    x[:, :, 9, :] = np.random.default_rng(1).standard_normal((30, 2, 2)).astype(np.float32)
    out = run_cf32(pkg, x)
    ref = oracle.xengine_cf32(x)
    f32_tolerance_check(out, ref, 64)
    b = 9 * 10 // 2 + 9
    mask = np.ones(out.shape[1], bool)
    mask[b] = False
    assert not out[:, mask].any()


def test_overwrite_semantics_and_reuse(pkg):
    """d_vis is overwritten each call (reading R4); one handle serves several inputs and streams."""
    w = corrgen.scaled(corrgen.CONFIGS["c1"], n_chan=6, n_time=90)
    h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, "ci8")
    vis = h.empty_vis()
    s = torch.cuda.Stream()
    for k in range(3):
        x = w.generate(integration=k)
        d_in = torch.from_numpy(x).cuda()
        torch.cuda.synchronize()
        pkg.corr_xengine(h, d_in, vis, stream=s)
        s.synchronize()
        assert np.array_equal(vis.cpu().numpy(), oracle.xengine_ci8(x))
    pkg.corr_destroy(h)


def test_stream_run_matches_oracle(pkg):
    """Streaming driver: 5 integrations through pinned host buffers, cf32 and ci8."""
    for dtype, key in (("cf32", "c5"), ("ci8", "c2")):
        w = corrgen.scaled(corrgen.CONFIGS[key], n_chan=8, n_time=60)
        xs = [w.generate(integration=k) for k in range(5)]
        h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, dtype)
        pinned = [torch.from_numpy(x).pin_memory() for x in xs]
        d_vis, stats = h.stream_run(pinned)
        out = d_vis.cpu().numpy()
        pkg.corr_destroy(h)
        assert stats["device_s"] > 0 and stats["kernel_s"] > 0
        for k, x in enumerate(xs):
            if dtype == "ci8":
                assert np.array_equal(out[k], oracle.xengine_ci8(x))
            else:
                f32_tolerance_check(out[k], oracle.xengine_cf32(x), w.n_inputs)


def test_abi_errors_on_device(pkg):
    L = pkg.lib()
    h = pkg.corr_create(64, 2, 10, "ci8")
    good = torch.zeros(h.in_bytes + 64, dtype=torch.int8, device="cuda")
    vis = h.empty_vis()
    assert L.corr_xengine(h._h, None, vis.data_ptr(), None) == pkg.CORR_EINVAL
    assert L.corr_xengine(h._h, good.data_ptr() + 1, vis.data_ptr(), None) == pkg.CORR_EINVAL
    assert L.corr_xengine(None, good.data_ptr(), vis.data_ptr(), None) == pkg.CORR_EINVAL
    assert L.corr_xengine(h._h, good.data_ptr(), good.data_ptr(), None) == pkg.CORR_EINVAL
    assert b"corr_xengine" in L.corr_last_error()
    pkg.corr_destroy(h)
    for bad in [(48, 2, 10, "ci8"), (64, 2, 70000, "ci8"), (0, 1, 1, "ci8"), (64, 1, 1, 7)]:
        with pytest.raises(pkg.CorrError):
            pkg.corr_create(*bad)
    assert L.corr_destroy(None) == pkg.CORR_OK


def test_mma_probe_runs_at_the_tensor_rate(pkg):
    """corr_probe_mma: one thread per SM issues M=128,N=256,K=32 int8 MMAs back to back; the tensor pipe needs
    128 cycles for each (8192 MACs per cycle per SM), MN-major operands included."""
    r = pkg.probe_mma(128, 256, True, 8192, random_fill=True)
    assert 120.0 <= r["cycles_per_mma"] <= 150.0, r
    assert r["tops"] > 3000.0, r


# Every plan of the diag schedule (N_I <= 64): gsize adjacent panels per item x time slices.  Small inputs
# default to whole integrations of 1-2 panels; "4,s" is what the large configs (c2) run, incl. the reduce-add path.
@pytest.mark.parametrize("plan", ["4,1", "4,3", "2,1", "2,2", "1,1", "1,4"])
@pytest.mark.parametrize("N,C,T", [(64, 11, 700), (32, 13, 530), (64, 1, 129)])
def test_ci8_diag_plans_bit_exact(pkg, plan, N, C, T):
    g, sl = (int(v) for v in plan.split(","))
    w = corrgen.scaled(corrgen.CONFIGS["c2"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    out = run_ci8(pkg, x, options=[(pkg.CORR_OPT_DIAG_PLAN, 256 * g + sl)])
    assert np.array_equal(out, oracle.xengine_ci8(x, threads=_threads()))


# Mixed plans (inputs > 64 MB with more panel groups than SMs): a x 148 groups run as whole integrations with plain
# stores, the left-over groups as time slices that reduce-add into their zeroed channels -- in ONE launch.
@pytest.mark.parametrize("N,C,T,mix", [(64, 700, 800, 1), (32, 1300, 900, 1), (64, 700, 800, 0)])
def test_ci8_mixed_whole_and_sliced_groups_bit_exact(pkg, N, C, T, mix):
    w = corrgen.scaled(corrgen.CONFIGS["c2"], n_inputs=N, n_chan=C, n_time=T)
    x = w.generate()
    out = run_ci8(pkg, x, options=[(pkg.CORR_OPT_MIX, mix)])
    assert np.array_equal(out, oracle.xengine_ci8(x, threads=_threads()))


def test_set_option_rejects_bad_arguments(pkg):
    h = pkg.corr_create(64, 2, 100, "ci8")
    for key, value in [(99, 1), (pkg.CORR_OPT_DIAG_PLAN, 256 * 3 + 1), (pkg.CORR_OPT_DIAG_PLAN, 256 * 4 + 65), (pkg.CORR_OPT_UNITS, -1)]:
        with pytest.raises(pkg.CorrError) as e:
            h.set_option(key, value)
        assert e.value.status == pkg.CORR_EINVAL
    pkg.corr_destroy(h)


# N_I = 64 float path (xengine_f32_n64_kernel: 7-channel groups, time slices with reduce-add): group tails (C not a
# multiple of 7), slice tails, one slice (plain stores) and many; and the generic 4 x 4 kernel forced on the same shapes.
@pytest.mark.parametrize("generic", [False, True])
# (1100, 70) and (1040, 16): more groups than SMs -- whole groups with plain stores plus sliced left-over groups in one launch
@pytest.mark.parametrize("C,T", [(1, 1), (7, 16), (8, 17), (15, 100), (150, 33), (23, 700), (300, 260), (1100, 70), (1040, 16)])
def test_cf32_n64_paths_within_tolerance(pkg, generic, C, T):
    w = corrgen.scaled(corrgen.CONFIGS["c5"], n_inputs=64, n_chan=C, n_time=T)
    x = w.generate()
    out = run_cf32(pkg, x, options=[(pkg.CORR_OPT_F32_GENERIC, 1)] if generic else ())
    f32_tolerance_check(out, oracle.xengine_cf32(x, threads=_threads()), 64)


def test_ci8_cuda_graph_with_dependent_launches(pkg):
    """Calls captured into a CUDA graph launch programmatically (the next kernel may start while the preceding one
    drains): results must not depend on it -- the same d_vis written by consecutive calls (write after write), and an
    input produced by the preceding kernel of the stream (standalone corner turn -> X-engine)."""
    w = corrgen.scaled(corrgen.CONFIGS["c1"], n_chan=24, n_time=300)
    xs = [w.generate(integration=k) for k in range(3)]
    refs = [oracle.xengine_ci8(x, threads=_threads()) for x in xs]
    h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, "ci8")
    ht = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, "ci8")
    ht.set_turn(pkg.CORR_TURN_STANDALONE)
    d = [torch.from_numpy(x).cuda() for x in xs]
    va, vb, vc = h.empty_vis(), h.empty_vis(), h.empty_vis()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        h.xengine(d[0], va, s)
        ht.xengine(d[2], vc, s)   # warm-up outside the capture (allocates the turn scratch)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            h.xengine(d[0], va, s)
            h.xengine(d[1], va, s)     # same output buffer as the call before
            h.xengine(d[2], vb, s)
            ht.xengine(d[0], vc, s)    # corner-turn kernel, then the X-engine on its output
        for buf in (va, vb, vc):
            buf.fill_(-0x55555555)
        g.replay()
        g.replay()
        torch.cuda.synchronize()
    assert np.array_equal(va.cpu().numpy(), refs[1])
    assert np.array_equal(vb.cpu().numpy(), refs[2])
    assert np.array_equal(vc.cpu().numpy(), refs[0])
    del g
    pkg.corr_destroy(h)
    pkg.corr_destroy(ht)
