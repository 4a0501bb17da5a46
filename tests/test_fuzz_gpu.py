"""Seeded random shapes, plan options, batch sizes and channel windows through the C ABI, each checked element by element
against the CPU oracle.  plan_i8 / plan_f32 choose among many schedule families from modelled times and thresholds; the
hand-picked shapes of the parity tests sit on the thresholds known when they were written, this file walks across them
(N_I 32..4096, T including 1, 31..33, 1025..2047, >= 2048 and the int8 limit 65535, ragged channel counts, every legal
corr_set_option combination).  The case list is a pure function of the seed below, so a failure reproduces by its index.

Outputs are poison-filled before the call; channels are compared in a random contiguous block sized so that the oracle
needs a fraction of a second (the whole cube when it is small), and no element anywhere may still hold the poison."""
from __future__ import annotations

import numpy as np
import pytest

import corrgen
import oracle
from parity_util import f32_tolerance_check

torch = pytest.importorskip("torch")

SEED = 20261106
N_CASES = 96
POISON = -0x55555555
CHECK_CMACS = 2.5e8          # oracle work per case, about 0.1 s on a 16-core host


@pytest.fixture(scope="module")
def pkg():
    import paper_0906_1887_b200 as p
    p.lib()
    return p


def _cases():
    rng = np.random.default_rng(SEED)
    out = []
    for k in range(N_CASES):
        dtype = rng.choice(["ci8", "ci8", "ci8", "ci4", "cf32"])
        r = rng.random()
        if dtype == "cf32":
            N = 32 * int(rng.integers(1, 9)) if r < 0.6 else 32 * int(rng.integers(8, 33))       # <= 256 | 256..1024
        elif r < 0.55:
            N = 32 * int(rng.integers(1, 17))                                                     # 32..512
        elif r < 0.9:
            N = 32 * int(rng.integers(17, 41))                                                    # 544..1280
        else:
            N = 32 * int(rng.integers(41, 129))                                                   # 1312..4096
        t_class = int(rng.integers(0, 8))
        T = [1, 31, 32, 33, int(rng.integers(34, 1025)), int(rng.integers(1025, 2048)), int(rng.integers(2048, 4300)),
             int(rng.integers(34, 400))][t_class]
        if dtype == "cf32":
            T = min(T, 600)
        nb = N * (N + 1) // 2
        sample = {"ci8": 2, "ci4": 1, "cf32": 8}[dtype]
        c_max = max(1, min(int(48e6 // (T * N * sample)), int(64e6 // (nb * 8)), 300))          # input <= 48 MB, output <= 64 MB
        C = int(rng.integers(1, c_max + 1))
        # a few regimes are too rare to leave to chance: inputs > 64 MB at N_I <= 64 (the large-input branch of the planner)
        # and integrations at the int32-safe limit
        if k in (5, 29, 53):
            dtype, N, T, C = "ci8", (64, 32, 64)[k // 24], int(rng.integers(2500, 4000)), int(rng.integers(300, 420))
        if k in (7, 31):
            dtype, N, T, C = ("ci8", "ci4")[k // 24], (64, 32)[k // 24], int(rng.integers(60000, 65536)), int(rng.integers(1, 4))
        opts = []
        if dtype != "cf32":
            for name, values in (("CORR_OPT_PAIRS", (0, 1, 2)), ("CORR_OPT_WIDE", (0, 1, 2)), ("CORR_OPT_RESIDENT", (0, 1, 2)),
                                 ("CORR_OPT_MIX", (0, 1)), ("CORR_OPT_COLLECT", (0, 1)), ("CORR_OPT_PDL", (0, 1, 2)),
                                 ("CORR_OPT_UNITS", (0, 7, 40))):
                if rng.random() < 0.3:
                    opts.append((name, int(rng.choice(values))))
            if N <= 64 and rng.random() < 0.4:
                opts.append(("CORR_OPT_DIAG_PLAN", 256 * int(rng.choice([1, 2, 4])) + int(rng.choice([0, 1, 2, 3, 5]))))
        elif rng.random() < 0.3:
            opts.append(("CORR_OPT_F32_GENERIC", 1))
        window = None
        if rng.random() < 0.2 and C >= 2:
            cw = int(rng.integers(1, C))
            window = (int(rng.integers(0, C - cw + 1)), cw)                                       # (chan0, channels owned)
        n_batch = 1
        if dtype == "ci8" and window is None and T * C * N * 2 <= (1 << 20) and rng.random() < 0.5:
            n_batch = int(rng.integers(2, 71))
        turn = bool(dtype == "ci8" and window is None and n_batch == 1 and rng.random() < 0.15 and not (N == 32 and C % 2))
        out.append(dict(k=k, dtype=dtype, N=N, C=C, T=T, opts=opts, window=window, n_batch=n_batch, turn=turn))
    return out


CASES = _cases()


def _generate(c, seed):
    if c["dtype"] == "cf32":
        return corrgen.gauss_f32(c["T"], c["C"], c["N"], seed, 0.70710678, tone_amp=0.5)
    if c["dtype"] == "ci4":
        return corrgen.uniform_i8(c["T"], c["C"], c["N"], seed, 7)
    return corrgen.uniform_i8(c["T"], c["C"], c["N"], seed, 127)


def _oracle(c, x, c0, c1):
    th = oracle.host_threads()
    if c["dtype"] == "cf32":
        return oracle.xengine_cf32(x, c0, c1, threads=th)
    if c["dtype"] == "ci4":
        return oracle.xengine_ci4(corrgen.pack_ci4(x), c0, c1, threads=th)
    return oracle.xengine_ci8(x, c0, c1, threads=th)


def _compare(c, got, x, chan0, rng):
    """got: [Cw][nb][2] of the handle's channels chan0 .. chan0 + Cw - 1 of cube x."""
    Cw = got.shape[0]
    if c["dtype"] == "cf32":
        assert not np.isnan(got).any(), "an output element was never written"
    else:
        assert not (got == POISON).any(), "an output element was never written"
    n_check = int(max(1, min(Cw, CHECK_CMACS // (c["T"] * c["N"] * (c["N"] + 1) // 2 + 1))))
    blocks = {int(rng.integers(0, Cw - n_check + 1)), Cw - n_check}              # a random block and the one that ends the cube
    for b0 in sorted(blocks):
        want = _oracle(c, x, chan0 + b0, chan0 + b0 + n_check)
        if c["dtype"] == "cf32":
            f32_tolerance_check(got[b0:b0 + n_check], want, c["N"], rel=1e-5)
        else:
            assert np.array_equal(got[b0:b0 + n_check], want), f"channels {b0}..{b0 + n_check - 1}"


@pytest.mark.gpu
@pytest.mark.parametrize("c", CASES, ids=lambda c: f"{c['k']}-{c['dtype']}-N{c['N']}-C{c['C']}-T{c['T']}")
def test_random_case_matches_the_oracle(pkg, c):
    rng = np.random.default_rng(SEED + 1 + c["k"])
    chan0, Cw = c["window"] if c["window"] else (0, c["C"])
    h = pkg.corr_create(c["N"], Cw, c["T"], c["dtype"])
    try:
        for name, value in c["opts"]:
            h.set_option(getattr(pkg, name), value)
        if c["window"]:
            h.set_chan_window(c["C"], chan0)
        if c["turn"]:
            h.set_turn(pkg.CORR_TURN_STANDALONE)
        fill = float("nan") if c["dtype"] == "cf32" else POISON
        if c["n_batch"] == 1:
            x = _generate(c, seed=c["k"])
            d_in = torch.from_numpy(corrgen.pack_ci4(x) if c["dtype"] == "ci4" else x).cuda()
            vis = h.empty_vis()
            vis.fill_(fill)
            pkg.corr_xengine(h, d_in, vis)
            torch.cuda.synchronize()
            _compare(c, vis.cpu().numpy(), x, chan0, rng)
        else:
            xs = [_generate(c, seed=1000 * c["k"] + b) for b in range(c["n_batch"])]
            d_in = [torch.from_numpy(x).cuda() for x in xs]
            d_vis = [h.empty_vis() for _ in xs]
            for v in d_vis:
                v.fill_(fill)
            pkg.corr_xengine_batch(h, d_in, d_vis)
            torch.cuda.synchronize()
            for b in {0, c["n_batch"] - 1, int(rng.integers(0, c["n_batch"]))}:
                _compare(c, d_vis[b].cpu().numpy(), xs[b], 0, rng)
    finally:
        pkg.corr_destroy(h)


def test_the_case_list_spans_the_plan_families():
    """The generator above is only useful if it reaches every regime; this pins that (no GPU work)."""
    ci8 = [c for c in CASES if c["dtype"] == "ci8"]
    assert len(CASES) >= 80 and len(ci8) >= 40
    assert {c["dtype"] for c in CASES} == {"ci8", "ci4", "cf32"}
    assert any(c["N"] <= 64 for c in ci8) and any(128 <= c["N"] < 512 for c in ci8) and any(c["N"] >= 512 for c in ci8)
    assert any(c["N"] > 2048 for c in CASES if c["dtype"] != "cf32")
    assert any(c["N"] >= 256 for c in CASES if c["dtype"] == "cf32")
    for lo, hi in ((1, 1), (31, 33), (1025, 2047), (2048, 65535), (60000, 65535)):
        assert any(lo <= c["T"] <= hi for c in CASES if c["dtype"] != "cf32"), (lo, hi)
    assert any(c["n_batch"] > 64 for c in CASES) and any(c["window"] for c in CASES) and any(c["turn"] for c in CASES)
    assert any(c["T"] * c["C"] * c["N"] * 2 > (64 << 20) for c in ci8)
