"""The C generator (corrgen/gen.c) against its numpy mirror and its stated recipe."""
import numpy as np
import pytest

import corrgen


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4"])
def test_c_matches_numpy_int8(name):
    w = corrgen.scaled(corrgen.CONFIGS[name], n_time=37, n_chan=5, n_inputs=8)
    got = w.generate()
    if w.kind == "uniform":
        want = corrgen.uniform_i8_numpy(37, 5, 8, w.seed, w.clip)
    else:
        want = corrgen.gauss_i8_numpy(37, 5, 8, w.seed, w.sigma, w.clip, w.tone_amp)
    assert got.dtype == np.int8 and got.shape == (37, 5, 8, 2)
    assert np.array_equal(got, want)
    assert got.min() >= -w.clip and got.max() <= w.clip


def test_c_matches_numpy_f32():
    w = corrgen.scaled(corrgen.CONFIGS["c5"], n_time=29, n_chan=4, n_inputs=8)
    got = w.generate(integration=2)
    want = corrgen.gauss_f32_numpy(29, 4, 8, w.seed + 2 * 1000003, w.sigma, w.tone_amp)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-6)


def test_counter_based_slices_and_threads():
    """Any time range regenerates on its own; thread count changes nothing."""
    w = corrgen.scaled(corrgen.CONFIGS["c2"], n_time=64, n_chan=3, n_inputs=4)
    whole = w.generate(threads=1)
    assert np.array_equal(w.generate(threads=4), whole)
    assert np.array_equal(w.generate(t_begin=10, t_end=33), whole[10:33])


def test_distinct_integrations_and_seeds():
    w = corrgen.scaled(corrgen.CONFIGS["c5"], n_time=16, n_chan=2, n_inputs=4)
    assert not np.array_equal(w.generate(0), w.generate(1))
    assert np.array_equal(w.generate(1), w.generate(1))


def test_moments():
    w = corrgen.scaled(corrgen.CONFIGS["c1"], n_time=512, n_chan=8, n_inputs=32)
    x = w.generate().astype(np.float64)
    assert abs(x.mean()) < 0.05
    assert 2.7 < x.std() < 3.1          # sigma 3 clipped at +-7
    u = corrgen.scaled(corrgen.CONFIGS["c3"], n_time=256, n_chan=4, n_inputs=32).generate()
    assert u.min() == -127 and u.max() == 127 and abs(u.astype(np.float64).mean()) < 1.5
    f = corrgen.scaled(corrgen.CONFIGS["c5"], n_time=256, n_chan=16, n_inputs=16, tone_amp=0.0).generate()
    power = (f.astype(np.float64) ** 2).sum(axis=-1).mean()
    assert 0.97 < power < 1.03          # CN(0,1): total variance 1


def test_config_table_matches_baseline():
    c = corrgen.CONFIGS
    assert (c["c1"].n_inputs, c["c1"].n_chan, c["c1"].n_time) == (32, 128, 1000)
    assert (c["c2"].n_inputs, c["c2"].n_chan, c["c2"].n_time) == (64, 768, 10000)
    assert (c["c3"].n_inputs, c["c3"].n_chan, c["c3"].n_time) == (256, 512, 4000)
    assert (c["c4"].n_inputs, c["c4"].n_chan, c["c4"].n_time) == (1024, 128, 1000)
    assert (c["c5"].n_inputs, c["c5"].n_chan, c["c5"].n_time, c["c5"].n_integrations) == (64, 1536, 500, 20)
    assert c["c2"].in_bytes == 983040000 and c["c2"].cmacs == 10000 * 768 * 2080
    assert c["c4"].vis_bytes == 537395200
