"""Seeded generators: determinism, ranges, shapes (no method arithmetic in synth).  -m "not gpu" """
import numpy as np

from inputs import synth


def test_image_recipe():
    a = synth.make_image(128, 1001)
    b = synth.make_image(128, 1001)
    assert np.array_equal(a, b) and a.dtype == np.complex128 and a.shape == (128, 128)
    assert np.all(a.imag == 0) and a.real.max() > 0.5
    assert np.count_nonzero(a) <= 20 + 3 * (2 * 24 + 3) ** 2
    assert not np.array_equal(a, synth.make_image(128, 1002))


def test_uv_gaussian_truncation_and_dtype():
    for cfg_i, M in [(1, 10_000), (2, 50_000), (4, 200_000)]:
        cfg = synth.CONFIGS[cfg_i]
        uv = synth.make_uv(cfg, M)
        assert uv.shape == (M, 2) and uv.dtype == synth.real_dtype(cfg.dtype)
        assert np.abs(uv).max() < cfg.K / 2 - cfg.J
        assert abs(uv.std() / (cfg.K / cfg.sigma_div) - 1) < 0.1
        assert np.array_equal(uv, synth.make_uv(cfg, M))


def test_rotation_synthesis_tracks():
    cfg = synth.CONFIGS[3]
    uv = synth.make_uv(cfg, 200_000)
    assert uv.dtype == np.float32 and np.abs(uv).max() <= 0.8 * cfg.K / 2 * 1.0001
    # 27 antennas -> 351 baselines x 10 channels per time step, time-major
    assert len(synth._antennas_y27()) == 27
    cfg5 = synth.CONFIGS[5]
    assert len(synth._antennas_ska197(cfg5.seed)) == 197
    uv5 = synth.make_uv(cfg5, 300_000)
    assert np.abs(uv5).max() <= 0.8 * cfg5.K / 2 * 1.0001
    w = synth.make_weights(cfg, 1000)
    assert w.dtype == np.float32 and 0.5 <= w.min() and w.max() <= 1.5


def test_full_track_lengths_cover_the_configs():
    """351 x 2880 x 10 >= 1e7 and 19306 x 2880 x 9 >= 5e8."""
    assert 27 * 26 // 2 * 2880 * 10 >= synth.CONFIGS[3].M
    assert 197 * 196 // 2 * 2880 * 9 >= synth.CONFIGS[5].M


def test_noise_level():
    rng = synth.rng_for(1, 1)
    y = rng.standard_normal(20000) + 1j * rng.standard_normal(20000)
    yn = synth.add_noise(y, 30.0, 5)
    assert abs(np.linalg.norm(yn - y) / np.linalg.norm(y) / 10 ** (-1.5) - 1) < 0.03
