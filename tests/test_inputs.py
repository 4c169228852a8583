"""Pins for the seeded input generators: Eisenstein-Hu no-wiggle numbers,
sigma8 normalisation, and statistics of the counter-based Gaussian field."""
import numpy as np
import pytest

import fpm_inputs as fi


def test_eisenstein_hu_nowiggle_numbers():
    s, alpha = fi.eh_sound_horizon_and_alpha()
    assert s == pytest.approx(150.375, abs=1e-3)
    assert alpha == pytest.approx(0.79793, abs=1e-5)
    t = fi.eh_nowiggle_transfer([1e-6, 0.01, 0.1, 1.0])
    assert t[0] == pytest.approx(1.0, abs=1e-4)
    assert t[1:] == pytest.approx([0.784518, 0.132328, 0.004608], abs=2e-6)
    assert fi.sigma_r(8.0, fi.power_amplitude()) == pytest.approx(0.8159, rel=1e-12)
    assert fi.linear_power([0.1, 0.02]) == pytest.approx([5838.28, 23951.99], rel=1e-5)
    assert fi.linear_power(0.0) == 0.0


def test_counter_generator_is_size_independent_and_normal():
    a = fi.counter_normal(1, np.arange(1000, dtype=np.uint64))
    b = fi.counter_normal(1, np.arange(200000, dtype=np.uint64))
    assert np.array_equal(a, b[:1000])
    assert not np.array_equal(a, fi.counter_normal(2, np.arange(1000, dtype=np.uint64)))
    assert abs(b.mean()) < 4 / np.sqrt(b.size)
    assert b.var() == pytest.approx(1.0, abs=0.02)
    assert np.mean(b ** 4) == pytest.approx(3.0, abs=0.15)
    u = fi.counter_uniform(3, np.arange(100000, dtype=np.uint64))
    assert 0 < u.min() and u.max() < 1 and u.mean() == pytest.approx(0.5, abs=0.01)


def test_linear_field_variance_matches_the_mode_sum():
    n, box = 32, 100.0
    d = fi.linear_field(n, box, seed=1)
    assert d.dtype == np.float32 and d.shape == (n, n, n)
    assert abs(float(d.mean())) < 1e-6
    f = np.fft.fftfreq(n, 1.0 / n)
    k = 2 * np.pi / box * np.sqrt(f[:, None, None] ** 2 + f[None, :, None] ** 2 + f[None, None, :] ** 2)
    expect = fi.linear_power(k).sum() / box ** 3
    assert float(d.astype(np.float64).var()) == pytest.approx(expect, rel=0.05)
    assert np.array_equal(d, fi.linear_field(n, box, seed=1))


def test_configs_match_baseline_json():
    c = fi.CONFIGS
    assert (c["C1"].np_side, c["C1"].ng, c["C1"].box, c["C1"].lpt_order, c["C1"].n_steps) == (32, 32, 100.0, 1, 5)
    assert (c["C3"].np_side, c["C3"].ng, c["C3"].resolution_factor) == (256, 512, 2)
    assert (c["C4"].np_side, c["C4"].n_steps, c["C4"].backward) == (512, 40, True)
    assert c["C5"].n_particles == 1024 ** 3
    st = c["C2"].stages()
    assert len(st) == 11 and st[0] == 0.1 and st[-1] == pytest.approx(1.0)


def test_random_particles_in_range():
    for cl in (False, True):
        p = fi.random_particles(5000, 32, 7, clustered=cl)
        assert p.dtype == np.float32 and p.shape == (3, 5000)
        assert p.min() >= 0 and p.max() < 32
