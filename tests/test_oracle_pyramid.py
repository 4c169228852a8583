"""Pins of the multi-grid pyramid oracle (Eq. 6-9, Alg. 2-3 PAPER.md:247-305;
DESIGN.md reading R14: the order-6 B-spline two-scale mask [1, 6, 15, 20, 15, 6, 1]/64 per axis)."""
import numpy as np
import pytest
import scipy.ndimage as ndi

import fpm_inputs as fi

OM = 0.3075
H1 = np.array([1, 6, 15, 20, 15, 6, 1], dtype=np.float64) / 64.0


def test_reduce_of_a_plane_wave_is_the_closed_form_filter_response(oracle):
    """Stride-2 convolution of exp(i w.x) with h (x) h (x) h: amplitude prod_d cos^6(w_d / 2) (the symbol of the
    binomial mask), sampled at 2 X.  Fails on a shifted or mis-normalised kernel or a wrong stride."""
    n = 16
    x = np.arange(n)
    for (a, b, c) in [(1, 0, 0), (0, 2, 0), (1, 2, 3), (3, 3, 1)]:
        w = 2 * np.pi * np.array([a, b, c]) / n
        field = np.cos(w[0] * x[:, None, None] + w[1] * x[None, :, None] + w[2] * x[None, None, :] + 0.3)
        amp = np.prod(np.cos(w / 2) ** 6)
        X = 2 * np.arange(n // 2)
        expect = amp * np.cos(w[0] * X[:, None, None] + w[1] * X[None, :, None] + w[2] * X[None, None, :] + 0.3)
        assert np.max(np.abs(oracle.reduce(field, 1) - expect)) < 1e-14


def test_reduce_equals_a_library_convolution_then_subsampling(oracle):
    rng = np.random.default_rng(1)
    field = rng.standard_normal((16, 16, 16))
    k3 = H1[:, None, None] * H1[None, :, None] * H1[None, None, :]
    lib = ndi.convolve(field, k3, mode="wrap")[::2, ::2, ::2]       # symmetric kernel: correlation = convolution
    assert np.max(np.abs(oracle.reduce(field, 1) - lib)) < 1e-14
    lib2 = ndi.convolve(lib, k3, mode="wrap")[::2, ::2, ::2]
    assert np.max(np.abs(oracle.reduce(field, 2) - lib2)) < 1e-14     # Alg. 2: f = 2 consecutive passes


def test_reduce_keeps_the_mean_and_expand_keeps_a_constant(oracle):
    rng = np.random.default_rng(2)
    field = rng.standard_normal((16, 16, 16)) + 3.0
    assert oracle.reduce(field, 2).mean() == pytest.approx(field.mean(), rel=1e-13)
    up = oracle.expand(np.full((4, 4, 4), 2.5), 2)
    assert up.shape == (16, 16, 16) and np.max(np.abs(up - 2.5)) < 1e-14       # both polyphases of 2h sum to 1
    assert oracle.expand(field[:8, :8, :8], 1).mean() == pytest.approx(field[:8, :8, :8].mean(), rel=1e-13)


def test_expand_is_eight_times_the_transpose_of_reduce(oracle):
    """TransposedConv3D with 8 K (Alg. 2): <REDUCE a, b> = <a, EXPAND b> / 8^f."""
    rng = np.random.default_rng(3)
    for f in (1, 2):
        a = rng.standard_normal((16, 16, 16))
        b = rng.standard_normal((16 >> f,) * 3)
        lhs = np.sum(oracle.reduce(a, f) * b)
        rhs = np.sum(a * oracle.expand(b, f)) / 8.0 ** f
        assert lhs == pytest.approx(rhs, rel=1e-12)


def test_expand_of_a_coarse_plane_wave(oracle):
    """Zero insertion doubles the spectrum (w and w + pi), the mask 2h weighs the two images by cos^6(w/2) and
    sin^6(w/2): EXPAND(cos(2 w X)) = cos^6(w/2) cos(w x) + sin^6(w/2) cos((w + pi) x) along one axis."""
    m = 8
    X = np.arange(m)
    k = 1
    w = 2 * np.pi * k / (2 * m)                           # fine-grid frequency of the coarse wave
    coarse = np.cos(2 * w * X)[:, None, None] * np.ones((m, m, m))
    x = np.arange(2 * m)
    expect = (np.cos(w / 2) ** 6 * np.cos(w * x) + np.sin(w / 2) ** 6 * np.cos((w + np.pi) * x))[:, None, None] * np.ones((2 * m,) * 3)
    assert np.max(np.abs(oracle.expand(coarse, 1) - expect)) < 1e-14


def test_laplacian_pyramid_reconstructs_exactly(oracle):
    """Eq. 8-9: g_l = L_l + EXPAND(g_{l+1}) recovers g_0 from (L_0, L_1, g_2) -- 'the negligible
    residuals show that the reconstruction of the fields is exact'."""
    rng = np.random.default_rng(4)
    g0 = rng.standard_normal((16, 16, 16))
    g1 = oracle.reduce(g0, 1)
    g2 = oracle.reduce(g1, 1)
    L0 = g0 - oracle.expand(g1, 1)
    L1 = g1 - oracle.expand(g2, 1)
    r1 = L1 + oracle.expand(g2, 1)
    r0 = L0 + oracle.expand(r1, 1)
    assert np.max(np.abs(r0 - g0)) < 1e-14
    assert np.max(np.abs(oracle.reduce(g0, 2) - g2)) == 0.0


def test_pyramid_force_with_zero_levels_is_the_single_grid_force(oracle):
    rho = 1.0 + 0.1 * fi.linear_field(8, 50.0, seed=2).astype(np.float64)
    single = oracle.force_grids(rho, scale=1.5 * OM)
    pyr = oracle.force_grids_pyramid(rho, levels=0, scale=1.5 * OM)
    for d in range(3):
        assert np.max(np.abs(pyr[d] - single[d])) < 1e-13 * np.max(np.abs(single[d]))


@pytest.mark.parametrize("levels", [1, 2])
def test_pyramid_force_is_close_to_the_single_grid_force(oracle, levels):
    """PAPER.md:313 / Fig. 6-7: 'the pyramid implementation shows higher residuals than the single mesh
    implementation, but they are sub-percent'.  With the exact symbols (-1/k^2, ik: FPM_KERNEL_NAIVE) the coarse
    and the fine mesh solve the same continuum problem and only the mask's aliasing separates them: 0.1 %.  With
    the finite-difference symbols of Eq. 4-5 the coarse mesh has 2^f times the discretisation step, which shows
    up at the per-cent level on a 32^3 mesh.  Also pins the units reading (coarse force x 2^f): without the
    factor the long-range part would be off by 2^f and the error of order one."""
    cfg = fi.CONFIGS["C1"]
    delta = fi.linear_field(cfg.np_side, cfg.box, cfg.seed).astype(np.float64)
    pos, _ = oracle.lpt_init(delta, cfg.ng, OM, 0.5, 1)          # a moderately evolved particle set
    rho = oracle.paint(pos, cfg.ng)
    for mode, tol in ((1, 3e-3), (0, 5e-2)):
        single = oracle.force_grids(rho, mode=mode, scale=1.5 * OM)
        pyr = oracle.force_grids_pyramid(rho, levels=levels, mode=mode, scale=1.5 * OM)
        num = sum(np.sum((pyr[d] - single[d]) ** 2) for d in range(3))
        den = sum(np.sum(single[d] ** 2) for d in range(3))
        assert np.sqrt(num / den) < tol, (mode, np.sqrt(num / den))
    f_single = oracle.force(pos, cfg.ng, mode=1, scale=1.5 * OM)
    f_pyr = oracle.force_pyramid(pos, cfg.ng, levels=levels, mode=1, scale=1.5 * OM)
    assert np.linalg.norm(f_pyr - f_single) / np.linalg.norm(f_single) < 3e-3
