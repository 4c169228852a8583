"""GPU parity: hand-written 3-D r2c / c2r (libfpm) vs the float64 oracle.

Tolerance: relative L2 <= 1e-5 is the north_star bound on density and forces; a float32 FFT of
N <= 1024 points per axis has relative L2 error ~ 1e-7 sqrt(log2 N^3), so 2e-6 is asserted here.
"""
import numpy as np
import pytest

from gpu_util import dev, host, rel_l2

pytestmark = pytest.mark.gpu
TOL = 2e-6


@pytest.fixture(scope="module")
def fpm():
    import paper_2010_11847_b200 as fpm
    return fpm


@pytest.mark.parametrize("ng", [8, 16, 32, 64, 128, 256])
def test_r2c_and_c2r_match_oracle(fpm, oracle, ng):
    rng = np.random.default_rng(ng)
    rho = (rng.standard_normal((ng, ng, ng)) + 1.0).astype(np.float32)
    ctx = fpm.FPM(ng, workspace=False)
    got = host(ctx.fft_r2c(dev(rho)))
    ref = oracle.fft_r2c(rho.astype(np.float64))
    assert got.shape == (ng, ng, ng // 2 + 1)
    assert rel_l2(got, ref) < TOL
    assert np.max(np.abs(got - ref)) < 1e-5 * np.max(np.abs(ref))
    # inverse on a Hermitian spectrum (fp32-rounded oracle spectrum)
    spec = ref.astype(np.complex64)
    back = host(ctx.fft_c2r(dev(spec)))
    ref_back = oracle.fft_c2r(spec.astype(np.complex128))
    assert rel_l2(back, ref_back) < TOL
    # round trip
    rt = host(ctx.fft_c2r(ctx.fft_r2c(dev(rho)), clobber=True))
    assert rel_l2(rt, rho) < TOL


@pytest.mark.parametrize("ng", [16, 64])
def test_c2r_of_a_non_hermitian_spectrum_follows_the_stated_contract(fpm, oracle, ng):
    """include/fpm.h, fpm_fft_c2r: on a spectrum whose kz = 0 / Nyquist planes are not Hermitian the result is
    the real part of the inverse of the conjugate-completed spectrum -- what the oracle computes (pinned
    against numpy.fft.ifftn in tests/test_oracle_fft.py)."""
    rng = np.random.default_rng(ng + 1)
    spec = (rng.standard_normal((ng, ng, ng // 2 + 1)) + 1j * rng.standard_normal((ng, ng, ng // 2 + 1))).astype(np.complex64)
    ctx = fpm.FPM(ng, workspace=False)
    got = host(ctx.fft_c2r(dev(spec)))
    ref = oracle.fft_c2r(spec.astype(np.complex128))
    assert rel_l2(got, ref) < TOL
    assert np.max(np.abs(got - ref)) < 1e-5 * np.max(np.abs(ref))


def test_delta_and_plane_wave_closed_forms(fpm):
    ng = 64
    ctx = fpm.FPM(ng, workspace=False)
    rho = np.zeros((ng, ng, ng), dtype=np.float32)
    rho[0, 0, 0] = 1.0
    got = host(ctx.fft_r2c(dev(rho)))
    assert np.max(np.abs(got - 1.0)) < 1e-6
    x = np.arange(ng)
    rho = np.cos(2 * np.pi * (3 * x[:, None, None] + 5 * x[None, :, None] + 7 * x[None, None, :]) / ng).astype(np.float32)
    got = host(ctx.fft_r2c(dev(rho)))
    expect = np.zeros_like(got)
    expect[3, 5, 7] = ng ** 3 / 2
    assert np.max(np.abs(got - expect)) < 2e-6 * ng ** 3


@pytest.mark.parametrize("ng", [512, 1024])
def test_full_size_sampled_outputs_and_roundtrip(fpm, ng):
    """At the bench sizes (C4: 512, C5: 1024 -- Plan<1024>, the 128 KB column tiles and the M = 512 z pass)
    the oracle computes sampled output bins one by one (direct DFT sums)."""
    import torch
    rng = np.random.default_rng(1)
    rho = rng.standard_normal((ng, ng, ng), dtype=np.float32)
    ctx = fpm.FPM(ng, workspace=False)
    d_rho = dev(rho)
    spec = ctx.fft_r2c(d_rho)
    x = np.arange(ng)
    r64 = rho.astype(np.float64)
    scale = np.sqrt(ng ** 3)
    h = ng // 2
    for (a, b, c) in [(0, 0, 0), (1, 2, 3), (ng - 1, h, h), (h + 1, 13, 0), (100, 300, 77), (h, h, h)]:
        ea = np.exp(-2j * np.pi * a * x / ng)
        eb = np.exp(-2j * np.pi * b * x / ng)
        ec = np.exp(-2j * np.pi * c * x / ng)
        ref = np.einsum("x,y,z,xyz->", ea, eb, ec, r64, optimize=True)
        got = complex(spec[a, b, c].item())
        assert abs(got - ref) < 2e-5 * scale
    back = ctx.fft_c2r(spec, clobber=True)
    err = torch.linalg.vector_norm(back - d_rho) / torch.linalg.vector_norm(d_rho)
    assert err.item() < TOL
