"""Pins for the oracle's FFT: brute-force DFT on tiny grids, the library
transform on larger ones, closed forms (delta, cosine), Parseval, round trip."""
import numpy as np
import pytest


def brute_dft3(rho):
    """delta_hat(k) = sum_x rho(x) exp(-2 pi i n.x/ng), written as three dense DFT matrices."""
    ng = rho.shape[0]
    j = np.arange(ng)
    w = np.exp(-2j * np.pi * np.outer(j, j) / ng)
    full = np.einsum("ax,by,cz,xyz->abc", w, w, w, rho.astype(np.complex128))
    return full[:, :, : ng // 2 + 1]


@pytest.mark.parametrize("ng", [2, 4, 8])
def test_r2c_equals_brute_force_dft(oracle, ng):
    rng = np.random.default_rng(ng)
    rho = rng.standard_normal((ng, ng, ng))
    ref = brute_dft3(rho)
    assert np.max(np.abs(oracle.fft_r2c(rho) - ref)) <= 1e-12 * np.max(np.abs(ref))


@pytest.mark.parametrize("ng", [16, 32])
def test_radix2_equals_naive_and_library(oracle, ng):
    rng = np.random.default_rng(100 + ng)
    rho = rng.standard_normal((ng, ng, ng))
    fast = oracle.fft_r2c(rho)
    lib = np.fft.rfftn(rho)
    assert np.max(np.abs(fast - lib)) <= 1e-12 * np.max(np.abs(lib))
    if ng == 16:
        naive = oracle.fft_r2c(rho, force_naive=True)
        assert np.max(np.abs(fast - naive)) <= 1e-12 * np.max(np.abs(lib))
        assert np.max(np.abs(naive - brute_dft3(rho))) <= 1e-11 * np.max(np.abs(lib))


@pytest.mark.parametrize("ng", [4, 8, 16, 64])
def test_round_trip_and_inverse_normalisation(oracle, ng):
    rng = np.random.default_rng(7 + ng)
    rho = rng.standard_normal((ng, ng, ng))
    back = oracle.fft_c2r(oracle.fft_r2c(rho))
    assert np.max(np.abs(back - rho)) < 1e-12
    # inverse against the library on a Hermitian spectrum
    spec = np.fft.rfftn(rho)
    assert np.max(np.abs(oracle.fft_c2r(spec) - np.fft.irfftn(spec, s=rho.shape, axes=(0, 1, 2)))) < 1e-12


def test_delta_function_maps_to_ones_and_shift_theorem(oracle):
    ng = 16
    rho = np.zeros((ng, ng, ng))
    rho[0, 0, 0] = 1.0
    assert np.max(np.abs(oracle.fft_r2c(rho) - 1.0)) < 1e-13
    rho[:] = 0
    rho[3, 5, 2] = 1.0  # sign convention: exp(-i k.x)
    k = np.fft.fftfreq(ng, 1.0 / ng)
    kz = np.arange(ng // 2 + 1)
    ref = np.exp(-2j * np.pi * (3 * k[:, None, None] + 5 * k[None, :, None] + 2 * kz[None, None, :]) / ng)
    assert np.max(np.abs(oracle.fft_r2c(rho) - ref)) < 1e-13


def test_single_cosine_gives_two_spikes(oracle):
    ng = 16
    x = np.arange(ng)
    rho = np.cos(2 * np.pi * 3 * x / ng)[:, None, None] * np.ones((1, ng, ng))
    spec = oracle.fft_r2c(rho)
    expect = np.zeros_like(spec)
    expect[3, 0, 0] = expect[ng - 3, 0, 0] = ng ** 3 / 2
    assert np.max(np.abs(spec - expect)) < 1e-9


def test_parseval_with_half_space_weights(oracle):
    ng = 16
    rng = np.random.default_rng(3)
    rho = rng.standard_normal((ng, ng, ng))
    spec = oracle.fft_r2c(rho)
    w = np.full(ng // 2 + 1, 2.0)
    w[0] = w[-1] = 1.0
    assert np.sum(w * np.abs(spec) ** 2) / ng ** 3 == pytest.approx(np.sum(rho ** 2), rel=1e-12)


def test_c2r_of_a_spectrum_that_is_not_hermitian_on_the_kz_0_and_nyquist_planes(oracle):
    """The contract include/fpm.h states for fpm_fft_c2r on inputs that are not the spectrum of a real
    field: the result is the real part of the inverse transform of the spectrum completed by
    a(-k) = conj(a(k)) for 0 < kz < ng/2, with the planes kz = 0 and kz = ng/2 taken as stored.
    Pinned against numpy.fft.ifftn of the explicitly completed full spectrum."""
    ng = 8
    rng = np.random.default_rng(11)
    half = rng.standard_normal((ng, ng, ng // 2 + 1)) + 1j * rng.standard_normal((ng, ng, ng // 2 + 1))
    full = np.zeros((ng, ng, ng), dtype=np.complex128)
    full[:, :, : ng // 2 + 1] = half
    idx = (-np.arange(ng)) % ng
    for z in range(ng // 2 + 1, ng):
        full[:, :, z] = np.conj(half[idx][:, idx][:, :, ng - z])
    ref = np.fft.ifftn(full).real
    assert np.max(np.abs(oracle.fft_c2r(half) - ref)) < 1e-13
    assert np.max(np.abs(oracle.fft_c2r(half, force_naive=True) - ref)) < 1e-13
