"""Pins for the force kernel and one force evaluation."""
import numpy as np
import pytest

import fpm_inputs as fi


def potential_from_density(oracle, rho, mode):
    """phi with phi_hat = -delta_hat / K^2, recovered from the oracle's own force spectrum is not
    possible without dividing by g; instead build phi with numpy from the printed Eq. 4."""
    ng = rho.shape[0]
    w = 2 * np.pi * np.fft.fftfreq(ng)
    wz = 2 * np.pi * np.arange(ng // 2 + 1) / ng
    if mode == 0:
        k2 = (2 * np.sin(w / 2))[:, None, None] ** 2 + (2 * np.sin(w / 2))[None, :, None] ** 2 + (2 * np.sin(wz / 2))[None, None, :] ** 2
    else:
        k2 = w[:, None, None] ** 2 + w[None, :, None] ** 2 + wz[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    phik = -np.fft.rfftn(rho) / k2
    phik[0, 0, 0] = 0.0
    return np.fft.irfftn(phik, s=rho.shape, axes=(0, 1, 2))


def test_eq4_is_the_inverse_of_the_7_point_laplacian_and_eq5_the_4_point_gradient(oracle):
    """FFT-free reading check: F_d = -D1_d phi with D1 the real-space stencil
    (-phi[+2] + 8 phi[+1] - 8 phi[-1] + phi[-2])/12, and the 7-point Laplacian of phi is rho - mean."""
    ng = 16
    rng = np.random.default_rng(0)
    rho = rng.standard_normal((ng, ng, ng)) + 1.0
    F = oracle.force_grids(rho, mode=0, scale=1.0)
    # the potential whose 7-point Laplacian is rho - mean, solved without any FFT symbol:
    phi = potential_from_density(oracle, rho, 0)
    lap = -6 * phi
    for d in range(3):
        lap = lap + np.roll(phi, 1, d) + np.roll(phi, -1, d)
    assert np.max(np.abs(lap - (rho - rho.mean()))) < 1e-12
    for d in range(3):
        grad = (-np.roll(phi, -2, d) + 8 * np.roll(phi, -1, d) - 8 * np.roll(phi, 1, d) + np.roll(phi, 2, d)) / 12
        assert np.max(np.abs(F[d] + grad)) < 1e-12 * max(1.0, np.max(np.abs(grad)))


def test_naive_kernel_is_ik_over_k2_with_nyquist_zeroed(oracle):
    ng = 8
    rng = np.random.default_rng(1)
    dk = np.fft.rfftn(rng.standard_normal((ng, ng, ng)))
    fk = oracle.apply_force_kernel(dk, mode=1, scale=2.0)
    n = np.fft.fftfreq(ng, 1.0 / ng)
    nz = np.arange(ng // 2 + 1.0)
    w = [2 * np.pi * n[:, None, None] / ng, 2 * np.pi * n[None, :, None] / ng, 2 * np.pi * nz[None, None, :] / ng]
    k2 = w[0] ** 2 + w[1] ** 2 + w[2] ** 2
    k2[0, 0, 0] = np.inf
    for d in range(3):
        g = np.broadcast_to(w[d], dk.shape).copy()
        idx = [slice(None)] * 3
        idx[d] = ng // 2
        g[tuple(idx)] = 0.0
        assert np.allclose(fk[d], 2.0 * 1j * g * dk / k2, rtol=1e-13, atol=1e-13)
    # mixed mode: Eq. 5 gradient over k^2
    fm = oracle.apply_force_kernel(dk, mode=2, scale=1.0)
    g5 = (8 * np.sin(w[0]) - np.sin(2 * w[0])) / 6
    g5 = np.broadcast_to(g5, dk.shape).copy()
    g5[ng // 2] = 0.0
    assert np.allclose(fm[0], 1j * g5 * dk / k2, rtol=1e-13, atol=1e-13)


@pytest.mark.parametrize("B", [1, 2])
def test_zero_force_on_unperturbed_lattice(oracle, B):
    nps = 8
    g = np.arange(nps, dtype=np.float64) * B
    q = np.stack(np.meshgrid(g, g, g, indexing="ij")).reshape(3, -1)
    for mode in (0, 1, 2):
        f = oracle.force(q, nps * B, mode=mode, scale=1.5 * 0.3075, mass=float(B ** 3))
        assert np.max(np.abs(f)) < 1e-13


def test_net_momentum_is_conserved(oracle):
    ng = 16
    pos = fi.random_particles(2000, ng, seed=3, clustered=True).astype(np.float64)
    for mode in (0, 1, 2):
        f = oracle.force(pos, ng, mode=mode, scale=1.0, mass=1.0)
        assert np.max(np.abs(f.sum(axis=1))) < 1e-12 * np.sqrt(np.mean(f ** 2)) * f.shape[1]


def _point_force_ratio(oracle, ng, mode, r, ndir, rng):
    src = np.array([[ng / 2 + 0.31], [ng / 2 - 0.17], [ng / 2 + 0.08]])
    rho = oracle.paint(src, ng)
    F = oracle.force_grids(rho, mode=mode, scale=1.0)
    u = rng.standard_normal((3, ndir))
    u /= np.linalg.norm(u, axis=0)
    tgt = src + r * u
    fr = sum(oracle.readout(F[d], tgt) * u[d] for d in range(3))
    return fr / (-1.0 / (4 * np.pi * r * r))


def test_single_particle_force_follows_inverse_square_law(oracle):
    """lap phi = delta (unit mass, scale 1) => radial force -1/(4 pi r^2) towards the source at
    separations of several cells; the slow deficit is the uniform background + periodic images."""
    rng = np.random.default_rng(5)
    ng = 64
    for mode in (0, 2):
        for r, tol in ((4.0, 0.04), (6.0, 0.03), (8.0, 0.03)):
            ratio = _point_force_ratio(oracle, ng, mode, r, 200, rng)
            assert np.mean(ratio) == pytest.approx(1.0, abs=tol)
            assert np.all(ratio > 0.8)          # attractive in every direction
    ratio = _point_force_ratio(oracle, ng, 1, 6.0, 400, rng)   # ik kernel: only the angle average
    assert np.mean(ratio) == pytest.approx(1.0, abs=0.06)


def test_force_points_towards_overdensity(oracle):
    ng = 32
    src = np.array([[10.0], [10.0], [10.0]])
    F = oracle.force_grids(oracle.paint(src, ng), mode=0, scale=1.0)
    assert oracle.readout(F[0], np.array([[14.0], [10.0], [10.0]]))[0] < 0
    assert oracle.readout(F[0], np.array([[6.0], [10.0], [10.0]]))[0] > 0
    assert oracle.readout(F[2], np.array([[10.0], [10.0], [15.0]]))[0] < 0
