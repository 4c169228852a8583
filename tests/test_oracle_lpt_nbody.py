"""Pins for LPT initial conditions, the whole-run driver and P(k)."""
import math

import numpy as np
import pytest

import fpm_inputs as fi

OM = 0.3075


def test_lpt_two_cosines_closed_form(oracle):
    """delta = A cos(kx x) + B cos(ky y): psi1_x = -A sin(kx x)/kx,
    psi2_x = A B kx sin(kx x) cos(ky y)/(kx^2+ky^2); the 2LPT source vanishes for one plane wave."""
    n = 16
    A, Bc = 0.03, 0.02
    kx, ky = 2 * np.pi * 2 / n, 2 * np.pi * 3 / n
    x = np.arange(n)[:, None, None] * np.ones((n, n, n))
    y = np.arange(n)[None, :, None] * np.ones((n, n, n))
    delta = A * np.cos(kx * x) + Bc * np.cos(ky * y)
    psi1, psi2 = oracle.lpt_displacements(delta, order=2)
    assert np.max(np.abs(psi1[0] + A * np.sin(kx * x) / kx)) < 1e-14
    assert np.max(np.abs(psi1[1] + Bc * np.sin(ky * y) / ky)) < 1e-14
    assert np.max(np.abs(psi1[2])) < 1e-14
    k2 = kx * kx + ky * ky
    assert np.max(np.abs(psi2[0] - A * Bc * kx * np.sin(kx * x) * np.cos(ky * y) / k2)) < 1e-15
    assert np.max(np.abs(psi2[1] - A * Bc * ky * np.cos(kx * x) * np.sin(ky * y) / k2)) < 1e-15
    assert np.max(np.abs(psi2[2])) < 1e-15
    _, p2 = oracle.lpt_displacements(A * np.cos(kx * x), order=2)
    assert np.max(np.abs(p2)) < 1e-16


def test_lpt_divergence_of_psi1_is_minus_delta(oracle):
    n = 16
    delta = fi.linear_field(n, 100.0, seed=2).astype(np.float64)
    psi1, _ = oracle.lpt_displacements(delta, order=1)
    k = 2 * np.pi * np.fft.fftfreq(n)
    kz = 2 * np.pi * np.arange(n // 2 + 1) / n
    ks = [k[:, None, None], k[None, :, None], kz[None, None, :]]
    div = sum(1j * ks[d] * np.fft.rfftn(psi1[d]) for d in range(3))
    dk = np.fft.rfftn(delta)
    # exact except on Nyquist planes, where i k_d is zeroed (R9 reading)
    inner = (slice(1, n // 2), slice(1, n // 2), slice(1, n // 2))
    assert np.max(np.abs(div[inner] + dk[inner])) < 1e-10 * np.max(np.abs(dk))


def test_lpt_init_positions_and_momenta(oracle):
    """x = q B + B (D1 psi1 + D2 psi2), p = a^2 E B (f1 D1 psi1 + f2 D2 psi2) in mesh cells."""
    n, ng, a0 = 8, 16, 0.1
    delta = 0.05 * fi.linear_field(n, 50.0, seed=3).astype(np.float64)
    psi1, psi2 = oracle.lpt_displacements(delta, order=2)
    g = oracle.growth(OM, a0)
    pos, mom = oracle.lpt_init(delta, ng, OM, a0, 2)
    q = np.stack(np.meshgrid(*[np.arange(n) * 2.0] * 3, indexing="ij")).reshape(3, -1)
    disp = (g["D1"] * psi1 + g["D2"] * psi2).reshape(3, -1) * 2
    assert np.allclose(np.mod(q + disp, ng), pos, atol=1e-12)
    vel = a0 ** 2 * g["E"] * (g["f1"] * g["D1"] * psi1 + g["f2"] * g["D2"] * psi2).reshape(3, -1) * 2
    assert np.allclose(vel, mom, rtol=1e-12, atol=1e-15)
    pos1, mom1 = oracle.lpt_init(delta, ng, OM, a0, 1)
    assert np.allclose(np.mod(q + (g["D1"] * psi1).reshape(3, -1) * 2, ng), pos1, atol=1e-12)


def _plane_wave_growth(oracle, n, mode_number, n_steps=5):
    A = 1e-4
    x = np.arange(n)[:, None, None] * np.ones((n, n, n))
    kx = 2 * np.pi * mode_number / n
    delta = A * np.cos(kx * x)
    a0 = 0.1
    pos, mom = oracle.lpt_init(delta, n, OM, a0, 1)
    stages = np.linspace(a0, 1.0, n_steps + 1)
    pos, mom, traj = oracle.nbody(pos, mom, n, n, OM, stages, return_traj=True)
    q = x.reshape(-1)
    basis = -A * np.sin(kx * q) / kx          # psi1_x
    out = []
    for j, a in enumerate(stages):
        disp = traj[j, 0] - q
        disp = (disp + n / 2) % n - n / 2
        out.append(np.dot(disp, basis) / np.dot(basis, basis) / oracle.growth(OM, a)["D1"])
    return np.array(out)


@pytest.mark.parametrize("order,n,ng", [(1, 8, 8), (2, 8, 8), (1, 8, 16), (2, 8, 16)])
def test_lpt_momenta_are_the_time_derivative_of_the_lpt_positions(oracle, order, n, ng):
    """Independent pin of the momentum coefficients a^2 E f1 D1 and a^2 E f2 D2 (Alg. 4, PAPER.md:363-383;
    R0: p = a^2 dx/dt / H0 = a^3 E dx/da): a 4th-order central difference in a0 of the oracle's own LPT
    POSITIONS must reproduce its momenta.  E(a) is typed out from its definition (R0), not taken from
    oracle.growth, so a wrong f1, f2, D2 normalisation or a missing factor of a fails here (the D(a) pin
    of the plane-wave test cannot see f(a): f1(0.1) = 0.9988)."""
    a0, h = 0.1, 2e-3
    delta = 0.05 * fi.linear_field(n, 50.0, seed=3).astype(np.float64)

    def x_of(a):
        return oracle.lpt_init(delta, ng, OM, a, order)[0]

    def wrapped_diff(u, v):
        d = u - v
        return d - ng * np.round(d / ng)

    dxda = (8.0 * wrapped_diff(x_of(a0 + h), x_of(a0 - h)) - wrapped_diff(x_of(a0 + 2 * h), x_of(a0 - 2 * h))) / (12.0 * h)
    e_of_a = math.sqrt(OM / a0 ** 3 + 1.0 - OM)
    _, mom = oracle.lpt_init(delta, ng, OM, a0, order)
    assert np.max(np.abs(a0 ** 3 * e_of_a * dxda - mom)) < 1e-6 * np.max(np.abs(mom))


def test_small_plane_wave_follows_linear_growth(oracle):
    """ICs from the Zel'dovich approximation at a = 0.1, 5 steps to a = 1: the displacement
    amplitude tracks D1(a) up to the paint x readout window and the finite-difference kernels,
    a deficit of order omega^2 that must quarter when omega is halved (R4 pin)."""
    r2 = _plane_wave_growth(oracle, 32, 2)
    r1 = _plane_wave_growth(oracle, 32, 1)
    assert r1[0] == pytest.approx(1.0, abs=1e-9) and r2[0] == pytest.approx(1.0, abs=1e-9)
    # bounded by the paint x readout window sinc^4(omega/2) itself
    for r, m in ((r1, 1), (r2, 2)):
        window = np.sinc(m / 32.0) ** 4          # np.sinc(x) = sin(pi x)/(pi x)
        assert np.all(r[1:] < 1.0) and np.all(r[1:] > window)
    assert np.all(np.diff(r1) < 0)            # slowly accumulating deficit, never growth
    assert (1 - r2[-1]) / (1 - r1[-1]) == pytest.approx(4.0, rel=0.1)


def test_nbody_equals_manual_kick_drift_kick(oracle):
    n, ng = 8, 8
    delta = 0.5 * fi.linear_field(n, 50.0, seed=4).astype(np.float64)
    pos0, mom0 = oracle.lpt_init(delta, ng, OM, 0.2, 1)
    stages = [0.2, 0.5, 1.0]
    pos, mom = oracle.nbody(pos0, mom0, ng, n, OM, stages)
    x, p = pos0.copy(), mom0.copy()
    f = oracle.force(x, ng, scale=1.5 * OM)
    for j in range(2):
        ai, af = stages[j], stages[j + 1]
        ah = math.sqrt(ai * af)
        p = oracle.kick(p, f, oracle.kick_factor(OM, ai, ai, ah))
        x = oracle.drift(x, p, oracle.drift_factor(OM, ai, ah, af), ng)
        f = oracle.force(x, ng, scale=1.5 * OM)
        p = oracle.kick(p, f, oracle.kick_factor(OM, ah, af, af))
    assert np.allclose(x, pos, atol=1e-13) and np.allclose(p, mom, atol=1e-13)


def test_drift_wraps_into_box(oracle):
    pos = np.array([[7.5, 0.25], [0.0, 7.9], [3.0, 3.0]])
    mom = np.array([[1.0, -1.0], [0.0, 1.0], [-4.0, 13.0]])
    out = oracle.drift(pos, mom, 1.0, 8)
    assert np.allclose(out, [[0.5, 7.25], [0.0, 0.9], [7.0, 0.0]])
    assert np.all(out >= 0) and np.all(out < 8)


def test_power_spectrum_of_a_single_mode_and_of_the_linear_field(oracle):
    n, box = 16, 100.0
    x = np.arange(n)[:, None, None] * np.ones((n, n, n))
    amp = 0.1
    mesh = 1.0 + amp * np.cos(2 * np.pi * 3 * x / n)
    k, pk, nm = oracle.power(mesh, box)
    # |delta_k|^2 = (amp n^3/2)^2 at +-3 on the x axis; bin 3 holds those 2 modes among nm[2]
    assert pk[2] * nm[2] == pytest.approx(2 * (amp / 2) ** 2 * box ** 3, rel=1e-12)
    assert np.all(pk[np.arange(n // 2) != 2] < 1e-25)
    assert nm[0] == 6 + 12 + 8 - 8       # |n| in [0.5, 1.5): 6 axis + 12 face-diagonal modes
    # measured spectrum of the seeded Gaussian field follows the input P(k) within cosmic variance
    n, box = 64, 400.0
    d = fi.linear_field(n, box, seed=1).astype(np.float64)
    k, pk, nm = oracle.power(1.0 + d, box)
    sel = (nm > 200) & (np.arange(n // 2) < n // 2 - 2)
    ratio = pk[sel] / fi.linear_power(k[sel])
    assert np.all(np.abs(ratio - 1) < 5 * np.sqrt(2.0 / nm[sel]) + 0.03)
    # cross spectrum with itself is the auto spectrum (Eq. 11: r_c = 1)
    _, pab, _ = oracle.power(1.0 + d, box, mesh_b=1.0 + d)
    assert np.allclose(pab, pk, rtol=1e-12)


def test_batch_of_runs_equals_the_single_runs_and_its_members_are_independent(oracle):
    """N2 pin: the batch is defined as B independent runs, so member b must be bit-for-bit the single run of
    its inputs, and changing one member's input must leave every other member's output untouched."""
    n, ng = 8, 8
    stages = [0.1, 0.4, 0.7, 1.0]
    states = [oracle.lpt_init(0.5 * fi.linear_field(n, 60.0, seed=s).astype(np.float64), ng, OM, 0.1, 2) for s in (1, 2, 3)]
    pos = np.stack([p for p, _ in states])
    mom = np.stack([m for _, m in states])
    bp, bm = oracle.nbody_batch(pos, mom, ng, n, OM, stages)
    for b in range(3):
        sp, sm = oracle.nbody(pos[b], mom[b], ng, n, OM, stages)
        assert np.array_equal(bp[b], sp) and np.array_equal(bm[b], sm)
    pos2 = pos.copy()
    pos2[1] = np.mod(pos2[1] + 0.37, ng)
    cp, cm = oracle.nbody_batch(pos2, mom, ng, n, OM, stages)
    assert np.array_equal(cp[0], bp[0]) and np.array_equal(cp[2], bp[2]) and not np.array_equal(cp[1], bp[1])
