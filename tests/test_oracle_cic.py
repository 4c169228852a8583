"""Pins for CIC paint / readout and their adjoints."""
import numpy as np
import pytest

import fpm_inputs as fi


def lattice(np_side, B=1):
    g = np.arange(np_side, dtype=np.float64) * B
    q = np.stack(np.meshgrid(g, g, g, indexing="ij")).reshape(3, -1)
    return q


def test_mass_conservation(oracle):
    pos = fi.random_particles(4096, 16, seed=5, clustered=True).astype(np.float64)
    assert oracle.paint(pos, 16).sum() == pytest.approx(4096.0, rel=1e-13)
    q = lattice(8, 2) + 0.3
    assert oracle.paint(q, 16, mass_const=8.0).sum() == pytest.approx(4096.0, rel=1e-13)
    m = np.linspace(0.5, 2.0, 4096)
    assert oracle.paint(pos, 16, mass=m).sum() == pytest.approx(m.sum(), rel=1e-13)


def test_particle_on_cell_corner_and_trilinear_weights(oracle):
    pos = np.array([[3.0], [15.0], [0.0]])
    mesh = oracle.paint(pos, 16)
    assert mesh[3, 15, 0] == 1.0 and np.count_nonzero(mesh) == 1
    # generic point: weights are the products of (1-t, t), wrapped periodically
    pos = np.array([[15.25], [2.5], [7.75]])
    mesh = oracle.paint(pos, 16)
    assert mesh[15, 2, 7] == pytest.approx(0.75 * 0.5 * 0.25)
    assert mesh[0, 3, 8] == pytest.approx(0.25 * 0.5 * 0.75)
    assert mesh[0, 2, 7] == pytest.approx(0.25 * 0.5 * 0.25)
    assert np.count_nonzero(mesh) == 8


def test_unperturbed_lattice(oracle):
    assert np.all(oracle.paint(lattice(8), 8) == 1.0)
    mesh = oracle.paint(lattice(8, 2), 16, mass_const=8.0)   # B = 2: pure Nyquist pattern
    assert np.all(mesh[::2, ::2, ::2] == 8.0) and mesh.sum() == 4096.0
    assert np.count_nonzero(mesh) == 512


def test_readout_constant_and_linear_ramp(oracle):
    ng = 16
    pos = fi.random_particles(500, ng, seed=9).astype(np.float64)
    assert np.allclose(oracle.readout(np.full((ng, ng, ng), 2.5), pos), 2.5, rtol=1e-14)
    inner = pos[:, np.all(pos < ng - 1, axis=0)]
    for d in range(3):
        shape = [1, 1, 1]
        shape[d] = ng
        ramp = np.arange(ng, dtype=np.float64).reshape(shape) * np.ones((ng, ng, ng))
        assert np.allclose(oracle.readout(ramp, inner), inner[d], rtol=1e-13)


def test_paint_readout_are_an_adjoint_pair(oracle):
    ng, n = 16, 3000
    rng = np.random.default_rng(2)
    pos = fi.random_particles(n, ng, seed=4, clustered=True).astype(np.float64)
    m, y = rng.standard_normal(n), rng.standard_normal((ng, ng, ng))
    lhs = np.sum(oracle.paint(pos, ng, mass=m) * y)
    rhs = np.sum(m * oracle.readout(y, pos))
    assert lhs == pytest.approx(rhs, rel=1e-12)


def test_adjoint_position_gradients_vs_finite_differences(oracle):
    ng, n = 8, 40
    rng = np.random.default_rng(11)
    pos = rng.uniform(0.05, 0.95, (3, n)) + rng.integers(0, ng, (3, n))  # away from cell faces
    m = rng.uniform(0.5, 2.0, n)
    gbar = rng.standard_normal((ng, ng, ng))     # dL/drho  for L = <paint(x) m, gbar>
    vbar = rng.standard_normal(n)                # dL/dout  for L = <readout(F, x), vbar>
    F = rng.standard_normal((ng, ng, ng))
    gpos_p, gmass_p = oracle.paint_adjoint(pos, ng, gbar, mass=m)
    gmesh_r, gpos_r = oracle.readout_adjoint(F, pos, vbar)
    assert np.allclose(gmass_p, oracle.readout(gbar, pos), rtol=1e-14)
    assert np.allclose(gmesh_r, oracle.paint(pos, ng, mass=vbar), rtol=1e-14)
    eps = 1e-6
    for d in range(3):
        for p in (0, 7, 23):
            xp, xm = pos.copy(), pos.copy()
            xp[d, p] += eps
            xm[d, p] -= eps
            fd_p = (np.sum(oracle.paint(xp, ng, mass=m) * gbar) - np.sum(oracle.paint(xm, ng, mass=m) * gbar)) / (2 * eps)
            fd_r = (np.sum(oracle.readout(F, xp) * vbar) - np.sum(oracle.readout(F, xm) * vbar)) / (2 * eps)
            assert gpos_p[d, p] == pytest.approx(fd_p, rel=1e-7, abs=1e-8)
            assert gpos_r[d, p] == pytest.approx(fd_r, rel=1e-7, abs=1e-8)


def test_readout_adjoint_accumulates_into_grad_mesh(oracle):
    ng, n = 8, 50
    rng = np.random.default_rng(1)
    pos = rng.uniform(0, ng, (3, n))
    vbar = rng.standard_normal(n)
    base = rng.standard_normal((ng, ng, ng))
    gm, _ = oracle.readout_adjoint(np.zeros((ng, ng, ng)), pos, vbar, grad_mesh=base)
    assert np.allclose(gm - base, oracle.paint(pos, ng, mass=vbar), atol=1e-14)
