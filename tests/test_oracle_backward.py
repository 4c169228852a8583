"""Pins of the oracle's reverse mode against central
finite differences of the oracle's own FORWARD functions in float64, and against the per-operator
adjoint identities.  A wrong sign, a missing term (direct dW/dx term, mesh term, the 2LPT product
rule) or a transposed kernel fails the directional-derivative checks below."""
import numpy as np
import pytest

import fpm_inputs as fi

OM = 0.3075


def _periodic_objective(pos, mom, w, u, ng):
    """L = sum w cos(2 pi x / ng) + sum u p : smooth across the periodic wrap."""
    return float(np.sum(w * np.cos(2 * np.pi * pos / ng)) + np.sum(u * mom))


def _periodic_objective_grad(pos, w, u, ng):
    return -w * (2 * np.pi / ng) * np.sin(2 * np.pi * pos / ng), u.copy()


@pytest.mark.parametrize("ng,n,mass,mode", [(8, 40, 1.0, 0), (16, 300, 8.0, 0), (8, 40, 1.0, 1), (8, 40, 1.0, 2)])
def test_force_vjp_matches_finite_differences(oracle, ng, n, mass, mode):
    rng = np.random.default_rng(5)
    pos = rng.uniform(0.05, ng - 0.05, size=(3, n))
    pos = np.where(np.abs(pos - np.round(pos)) < 0.02, pos + 0.05, pos)   # stay off cell faces
    v = rng.standard_normal((3, n))
    dx = rng.standard_normal((3, n))
    eps = 1e-6
    fp = oracle.force(pos + eps * dx, ng, mode=mode, scale=1.5 * OM, mass=mass)
    fm = oracle.force(pos - eps * dx, ng, mode=mode, scale=1.5 * OM, mass=mass)
    lhs = float(np.sum(v * (fp - fm) / (2 * eps)))
    gx = oracle.force_vjp(pos, ng, v, mode=mode, scale=1.5 * OM, mass=mass)
    rhs = float(np.sum(gx * dx))
    assert lhs == pytest.approx(rhs, rel=2e-6, abs=1e-10)


def test_force_vjp_is_linear_in_the_cotangent_and_zero_for_zero(oracle):
    rng = np.random.default_rng(6)
    ng, n = 8, 30
    pos = rng.uniform(0, ng, size=(3, n))
    v1, v2 = rng.standard_normal((3, n)), rng.standard_normal((3, n))
    g1 = oracle.force_vjp(pos, ng, v1)
    g2 = oracle.force_vjp(pos, ng, v2)
    g12 = oracle.force_vjp(pos, ng, 2.0 * v1 - 3.0 * v2)
    assert np.allclose(g12, 2.0 * g1 - 3.0 * g2, rtol=1e-12, atol=1e-14)
    assert np.all(oracle.force_vjp(pos, ng, np.zeros((3, n))) == 0.0)


@pytest.mark.parametrize("np_side,ng,n_steps", [(4, 4, 2), (4, 8, 2), (8, 8, 3)])
def test_nbody_vjp_matches_finite_differences(oracle, np_side, ng, n_steps):
    rng = np.random.default_rng(7)
    n = np_side ** 3
    B = ng // np_side
    q = np.stack(np.meshgrid(*[np.arange(np_side) * B] * 3, indexing="ij")).reshape(3, n).astype(float)
    pos0 = (q + rng.uniform(0.1, 0.4, size=(3, n))) % ng
    mom0 = 0.05 * rng.standard_normal((3, n))
    stages = np.linspace(0.2, 0.8, n_steps + 1)
    w, u = rng.standard_normal((3, n)), rng.standard_normal((3, n))

    def loss(p0, m0):
        pf, mf = oracle.nbody(p0, m0, ng, np_side, OM, stages)
        return _periodic_objective(pf, mf, w, u, ng)

    pf, mf, traj = oracle.nbody(pos0, mom0, ng, np_side, OM, stages, return_traj=True)
    assert np.array_equal(traj[0], pos0) and np.array_equal(traj[-1], pf)
    gxf, gpf = _periodic_objective_grad(pf, w, u, ng)
    gx0, gp0 = oracle.nbody_vjp(traj, ng, np_side, OM, stages, gxf, gpf)
    for seed in (1, 2):
        r = np.random.default_rng(seed)
        dx, dp = r.standard_normal((3, n)), r.standard_normal((3, n))
        eps = 1e-6
        fd = (loss(pos0 + eps * dx, mom0 + eps * dp) - loss(pos0 - eps * dx, mom0 - eps * dp)) / (2 * eps)
        an = float(np.sum(gx0 * dx) + np.sum(gp0 * dp))
        assert fd == pytest.approx(an, rel=1e-6, abs=1e-9)


def test_nbody_vjp_with_zero_steps_is_the_identity(oracle):
    rng = np.random.default_rng(8)
    n = 64
    traj = rng.uniform(0, 4, size=(1, 3, n))
    gx, gp = rng.standard_normal((3, n)), rng.standard_normal((3, n))
    ox, op = oracle.nbody_vjp(traj, 4, 4, OM, [0.5], gx, gp)
    assert np.array_equal(ox, gx) and np.array_equal(op, gp)


@pytest.mark.parametrize("order,np_side,ng", [(1, 8, 8), (2, 8, 8), (2, 8, 16)])
def test_lpt_init_vjp_matches_finite_differences(oracle, order, np_side, ng):
    rng = np.random.default_rng(9)
    delta = 0.3 * rng.standard_normal((np_side,) * 3)
    n = np_side ** 3
    w, u = rng.standard_normal((3, n)), rng.standard_normal((3, n))
    a0 = 0.3

    def loss(d):
        p, m = oracle.lpt_init(d, ng, OM, a0, order)
        return _periodic_objective(p, m, w, u, ng)

    pos, mom = oracle.lpt_init(delta, ng, OM, a0, order)
    gx, gp = _periodic_objective_grad(pos, w, u, ng)
    gd = oracle.lpt_init_vjp(delta, ng, OM, a0, order, gx, gp)
    for seed in (3, 4):
        dd = np.random.default_rng(seed).standard_normal(delta.shape)
        eps = 1e-6
        fd = (loss(delta + eps * dd) - loss(delta - eps * dd)) / (2 * eps)
        assert fd == pytest.approx(float(np.sum(gd * dd)), rel=1e-6, abs=1e-9)
    # the mean of delta_lin carries no information (k = 0 is discarded): its gradient sums to zero
    assert abs(gd.sum()) < 1e-9 * np.abs(gd).sum()


def test_end_to_end_gradient_of_the_density_objective(oracle):
    """C4's objective at toy size: L = sum(final density x seeded weight field) w.r.t. delta_lin."""
    np_side = ng = 8
    box = 50.0
    delta = fi.linear_field(np_side, box, 3).astype(np.float64)
    wfield = fi.weight_field(ng, 101).astype(np.float64)
    stages = np.linspace(0.1, 1.0, 4)

    def loss(d):
        p, m = oracle.lpt_init(d, ng, OM, 0.1, 2)
        pf, _ = oracle.nbody(p, m, ng, np_side, OM, stages)
        return float(np.sum(oracle.paint(pf, ng) * wfield))

    p, m = oracle.lpt_init(delta, ng, OM, 0.1, 2)
    pf, mf, traj = oracle.nbody(p, m, ng, np_side, OM, stages, return_traj=True)
    gxf, _ = oracle.paint_adjoint(pf, ng, wfield)
    gx0, gp0 = oracle.nbody_vjp(traj, ng, np_side, OM, stages, gxf, np.zeros_like(gxf))
    gd = oracle.lpt_init_vjp(delta, ng, OM, 0.1, 2, gx0, gp0)
    dd = np.random.default_rng(11).standard_normal(delta.shape)
    eps = 1e-6
    fd = (loss(delta + eps * dd) - loss(delta - eps * dd)) / (2 * eps)
    assert fd == pytest.approx(float(np.sum(gd * dd)), rel=1e-5)
