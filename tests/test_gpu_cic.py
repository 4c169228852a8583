"""GPU parity: CIC paint / readout and their adjoints vs the oracle (R1, R10, R11).
Tolerance: relative L2 <= 1e-5 (north_star); fp32 weights and atomic ordering give ~1e-7."""
import numpy as np
import pytest

import fpm_inputs as fi
from gpu_util import dev, host, rel_l2

pytestmark = pytest.mark.gpu
TOL = 1e-5


@pytest.fixture(scope="module")
def fpm():
    import paper_2010_11847_b200 as fpm
    return fpm


@pytest.mark.parametrize("ng,n,clustered", [(16, 1000, False), (32, 20011, True), (64, 300007, True), (128, 2 ** 21, False)])
def test_paint_matches_oracle(fpm, oracle, ng, n, clustered):
    pos = fi.random_particles(n, ng, seed=ng + n, clustered=clustered)
    ctx = fpm.FPM(ng, workspace=False)
    got = host(ctx.paint(dev(pos)))
    ref = oracle.paint(pos.astype(np.float64), ng, mass_const=1.0)
    assert rel_l2(got, ref) < TOL
    assert abs(got.astype(np.float64).sum() - n) < 1e-5 * n


def test_paint_with_masses_resolution_factor_and_edges(fpm, oracle):
    ng, nps = 32, 16
    ctx = fpm.FPM(ng, nps, workspace=False)
    n = nps ** 3
    pos = fi.random_particles(n, ng, seed=77, clustered=True)
    # default mass is B^3 = 8 so the mean density is 1
    got = host(ctx.paint(dev(pos)))
    assert rel_l2(got, oracle.paint(pos.astype(np.float64), ng, mass_const=8.0)) < TOL
    assert got.mean() == pytest.approx(1.0, rel=1e-5)
    m = np.linspace(-1.0, 2.0, n).astype(np.float32)
    got = host(ctx.paint(dev(pos), dev(m)))
    ref = oracle.paint(pos.astype(np.float64), ng, mass=m.astype(np.float64))
    assert rel_l2(got, ref) < TOL
    # degenerate inputs: no particles; particles on corners and on the last cell (periodic wrap)
    import torch
    empty = torch.empty(3, 0, dtype=torch.float32, device="cuda")
    assert float(ctx.paint(empty).abs().max()) == 0.0
    edge = np.array([[0.0, 31.0, 31.5, 31.999998], [0.0, 31.0, 0.25, 31.999998], [0.0, 31.0, 31.75, 0.0]], dtype=np.float32)
    got = host(ctx.paint(dev(edge), dev(np.ones(4, dtype=np.float32))))
    ref = oracle.paint(edge.astype(np.float64), ng, mass_const=1.0)
    assert np.max(np.abs(got - ref)) < 1e-6
    assert got[0, 0, 0] == pytest.approx(ref[0, 0, 0]) and got.sum() == pytest.approx(4.0, rel=1e-6)


def test_lattice_paints_to_uniform_density(fpm):
    ng = 32
    g = np.arange(ng, dtype=np.float32)
    q = np.stack(np.meshgrid(g, g, g, indexing="ij")).reshape(3, -1)
    ctx = fpm.FPM(ng, workspace=False)
    assert np.all(host(ctx.paint(dev(q))) == 1.0)


@pytest.mark.parametrize("ng,n", [(16, 999), (64, 100003)])
def test_readout_matches_oracle(fpm, oracle, ng, n):
    rng = np.random.default_rng(ng)
    mesh = rng.standard_normal((ng, ng, ng)).astype(np.float32)
    pos = fi.random_particles(n, ng, seed=5, clustered=True)
    ctx = fpm.FPM(ng, workspace=False)
    got = host(ctx.readout(dev(mesh), dev(pos)))
    ref = oracle.readout(mesh.astype(np.float64), pos.astype(np.float64))
    assert rel_l2(got, ref) < TOL
    assert np.max(np.abs(got - ref)) < 2e-6 * np.max(np.abs(ref))


def test_adjoints_match_oracle_and_dot_product_identity(fpm, oracle):
    ng, n = 32, 50021
    rng = np.random.default_rng(3)
    pos = fi.random_particles(n, ng, seed=8, clustered=True)
    m = rng.uniform(0.5, 2.0, n).astype(np.float32)
    gbar = rng.standard_normal((ng, ng, ng)).astype(np.float32)
    vbar = rng.standard_normal(n).astype(np.float32)
    F = rng.standard_normal((ng, ng, ng)).astype(np.float32)
    ctx = fpm.FPM(ng, workspace=False)
    p64 = pos.astype(np.float64)
    gpos, gmass = ctx.paint_adjoint(dev(pos), dev(gbar), mass=dev(m))
    rpos, rmass = oracle.paint_adjoint(p64, ng, gbar.astype(np.float64), mass=m.astype(np.float64))
    assert rel_l2(host(gpos), rpos) < TOL and rel_l2(host(gmass), rmass) < TOL
    base = rng.standard_normal((ng, ng, ng)).astype(np.float32)
    gm, gp = ctx.readout_adjoint(dev(F), dev(pos), dev(vbar), grad_mesh=dev(base))
    rm, rp = oracle.readout_adjoint(F.astype(np.float64), p64, vbar.astype(np.float64), grad_mesh=base.astype(np.float64))
    assert rel_l2(host(gm), rm) < TOL and rel_l2(host(gp), rp) < TOL
    # <paint(x) m, y> = <m, readout(y, x)> on the GPU path itself
    lhs = float((ctx.paint(dev(pos), dev(m)).double() * dev(gbar).double()).sum())
    rhs = float((dev(m).double() * ctx.readout(dev(gbar), dev(pos)).double()).sum())
    assert lhs == pytest.approx(rhs, rel=1e-5)


@pytest.mark.parametrize("mode", ["fixed", "float"])
def test_brick_paint_with_resolution_factor_two(fpm, oracle, mode):
    """A full lattice particle set on a mesh twice as fine (C3's regime: 1/8 particle per cell) takes
    the sub-brick window path; displaced lattice with a few multi-cell outliers, against the oracle."""
    import paper_2010_11847_b200 as m
    nps, ng = 32, 64
    n = nps ** 3
    rng = np.random.default_rng(7)
    q = np.stack(np.meshgrid(*[np.arange(nps) * 2.0] * 3, indexing="ij")).reshape(3, n)
    pos = q + rng.normal(0.0, 0.8, size=(3, n))
    pos[:, ::97] += rng.normal(0.0, 6.0, size=(3, len(range(0, n, 97))))     # outliers leave the window
    pos = np.mod(pos, ng).astype(np.float32)
    ctx = m.FPM(ng, nps, paint_mode=m.PAINT_BRICK_FIXED if mode == "fixed" else m.PAINT_BRICK_FLOAT)
    got = host(ctx.paint(dev(pos)))
    ref = oracle.paint(pos.astype(np.float64), ng, mass_const=8.0)
    assert rel_l2(got, ref) < TOL
    assert abs(got.astype(np.float64).sum() - 8.0 * n) < 1e-5 * 8.0 * n
    mass = rng.standard_normal(n).astype(np.float32)                         # signed per-particle masses
    got = host(ctx.paint(dev(pos), mass=dev(mass)))
    ref = oracle.paint(pos.astype(np.float64), ng, mass=mass.astype(np.float64))
    assert rel_l2(got, ref) < TOL
