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


def _lattice(nps, ng, sigma, seed):
    rng = np.random.default_rng(seed)
    q = np.stack(np.meshgrid(*[np.arange(nps) * float(ng // nps)] * 3, indexing="ij")).reshape(3, -1)
    return np.mod(q + rng.normal(0.0, sigma, size=q.shape), ng).astype(np.float32)


@pytest.mark.parametrize("nps,ng", [(32, 32), (64, 64), (32, 64)])
def test_brick_paint_max_abs_error_and_window_wrap(fpm, oracle, nps, ng):
    """Max-abs (not only L2) bound on the brick-window paint.  np = ng = 32: the 40-cell window is wider than
    the box, so window cells alias and the flush must still add every deposit once.  Fixed-point quantum is
    2^-19 m (2^-21 m at B = 2) per deposit and a cell of this cloud receives < 64 deposits."""
    m0 = float((ng // nps) ** 3)
    for sigma in (0.4, 2.5):          # inside the window / many particles on the slow path
        pos = _lattice(nps, ng, sigma, seed=nps + ng)
        ref = oracle.paint(pos.astype(np.float64), ng, mass_const=m0)
        for mode in (fpm.PAINT_BRICK_FIXED, fpm.PAINT_BRICK_FLOAT, fpm.PAINT_DIRECT):
            ctx = fpm.FPM(ng, nps, workspace=False, paint_mode=mode)
            got = host(ctx.paint(dev(pos))).astype(np.float64)
            assert np.max(np.abs(got - ref)) < 2e-6 * np.max(ref) + 64 * 2.0 ** -20 * m0, (sigma, mode)
            assert rel_l2(got, ref) < TOL


def test_fixed_point_window_cannot_overflow(fpm, oracle):
    """All 4096 particles of a brick in ONE cell (the case the scale 2^19 / m is derived for), with the
    constant mass, with equal negative masses and with alternating signs."""
    nps = ng = 64
    n = nps ** 3
    pos = np.empty((3, n), dtype=np.float32)
    pos[0], pos[1], pos[2] = 20.25, 21.5, 22.75
    ctx = fpm.FPM(ng, nps, workspace=False, paint_mode=fpm.PAINT_BRICK_FIXED)
    p64 = pos.astype(np.float64)
    cases = [None, -np.ones(n, dtype=np.float32), np.where(np.arange(n) % 2 == 0, 1.0, -1.0).astype(np.float32),
             np.full(n, 32768.0, dtype=np.float32)]
    for mass in cases:
        got = host(ctx.paint(dev(pos), None if mass is None else dev(mass))).astype(np.float64)
        ref = oracle.paint(p64, ng, mass=None if mass is None else mass.astype(np.float64), mass_const=1.0)
        scale = max(np.max(np.abs(ref)), float(n) * (1.0 if mass is None else float(np.max(np.abs(mass)))) / 64)
        assert np.max(np.abs(got - ref)) < 2e-6 * scale
        assert np.count_nonzero(got) <= 8


def test_paint_with_badly_conditioned_and_non_finite_masses(fpm, oracle):
    """a brick with one huge outlier must not coarsen its ordinary deposits, and NaN/Inf masses
    must propagate (AUTO keeps the fixed-point window only for well-conditioned bricks)."""
    nps = ng = 64
    n = nps ** 3
    pos = _lattice(nps, ng, 0.7, seed=5)
    rng = np.random.default_rng(9)
    mass = np.exp(rng.normal(0.0, 1.0, n)).astype(np.float32)            # log-normal, heavy-ish tail
    mass[12345] = 1.0e6                                                   # one outlier
    mass[54321] = -3.0e5
    ctx = fpm.FPM(ng, nps, workspace=False)                               # PAINT_AUTO
    got = host(ctx.paint(dev(pos), dev(mass))).astype(np.float64)
    ref = oracle.paint(pos.astype(np.float64), ng, mass=mass.astype(np.float64))
    # well away from the outliers the error must stay at the level of ordinary masses (mean ~ 1.6):
    # 2^-18 mean|m| per deposit, < 64 deposits per cell; near them fp32 rounding of the outlier itself
    err = np.abs(got - ref)
    assert np.max(err - 2e-7 * np.abs(ref)) < 64 * 2.0 ** -18 * 2.0
    assert rel_l2(got, ref) < 1e-6
    bad = mass.copy()
    bad[777] = np.nan
    bad[100000] = np.inf
    got = host(ctx.paint(dev(pos), dev(bad)))
    i777 = np.floor(pos[:, 777]).astype(int)
    i1e5 = np.floor(pos[:, 100000]).astype(int)
    assert np.isnan(got[tuple(i777)]) and not np.isfinite(got[tuple(i1e5)])
    finite_ref = oracle.paint(pos.astype(np.float64), ng, mass=np.where(np.isfinite(bad), mass, 0.0).astype(np.float64))
    ok = np.isfinite(got)
    assert ok.sum() >= got.size - 16
    assert np.max(np.abs(got[ok] - finite_ref[ok]) - 2e-7 * np.abs(finite_ref[ok])) < 1e-3
