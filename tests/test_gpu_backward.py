"""GPU parity of the reverse-mode drivers
against the float64 oracle on the same fp32 inputs.  Tolerance: relative L2 <= 1e-4 (R12)."""
import numpy as np
import pytest

import fpm_inputs as fi
from gpu_util import dev, host, rel_l2

pytestmark = pytest.mark.gpu
OM = fi.COSMO["omega_m"]
TOL = 1e-4


@pytest.fixture(scope="module")
def fpm():
    import paper_2010_11847_b200 as m
    return m


@pytest.mark.parametrize("ng,nps,n,force_path", [(16, 16, 700, 0), (32, 32, 32 ** 3, 0), (32, 32, 32 ** 3, 1), (64, 32, 32 ** 3, 1)])
def test_force_vjp_matches_oracle(fpm, oracle, ng, nps, n, force_path):
    pos = fi.random_particles(n, ng, 21, clustered=True)
    v = np.random.default_rng(22).standard_normal((3, n)).astype(np.float32)
    ctx = fpm.FPM(ng, nps, force_path=force_path)
    mass = float((ng // nps) ** 3)
    got = host(ctx.force_vjp(dev(pos), dev(v), coef=0.37))
    ref = 0.37 * oracle.force_vjp(pos.astype(np.float64), ng, v.astype(np.float64), scale=1.5 * OM, mass=mass)
    assert rel_l2(got, ref) < TOL


@pytest.mark.parametrize("mode", [1, 2])
def test_force_vjp_other_kernel_modes(fpm, oracle, mode):
    """NAIVE (i k, -1/k^2) takes the three-transform adjoint path, MIXED the stencil-divergence path."""
    ng = nps = 32
    n = nps ** 3
    pos = fi.random_particles(n, ng, 23, clustered=True)
    v = np.random.default_rng(24).standard_normal((3, n)).astype(np.float32)
    for force_path in (0, 1):
        ctx = fpm.FPM(ng, nps, kernel_mode=mode, force_path=force_path)
        got = host(ctx.force_vjp(dev(pos), dev(v), coef=1.3))
        ref = 1.3 * oracle.force_vjp(pos.astype(np.float64), ng, v.astype(np.float64), mode=mode, scale=1.5 * OM)
        assert rel_l2(got, ref) < TOL


def test_force_vjp_accumulates_into_grad_pos(fpm):
    ng, n = 16, 500
    pos = dev(fi.random_particles(n, ng, 5))
    v = dev(np.random.default_rng(6).standard_normal((3, n)).astype(np.float32))
    ctx = fpm.FPM(ng, ng)
    g1 = ctx.force_vjp(pos, v)
    import torch
    g0 = torch.ones(3, n, device="cuda")
    g2 = ctx.force_vjp(pos, v, grad_pos=g0.clone())
    assert float((g2 - g1 - g0).abs().max()) <= 1e-5 * float(g1.abs().max())


@pytest.mark.parametrize("np_side,ng,n_steps,force_path", [(32, 32, 3, 0), (32, 32, 3, 1), (32, 64, 2, 1)])
def test_nbody_vjp_matches_oracle(fpm, oracle, np_side, ng, n_steps, force_path):
    import torch
    cfg = fi.Config("T", np_side, ng, 100.0, 2, n_steps)
    delta = fi.linear_field(np_side, cfg.box, 2)
    ctx = fpm.FPM(ng, np_side, box=cfg.box, force_path=force_path)
    pos, mom = ctx.lpt_init(dev(delta), cfg.a0, 2)
    n = np_side ** 3
    stages = cfg.stages()
    traj = torch.empty(n_steps + 1, 3, n, device="cuda")
    ctx.nbody(pos, mom, stages, traj=traj)
    rng = np.random.default_rng(31)
    gx, gp = rng.standard_normal((3, n)).astype(np.float32), rng.standard_normal((3, n)).astype(np.float32)
    dgx, dgp = dev(gx), dev(gp)
    ctx.nbody_vjp(traj, stages, dgx, dgp)
    # the oracle differentiates along the SAME (GPU, fp32) trajectory, widened
    rgx, rgp = oracle.nbody_vjp(host(traj).astype(np.float64), ng, np_side, OM, stages,
                                gx.astype(np.float64), gp.astype(np.float64))
    assert rel_l2(host(dgx), rgx) < TOL
    assert rel_l2(host(dgp), rgp) < TOL


def test_nbody_vjp_grad_mom_zero_flag_changes_nothing(fpm):
    """FPM_VJP_GRAD_MOM_ZERO skips the last force VJP, which adds kf * J^T 0 = 0 when grad_mom enters as zeros."""
    import torch
    cfg = fi.Config("T", 32, 32, 100.0, 2, 3)
    ctx = fpm.FPM(32, 32, box=cfg.box, force_path=1)
    pos, mom = ctx.lpt_init(dev(fi.linear_field(32, cfg.box, 2)), cfg.a0, 2)
    n, stages = 32 ** 3, cfg.stages()
    traj = torch.empty(4, 3, n, device="cuda")
    ctx.nbody(pos, mom, stages, traj=traj)
    gx = np.random.default_rng(5).standard_normal((3, n)).astype(np.float32)
    a_gx, a_gp = dev(gx), torch.zeros(3, n, device="cuda")
    b_gx, b_gp = dev(gx), torch.zeros(3, n, device="cuda")
    before = ctx.launch_count()
    ctx.nbody_vjp(traj, stages, a_gx, a_gp)
    mid = ctx.launch_count()
    ctx.nbody_vjp(traj, stages, b_gx, b_gp, grad_mom_is_zero=True)
    after = ctx.launch_count()
    assert after - mid < mid - before                    # one backward force evaluation fewer
    assert rel_l2(host(b_gx), host(a_gx)) < 1e-6 and rel_l2(host(b_gp), host(a_gp)) < 1e-6


def test_binding_refuses_wrongly_shaped_arrays(fpm):
    """a wrong shape must be an FpmError, not an out-of-bounds device access."""
    import torch
    ctx = fpm.FPM(32, 32)
    n = 32 ** 3
    pos, mom = torch.zeros(3, n, device="cuda"), torch.zeros(3, n, device="cuda")
    with pytest.raises(fpm.FpmError):
        ctx.nbody(pos[:, : n - 1].contiguous(), mom, [0.1, 0.2])
    with pytest.raises(fpm.FpmError):
        ctx.nbody(pos, mom, [0.1, 0.2], traj=torch.zeros(1, 3, n, device="cuda"))
    with pytest.raises(fpm.FpmError):
        ctx.paint(pos, out=torch.zeros(16, 16, 16, device="cuda"))
    with pytest.raises(fpm.FpmError):
        ctx.paint(torch.zeros(n, 3, device="cuda"))
    with pytest.raises(fpm.FpmError):
        ctx.fft_r2c(torch.zeros(32, 32, 16, device="cuda"))
    with pytest.raises(fpm.FpmError):
        ctx.nbody_vjp(torch.zeros(2, 3, n, device="cuda"), [0.1, 0.2, 0.3], pos, mom)
    with pytest.raises(fpm.FpmError):
        ctx.lpt_init(torch.zeros(16, 16, 16, device="cuda"), 0.1, 2)


@pytest.mark.parametrize("order,np_side,ng", [(1, 32, 32), (2, 32, 32), (2, 32, 64), (2, 64, 64)])
def test_lpt_init_vjp_matches_oracle(fpm, oracle, order, np_side, ng):
    delta = fi.linear_field(np_side, 100.0, 4)
    n = np_side ** 3
    rng = np.random.default_rng(41)
    gx, gp = rng.standard_normal((3, n)).astype(np.float32), rng.standard_normal((3, n)).astype(np.float32)
    ctx = fpm.FPM(ng, np_side)
    got = host(ctx.lpt_init_vjp(dev(delta), 0.1, order, dev(gx), dev(gp)))
    ref = oracle.lpt_init_vjp(delta.astype(np.float64), ng, OM, 0.1, order, gx.astype(np.float64), gp.astype(np.float64))
    assert rel_l2(got, ref) < TOL


def test_gradient_of_density_objective_C1(fpm, oracle):
    """C4's objective at C1 size: L = sum(final density x seeded weight field), gradient w.r.t. the
    linear field through adjoint paint -> nbody_vjp -> lpt_init_vjp, against the oracle chain and a
    float64 directional finite difference of the oracle forward model."""
    import torch
    cfg = fi.CONFIGS["C1"]
    ng, nps = cfg.ng, cfg.np_side
    delta = fi.linear_field(nps, cfg.box, cfg.seed)
    wfield = fi.weight_field(ng, 101)
    stages = cfg.stages()
    ctx = fpm.FPM(ng, nps, box=cfg.box, force_path=1)
    ddelta = dev(delta)
    pos, mom = ctx.lpt_init(ddelta, cfg.a0, cfg.lpt_order)
    n = nps ** 3
    traj = torch.empty(cfg.n_steps + 1, 3, n, device="cuda")
    ctx.nbody(pos, mom, stages, traj=traj)
    gx, _ = ctx.paint_adjoint(pos, dev(wfield), want_grad_mass=False)
    gp = torch.zeros_like(gx)
    ctx.nbody_vjp(traj, stages, gx, gp)
    gd = host(ctx.lpt_init_vjp(ddelta, cfg.a0, cfg.lpt_order, gx, gp)).astype(np.float64)

    d64, w64 = delta.astype(np.float64), wfield.astype(np.float64)
    p, m = oracle.lpt_init(d64, ng, OM, cfg.a0, cfg.lpt_order)
    pf, mf, otraj = oracle.nbody(p, m, ng, nps, OM, stages, return_traj=True)
    ogx, _ = oracle.paint_adjoint(pf, ng, w64)
    ogx0, ogp0 = oracle.nbody_vjp(otraj, ng, nps, OM, stages, ogx, np.zeros_like(ogx))
    ogd = oracle.lpt_init_vjp(d64, ng, OM, cfg.a0, cfg.lpt_order, ogx0, ogp0)
    assert rel_l2(gd, ogd) < 1e-3     # fp32 trajectory vs float64 trajectory through 5 nonlinear steps

    def loss(d):
        pp, mm = oracle.lpt_init(d, ng, OM, cfg.a0, cfg.lpt_order)
        pff, _ = oracle.nbody(pp, mm, ng, nps, OM, stages)
        return float(np.sum(oracle.paint(pff, ng) * w64))

    dd = np.random.default_rng(51).standard_normal(d64.shape)
    eps = 1e-5
    fd = (loss(d64 + eps * dd) - loss(d64 - eps * dd)) / (2 * eps)
    assert float(np.sum(gd * dd)) == pytest.approx(fd, rel=2e-3)
