"""GPU parity: transfer function, one force evaluation, kick, drift, LPT and whole runs vs the
oracle.  Tolerances are the north_star's: relative L2 <= 1e-5
on density and forces per step; final positions within 1e-3 cell and P(k) within 1e-4 per bin."""
import numpy as np
import pytest

import fpm_inputs as fi
from gpu_util import dev, host, periodic_dist, rel_l2

pytestmark = pytest.mark.gpu
OM = fi.COSMO["omega_m"]


@pytest.fixture(scope="module")
def fpm():
    import paper_2010_11847_b200 as fpm
    return fpm


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_apply_force_kernel_matches_oracle(fpm, oracle, mode):
    ng = 32
    rng = np.random.default_rng(mode)
    dk = np.fft.rfftn(rng.standard_normal((ng, ng, ng))).astype(np.complex64)
    ctx = fpm.FPM(ng, kernel_mode=mode, workspace=False)
    got = ctx.apply_force_kernel(dev(dk), scale=1.5 * OM)
    ref = oracle.apply_force_kernel(dk.astype(np.complex128), mode=mode, scale=1.5 * OM)
    for d in range(3):
        g = host(got[d])
        assert rel_l2(g, ref[d]) < 1e-6
        idx = [slice(None)] * 3
        idx[d] = ng // 2
        assert np.all(g[tuple(idx)] == 0)            # Nyquist plane of axis d is exactly zero
        assert g[0, 0, 0] == 0


def test_growth_and_factors_match_oracle(fpm, oracle):
    ctx = fpm.FPM(16, workspace=False)
    for a in (0.1, 0.37, 1.0):
        g, r = ctx.growth(a), oracle.growth(OM, a)
        for k in r:
            assert g[k] == pytest.approx(r[k], rel=1e-7)
    assert ctx.drift_factor(0.1, 0.2, 0.3) == pytest.approx(oracle.drift_factor(OM, 0.1, 0.2, 0.3), rel=1e-7)
    assert ctx.kick_factor(0.1, 0.2, 0.3) == pytest.approx(oracle.kick_factor(OM, 0.1, 0.2, 0.3), rel=1e-7)
    cq = fpm.FPM(16, factor_mode=1, workspace=False)
    assert cq.drift_factor(0.1, 0.2, 0.3) == pytest.approx(oracle.drift_factor(OM, 0.1, 0.2, 0.3, 1), rel=1e-9)
    assert cq.kick_factor(0.1, 0.2, 0.3) == pytest.approx(oracle.kick_factor(OM, 0.1, 0.2, 0.3, 1), rel=1e-9)


def test_step_factors_are_the_merged_leapfrog_factors(fpm, oracle):
    """fpm_step_factors (R6): half step at sqrt(a_j a_j+1); the second half kick of step j-1 and the first of
    step j share one force evaluation.  Rebuilt here from the oracle's kick/drift factors."""
    stages = fi.CONFIGS["C2"].stages()
    n = len(stages) - 1
    for factor_mode in (0, 1):
        ctx = fpm.FPM(16, factor_mode=factor_mode, workspace=False)
        got = ctx.step_factors(stages)
        assert len(got) == n + 1
        pending = 0.0
        for j in range(n + 1):
            kf, dr = pending, 0.0
            if j < n:
                ai, af = stages[j], stages[j + 1]
                ah = (ai * af) ** 0.5
                kf += oracle.kick_factor(OM, ai, ai, ah, factor_mode)
                dr = oracle.drift_factor(OM, ai, ah, af, factor_mode)
                pending = oracle.kick_factor(OM, ah, af, af, factor_mode)
            assert got[j][0] == pytest.approx(kf, rel=1e-7) and got[j][1] == pytest.approx(dr, rel=1e-7, abs=0.0)
    assert got[n][1] == 0.0
    assert ctx.step_factors([0.5]) == [(0.0, 0.0)]
    with pytest.raises(fpm.FpmError):
        ctx.step_factors([0.1, -0.2])


@pytest.mark.parametrize("force_path", [0, 1])
@pytest.mark.parametrize("ng,nps,mode", [(32, 32, 0), (64, 32, 0), (64, 64, 1), (64, 64, 2), (128, 128, 0)])
def test_force_evaluation_matches_oracle(fpm, oracle, ng, nps, mode, force_path):
    """paint -> r2c -> kernel -> 3 c2r -> readout at a clustered (a ~ 1-like) particle set, with the
    transfer function as its own kernel (force_path 0) and fused into the FFT passes (1)."""
    n = nps ** 3
    pos = fi.random_particles(n, ng, seed=ng + mode, clustered=True)
    ctx = fpm.FPM(ng, nps, kernel_mode=mode, force_path=force_path)
    got = host(ctx.force(dev(pos)))
    ref, rho = oracle.force(pos.astype(np.float64), ng, mode=mode, scale=1.5 * OM,
                            mass=float((ng // nps) ** 3), return_rho=True)
    assert rel_l2(host(ctx.workspace_density()), rho) < 1e-5
    assert rel_l2(got, ref) < 1e-5
    # net momentum conservation on the GPU path itself
    assert np.max(np.abs(got.astype(np.float64).sum(axis=1))) < 1e-4 * np.sqrt(np.mean(ref ** 2)) * n


@pytest.mark.parametrize("ng,nps,mode", [(64, 64, 0), (64, 32, 1), (128, 128, 0), (128, 64, 2)])
def test_fused_force_through_the_global_tile_movers_matches_oracle(fpm, oracle, ng, nps, mode):
    """The chain a driver without cuTensorMapEncodeTiled gets (fpm_set_tile_movers(FPM_MOVERS_GLOBAL): forward y
    by launch_cols, fft_x_force_kernel, fft_y_inv3_pair_kernel), against the oracle like the default chain --
    both the planar force meshes (fpm_force) and the interleaved mesh of the step kernels (fpm_pm_step) -- and
    the potential solve of fpm_force_vjp through the same movers."""
    import torch
    n = nps ** 3
    pos = fi.random_particles(n, ng, seed=ng + mode, clustered=True)
    ctx = fpm.FPM(ng, nps, kernel_mode=mode, force_path=fpm.FORCE_FUSED)
    assert ctx.tile_movers() == fpm.MOVERS_TENSOR_MAPS          # what a B200 driver provides
    ctx.set_tile_movers(fpm.MOVERS_GLOBAL)
    assert ctx.tile_movers() == fpm.MOVERS_GLOBAL
    mass = float((ng // nps) ** 3)
    ref = oracle.force(pos.astype(np.float64), ng, mode=mode, scale=1.5 * OM, mass=mass)
    d_pos = dev(pos)
    planar = host(ctx.force(d_pos))
    step = torch.zeros_like(d_pos)
    ctx.pm_step(d_pos.clone(), step, 1.0, 0.0)                  # mom = 0 + f(pos) * 1
    for got in (planar, host(step)):
        assert rel_l2(got, ref) < 1e-5
        assert np.max(np.abs(got - ref)) < 1e-5 * np.max(np.abs(ref))
    v = np.random.default_rng(5).standard_normal((3, n)).astype(np.float32)
    got = host(ctx.force_vjp(d_pos, dev(v), coef=0.37))
    ref = 0.37 * oracle.force_vjp(pos.astype(np.float64), ng, v.astype(np.float64), mode=mode, scale=1.5 * OM, mass=mass)
    assert rel_l2(got, ref) < 1e-4
    ctx.set_tile_movers(fpm.MOVERS_AUTO)
    assert ctx.tile_movers() == fpm.MOVERS_TENSOR_MAPS
    assert rel_l2(host(ctx.force(d_pos)), planar) < 1e-6
    with pytest.raises(fpm.FpmError):
        ctx.set_tile_movers(7)


def test_zero_force_on_lattice(fpm):
    for ng, nps in ((32, 32), (32, 16)):
        b = ng // nps
        g = np.arange(nps, dtype=np.float32) * b
        q = np.stack(np.meshgrid(g, g, g, indexing="ij")).reshape(3, -1)
        ctx = fpm.FPM(ng, nps)
        assert float(ctx.force(dev(q)).abs().max()) < 1e-6


def test_kick_and_drift_match_oracle(fpm, oracle):
    ng, n = 64, 100003           # odd n: exercises the unaligned / tail path
    rng = np.random.default_rng(0)
    pos = fi.random_particles(n, ng, seed=1)
    mom = rng.standard_normal((3, n)).astype(np.float32) * 3
    f = rng.standard_normal((3, n)).astype(np.float32)
    ctx = fpm.FPM(ng, workspace=False)
    ai, ac, af = 0.3, 0.35, 0.4
    got_p = host(ctx.kick(dev(mom), dev(f), ai, ac, af))
    ref_p = oracle.kick(mom.astype(np.float64), f.astype(np.float64), oracle.kick_factor(OM, ai, ac, af))
    assert rel_l2(got_p, ref_p) < 1e-6
    got_x = host(ctx.drift(dev(pos), dev(mom), ai, ac, af))
    ref_x = oracle.drift(pos.astype(np.float64), mom.astype(np.float64), oracle.drift_factor(OM, ai, ac, af), ng)
    assert np.max(periodic_dist(got_x, ref_x, ng)) < 2e-5
    assert got_x.min() >= 0 and got_x.max() < ng
    # large momenta wrap several boxes
    big = (mom * 1000).astype(np.float32)
    got_x = host(ctx.drift(dev(pos), dev(big), ai, ac, af))
    assert got_x.min() >= 0 and got_x.max() < ng


@pytest.mark.parametrize("name,order", [("C1", 1), ("C1", 2)])
def test_lpt_init_matches_oracle(fpm, oracle, name, order):
    cfg = fi.CONFIGS[name]
    delta = fi.linear_field(cfg.np_side, cfg.box, cfg.seed)
    ctx = fpm.FPM(cfg.ng, cfg.np_side, box=cfg.box)
    pos, mom = ctx.lpt_init(dev(delta), cfg.a0, order)
    rpos, rmom = oracle.lpt_init(delta.astype(np.float64), cfg.ng, OM, cfg.a0, order)
    assert np.max(periodic_dist(host(pos), rpos, cfg.ng)) < 2e-5
    assert rel_l2(host(mom), rmom) < 1e-5


def test_lpt_init_with_resolution_factor_two(fpm, oracle):
    nps, ng, box = 32, 64, 100.0
    delta = fi.linear_field(nps, box, 2)
    ctx = fpm.FPM(ng, nps, box=box)
    pos, mom = ctx.lpt_init(dev(delta), 0.1, 2)
    rpos, rmom = oracle.lpt_init(delta.astype(np.float64), ng, OM, 0.1, 2)
    assert np.max(periodic_dist(host(pos), rpos, ng)) < 4e-5
    assert rel_l2(host(mom), rmom) < 1e-5


def _run_config(fpm, oracle, cfg, order, force_path=0):
    delta = fi.linear_field(cfg.np_side, cfg.box, cfg.seed)
    ctx = fpm.FPM(cfg.ng, cfg.np_side, box=cfg.box, force_path=force_path)
    pos, mom = ctx.lpt_init(dev(delta), cfg.a0, order)
    # the oracle starts from the SAME fp32 initial state, widened
    p0, m0 = host(pos).astype(np.float64), host(mom).astype(np.float64)
    stages = cfg.stages()
    ctx.nbody(pos, mom, stages)
    rpos, rmom = oracle.nbody(p0, m0, cfg.ng, cfg.np_side, OM, stages)
    return ctx, host(pos), host(mom), rpos, rmom


@pytest.mark.parametrize("force_path", [0, 1])
def test_full_run_C1_matches_oracle(fpm, oracle, force_path):
    cfg = fi.CONFIGS["C1"]
    ctx, pos, mom, rpos, rmom = _run_config(fpm, oracle, cfg, cfg.lpt_order, force_path)
    dist = periodic_dist(pos, rpos, cfg.ng)
    assert dist.max() < 1e-3, f"max {dist.max():.2e} rms {np.sqrt((dist**2).mean()):.2e}"
    assert rel_l2(mom, rmom) < 1e-4
    b3 = float(cfg.resolution_factor ** 3)
    k, pk_ref, nm = oracle.power(oracle.paint(rpos, cfg.ng, mass_const=b3), cfg.box)
    _, pk_got, _ = oracle.power(oracle.paint(pos.astype(np.float64), cfg.ng, mass_const=b3), cfg.box)
    assert np.max(np.abs(pk_got / pk_ref - 1)) < 1e-4


@pytest.mark.parametrize("np_side,ng", [(64, 64), (32, 64)])
def test_short_run_fused_path_spanning_several_bricks(fpm, oracle, np_side, ng):
    """4 FastPM steps through the fused path (interleaved force mesh, pipelined brick readout)."""
    cfg = fi.Config("T", np_side, ng, 100.0, 2, 4)
    ctx, pos, mom, rpos, rmom = _run_config(fpm, oracle, cfg, 2, force_path=1)
    dist = periodic_dist(pos, rpos, cfg.ng)
    assert dist.max() < 1e-3, f"max {dist.max():.2e}"
    assert rel_l2(mom, rmom) < 1e-4


@pytest.mark.parametrize("force_path", [0, 1])
def test_pm_step_with_arbitrary_particle_count(fpm, oracle, force_path):
    """n is not a lattice set: the generic (non-brick) kernels run; one PM step against the oracle."""
    ng, n = 32, 5003
    pos = fi.random_particles(n, ng, 17, clustered=True)
    mom = (0.1 * np.random.default_rng(3).standard_normal((3, n))).astype(np.float32)
    ctx = fpm.FPM(ng, ng, force_path=force_path)
    kf, dr = ctx.kick_factor(0.2, 0.2, 0.3), ctx.drift_factor(0.2, 0.25, 0.3)
    dpos, dmom = dev(pos), dev(mom)
    ctx.pm_step(dpos, dmom, kf, dr)
    f = oracle.force(pos.astype(np.float64), ng, scale=1.5 * OM, mass=1.0)
    rmom = oracle.kick(mom.astype(np.float64), f, kf)
    rpos = oracle.drift(pos.astype(np.float64), rmom, dr, ng)
    assert rel_l2(host(dmom), rmom) < 1e-5
    assert periodic_dist(host(dpos), rpos, ng).max() < 1e-4


def test_full_run_C2_matches_oracle(fpm, oracle):
    """BASELINE.json configs[1]: 128^3 / 128^3, 2LPT, 10 steps to a = 1, through the fused path."""
    cfg = fi.CONFIGS["C2"]
    ctx, pos, mom, rpos, rmom = _run_config(fpm, oracle, cfg, cfg.lpt_order, force_path=1)
    dist = periodic_dist(pos, rpos, cfg.ng)
    rms, p9999 = np.sqrt((dist ** 2).mean()), np.quantile(dist, 0.9999)
    assert dist.max() < 1e-3, f"max {dist.max():.2e} p99.99 {p9999:.2e} rms {rms:.2e}"
    assert rel_l2(mom, rmom) < 1e-4
    k, pk_ref, nm = oracle.power(oracle.paint(rpos, cfg.ng), cfg.box)
    _, pk_got, _ = oracle.power(oracle.paint(pos.astype(np.float64), cfg.ng), cfg.box)
    assert np.max(np.abs(pk_got / pk_ref - 1)) < 1e-4


def test_full_run_naive_kernel_and_quinn_factors(fpm, oracle):
    """C1 through the fused path with the other option of each switch: -1/k^2, ik kernels (R3d) and the
    plain Quinn et al. kick/drift integrals (R4)."""
    cfg = fi.CONFIGS["C1"]
    delta = fi.linear_field(cfg.np_side, cfg.box, cfg.seed)
    ctx = fpm.FPM(cfg.ng, cfg.np_side, box=cfg.box, kernel_mode=fpm.KERNEL_NAIVE, factor_mode=fpm.FACTORS_QUINN,
                  force_path=1)
    pos, mom = ctx.lpt_init(dev(delta), cfg.a0, cfg.lpt_order)
    p0, m0 = host(pos).astype(np.float64), host(mom).astype(np.float64)
    ctx.nbody(pos, mom, cfg.stages())
    rpos, rmom = oracle.nbody(p0, m0, cfg.ng, cfg.np_side, OM, cfg.stages(), mode=oracle.KERNEL_NAIVE,
                              factor_mode=oracle.FACTORS_QUINN)
    assert periodic_dist(host(pos), rpos, cfg.ng).max() < 1e-3
    assert rel_l2(host(mom), rmom) < 1e-4
