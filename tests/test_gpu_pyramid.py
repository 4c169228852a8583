"""the multi-grid pyramid (Eq. 6-9; Alg. 2-3) on the GPU
against the float64 oracle (pinned in tests/test_oracle_pyramid.py), and the paper's accuracy claim
(pyramid residuals 'sub-percent') as a study of the pyramid force against the single-mesh force."""
import numpy as np
import pytest

import fpm_inputs as fi
from gpu_util import dev, host, rel_l2

pytestmark = pytest.mark.gpu
OM = fi.COSMO["omega_m"]


@pytest.fixture(scope="module")
def fpm():
    import paper_2010_11847_b200 as m
    return m


@pytest.mark.parametrize("ng,levels", [(32, 1), (32, 2), (64, 2), (64, 3)])
def test_reduce_and_expand_match_oracle(fpm, oracle, ng, levels):
    rng = np.random.default_rng(ng + levels)
    fine = rng.standard_normal((ng, ng, ng)).astype(np.float32)
    nc = ng >> levels
    coarse = rng.standard_normal((nc, nc, nc)).astype(np.float32)
    ctx = fpm.FPM(ng)
    got = host(ctx.reduce(dev(fine), levels))
    ref = oracle.reduce(fine.astype(np.float64), levels)
    assert got.shape == (nc, nc, nc)
    assert np.max(np.abs(got - ref)) < 2e-6 * np.max(np.abs(ref))
    got = host(ctx.expand(dev(coarse), levels))
    ref = oracle.expand(coarse.astype(np.float64), levels)
    assert got.shape == (ng, ng, ng)
    assert np.max(np.abs(got - ref)) < 2e-6 * np.max(np.abs(ref))
    # Eq. 9 on the GPU path itself: g0 = L0 + EXPAND(g1) with L0 = g0 - EXPAND(REDUCE(g0))
    d_fine = dev(fine)
    low = ctx.expand(ctx.reduce(d_fine, 1), 1)
    lap = d_fine - low
    assert float((lap + low - d_fine).abs().max()) < 1e-6
    # zero levels: a copy
    assert np.array_equal(host(ctx.reduce(d_fine, 0)), fine)


@pytest.mark.parametrize("ng,nps,mode,levels", [(64, 32, 0, 1), (64, 64, 0, 2), (64, 64, 1, 2), (128, 64, 2, 2)])
def test_pyramid_force_matches_oracle(fpm, oracle, ng, nps, mode, levels):
    n = nps ** 3
    pos = fi.random_particles(n, ng, seed=ng + mode + levels, clustered=True)
    ctx = fpm.FPM(ng, nps, kernel_mode=mode)
    got = host(ctx.force_pyramid(dev(pos), levels)).astype(np.float64)
    ref = oracle.force_pyramid(pos.astype(np.float64), ng, levels=levels, mode=mode, scale=1.5 * OM,
                               mass=float((ng // nps) ** 3))
    assert rel_l2(got, ref) < 1e-5
    assert np.max(np.abs(got - ref)) < 1e-5 * np.max(np.abs(ref))
    if levels == 2 and mode == 0:
        single = host(ctx.force(dev(pos)))
        assert rel_l2(host(ctx.force_pyramid(dev(pos), 0)), single) < 1e-6      # no levels: the single-mesh force
    with pytest.raises(fpm.FpmError):
        ctx.force_pyramid(dev(pos), 5)                                           # ng >> levels must stay >= 8


def test_accuracy_of_the_pyramid_force_in_the_papers_configuration(fpm):
    """400 Mpc/h box, 128^3 mesh, force resolution 1, two reduction levels (global mesh 4x
    coarser).  The pyramid force against the single-mesh force at a = 0.1 (the first step) and at a = 1."""
    import torch
    ng = 128
    delta = dev(fi.linear_field(ng, 400.0, 1))
    stages = [0.1 + 0.09 * j for j in range(11)]
    for mode, tol in ((fpm.KERNEL_PAPER, 3e-2), (fpm.KERNEL_NAIVE, 5e-3)):
        ctx = fpm.FPM(ng, ng, omega_m=OM, box=400.0, kernel_mode=mode, force_path=fpm.FORCE_FUSED)
        pos, mom = ctx.lpt_init(delta, 0.1, 1)
        errs = []
        for evolve in (False, True):
            if evolve:
                ctx.nbody(pos, mom, stages)
            single = ctx.force(pos)
            pyr = ctx.force_pyramid(pos, 2)
            errs.append(float(torch.linalg.vector_norm(pyr - single) / torch.linalg.vector_norm(single)))
        print(f"pyramid vs single-mesh force, 128^3, kernel mode {mode}: rel-L2 {errs[0]:.2e} at a=0.1, {errs[1]:.2e} at a=1")
        assert max(errs) < tol


def test_pyramid_run_against_single_mesh_run_by_the_papers_own_metric(fpm, oracle):
    """PAPER.md:311-338 (section 6.1, Eq. 10-11, Fig. 7): a 5-step run from z = 9 to z = 0 on a 128^3 mesh in a
    400 Mpc/h box, 1LPT initial conditions, force resolution 1 -- once with the single-mesh force and once with
    the pyramid force (two reduction levels) -- compared by the transfer function T_f = sqrt(P_a / P_b) and the
    cross-correlation r_c = P_ab / sqrt(P_a P_b) of the final densities.  The paper reports both within 1e-4 of 1
    "across all scales" against FastPM, r_c "starting to deviate marginally on small scales", and the residuals
    of Fig. 6 "sub-percent".  This is the one check of reading R14 (the B-spline mask, the 2^levels force unit)
    against numbers the paper prints rather than against the oracle's restatement of the same reading: a wrong
    unit factor or a non-interpolating mask moves T_f by tens of percent on the scales the coarse mesh serves.
    Measured: with the exact symbols (-1/k^2, ik) on both meshes the reading is sub-percent on every scale; with
    Eq. 4-5 on both meshes T_f peaks at 2 % near k = 0.1 h/Mpc, where the 4x coarser mesh's finite-difference
    symbols differ from the fine mesh's at the same physical k (the paper does not say which kernels its coarse
    level uses) -- DESIGN.md R14.  Both runs share the kick/drift arithmetic below (fpm_step_factors)."""
    import torch
    ng, box = 128, 400.0
    delta = dev(fi.linear_field(ng, box, 1))
    stages = [0.1 + 0.18 * j for j in range(6)]
    worst = {}
    for mode in (fpm.KERNEL_NAIVE, fpm.KERNEL_PAPER):
        ctx = fpm.FPM(ng, ng, omega_m=OM, box=box, kernel_mode=mode, force_path=fpm.FORCE_FUSED)
        fac = ctx.step_factors(stages)
        rho = {}
        for name, force in (("single", ctx.force), ("pyramid", lambda p: ctx.force_pyramid(p, 2))):
            pos, mom = ctx.lpt_init(delta, 0.1, 1)
            for kf, df in fac:
                mom += force(pos) * kf
                pos = torch.remainder(pos + mom * df, float(ng))
                pos = torch.where(pos >= ng, pos - ng, pos).contiguous()
            rho[name] = host(ctx.paint(pos)).astype(np.float64)
        k, pa, _ = oracle.power(rho["pyramid"], box)
        _, pb, _ = oracle.power(rho["single"], box)
        _, pab, _ = oracle.power(rho["pyramid"], box, rho["single"])
        tf = np.sqrt(pa / pb)
        rc = pab / np.sqrt(pa * pb)
        worst[mode] = (float(np.abs(tf - 1).max()), float((1 - rc).max()))
        print(f"pyramid vs single-mesh run, 128^3 / 400 Mpc/h / 5 steps, kernel mode {mode}: max |T_f - 1| = "
              f"{worst[mode][0]:.2e} at k = {k[int(np.abs(tf - 1).argmax())]:.3f} h/Mpc, max 1 - r_c = "
              f"{worst[mode][1]:.2e} at k = {k[int((1 - rc).argmax())]:.3f} h/Mpc")
    # measured on a B200: 3.9e-4 / 8.3e-6 with the exact symbols, 2.1e-2 / 2.8e-3 with Eq. 4-5
    assert worst[fpm.KERNEL_NAIVE][0] < 1e-3 and worst[fpm.KERNEL_NAIVE][1] < 1e-4      # the paper's "within 0.01 %" order
    assert worst[fpm.KERNEL_PAPER][0] < 3e-2 and worst[fpm.KERNEL_PAPER][1] < 1e-2
