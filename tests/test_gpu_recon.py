"""GPU parity of the MAP-reconstruction calls (Eq. 12, Listing 7.1)
against the float64 oracle on the same fp32 inputs."""
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


def _problem(np_side, ng, box, n_steps, sigma, oracle):
    truth = fi.linear_field(np_side, box, 6)
    stages = list(np.linspace(0.1, 1.0, n_steps + 1))
    p, m = oracle.lpt_init(truth.astype(np.float64), ng, OM, stages[0], 2)
    pf, _ = oracle.nbody(p, m, ng, np_side, OM, stages)
    data = (oracle.paint(pf, ng, mass_const=float((ng // np_side) ** 3)) + fi.noise_field(ng, sigma)).astype(np.float32)
    return truth, stages, data, fi.inverse_prior_power(np_side, box)


# gradient tolerance: the GPU differentiates along its own fp32 trajectory, the oracle along its float64
# one (with the SAME trajectory the drivers agree to 1e-4, tests/test_gpu_backward.py); dW/dx of CIC jumps
# at cell faces, and with two mesh cells per particle spacing (B = 2) twice as many faces are crossed.
@pytest.mark.parametrize("np_side,ng,n_steps,force_path,gtol", [(32, 32, 3, 1, 1e-3), (32, 32, 3, 0, 1e-3),
                                                                 (32, 64, 2, 1, 1e-2)])
def test_loss_and_gradient_match_oracle(fpm, oracle, np_side, ng, n_steps, force_path, gtol):
    box, sigma = 100.0, 0.7
    truth, stages, data, ip = _problem(np_side, ng, box, n_steps, sigma, oracle)
    s = (0.5 * fi.linear_field(np_side, box, 8)).astype(np.float32)
    ctx = fpm.FPM(ng, np_side, box=box, force_path=force_path)
    (chi2, prior), grad = ctx.recon_loss_grad(dev(s), dev(data), sigma, dev(ip), stages, 2)
    (rchi2, rprior), rgrad = oracle.recon_loss_grad(s.astype(np.float64), ng, OM, stages[0], 2, stages,
                                                    data.astype(np.float64), sigma, ip.astype(np.float64))
    assert chi2 == pytest.approx(rchi2, rel=1e-4)      # fp32 run vs float64 run, summed over the mesh
    assert prior == pytest.approx(rprior, rel=1e-5)
    assert rel_l2(host(grad), rgrad) < gtol
    # and against a float64 directional finite difference of the oracle's loss
    d64, s64, ip64 = data.astype(np.float64), s.astype(np.float64), ip.astype(np.float64)
    dd = np.random.default_rng(12).standard_normal(s64.shape)
    eps = 1e-5
    lp = sum(oracle.recon_loss_grad(s64 + eps * dd, ng, OM, stages[0], 2, stages, d64, sigma, ip64)[0])
    lm = sum(oracle.recon_loss_grad(s64 - eps * dd, ng, OM, stages[0], 2, stages, d64, sigma, ip64)[0])
    assert float(np.sum(host(grad).astype(np.float64) * dd)) == pytest.approx((lp - lm) / (2 * eps), rel=10 * gtol)


def test_adam_step_matches_oracle(fpm, oracle):
    import torch
    rng = np.random.default_rng(3)
    n = 100003
    x, g1, g2 = (rng.standard_normal(n).astype(np.float32) for _ in range(3))
    ctx = fpm.FPM(16, 16)
    dx, dm, dv = dev(x), torch.zeros(n, device="cuda"), torch.zeros(n, device="cuda")
    rx, rm, rv = x.astype(np.float64), np.zeros(n), np.zeros(n)
    for t, g in ((1, g1), (2, g2)):
        ctx.adam_step(dx, dev(g), dm, dv, 0.1, t)
        rx, rm, rv = oracle.adam_step(rx, g.astype(np.float64), rm, rv, 0.1, t)
    assert rel_l2(host(dx), rx) < 1e-6 and rel_l2(host(dm), rm) < 1e-6 and rel_l2(host(dv), rv) < 1e-6


def test_adam_step_refuses_short_state_tensors(fpm):
    """grad, m and v are indexed up to x.numel() behind the C-ABI: a short one must be refused by the binding."""
    import torch
    ctx = fpm.FPM(16)
    x = torch.zeros(4096, device="cuda")
    ok = torch.zeros(4096, device="cuda")
    short = torch.zeros(4095, device="cuda")
    for args in ((short, ok, ok), (ok, short, ok), (ok, ok, short)):
        with pytest.raises(fpm.FpmError, match="expected 4096 elements"):
            ctx.adam_step(x, *args, 0.1, 1)
    ctx.adam_step(x, ok, ok.clone(), ok.clone(), 0.1, 1)


def test_reconstruction_loop_descends_like_the_oracle(fpm, oracle):
    """12 Adam iterations from s = 0 (Listing 7.1 train loop): GPU and oracle losses track each other."""
    import torch
    np_side = ng = 32
    box, sigma, lr = 100.0, 0.7, 0.05
    truth, stages, data, ip = _problem(np_side, ng, box, 3, sigma, oracle)
    ctx = fpm.FPM(ng, np_side, box=box, force_path=1)
    s = torch.zeros(np_side, np_side, np_side, device="cuda")
    m, v = torch.zeros_like(s), torch.zeros_like(s)
    d_data, d_ip = dev(data), dev(ip)
    rs = np.zeros((np_side,) * 3)
    rm, rv = np.zeros_like(rs), np.zeros_like(rs)
    gl, ol = [], []
    for t in range(1, 13):
        (a, b), g = ctx.recon_loss_grad(s, d_data, sigma, d_ip, stages, 2)
        ctx.adam_step(s, g, m, v, lr, t)
        gl.append(a + b)
        (ra, rb), rg = oracle.recon_loss_grad(rs, ng, OM, stages[0], 2, stages, data.astype(np.float64), sigma,
                                              ip.astype(np.float64))
        rs, rm, rv = oracle.adam_step(rs, rg, rm, rv, lr, t)
        ol.append(ra + rb)
    assert gl[-1] < 0.9 * gl[0] and all(b < a for a, b in zip(gl, gl[1:]))
    assert np.allclose(gl, ol, rtol=2e-3)
    assert rel_l2(host(s), rs) < 1e-2


def test_reconstruction_recovers_the_large_scale_field(fpm, oracle):
    """The paper's toy problem (Fig. 13-14) at 64^3: 200 Adam iterations from s = 0 on
    synthetic data (own forward run of a seeded truth + unit Gaussian noise).  The cross-correlation
    coefficient r_c (Eq. 11) of the reconstruction with the truth must be close to 1 on
    large scales ("the reconstruction is near perfect on the large scales") and the
    likelihood term must reach the noise level, chi2 ~ n_cells / 2."""
    import torch
    n, box, sigma, lr = 64, 200.0, 1.0, 0.02
    stages = [0.1 + j * 0.9 / 5 for j in range(6)]
    ctx = fpm.FPM(n, n, box=box, force_path=1)
    truth = fi.linear_field(n, box, 6)
    p, m = ctx.lpt_init(dev(truth), stages[0], 2)
    ctx.nbody(p, m, stages)
    data = ctx.paint(p) + dev(fi.noise_field(n, sigma))
    ip = dev(fi.inverse_prior_power(n, box))
    s = torch.zeros(n, n, n, device="cuda")
    am, av = torch.zeros_like(s), torch.zeros_like(s)
    first = None
    for t in range(1, 201):
        (chi2, prior), g = ctx.recon_loss_grad(s, data, sigma, ip, stages, 2)
        first = first if first is not None else chi2 + prior
        ctx.adam_step(s, g, am, av, lr, t)
    assert chi2 + prior < 0.3 * first
    assert 0.4 * n ** 3 < chi2 < 0.6 * n ** 3
    rec, tru = host(s).astype(np.float64), truth.astype(np.float64)
    k, pab, _ = oracle.power(rec, box, tru)
    _, paa, _ = oracle.power(rec, box)
    _, pbb, _ = oracle.power(tru, box)
    rc = pab / np.sqrt(paa * pbb)
    assert np.all(rc[k < 0.12] > 0.9), rc[:6]
    assert rc[k < 0.2].min() > 0.75
