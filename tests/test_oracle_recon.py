"""Pins of the oracle's N1 functions (MAP reconstruction, Eq. 12, Listing 7.1):
the loss against its plain definition assembled from already-pinned pieces, the gradient against
central finite differences, the prior against its closed form, Adam against hand-computed steps."""
import numpy as np
import pytest

import fpm_inputs as fi

OM = 0.3075


def _setup(np_side=8, ng=8, box=50.0, n_steps=2, sigma=0.5):
    s = fi.linear_field(np_side, box, 5).astype(np.float64)
    truth = fi.linear_field(np_side, box, 6).astype(np.float64)
    stages = np.linspace(0.1, 1.0, n_steps + 1)
    inv_power = fi.inverse_prior_power(np_side, box).astype(np.float64)
    return s, truth, stages, inv_power, sigma


def _forward(oracle, s, ng, stages, order=2):
    p, m = oracle.lpt_init(s, ng, OM, stages[0], order)
    pf, _ = oracle.nbody(p, m, ng, s.shape[0], OM, stages)
    return oracle.paint(pf, ng, mass_const=float((ng // s.shape[0]) ** 3))


@pytest.mark.parametrize("np_side,ng", [(8, 8), (8, 16)])
def test_loss_is_eq12_assembled_from_pinned_pieces(oracle, np_side, ng):
    s, truth, stages, ip, sigma = _setup(np_side, ng)
    data = _forward(oracle, truth, ng, stages) + fi.noise_field(ng, sigma).astype(np.float64)
    (chi2, prior), _ = oracle.recon_loss_grad(s, ng, OM, stages[0], 2, stages, data, sigma, ip)
    rho = _forward(oracle, s, ng, stages)
    assert chi2 == pytest.approx(0.5 * np.sum((rho - data) ** 2) / sigma ** 2, rel=1e-12)
    sk = np.fft.fftn(s)                                   # full k-space, library routine
    ip_full = np.zeros(s.shape)
    nzh = np_side // 2 + 1
    ip_full[:, :, :nzh] = ip
    for z in range(nzh, np_side):                         # Hermitian half: inv_power is even in k
        ip_full[:, :, z] = ip[(-np.arange(np_side)) % np_side][:, (-np.arange(np_side)) % np_side, np_side - z]
    assert prior == pytest.approx(0.5 * np.sum(np.abs(sk) ** 2 * ip_full), rel=1e-12)


def test_prior_of_a_prior_sample_is_half_the_number_of_modes(oracle):
    """s drawn from the prior itself: <|s_k|^2 inv_power> = 1 per mode, so prior ~ (n^3 - 1)/2."""
    n, box = 16, 100.0
    s = fi.linear_field(n, box, 9).astype(np.float64)
    ip = fi.inverse_prior_power(n, box).astype(np.float64)
    data = np.ones((n, n, n))
    (_, prior), _ = oracle.recon_loss_grad(s, n, OM, 0.5, 1, [0.5], data, 1.0, ip)
    assert prior == pytest.approx(0.5 * (n ** 3 - 1), rel=5 * np.sqrt(2.0 / n ** 3))


@pytest.mark.parametrize("np_side,ng,order", [(8, 8, 1), (8, 8, 2), (8, 16, 2)])
def test_gradient_matches_finite_differences(oracle, np_side, ng, order):
    s, truth, stages, ip, sigma = _setup(np_side, ng)
    data = _forward(oracle, truth, ng, stages, order) + fi.noise_field(ng, sigma).astype(np.float64)

    def loss(x):
        (a, b), _ = oracle.recon_loss_grad(x, ng, OM, stages[0], order, stages, data, sigma, ip)
        return a + b

    _, g = oracle.recon_loss_grad(s, ng, OM, stages[0], order, stages, data, sigma, ip)
    for seed in (1, 2):
        d = np.random.default_rng(seed).standard_normal(s.shape)
        eps = 1e-6
        fd = (loss(s + eps * d) - loss(s - eps * d)) / (2 * eps)
        assert float(np.sum(g * d)) == pytest.approx(fd, rel=2e-6)


def test_gradient_vanishes_at_the_truth_without_noise_and_prior(oracle):
    s, truth, stages, ip, sigma = _setup()
    data = _forward(oracle, truth, 8, stages)
    (chi2, _), g = oracle.recon_loss_grad(truth, 8, OM, stages[0], 2, stages, data, sigma, 0.0 * ip)
    assert chi2 == 0.0 and np.max(np.abs(g)) == 0.0


def test_adam_first_steps_by_hand(oracle):
    x = np.array([1.0, -2.0, 0.5])
    g = np.array([0.3, -0.1, 0.0])
    m = v = np.zeros(3)
    lr, b1, b2, eps = 0.1, 0.9, 0.999, 1e-8
    x1, m1, v1 = oracle.adam_step(x, g, m, v, lr, 1)
    # step 1: m_hat = g, v_hat = g^2  ->  x -= lr g / (|g| + eps)
    assert x1 == pytest.approx(x - lr * g / (np.abs(g) + eps), rel=1e-14)
    assert m1 == pytest.approx(0.1 * g) and v1 == pytest.approx(0.001 * g * g)
    g2 = np.array([-0.2, 0.4, 0.1])
    x2, m2, v2 = oracle.adam_step(x1, g2, m1, v1, lr, 2)
    mh = (0.9 * 0.1 * g + 0.1 * g2) / (1 - 0.9 ** 2)
    vh = (0.999 * 0.001 * g * g + 0.001 * g2 * g2) / (1 - 0.999 ** 2)
    assert x2 == pytest.approx(x1 - lr * mh / (np.sqrt(vh) + eps), rel=1e-13)


def test_a_few_adam_iterations_reduce_the_loss(oracle):
    s, truth, stages, ip, sigma = _setup()
    data = _forward(oracle, truth, 8, stages) + fi.noise_field(8, sigma).astype(np.float64)
    x = np.zeros_like(s)
    m = v = np.zeros_like(s)
    losses = []
    for t in range(1, 9):
        (a, b), g = oracle.recon_loss_grad(x, 8, OM, stages[0], 2, stages, data, sigma, ip)
        losses.append(a + b)
        x, m, v = oracle.adam_step(x, g, m, v, 0.05, t)
    assert losses[-1] < 0.8 * losses[0]
