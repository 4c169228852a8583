"""Seeded input generators: counter-based noise, Eisenstein-Hu no-wiggle P(k), linear field.

Follows SURVEY.md section 8(c) R7-R8 (Alg. 4 lines 1-2 of the paper, PAPER.md:367-369:
"sample 3D normal random field of size N; scale g by power spectrum pk").  Library FFTs
(scipy) are used here because this is input manufacture, not a step of the method.
"""
import math

import numpy as np
import scipy.fft as sfft

from .configs import COSMO

_U64 = np.uint64
_GOLDEN = _U64(0x9E3779B97F4A7C15)


def _splitmix64(z):
    """SplitMix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (z + _GOLDEN).astype(_U64)
        z = ((z ^ (z >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)).astype(_U64)
        z = ((z ^ (z >> _U64(27))) * _U64(0x94D049BB133111EB)).astype(_U64)
        return z ^ (z >> _U64(31))


def counter_uniform(seed, index, stream=0):
    """Uniform in (0,1) keyed by (seed, stream, index): the same value at any array size."""
    index = np.asarray(index, dtype=_U64)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.asarray(_U64(seed) * _U64(0xD1342543DE82EF95) + _U64(stream), dtype=_U64))
        z = _splitmix64(index * _U64(0xA0761D6478BD642F) ^ key)
    return ((z >> _U64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def counter_normal(seed, index):
    """Standard normal keyed by (seed, index): Box-Muller on two counter uniforms, float64."""
    u1 = counter_uniform(seed, index, stream=1)
    u2 = counter_uniform(seed, index, stream=2)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


def _normal_grid(seed, n, dtype=np.float64, chunk=1 << 24):
    out = np.empty(n ** 3, dtype=dtype)
    for s in range(0, n ** 3, chunk):
        e = min(n ** 3, s + chunk)
        out[s:e] = counter_normal(seed, np.arange(s, e, dtype=np.uint64))
    return out.reshape(n, n, n)


# ----------------------------------------------------------------------------------------
# Eisenstein & Hu (1998) zero-baryon-oscillation ("no-wiggle") transfer function, R8.
# ----------------------------------------------------------------------------------------
def eh_sound_horizon_and_alpha(cosmo=COSMO):
    om, h, ob = cosmo["omega_m"], cosmo["h"], cosmo["omega_b"]
    omh2, obh2, fb = om * h * h, ob * h * h, ob / om
    s = 44.5 * math.log(9.83 / omh2) / math.sqrt(1.0 + 10.0 * obh2 ** 0.75)  # Mpc
    alpha = 1.0 - 0.328 * math.log(431.0 * omh2) * fb + 0.38 * math.log(22.3 * omh2) * fb * fb
    return s, alpha


def eh_nowiggle_transfer(k, cosmo=COSMO):
    """T(k), k in h/Mpc."""
    k = np.asarray(k, dtype=np.float64)
    om, h = cosmo["omega_m"], cosmo["h"]
    theta = cosmo["t_cmb"] / 2.7
    s, alpha = eh_sound_horizon_and_alpha(cosmo)
    kmpc = k * h  # 1/Mpc
    gamma_eff = om * h * (alpha + (1.0 - alpha) / (1.0 + (0.43 * kmpc * s) ** 4))
    q = k * theta * theta / gamma_eff
    l0 = np.log(2.0 * math.e + 1.8 * q)
    c0 = 14.2 + 731.0 / (1.0 + 62.5 * q)
    return l0 / (l0 + c0 * q * q)


def _tophat(x):
    x = np.asarray(x, dtype=np.float64)
    small = x < 1e-3
    xs = np.where(small, 1.0, x)
    w = 3.0 * (np.sin(xs) - xs * np.cos(xs)) / xs ** 3
    return np.where(small, 1.0 - x * x / 10.0, w)


def sigma_r(r, amplitude, cosmo=COSMO, nk=20000):
    """sqrt of (1/2pi^2) int k^2 P(k) W^2(kR) dk by log-k trapezoid over 1e-5..1e2 h/Mpc."""
    lnk = np.linspace(math.log(1e-5), math.log(1e2), nk)
    k = np.exp(lnk)
    pk = amplitude * k ** cosmo["n_s"] * eh_nowiggle_transfer(k, cosmo) ** 2
    integrand = k ** 3 * pk * _tophat(k * r) ** 2 / (2.0 * math.pi ** 2)
    return math.sqrt(np.trapezoid(integrand, lnk))


_AMP_CACHE = {}


def power_amplitude(cosmo=COSMO):
    """A in P = A k^ns T^2 fixed by sigma8 with a top-hat of 8 Mpc/h (a = 1)."""
    key = tuple(sorted(cosmo.items()))
    if key not in _AMP_CACHE:
        _AMP_CACHE[key] = (cosmo["sigma8"] / sigma_r(8.0, 1.0, cosmo)) ** 2
    return _AMP_CACHE[key]


def linear_power(k, cosmo=COSMO):
    """Linear P(k) at a = 1 in (Mpc/h)^3, k in h/Mpc; P(0) = 0."""
    k = np.asarray(k, dtype=np.float64)
    kk = np.where(k > 0, k, 1.0)
    p = power_amplitude(cosmo) * kk ** cosmo["n_s"] * eh_nowiggle_transfer(kk, cosmo) ** 2
    return np.where(k > 0, p, 0.0)


def linear_field(np_side, box, seed, cosmo=COSMO):
    """delta_L(x) at a = 1 on the Np^3 grid, float32 (R7).

    g ~ N(0,1) per cell from the counter generator; delta_k = g_k sqrt(P(k)/V_cell);
    the k = 0 mode is zero; the field is real by construction (irfftn of rfftn).
    """
    n = int(np_side)
    work = np.float64 if n <= 512 else np.float32
    g = _normal_grid(seed, n, dtype=work)
    gk = sfft.rfftn(g, workers=-1)
    del g
    kf = 2.0 * math.pi / box
    vcell = (box / n) ** 3
    fx = np.fft.fftfreq(n, 1.0 / n)
    fz = np.arange(n // 2 + 1, dtype=np.float64)
    for i in range(n):  # slab by slab to bound memory
        k2 = fx[i] ** 2 + fx[:, None] ** 2 + fz[None, :] ** 2
        amp = np.sqrt(linear_power(kf * np.sqrt(k2), cosmo) / vcell)
        gk[i] *= amp.astype(gk.real.dtype)
    gk[0, 0, 0] = 0.0
    out = sfft.irfftn(gk, s=(n, n, n), workers=-1)
    return np.ascontiguousarray(out, dtype=np.float32)


def inverse_prior_power(np_side, box, cosmo=COSMO):
    """Table 1/<|s_k|^2> of the Gaussian prior of N1 (Eq. 12; Listing 7.1 "r2c(var)^2/power")
    on the half-complex layout [n][n][n/2+1], float32: for the field of linear_field(), the unnormalised
    DFT has <|s_k|^2> = n^3 P(k) / V_cell.  The k = 0 entry is 0 (the mean is not constrained)."""
    n = int(np_side)
    kf = 2.0 * math.pi / box
    vcell = (box / n) ** 3
    fx = np.fft.fftfreq(n, 1.0 / n)
    fz = np.arange(n // 2 + 1, dtype=np.float64)
    k2 = fx[:, None, None] ** 2 + fx[None, :, None] ** 2 + fz[None, None, :] ** 2
    var = n ** 3 * linear_power(kf * np.sqrt(k2), cosmo) / vcell
    out = np.where(var > 0, 1.0 / np.where(var > 0, var, 1.0), 0.0)
    return np.ascontiguousarray(out, dtype=np.float32)


def noise_field(ng, sigma, seed=202):
    """Uncorrelated Gaussian data noise of standard deviation sigma on the Ng mesh."""
    return (sigma * _normal_grid(seed, int(ng), dtype=np.float64)).astype(np.float32)


def weight_field(ng, seed=101):
    """Seeded N(0,1) weight field on the Ng mesh (objective of C4's backward pass, R12)."""
    return _normal_grid(seed, int(ng), dtype=np.float32)


def random_particles(n, ng, seed, clustered=False):
    """[3][n] float32 positions in [0, ng): uniform, or a clustered mixture (blobs + background).

    Used by the kernel-level parity tests for paint/readout (uneven clustering, R1/R10).
    """
    idx = np.arange(n, dtype=np.uint64)
    pos = np.empty((3, n), dtype=np.float64)
    for d in range(3):
        pos[d] = counter_uniform(seed, idx, stream=10 + d) * ng
    if clustered:
        nblob = 8
        which = (counter_uniform(seed, idx, stream=20) * (nblob + 2)).astype(np.int64)
        cidx = np.arange(nblob, dtype=np.uint64)
        for d in range(3):
            centre = counter_uniform(seed + 7919, cidx, stream=30 + d) * ng
            off = counter_normal(seed + 104729 + d, idx) * (0.02 * ng + 0.5)
            blob = which < nblob
            pos[d] = np.where(blob, centre[np.minimum(which, nblob - 1)] + off, pos[d])
        pos = np.mod(pos, ng)
    out = pos.astype(np.float32)
    out[out >= ng] = 0.0  # float32 rounding of values just below ng
    return out
