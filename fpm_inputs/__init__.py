"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no paint, FFT-as-a-method-step,
force kernel, growth factors, kick/drift, LPT): it only manufactures the *inputs*
of the particle-mesh path -- the Gaussian linear field of Alg. 4 lines 1-2
(PAPER.md:367-369), weight fields, random particle clouds -- and names the
BASELINE.json configurations.  Neither `oracle/` nor `paper_2010_11847_b200/`
is imported from here, and neither of them imports the other.
"""
from .configs import CONFIGS, COSMO, Config
from .fields import (
    counter_normal,
    counter_uniform,
    eh_nowiggle_transfer,
    eh_sound_horizon_and_alpha,
    inverse_prior_power,
    linear_field,
    linear_power,
    noise_field,
    power_amplitude,
    random_particles,
    sigma_r,
    weight_field,
)

__all__ = [
    "CONFIGS", "COSMO", "Config",
    "counter_normal", "counter_uniform", "eh_nowiggle_transfer",
    "eh_sound_horizon_and_alpha", "inverse_prior_power", "linear_field", "linear_power", "noise_field",
    "power_amplitude", "random_particles", "sigma_r", "weight_field",
]
