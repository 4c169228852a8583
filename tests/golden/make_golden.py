"""Writes the stored expected values under tests/golden/ by calling ONLY oracle/ (and the seeded
input generators).  Run from the repo root:  python tests/golden/make_golden.py

The FlowPM paper prints no worked numeric example (every quantitative result is a plot), so these
fixtures are the float64 oracle's own outputs, frozen: they pin the oracle against silent changes of
its arithmetic (tests/test_golden.py) and give the GPU run a stored target.  Any later regeneration
must name, in its commit message, the passage or DESIGN.md reading that justifies the change.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import fpm_inputs as fi  # noqa: E402
import oracle  # noqa: E402


def c1_run():
    """BASELINE.json configs[0] (C1): 32^3 / 32^3, box 100 Mpc/h, 1LPT at a = 0.1, 5 steps to a = 1."""
    cfg = fi.CONFIGS["C1"]
    om = fi.COSMO["omega_m"]
    delta = fi.linear_field(cfg.np_side, cfg.box, cfg.seed).astype(np.float64)
    pos, mom = oracle.lpt_init(delta, cfg.ng, om, cfg.a0, cfg.lpt_order)
    pos, mom = oracle.nbody(pos, mom, cfg.ng, cfg.np_side, om, cfg.stages())
    k, pk, nm = oracle.power(oracle.paint(pos, cfg.ng), cfg.box)
    return k, pk, nm, pos, mom


def main():
    om = fi.COSMO["omega_m"]
    with open(os.path.join(HERE, "growth_table.txt"), "w") as f:
        f.write("# oracle.growth(omega_m = 0.3075, a): SURVEY.md 8(c) R5 (growth ODE, RK4, D1(1) = 1); paper silent\n")
        f.write("# (PAPER.md:29, 45 defer to Feng et al. 2016).  Written by tests/golden/make_golden.py.\n")
        f.write("# a D1 f1 D2 f2 E\n")
        for a in (0.1, 0.2, 0.3, 0.4, 0.5, 0.6, 0.7, 0.8, 0.9, 1.0):
            g = oracle.growth(om, a)
            f.write(f"{a:.1f} {g['D1']:.12e} {g['f1']:.12e} {g['D2']:.12e} {g['f2']:.12e} {g['E']:.12e}\n")
    k, pk, nm, pos, mom = c1_run()
    with open(os.path.join(HERE, "c1_oracle_power.txt"), "w") as f:
        f.write("# Final-density power spectrum of the float64 oracle run of C1 (BASELINE.json configs[0];\n")
        f.write("# Alg. 4 ICs PAPER.md:363-383, leapfrog PAPER.md:37-45, force PAPER.md:47-59; binning SURVEY.md R13).\n")
        f.write("# Written by tests/golden/make_golden.py.  bin k_mean[h/Mpc] P(k)[(Mpc/h)^3] N_modes\n")
        for i in range(len(k)):
            f.write(f"{i} {k[i]:.12e} {pk[i]:.12e} {int(nm[i])}\n")
    with open(os.path.join(HERE, "c1_oracle_state.txt"), "w") as f:
        f.write("# Final positions (mesh cells) and momenta of 8 particles of the same run: index x y z px py pz\n")
        for p in (0, 1, 33, 1057, 4000, 16384, 20011, 32767):
            f.write(f"{p} " + " ".join(f"{v:.12e}" for v in list(pos[:, p]) + list(mom[:, p])) + "\n")


if __name__ == "__main__":
    main()
