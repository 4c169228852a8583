"""Writes the stored expected values under tests/golden/ by calling ONLY oracle/ (and the seeded
input generators).  Run from the repo root:
    python tests/golden/make_golden.py                 # growth table + the C1 run (seconds)
    python tests/golden/make_golden.py --config C3     # full float64 run of C3 (minutes on 8-16 cores)
    python tests/golden/make_golden.py --config C4     # full float64 run of C4 (tens of minutes, ~25 GB)

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


SAMPLE_SEED, N_SAMPLE = 777, 2048


def sample_indices(n):
    """N_SAMPLE seeded particle (or cell) indices in [0, n), plus the first and last: the tests rebuild them."""
    u = fi.counter_uniform(SAMPLE_SEED, np.arange(N_SAMPLE, dtype=np.uint64), stream=40)
    idx = np.minimum((u * n).astype(np.int64), n - 1)
    return np.unique(np.concatenate([idx, [0, n - 1]]))


def big_run(name):
    """Full float64 oracle run of BASELINE.json's C3 / C4 (Alg. 4 ICs PAPER.md:363-383, leapfrog PAPER.md:37-45,
    force PAPER.md:47-59) from the seeded linear field; nothing is rounded to fp32 on the way.  Stores what
    a GPU run of the same configuration must land on (north_star: positions within 1e-3 cell, P(k) within
    1e-4 per bin; density and force within 1e-5 relative L2 per step):
      <name>_oracle_power.txt   final-density P(k) per bin (R13 binning)
      <name>_oracle_state.txt   initial and final (pos, mom) and the first force at N_SAMPLE seeded particles
      <name>_oracle_cells.txt   the density painted from the initial conditions at N_SAMPLE seeded cells,
                                with the global 2-norms of that density and force (denominators of rel-L2)."""
    import time
    cfg = fi.CONFIGS[name]
    om = fi.COSMO["omega_m"]
    tag = name.lower()
    t0 = time.time()
    delta = fi.linear_field(cfg.np_side, cfg.box, cfg.seed).astype(np.float64)
    pos0, mom0 = oracle.lpt_init(delta, cfg.ng, om, cfg.a0, cfg.lpt_order)
    del delta
    print(f"[{name}] lpt_init {time.time() - t0:.0f} s", flush=True)
    mass = float(cfg.resolution_factor ** 3)
    f0, rho0 = oracle.force(pos0, cfg.ng, scale=1.5 * om, mass=mass, return_rho=True)
    print(f"[{name}] first force {time.time() - t0:.0f} s", flush=True)
    pidx = sample_indices(cfg.n_particles)
    cidx = sample_indices(cfg.ng ** 3)
    rho_s = rho0.reshape(-1)[cidx].copy()
    rho_norm, f_norm = float(np.sqrt(np.sum(rho0 ** 2))), float(np.sqrt(np.sum(f0 ** 2)))
    rho_max, f_max = float(np.max(np.abs(rho0))), float(np.max(np.abs(f0)))
    f0_s = f0[:, pidx].copy()
    p0_s, m0_s = pos0[:, pidx].copy(), mom0[:, pidx].copy()
    del f0, rho0
    pos, mom = oracle.nbody(pos0, mom0, cfg.ng, cfg.np_side, om, cfg.stages())
    del pos0, mom0
    print(f"[{name}] nbody {time.time() - t0:.0f} s", flush=True)
    k, pk, nm = oracle.power(oracle.paint(pos, cfg.ng, mass_const=mass), cfg.box)
    head = (f"# float64 oracle run of {name} (BASELINE.json configs; {cfg.np_side}^3 particles on a {cfg.ng}^3 mesh, box "
            f"{cfg.box:g} Mpc/h, {cfg.lpt_order}LPT at a = {cfg.a0}, {cfg.n_steps} steps to a = {cfg.a1}, seed {cfg.seed}).\n"
            f"# Written by `python tests/golden/make_golden.py --config {name}` (calls only oracle/ and fpm_inputs/).\n")
    with open(os.path.join(HERE, f"{tag}_oracle_power.txt"), "w") as f:
        f.write(head + "# Final-density power spectrum (PAPER.md:325-333 Eq. 10; binning SURVEY.md R13).\n"
                "# bin k_mean[h/Mpc] P(k)[(Mpc/h)^3] N_modes\n")
        for i in range(len(k)):
            f.write(f"{i} {k[i]:.12e} {pk[i]:.12e} {int(nm[i])}\n")
    with open(os.path.join(HERE, f"{tag}_oracle_state.txt"), "w") as f:
        f.write(head + f"# Seeded particle sample (make_golden.sample_indices): initial state (Alg. 4), force at the initial\n"
                "# positions (already x 1.5 Omega_m, PAPER.md:49-59) and final state, mesh-cell units.\n"
                "# index x0 y0 z0 px0 py0 pz0 fx0 fy0 fz0 x y z px py pz\n")
        for j, p in enumerate(pidx):
            vals = list(p0_s[:, j]) + list(m0_s[:, j]) + list(f0_s[:, j]) + list(pos[:, p]) + list(mom[:, p])
            f.write(f"{p} " + " ".join(f"{v:.12e}" for v in vals) + "\n")
    with open(os.path.join(HERE, f"{tag}_oracle_cells.txt"), "w") as f:
        f.write(head + "# Density painted from the initial conditions (PAPER.md:47) at a seeded cell sample.\n"
                f"# norms: rho_l2 {rho_norm:.12e} rho_maxabs {rho_max:.12e} force_l2 {f_norm:.12e} force_maxabs {f_max:.12e}\n"
                "# flat_cell_index rho\n")
        for c, v in zip(cidx, rho_s):
            f.write(f"{c} {v:.12e}\n")
    print(f"[{name}] done {time.time() - t0:.0f} s", flush=True)


def big_gradient(name):
    """Float64 oracle gradient of BASELINE.json's backward objective at C3 size (configs[3] words it for C4, whose
    float64 reverse run would take hours): L = sum(final density x seeded N(0,1) weight field, seed 101) with
    respect to the linear field, through paint_adjoint -> nbody_vjp -> lpt_init_vjp (
    PAPER.md:21-23, 401, 586).  Stores the gradient at N_SAMPLE seeded lattice points and its 2-norm:
      <name>_oracle_gradient.txt"""
    import time
    cfg = fi.CONFIGS[name]
    om = fi.COSMO["omega_m"]
    t0 = time.time()
    delta = fi.linear_field(cfg.np_side, cfg.box, cfg.seed).astype(np.float64)
    w = fi.weight_field(cfg.ng, 101).astype(np.float64)
    mass = float(cfg.resolution_factor ** 3)
    pos, mom = oracle.lpt_init(delta, cfg.ng, om, cfg.a0, cfg.lpt_order)
    pf, _, traj = oracle.nbody(pos, mom, cfg.ng, cfg.np_side, om, cfg.stages(), return_traj=True)
    del pos, mom
    print(f"[{name} gradient] forward {time.time() - t0:.0f} s", flush=True)
    loss = float(np.sum(oracle.paint(pf, cfg.ng, mass_const=mass) * w))
    gx, _ = oracle.paint_adjoint(pf, cfg.ng, w, mass_const=mass)
    del pf
    gx0, gp0 = oracle.nbody_vjp(traj, cfg.ng, cfg.np_side, om, cfg.stages(), gx, np.zeros_like(gx))
    del traj, gx
    print(f"[{name} gradient] nbody_vjp {time.time() - t0:.0f} s", flush=True)
    gd = oracle.lpt_init_vjp(delta, cfg.ng, om, cfg.a0, cfg.lpt_order, gx0, gp0)
    idx = sample_indices(cfg.n_particles)
    flat = gd.reshape(-1)
    with open(os.path.join(HERE, f"{name.lower()}_oracle_gradient.txt"), "w") as f:
        f.write(f"# float64 oracle: d/d(delta_lin) of L = sum(final density x weight field seed 101) for {name} "
                f"({cfg.np_side}^3 particles on a {cfg.ng}^3 mesh, {cfg.n_steps} steps), SURVEY.md 8(c) R12.\n"
                f"# Written by `python tests/golden/make_golden.py --config {name} --gradient` (calls only oracle/ and fpm_inputs/).\n"
                f"# norms: loss {loss:.12e} grad_l2 {float(np.sqrt(np.sum(gd ** 2))):.12e} grad_maxabs {float(np.max(np.abs(gd))):.12e}\n"
                "# flat_lattice_index gradient\n")
        for i in idx:
            f.write(f"{i} {flat[i]:.12e}\n")
    print(f"[{name} gradient] done {time.time() - t0:.0f} s", flush=True)


def main():
    import argparse
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default=None, choices=["C3", "C4"])
    ap.add_argument("--gradient", action="store_true", help="the reverse-mode gradient of the C4 objective at this config")
    args = ap.parse_args()
    if args.config and args.gradient:
        big_gradient(args.config)
        return
    if args.config:
        big_run(args.config)
        return
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
