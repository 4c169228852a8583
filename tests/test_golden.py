"""Stored expected values (tests/golden/, written by tests/golden/make_golden.py from oracle/ only).
The paper prints no worked example, so the fixtures freeze the pinned float64 oracle; the GPU run of
the same configuration must land on them within the north_star tolerances."""
import os

import numpy as np
import pytest

import fpm_inputs as fi

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
OM = fi.COSMO["omega_m"]


def _load(name):
    return np.loadtxt(os.path.join(GOLD, name), comments="#")


def test_oracle_growth_matches_stored_table(oracle):
    for a, d1, f1, d2, f2, e in _load("growth_table.txt"):
        g = oracle.growth(OM, float(a))
        assert [g["D1"], g["f1"], g["D2"], g["f2"], g["E"]] == pytest.approx([d1, f1, d2, f2, e], rel=1e-10)


def test_oracle_c1_run_matches_stored_power_and_state(oracle):
    cfg = fi.CONFIGS["C1"]
    delta = fi.linear_field(cfg.np_side, cfg.box, cfg.seed).astype(np.float64)
    pos, mom = oracle.lpt_init(delta, cfg.ng, OM, cfg.a0, cfg.lpt_order)
    pos, mom = oracle.nbody(pos, mom, cfg.ng, cfg.np_side, OM, cfg.stages())
    _, pk, _ = oracle.power(oracle.paint(pos, cfg.ng), cfg.box)
    assert pk == pytest.approx(_load("c1_oracle_power.txt")[:, 2], rel=1e-9)
    for row in _load("c1_oracle_state.txt"):
        p = int(row[0])
        assert list(pos[:, p]) + list(mom[:, p]) == pytest.approx(list(row[1:]), rel=1e-9, abs=1e-9)


@pytest.mark.gpu
def test_gpu_c1_run_lands_on_the_stored_oracle_values(oracle):
    """GPU C1 run from its own (fp32) LPT initial conditions vs the stored float64 run: P(k) within
    1e-4 per bin and the sampled particles within 1e-3 cell (north_star)."""
    import torch

    import paper_2010_11847_b200 as fpm
    cfg = fi.CONFIGS["C1"]
    for force_path in (fpm.FORCE_UNFUSED, fpm.FORCE_FUSED):
        ctx = fpm.FPM(cfg.ng, cfg.np_side, omega_m=OM, box=cfg.box, force_path=force_path)
        pos, mom = ctx.lpt_init(torch.from_numpy(fi.linear_field(cfg.np_side, cfg.box, cfg.seed)).cuda(),
                                cfg.a0, cfg.lpt_order)
        ctx.nbody(pos, mom, cfg.stages())
        hp = pos.cpu().numpy().astype(np.float64)
        _, pk, _ = oracle.power(oracle.paint(hp, cfg.ng), cfg.box)
        assert np.max(np.abs(pk / _load("c1_oracle_power.txt")[:, 2] - 1)) < 1e-4
        for row in _load("c1_oracle_state.txt"):
            d = np.abs(hp[:, int(row[0])] - row[1:4])
            assert np.max(np.minimum(d, cfg.ng - d)) < 1e-3
