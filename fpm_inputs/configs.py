"""The five BASELINE.json workloads as data."""
from dataclasses import dataclass

# Flat LCDM of every config (BASELINE.json `configs`); Omega_b and T_cmb complete the
# same Planck-2015 set.
COSMO = dict(omega_m=0.3075, h=0.6774, n_s=0.9667, sigma8=0.8159,
             omega_b=0.0486, t_cmb=2.7255)


@dataclass(frozen=True)
class Config:
    name: str
    np_side: int      # particles per side (Np)
    ng: int           # mesh cells per side (Ng)
    box: float        # Mpc/h
    lpt_order: int    # 1 or 2
    n_steps: int      # FastPM steps, linear in a
    a0: float = 0.1
    a1: float = 1.0
    seed: int = 1
    backward: bool = False

    @property
    def n_particles(self) -> int:
        return self.np_side ** 3

    @property
    def resolution_factor(self) -> int:
        return self.ng // self.np_side

    def stages(self):
        """a_j = a0 + j (a1 - a0)/n, j = 0..n  (n steps linear in a)."""
        n = self.n_steps
        return [self.a0 + j * (self.a1 - self.a0) / n for j in range(n + 1)]


CONFIGS = {
    "C1": Config("C1", 32, 32, 100.0, 1, 5),
    "C2": Config("C2", 128, 128, 200.0, 2, 10),
    "C3": Config("C3", 256, 512, 400.0, 2, 10),
    "C4": Config("C4", 512, 512, 1000.0, 2, 40, backward=True),
    "C5": Config("C5", 1024, 1024, 2000.0, 2, 10),
}
