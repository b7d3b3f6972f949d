"""The five BASELINE.json configurations, restated as data.

`mode` fields map to the C-ABI arguments of `cos_build`:
  lattice        0 = square (n_sub = 1), 1 = honeycomb (n_sub = 2, sublattice-summed)
  n_flavors      N_f
  alphas         None  -> uniform CoS (one propagator block, loop factor N_f, no shift edge)
                 tuple -> SB-CoS (N_f blocks, sigma_lambda = alpha_lambda / U, U = 1: reading G15)
  all_subsets    False -> single full-order output, True -> all 2^n - 1 subset readouts
"""
from dataclasses import dataclass, replace
from typing import Optional, Tuple


@dataclass(frozen=True)
class Workload:
    name: str
    n: int                  # perturbative order (interaction vertices)
    n_flavors: int
    lattice: int            # 0 square, 1 honeycomb
    L: int                  # linear size (sites for square, unit cells for honeycomb)
    t: float
    mu: float
    beta: float
    alphas: Optional[Tuple[float, ...]]
    all_subsets: bool
    batch: int
    seed: int
    U: float = 1.0          # reading G15: sigma = alpha / U with U = 1
    n_tau: int = 1024       # tau nodes of the lookup table (reading G18)

    @property
    def n_sub(self) -> int:
        return 2 if self.lattice == 1 else 1

    @property
    def d(self) -> int:
        """Dimension of one propagator block: endpoints (i, s)."""
        return self.n * self.n_sub

    @property
    def n_blocks(self) -> int:
        """Propagator blocks handed to cos_eval: 1 (uniform) or N_f (SB)."""
        return 1 if self.alphas is None else self.n_flavors

    @property
    def sigmas(self):
        return None if self.alphas is None else tuple(a / self.U for a in self.alphas)

    @property
    def n_out(self) -> int:
        return (1 << self.n) - 1 if self.all_subsets else 1

    def mu_eff(self):
        """Chemical potential entering each block's dispersion (reading G16:
        BASELINE wording mu_sigma = mu + alpha_sigma)."""
        if self.alphas is None:
            return (self.mu,)
        return tuple(self.mu + a for a in self.alphas)

    def scaled(self, **kw) -> "Workload":
        return replace(self, **kw)


CONFIGS = (
    Workload("cfg1_square_su2_n4", n=4, n_flavors=2, lattice=0, L=8, t=1.0, mu=0.0, beta=2.0,
             alphas=None, all_subsets=False, batch=1024, seed=0),
    Workload("cfg2_square_su2_n8_allsubsets", n=8, n_flavors=2, lattice=0, L=16, t=1.0, mu=-0.5, beta=5.0,
             alphas=None, all_subsets=True, batch=65536, seed=1),
    Workload("cfg3_honeycomb_sb2_n10", n=10, n_flavors=2, lattice=1, L=12, t=1.0, mu=0.0, beta=4.0,
             alphas=(0.3, -0.3), all_subsets=False, batch=16384, seed=2),
    Workload("cfg4_square_sb3_n10", n=10, n_flavors=3, lattice=0, L=16, t=1.0, mu=0.0, beta=4.0,
             alphas=(0.2, 0.0, -0.2), all_subsets=False, batch=8192, seed=3),
    Workload("cfg5_square_su2_n12", n=12, n_flavors=2, lattice=0, L=32, t=1.0, mu=0.0, beta=8.0,
             alphas=None, all_subsets=False, batch=64, seed=4),
)


def get_config(i: int) -> Workload:
    """1-based, as BASELINE.json / SURVEY.md number them."""
    return CONFIGS[i - 1]
