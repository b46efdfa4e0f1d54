"""The five synthetic workloads of BASELINE.json:configs, as plain data (no arithmetic).

The paper measures on unpublished random star fields; these seeded synthetic
fields stand in for them.  Used by tests/, bench.py and
__graft_entry__.py to drive both the CUDA library and the oracle with the same parameters.
"""
from dataclasses import dataclass
from typing import Optional, Tuple

MASS_EQUAL = 0
MASS_POWER_LAW = 1
MASS_BROKEN_POWER_LAW = 2


@dataclass(frozen=True)
class Workload:
    name: str
    N: int                 # number of point lenses (stars); 2N roots per phase
    kappa_star: float      # convergence in stars (sets the disk radius R = sqrt(N / kappa_star))
    kappa_s: float         # smooth convergence left after the compensating sheet
    gamma: float           # external shear
    num_phi: int           # phases on [0, 2 pi)
    mass_model: int
    mass_params: Optional[Tuple[float, ...]] = None
    seed: int = 0
    tol: float = 1e-12
    max_iter: int = 50


CONFIGS = {
    # "N=10 equal-mass ... kappa_*=0.4, kappa_s=0, gamma=0.3; 1000 phases; tol 1e-12, max_iter 50"
    "cfg1": Workload("cfg1", 10, 0.4, 0.0, 0.3, 1000, MASS_EQUAL),
    # "N=200 equal-mass, kappa_*=0.3, kappa_s=0.2, gamma=0.35; 4000 phases"
    "cfg2": Workload("cfg2", 200, 0.3, 0.2, 0.35, 4000, MASS_EQUAL),
    # "N=2000 Salpeter masses (m^-2.35 on [0.08, 1]), kappa_*=0.45, kappa_s=0, gamma=0.4; 5000 phases"
    "cfg3": Workload("cfg3", 2000, 0.45, 0.0, 0.4, 5000, MASS_POWER_LAW, (0.08, 1.0, 2.35)),
    # "N=10^4 Kroupa-like broken power law on [0.01, 1.5], kappa_*=0.2, kappa_s=0.5, gamma=0.55; 10000 phases"
    "cfg4": Workload("cfg4", 10000, 0.2, 0.5, 0.55, 10000, MASS_BROKEN_POWER_LAW,
                     (0.01, 0.08, 0.5, 1.5, 0.3, 1.3, 2.3)),
    # "N=5x10^4 equal-mass, kappa_*=0.6, kappa_s=0, gamma=0.25; 2000 phases"
    "cfg5": Workload("cfg5", 50000, 0.6, 0.0, 0.25, 2000, MASS_EQUAL),
}

# the configuration BASELINE.json's metric is quoted on ("at N=10^4 stars")
HEADLINE = "cfg4"
