"""The five BASELINE.json configs as seeded synthetic workloads.

Only input construction and the schedule parameters live here (no method arithmetic)."""
from dataclasses import dataclass
from typing import Callable

from . import lattices as L
from . import rng


@dataclass
class Workload:
    key: str
    description: str
    build: Callable[[], "L.TBModel"]
    batch: int
    n_moments: int          # N_m ("KPM order")
    dt: float
    n_steps: int
    order: int              # N_p Chebyshev terms per step: given by BASELINE.json (c1, c2), else the smallest N_p with
                            # |J_m(dE dt)| < 1e-15 for all m >= N_p [A5], evaluated once with scipy.special.jv at the
                            # generated model's dE (c3: x = 20 -> 50, c4: x = 16 -> 44, c5: dE = 10.7, x = 10.7 -> 36)
    path: str               # "vac" or "msd"
    config_id: int

    def phases(self, model, first_vector=0):
        return L.random_phase_vectors(model.N, self.batch, self.config_id, first_vector)


def _c1():
    return L.graphene(24, 24, hop=-2.7, W=1.0, seed=rng.stream_seed(1, 0), energy_scale=10.0)


def _c2():
    return L.square(1000, 1000, W=2.0, seed=rng.stream_seed(2, 0), energy_scale=5.1)


def _c3():
    return L.graphene(707, 707, hop=-2.7, vacancy_fraction=0.01, vacancy_seed=rng.stream_seed(3, 1),
                      energy_scale=10.0)


def _c4():
    return L.cubic(160, W=16.5, seed=rng.stream_seed(4, 0), energy_scale=16.0)


def _c5():
    return L.graphene_peierls_correlated(2828, 1414, config=5)


WORKLOADS = {
    "c1": Workload("c1", "graphene 24x24 four-atom cells (2304 orbitals), W=1 eV Anderson, dE=10 eV, "
                   "N_m=256, VAC 10 steps dt=1, N_p=64, B=1", _c1, 1, 256, 1.0, 10, 64, "vac", 1),
    "c2": Workload("c2", "square 1000x1000 (1e6 orbitals), W=2, dE=5.1, N_m=3000, VAC 20 steps dt=2, "
                   "N_p=40, B=1", _c2, 1, 3000, 2.0, 20, 40, "vac", 2),
    "c3": Workload("c3", "graphene 707x707 four-atom cells with 1% vacancies (1979403 orbitals), dE=10 eV, "
                   "N_m=2000, MSD 50 steps dt=2, N_p=50, B=1", _c3, 1, 2000, 2.0, 50, 50, "msd", 3),
    "c4": Workload("c4", "simple-cubic Anderson 160^3 (4.096e6 orbitals), W=16.5, dE=16, N_m=1000, "
                   "MSD 40 steps dt=1, N_p=44, B=4", _c4, 4, 1000, 1.0, 40, 44, "msd", 4),
    "c5": Workload("c5", "graphene 2828x1414 four-atom cells (15995168 orbitals), Peierls flux 1e-4/hexagon, "
                   "Gaussian-correlated potential, dE=10.7 eV, N_m=3000, VAC 30 steps dt=1, N_p=36 (tail rule), B=8",
                   _c5, 8, 3000, 1.0, 30, 36, "vac", 5),
}


def small_variant(key: str):
    """Reduced-size lattices of the same family, for parity cases the oracle finishes in seconds."""
    return {
        "c1": lambda: _c1(),
        "c2": lambda: L.square(120, 90, W=2.0, seed=rng.stream_seed(2, 0), energy_scale=5.1),
        "c3": lambda: L.graphene(40, 36, hop=-2.7, vacancy_fraction=0.01, vacancy_seed=rng.stream_seed(3, 1),
                                 energy_scale=10.0),
        "c4": lambda: L.cubic(20, W=16.5, seed=rng.stream_seed(4, 0), energy_scale=16.0),
        "c5": lambda: L.graphene_peierls_correlated(60, 32, config=5),
    }[key]()


# ------------------------------------------------------------------ the paper's two examples (section 5)
@dataclass
class Example:
    key: str
    description: str
    build: Callable[[float], "L.TBModel"]   # argument: linear scale factor (1.0 = the paper's size)
    batch: int              # N_r
    n_moments: int
    dts: tuple              # time steps (hbar / gamma)
    e_max: float            # energy grid -e_max .. e_max in steps of 0.02 gamma
    vac: bool
    msd: bool
    config_id: int

    def phases(self, model, first_vector=0):
        return L.random_phase_vectors(model.N, self.batch, self.config_id, first_vector)

    def energies(self):
        import numpy as np
        n = int(round(2 * self.e_max / 0.02)) + 1
        return np.linspace(-self.e_max, self.e_max, n)


def _e1(scale=1.0):
    n = max(8, int(round(2000 * scale)))
    return L.square(n, n, W=4.0, seed=rng.stream_seed(11, 0), energy_scale=6.1)


def _e2(scale=1.0):
    n = max(16, int(round(4000000 * scale)))
    return L.chain(n, W=4.0, seed=rng.stream_seed(12, 0), energy_scale=4.1)


EXAMPLES = {
    # 2000 x 2000 square lattice, W = 4, periodic, dE = 6.1, N_m = 1000, N_r = 1,
    # 20 steps of 0.2, energies -6 .. 6 step 0.02 (601 points), VAC and MSD
    "e1": Example("e1", "paper example 5.1: 2D square lattice 2000^2, W=4, dE=6.1, N_m=1000, 20 x dt=0.2, VAC+MSD",
                  _e1, 1, 1000, tuple([0.2] * 20), 6.0, True, True, 11),
    # chain of 4e6 sites, W = 4, periodic, dE = 4.1, N_m = 500, N_r = 2, 30 growing steps
    # 0.1 .. 1.0, 1 .. 10, 10 .. 100, energies -4 .. 4 step 0.02 (401 points), MSD only
    "e2": Example("e2", "paper example 5.2: 1D chain 4e6, W=4, dE=4.1, N_m=500, N_r=2, 30 growing steps, MSD",
                  _e2, 2, 500, tuple([0.1 * i for i in range(1, 11)] + [1.0 * i for i in range(1, 11)]
                                     + [10.0 * i for i in range(1, 11)]), 4.0, False, True, 12),
}
