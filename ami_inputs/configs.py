"""Parameter recipes of the five BASELINE.json configs.

Every input is seeded and synthetic.  The topology seeds below were chosen by
``tests/golden/choose_topology_seeds.py`` (which calls only ``oracle/``): the
first seed whose table is constructible (|alpha_p| = 1 at every summation) and,
for config 3, whose result contains a double pole, so that the derivative path
is measured.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

from . import diagrams as D
from .rng import SEED_BASE, energies, momenta

Q_EXT = (math.pi / 2, math.pi / 2)

# topology seeds: written by tests/golden/choose_topology_seeds.py
TOPOLOGY_SEEDS = {"cfg3": 2, "cfg4": 0, "cfg5": 0, "stress8": 0}


@dataclass
class Config:
    name: str
    diagram: D.Diagram
    t: float
    mu: float
    betas: tuple
    z_ext: np.ndarray  # complex128 [n_f][n_ext]
    n_samples: int
    e_reg: float = 0.0
    seed: int = SEED_BASE
    q: tuple = Q_EXT
    meta: dict = field(default_factory=dict)

    def energies(self, n=None, start=0) -> np.ndarray:
        """[n][n_eps] energies of a workload that supplies them directly (meta["energy_range"])."""
        return energies(self.seed, self.n_samples if n is None else n, self.diagram.n_eps,
                        self.meta["energy_range"], start)

    def momenta(self, n=None, start=0) -> np.ndarray:
        return momenta(self.seed, self.n_samples if n is None else n, self.diagram.n_int, start)


def _fermionic(n, beta):
    return 1j * (2 * n + 1) * math.pi / beta


def _bosonic(n, beta):
    return 1j * 2 * n * math.pi / beta


def get_config(name: str, **over) -> Config:
    if name == "cfg1":
        beta = 5.0
        c = Config("cfg1", D.self_energy_order2(), 1.0, 0.0, (beta,),
                   np.array([[_fermionic(0, beta)]]), 10_000, seed=SEED_BASE + 1)
    elif name == "cfg2_se":  # one (mu, beta) point of the sweep; callers vary mu/beta/N
        beta = over.pop("beta", 5.0)
        c = Config("cfg2_se", D.self_energy_order2(), 1.0, over.pop("mu", 0.0), (beta,),
                   np.array([[_fermionic(n, beta)] for n in range(8)]), 1_000_000, seed=SEED_BASE + 2)
    elif name == "cfg2_bubble":
        beta = over.pop("beta", 5.0)
        c = Config("cfg2_bubble", D.bubble(), 1.0, over.pop("mu", 0.0), (beta,),
                   np.array([[_bosonic(n, beta)] for n in range(8)]), 1_000_000, e_reg=1e-8,
                   seed=SEED_BASE + 2)
    elif name == "cfg2_bubble_doubled":
        beta = over.pop("beta", 5.0)
        c = Config("cfg2_bubble_doubled", D.doubled_line_bubble(), 1.0, over.pop("mu", 0.0), (beta,),
                   np.array([[_bosonic(n, beta)] for n in range(8)]), 1_000_000, e_reg=1e-8,
                   seed=SEED_BASE + 2)
    elif name == "cfg3":
        beta = 8.0
        c = Config("cfg3", D.random_self_energy(4, TOPOLOGY_SEEDS["cfg3"]), 1.0, 0.0, (beta,),
                   np.array([[_fermionic(0, beta)]]), 1_000_000, seed=SEED_BASE + 3)
    elif name == "cfg4":
        beta = 10.0
        c = Config("cfg4", D.random_self_energy(6, TOPOLOGY_SEEDS["cfg4"]), 1.0, -0.3, (beta,),
                   np.array([[_fermionic(0, beta)]]), 100_000, e_reg=1e-8, seed=SEED_BASE + 4)
    elif name == "cfg5":
        om = np.linspace(-4.0, 4.0, 64)
        c = Config("cfg5", D.random_self_energy(5, TOPOLOGY_SEEDS["cfg5"]), 1.0, 0.0,
                   (2.0, 5.0, 10.0, 20.0), (om + 0.1j).reshape(64, 1), 200_000, seed=SEED_BASE + 5)
    elif name == "paper_ex1":  # the paper's first example: energies drawn directly
        beta = 1.0            # in (-8, 8), 100 fermionic frequencies, beta = 1, N_E = 1e6; no dispersion step
        c = Config("paper_ex1", D.self_energy_order2(), 1.0, 0.0, (beta,),
                   np.array([[_fermionic(n, beta)] for n in range(100)]), 1_000_000, seed=SEED_BASE + 9,
                   meta={"energy_range": 8.0})
    elif name == "stress8":  # outside the graded configs: exercises table tiling
        beta = 5.0
        c = Config("stress8", D.random_self_energy(8, TOPOLOGY_SEEDS["stress8"]), 1.0, 0.0, (beta,),
                   np.array([[_fermionic(0, beta)]]), 20_000, seed=SEED_BASE + 8)
    else:
        raise KeyError(name)
    for k, v in over.items():
        setattr(c, k, v)
    return c


CONFIGS = ("cfg1", "cfg2_se", "cfg2_bubble", "cfg2_bubble_doubled", "cfg3", "cfg4", "cfg5")
