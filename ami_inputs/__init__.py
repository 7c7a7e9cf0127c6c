"""Seeded, synthetic input generators shared by the tests, the bench and both
implementations (the CPU oracle under ``oracle/`` and the CUDA path under
``paper_2311_17189_b200/``).

This package holds NONE of the method's arithmetic: no residues, no Fermi/Bose
functions, no dispersion.  It only produces

* momenta from a stateless counter-based generator (``rng``),
* labelled diagrams -- integer ``alpha``/``eps`` matrices -- either written out
  from the paper's own examples or drawn from a seeded random 1PI topology
  generator (``diagrams``),
* the parameter recipes of the five BASELINE.json configs (``configs``).

The recipes stand in for the paper's benchmark diagrams (Fig. 3,
an image that is not available) and its random example energies
(PAPER.md:270-271).
"""
from .rng import uniform01, momenta, SEED_BASE  # noqa: F401
from .diagrams import (  # noqa: F401
    Diagram,
    order1_line,
    bubble,
    doubled_line_bubble,
    self_energy_order2,
    self_energy_order2_doubled,
    random_self_energy,
    kron_identity,
)
from .configs import CONFIGS, get_config  # noqa: F401
