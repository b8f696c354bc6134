"""CPU oracle for the PIMD hot path of arXiv 2404.02628 -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with the
CUDA path in ``paper_2404_02628_b200``; neither imports the other.

``pimd_oracle.c`` holds the arithmetic (each function cites the passage of
PAPER.md it follows); this file is ctypes marshalling only.
``ideal_gas.py`` holds the exact finite-P ideal-gas reference energy.
"""
from .binding import (  # noqa: F401
    OracleError,
    build,
    conditioning,
    cycle_energies,
    cycle_energies_eq10,
    cycle_energy_eq7,
    eint,
    estimators,
    estimators_species,
    external_force_on,
    forces,
    forces_species,
    pair_histogram,
    philox_normal,
    philox_raw,
    potential,
    pr_matrix,
    set_pair_potential,
    step,
    stream_forces_on,
    vb,
)
