"""Seeded synthetic Poisson-Boltzmann inputs (BASELINE.json `configs`).

This package only *builds inputs* (dielectric maps, salt mask, charges, Dirichlet
ghost values).  It holds none of the solver's arithmetic, imports neither
`oracle/` nor `paper_1704_02745_b200/`, and hands byte-identical arrays to both.
"""
from .pb_inputs import (  # noqa: F401
    KBAR2_150MM_300K,
    PBInputs,
    born_ion,
    make_config,
    perturbed_charge_values,
    perturbed_charges,
    random_operator,
)
