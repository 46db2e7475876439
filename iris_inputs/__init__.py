"""Seeded synthetic inputs for the IRIS-SO hot path (shared by tests, bench, oracle and CUDA path).

This package holds *inputs only*: the observation parameter record, the rigid-rotor molecule
table that stands in for a LAMDA file (section 4.1), the five BASELINE.json
workload definitions and the seeded random-field recipe.  It contains
none of the method's arithmetic (no level balance, no profile, no transfer) and imports neither
``oracle`` nor ``paper_2607_01338_b200``.
"""
from .config import ObsConfig
from .molecule import rigid_rotor
from .fields import WORKLOADS, make_workload, make_fields, gaussian_random_field, weight_cube, lattice_to_columns

__all__ = ["ObsConfig", "rigid_rotor", "WORKLOADS", "make_workload", "make_fields",
           "gaussian_random_field", "weight_cube", "lattice_to_columns"]
