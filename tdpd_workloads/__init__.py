"""Seeded synthetic input generators shared by the CUDA path's tests/bench and by the oracle's tests.
Holds inputs only — none of the method's arithmetic ("Input recipe")."""
from .configs import (BASE_SEED, BODY_DOUBLE_POISEUILLE_Z, BODY_OFF, BODY_UNIFORM, MAX_SPECIES, MAX_TYPES,
                      Workload, config, fluid_params, lattice_centers, make_fluid, make_suspension,
                      rbc_params, small_suspension)
from .mesh import D0_RBC, evans_fung_inside, evans_fung_map, icosphere, random_rotations, rbc_mesh
