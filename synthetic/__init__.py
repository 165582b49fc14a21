"""Seeded synthetic inputs shared by the oracle tests and the CUDA-path tests/bench.

This package holds NO arithmetic of the Allegro method (no radial basis, no
spherical harmonics, no Clebsch-Gordan, no network): only hyper-parameter
tables, seeded positions/species/velocities and the seeded flat weight blob.
Both `oracle/` (test infrastructure) and `paper_2304_10061_b200/` (the
product) consume what is generated here; neither imports the other.
"""
from .configs import CONFIGS, Hparams, get_config, MASSES_AMU  # noqa: F401
from .systems import make_system, maxwell_boltzmann  # noqa: F401
from .weights import blob_num_floats, make_blob  # noqa: F401
