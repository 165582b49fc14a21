"""Hyper-parameter tables of the five BASELINE.json configs.

Pure data.  `Hparams` mirrors `allegro_hparams` of include/b200_allegro.h field by field.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Tuple


@dataclasses.dataclass
class Hparams:
    n_species: int
    l_max: int
    n_layers: int
    n_tensor: int
    n_bessel: int
    poly_p: int
    r_cut: float
    twobody_dims: Tuple[int, ...]      # hidden widths; last = latent width d
    latent_dims: Tuple[int, ...]       # per-layer latent MLP widths; last must equal d
    edge_dims: Tuple[int, ...]         # edge-energy MLP hidden widths; final ->1 implicit
    avg_num_neighbors: float           # c_env = 1/sqrt(this)
    resid_alpha: Tuple[float, ...]     # per layer
    # optional ordered species-pair cutoffs r_c[Z_centre][Z_neighbour] <= r_cut; None = flat r_cut
    r_cut_pair: Optional[Tuple[Tuple[float, ...], ...]] = None
    # optional trained Bessel angular frequencies w_n[Z_centre][Z_neighbour][n] in 1/A ("trainable
    # per-ordered-species-pair radial basis"); None = n pi / r_c of the pair
    bessel_freq_pair: Optional[Tuple[Tuple[Tuple[float, ...], ...], ...]] = None
    # optional atomic numbers per species: adds the ZBL pair repulsion; None = no ZBL term
    zbl_Z: Optional[Tuple[float, ...]] = None

    @property
    def d(self) -> int:
        return self.twobody_dims[-1]


@dataclasses.dataclass
class Config:
    index: int
    name: str
    hp: Hparams
    n_atoms: int
    density: float                     # atoms / A^3 of the water part (or of the whole box for cfg 4)
    kind: str                          # "water" | "solvated" | "random4"
    species_names: Tuple[str, ...]
    skin: float                        # Verlet skin for MD (A)
    rebuild_every: int
    dt_fs: float
    temperature: float
    pos_seed: int
    vel_seed: int
    weight_seed: int = 0
    # per-species energy scale/shift (SURVEY §8(d) "Energy scale"): the five configs use sigma_Z = 1 for every species
    # (RMS|F| is already O(1) eV/A with the seeded weights), mu_Z = -(1 + Z) eV.  Species-distinct sigma and
    # layer-distinct resid_alpha are exercised by tests/test_oracle_sigma_alpha.py and tests/test_gpu_sigma_alpha.py.
    sigma: float = 1.0

    def mu(self) -> List[float]:
        return [-(1.0 + z) for z in range(self.hp.n_species)]


# atomic masses (amu) by species name
MASSES_AMU = {"H": 1.008, "C": 12.011, "N": 14.007, "O": 15.999, "S": 32.06}

_RHO_W = 0.1
_AVG4 = 4.0 / 3.0 * math.pi * 4.0 ** 3 * 0.1     # 26.808257
_AVG6 = 4.0 / 3.0 * math.pi * 6.0 ** 3 * 0.08    # 72.382295


def _hp(S, lmax, nl, n, two, lat, edge, rc, avg):
    return Hparams(n_species=S, l_max=lmax, n_layers=nl, n_tensor=n, n_bessel=8, poly_p=6, r_cut=rc,
                   twobody_dims=tuple(two), latent_dims=tuple(lat), edge_dims=tuple(edge),
                   avg_num_neighbors=avg, resid_alpha=tuple([0.5] * nl))


CONFIGS: List[Config] = [
    Config(0, "water64", _hp(2, 1, 1, 8, [32, 32], [32], [16], 4.0, _AVG4),
           192, _RHO_W, "water", ("H", "O"), 1.0, 10, 0.5, 300.0, 1000, 2000),
    Config(1, "water4096", _hp(2, 2, 2, 32, [64, 128, 256], [256], [128], 4.0, _AVG4),
           12288, _RHO_W, "water", ("H", "O"), 1.0, 10, 0.5, 300.0, 1001, 2001),
    Config(2, "solvated100k", _hp(5, 2, 2, 64, [128, 256, 512], [512], [128], 4.0, _AVG4),
           100000, _RHO_W, "solvated", ("H", "C", "N", "O", "S"), 1.0, 10, 0.5, 300.0, 1002, 2002),
    Config(3, "solvated1M", _hp(5, 2, 2, 64, [128, 256, 512], [512], [128], 4.0, _AVG4),
           1000000, _RHO_W, "solvated", ("H", "C", "N", "O", "S"), 1.0, 10, 0.5, 300.0, 1003, 2003),
    Config(4, "tpstress50k", _hp(4, 3, 3, 64, [128, 256], [256], [128], 6.0, _AVG6),
           50000, 0.08, "random4", ("H", "C", "N", "O"), 1.0, 10, 0.5, 300.0, 1004, 2004),
]


# The paper's ordered-pair cutoffs restricted to water ("H-H 3.0, H-C 1.25, H-O 1.25, O-H 3.0", all
# others 4.0 Angstrom); species order of configs 0/1 is (H, O), rows = centre species.
WATER_PAIR_CUTOFFS = ((3.0, 1.25), (3.0, 4.0))


ATOMIC_NUMBERS = {"H": 1.0, "C": 6.0, "N": 7.0, "O": 8.0, "S": 16.0}


def get_config(index: int) -> Config:
    return CONFIGS[index]


def scaled_config(index: int, n_atoms: int) -> Config:
    """Same hyper-parameters and recipe as config `index` at a reduced atom count (parity tests at
    sizes the oracle finishes in seconds)."""
    c = dataclasses.replace(CONFIGS[index])
    c.n_atoms = n_atoms
    return c
