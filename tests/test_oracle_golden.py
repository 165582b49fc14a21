"""Pins of the oracle and the synthetic water recipe against numbers the paper prints (tests/golden/paper_values.txt,
each line with its PAPER.md citation).  The paper gives no worked numerical example of the model itself,
so these fix what it does print: neighbor counts of bulk water and the ordered-pair cutoffs."""
import os

import numpy as np

from oracle import allegro_oracle as O
from synthetic import CONFIGS, make_system
from synthetic.configs import WATER_PAIR_CUTOFFS, scaled_config


def _golden():
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as f:
        for line in f:
            line = line.split("#", 1)[0].split()
            if len(line) == 2:
                out[line[0]] = float(line[1])
    return out


def test_water_neighbor_count_matches_the_papers_bulk_water():
    """96 neighbors within 6 A and 20,834 atoms within 36 A.  Both numbers give the paper's number density
    (0.106 atoms/A^3); the oracle's list on the synthetic water box (0.1 atoms/A^3), rescaled by the density ratio,
    must reproduce the 96 (a half list, a double-counted image or a wrong cutoff test would be off by 2x or more)."""
    g = _golden()
    rho_paper = g["water_atoms_within_36A"] / (4.0 / 3.0 * np.pi * 36.0 ** 3)
    assert abs(g["water_neighbors_at_6A"] / (4.0 / 3.0 * np.pi * 6.0 ** 3) - rho_paper) < 0.002   # the two printed values agree
    cfg = scaled_config(1, 1536)
    pos, sp, box = make_system(cfg)
    assert box.min() >= 12.0
    ei, ej, es = O.neighbor_list(pos, box, 6.0)
    per_atom = ei.shape[0] / pos.shape[0]
    rho_ours = pos.shape[0] / float(np.prod(box))
    assert abs(per_atom * rho_paper / rho_ours - g["water_neighbors_at_6A"]) < 0.05 * g["water_neighbors_at_6A"], per_atom
    # every atom is a centre and the list is ordered: (i, j) present iff (j, i) present
    fwd = set(zip(ei.tolist(), ej.tolist(), map(tuple, es.tolist())))
    assert all((j, i, (-s[0], -s[1], -s[2])) in fwd for i, j, s in list(fwd)[:2000])


def test_pair_cutoffs_are_the_papers():
    """PAPER.md:222; species order of the water configs is (H, O), rows = centre species."""
    g = _golden()
    assert CONFIGS[1].hp.r_cut == g["default_cutoff_A"] and CONFIGS[1].hp.n_bessel == int(g["n_bessel"])
    assert WATER_PAIR_CUTOFFS == ((g["cutoff_HH_A"], g["cutoff_HO_A"]), (g["cutoff_OH_A"], g["default_cutoff_A"]))


def test_pair_reduction_is_about_the_papers_factor():
    """PAPER.md:182 ("approximately 3x"), counted by the oracle's list on synthetic water."""
    g = _golden()
    cfg = scaled_config(1, 1536)
    pos, sp, box = make_system(cfg)
    ei, ej, es = O.neighbor_list(pos, box, g["default_cutoff_A"])
    r = np.sqrt(((pos[ej] - pos[ei] + es * box) ** 2).sum(1))
    rc = np.array(WATER_PAIR_CUTOFFS)[sp[ei], sp[ej]]
    ratio = r.shape[0] / (r < rc).sum()
    assert abs(ratio - g["water_pair_reduction"]) < 0.5, ratio
