"""Pins for the oracle's ordered species-pair cutoffs ("independent cutoffs for each *ordered*
species pair", values PAPER.md:222; NEXT-1 reading in DESIGN.md: the pair's own cutoff enters the edge criterion,
the envelope argument and the Bessel functions)."""
import dataclasses

import numpy as np
import torch

from oracle import allegro_oracle as O
from synthetic import CONFIGS, make_system
from synthetic.configs import WATER_PAIR_CUTOFFS, scaled_config

from oracle_util import cluster, oracle_model


def _EF(m, pos, sp, box):
    return O.energy_forces(m, pos, sp, box, O.neighbor_list(pos, box, m.hp.r_cut))


def _hp(ci, pair):
    return dataclasses.replace(CONFIGS[ci].hp, r_cut_pair=pair)


def test_flat_matrix_equals_default():
    """r_c[Z_i][Z_j] = r_cut for every pair is the flat-cutoff model, bit for bit."""
    hp0 = CONFIGS[0].hp
    hp1 = _hp(0, ((4.0, 4.0), (4.0, 4.0)))
    pos, sp, box = cluster(14, 2, 5)
    m0, _ = oracle_model(hp0)
    m1, _ = oracle_model(hp1)
    E0, Ea0, F0 = _EF(m0, pos, sp, box)
    E1, Ea1, F1 = _EF(m1, pos, sp, box)
    assert E0 == E1 and np.array_equal(Ea0, Ea1) and np.array_equal(F0, F1)


def test_ordered_edge_sets_match_brute_force():
    """Edge (i, j) is kept iff r_ij < r_c[Z_i][Z_j] -- ordered: (H centre, O neighbour) uses 1.25, (O, H) 3.0."""
    hp = _hp(0, WATER_PAIR_CUTOFFS)
    cfg = scaled_config(0, 192)
    pos, sp, box = make_system(cfg)
    m, _ = oracle_model(hp)
    ei, ej, es = O.neighbor_list(pos, box, hp.r_cut)
    t = torch.from_numpy
    _, parts = m.edge_energies(t(pos), t(sp.astype(np.int64)), t(box), t(ei), t(ej), t(es), return_parts=True)
    kept = parts["idx"].numpy()
    rvec = pos[ej] - pos[ei] + es * box
    r = np.sqrt((rvec ** 2).sum(1))
    rc = np.array(WATER_PAIR_CUTOFFS)[sp[ei], sp[ej]]
    assert np.array_equal(kept, np.nonzero(r < rc)[0])
    # ordered asymmetry: O-centred pairs with an H neighbour outnumber H-centred pairs with an O neighbour
    n_HO = ((sp[ei[kept]] == 0) & (sp[ej[kept]] == 1)).sum()
    n_OH = ((sp[ei[kept]] == 1) & (sp[ej[kept]] == 0)).sum()
    assert n_OH > 2 * n_HO > 0


def test_water_pair_count_reduction():
    """the selected cutoffs reduce the number of ordered pairs by approximately 3x in liquid water."""
    cfg = scaled_config(1, 1536)
    pos, sp, box = make_system(cfg)
    ei, ej, es = O.neighbor_list(pos, box, 4.0)
    rvec = pos[ej] - pos[ei] + es * box
    r = np.sqrt((rvec ** 2).sum(1))
    rc = np.array(WATER_PAIR_CUTOFFS)[sp[ei], sp[ej]]
    ratio = r.shape[0] / (r < rc).sum()
    assert 2.2 < ratio < 4.0, ratio


def test_continuity_at_a_pair_cutoff():
    """Moving an H atom across r_c[O][H] = 3.0 of an O centre changes E continuously (C^2 envelope per pair)."""
    hp = _hp(0, WATER_PAIR_CUTOFFS)
    m, _ = oracle_model(hp, mu=[-1.0, -2.0])
    pos, sp, box = cluster(10, 2, 7)
    sp[0], sp[1] = 1, 0                       # atom 0: O centre, atom 1: H neighbour
    d = pos[1] - pos[0]
    d /= np.linalg.norm(d)
    Es = []
    for delta in (-2e-6, -1e-6, 0.0, 1e-6, 2e-6):
        p = pos.copy()
        p[1] = pos[0] + d * (3.0 + delta)
        Es.append(_EF(m, p, sp, box)[0])
    # no jump at the crossing: the energy differences stay on one straight line (slope = the force along d),
    # a discontinuity of E or of dE/dr at r_c[O][H] would show up as a second difference
    d1 = np.diff(Es)
    assert max(abs(d1)) < 1e-6 and max(abs(np.diff(d1))) < 1e-11, (d1, np.diff(d1))


def test_forces_finite_differences_with_pair_cutoffs():
    hp = _hp(0, WATER_PAIR_CUTOFFS)
    m, _ = oracle_model(hp, mu=[-1.0, -2.0])
    pos, sp, box = cluster(9, 2, 3, extent=3.5)
    E, _, F = _EF(m, pos, sp, box)
    h = 1e-4
    for a in (0, 4, 8):
        for k in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[a, k] += h
            pm[a, k] -= h
            fd = -(_EF(m, pp, sp, box)[0] - _EF(m, pm, sp, box)[0]) / (2 * h)
            assert abs(fd - F[a, k]) <= 1e-6 * max(1.0, np.abs(F).max()), (a, k, fd, F[a, k])
