"""Pins for the two parts of the oracle that uniform synthetic values cannot see (round-1 verdict): the per-species
energy scale sigma_{Z_i} of `E = sum_i (sigma_{Z_i} E_i + mu_{Z_i})` (indexed by the CENTRE's species,
also in the backward) and the per-LAYER residual coefficient alpha_L of SURVEY.md section 8(c) S7
(`x^L = c_old x^{L-1} + c_new u MLP`, c_old = 1/sqrt(1+alpha_L^2), c_new = alpha_L/sqrt(1+alpha_L^2)).

Each test compares the oracle with something that is not the oracle's own formula: an independent numpy scatter of the
sigma-free edge energies, linearity in sigma against per-species sub-system evaluations, the independent pair-potential
loop of P13 with a different alpha per layer, and central finite differences of E.  `test_wrong_sigma_index_would_fail`
and `test_alpha_order_matters` make sure the systems used can tell the right reading from the plausible wrong ones."""
import dataclasses
import math

import numpy as np
import pytest
import torch

from oracle import allegro_oracle as O
from synthetic import CONFIGS

from oracle_util import cluster, oracle_model, small_system
from test_oracle_model import _pair_energy

SIG2, MU2 = (0.7, 1.3), (-1.0, -2.5)
ALPHA = {1: (0.8,), 2: (0.3, 0.8), 3: (0.3, 0.8, 0.5)}


def _hp(ci):
    hp = CONFIGS[ci].hp
    return dataclasses.replace(hp, resid_alpha=ALPHA[hp.n_layers])


def _sig(S):
    return [0.7 + 0.6 * z / max(S - 1, 1) for z in range(S)]          # 0.7 .. 1.3, distinct per species


def _mu(S):
    return [-(1.0 + 1.5 * z) for z in range(S)]


def _edge_sums(m, pos, sp, box, nbr):
    """sum_j E_ij per centre by a plain numpy scatter of the oracle's (sigma-free) per-edge energies."""
    ei, ej, es = nbr
    t = torch.from_numpy
    Ee = m.edge_energies(t(pos), t(sp.astype(np.int64)), t(box), t(ei), t(ej), t(es)).numpy()
    Ei = np.zeros(pos.shape[0])
    np.add.at(Ei, ei, Ee)
    return Ee, Ei


@pytest.mark.parametrize("ci,n", [(0, 96), (1, 48), (4, 40)])
def test_sigma_scales_each_centre_by_its_own_species(ci, n):
    hp = _hp(ci)
    S = hp.n_species
    cfg, pos, sp, box = small_system(ci, n)
    nbr = O.neighbor_list(pos, box, hp.r_cut)
    sig, mu = np.array(_sig(S)), np.array(_mu(S))
    m, _ = oracle_model(hp, sigma=sig, mu=mu)
    m1, _ = oracle_model(hp, sigma=1.0, mu=mu)
    E, Ea, F = O.energy_forces(m, pos, sp, box, nbr)
    E1, Ea1, F1 = O.energy_forces(m1, pos, sp, box, nbr)
    _, Ei = _edge_sums(m, pos, sp, box, nbr)
    assert len(set(sp.tolist())) == S and np.abs(Ei).min() > 0
    # E-hat_i - mu_{Z_i} = sigma_{Z_i} * sum_j E_ij, atom by atom; and = sigma_{Z_i} x the sigma = 1 value
    np.testing.assert_allclose(Ea - mu[sp], sig[sp] * Ei, rtol=0, atol=1e-12 * np.abs(Ei).max())
    np.testing.assert_allclose(Ea - mu[sp], sig[sp] * (Ea1 - mu[sp]), rtol=0, atol=1e-12 * np.abs(Ei).max())
    assert E == pytest.approx(float((sig[sp] * Ei + mu[sp]).sum()), abs=1e-10)
    # forces are linear in sigma, and the coefficient of sigma_s is the force of the sub-system "centres of species s"
    # at sigma = 1 (strict locality): F(sigma) = sum_s sigma_s F_{centres of species s}
    Fsum = np.zeros_like(F)
    for s in range(S):
        _, _, Fs = O.energy_forces(m1, pos, sp, box, nbr, centers=np.nonzero(sp == s)[0])
        Fsum += sig[s] * Fs
    np.testing.assert_allclose(F, Fsum, rtol=0, atol=1e-11 * max(1.0, np.abs(F).max()))
    assert np.abs(F - F1).max() > 1e-3 * np.abs(F1).max()             # sigma does reach the forces


def test_doubling_sigma_of_one_species_touches_only_its_centres():
    hp = _hp(1)
    cfg, pos, sp, box = small_system(1, 48)
    nbr = O.neighbor_list(pos, box, hp.r_cut)
    mu = MU2
    ma, _ = oracle_model(hp, sigma=(0.7, 1.3), mu=mu)
    mb, _ = oracle_model(hp, sigma=(0.7, 2.6), mu=mu)                 # species 1 (O) doubled
    Ea_, Eaa, Fa = O.energy_forces(ma, pos, sp, box, nbr)
    Eb_, Eab, Fb = O.energy_forces(mb, pos, sp, box, nbr)
    H, Ox = sp == 0, sp == 1
    assert np.array_equal(Eaa[H], Eab[H])                             # centres of the other species: bit-identical
    np.testing.assert_allclose(Eab[Ox] - mu[1], 2.0 * (Eaa[Ox] - mu[1]), rtol=1e-13)
    # the force change is exactly the O-centred part at the old sigma
    _, _, FO = O.energy_forces(ma, pos, sp, box, nbr, centers=np.nonzero(Ox)[0])
    np.testing.assert_allclose(Fb - Fa, FO, rtol=0, atol=1e-11 * max(1.0, np.abs(Fa).max()))


def test_wrong_sigma_index_would_fail():
    """The systems above distinguish sigma_{Z_i} (centre) from sigma_{Z_j} (neighbour) and from a uniform sigma."""
    hp = _hp(1)
    cfg, pos, sp, box = small_system(1, 48)
    nbr = O.neighbor_list(pos, box, hp.r_cut)
    sig, mu = np.array(SIG2), np.array(MU2)
    m, _ = oracle_model(hp, sigma=sig, mu=mu)
    _, Ea, _ = O.energy_forces(m, pos, sp, box, nbr)
    Ee, Ei = _edge_sums(m, pos, sp, box, nbr)
    wrong_nb = np.zeros_like(Ei)
    np.add.at(wrong_nb, nbr[0], sig[sp[nbr[1]]] * Ee)                 # scaled by the neighbour's species
    scale = np.abs(Ei).max()
    assert np.abs((Ea - mu[sp]) - wrong_nb).max() > 1e-3 * scale
    assert np.abs((Ea - mu[sp]) - sig.mean() * Ei).max() > 1e-3 * scale
    assert np.abs((Ea - mu[sp]) - sig[::-1][sp] * Ei).max() > 1e-3 * scale


@pytest.mark.parametrize("ci", [0, 1])
def test_P13_pair_limit_with_distinct_sigma_mu_alpha(ci):
    """All path weights zero => E_ij depends on (r, Z_i, Z_j) only; the independent loop of test_oracle_model._pair_energy
    walks the blob itself and applies resid_alpha[L] layer by layer."""
    hp = _hp(ci)
    sig, mu = np.array(SIG2), np.array(MU2)
    m, blob = oracle_model(hp, sigma=sig, mu=mu, zero_alpha=True)
    pos, sp, box = cluster(9, hp.n_species, 21)
    ei, ej, es = O.neighbor_list(pos, box, hp.r_cut)
    E, Ea, F = O.energy_forces(m, pos, sp, box, (ei, ej, es))
    Epair = float(mu[sp].sum())
    Eat = mu[sp].copy()
    Fpair = np.zeros_like(F)
    for i, j in zip(ei, ej):
        rv = pos[j] - pos[i]
        r = np.linalg.norm(rv)
        e = sig[sp[i]] * _pair_energy(hp, blob, sp[i], sp[j], r)
        Epair += e; Eat[i] += e
        h = 1e-5
        dE = sig[sp[i]] * (_pair_energy(hp, blob, sp[i], sp[j], r + h) - _pair_energy(hp, blob, sp[i], sp[j], r - h)) / (2 * h)
        Fpair[i] += dE * rv / r
        Fpair[j] -= dE * rv / r
    assert abs(E - Epair) < 1e-11 * max(1, abs(Epair))
    np.testing.assert_allclose(Ea, Eat, atol=1e-11)
    np.testing.assert_allclose(F, Fpair, atol=1e-7 * max(1e-3, np.abs(F).max()))


def test_alpha_order_matters():
    """(0.3, 0.8) and (0.8, 0.3) give different energies, so a per-layer indexing slip cannot pass the pins above."""
    hp = _hp(1)
    hp_sw = dataclasses.replace(hp, resid_alpha=hp.resid_alpha[::-1])
    pos, sp, box = cluster(9, hp.n_species, 21)
    nbr = O.neighbor_list(pos, box, hp.r_cut)
    m, blob = oracle_model(hp, zero_alpha=True)
    msw, _ = oracle_model(hp_sw, zero_alpha=True)
    E = O.energy_forces(m, pos, sp, box, nbr)[0]
    Esw = O.energy_forces(msw, pos, sp, box, nbr)[0]
    assert abs(E - Esw) > 1e-4 * abs(E)
    # and the independent loop follows the swap
    i, j = int(nbr[0][0]), int(nbr[1][0])
    r = float(np.linalg.norm(pos[j] - pos[i]))
    assert _pair_energy(hp, blob, sp[i], sp[j], r) != _pair_energy(hp_sw, blob, sp[i], sp[j], r)


@pytest.mark.parametrize("ci", [0, 1, 4])
def test_P11_finite_differences_distinct_sigma_alpha(ci):
    hp = _hp(ci)
    S = hp.n_species
    m, _ = oracle_model(hp, sigma=_sig(S), mu=_mu(S))
    cfg, pos, sp, box = small_system(ci, 24)
    nbr = O.neighbor_list(pos, box, hp.r_cut + 0.01)
    E0, _, F = O.energy_forces(m, pos, sp, box, nbr)
    h = 1e-4
    g = np.random.default_rng(100 + ci)
    comps = [(a, c) for a in range(24) for c in range(3)]
    comps = [comps[k] for k in g.permutation(len(comps))[:24]]
    scale = np.sqrt((F ** 2).mean())
    assert scale > 1e-8
    for (a, c) in comps:
        pp = pos.copy(); pp[a, c] += h
        pm = pos.copy(); pm[a, c] -= h
        fd = -(O.energy_forces(m, pp, sp, box, nbr)[0] - O.energy_forces(m, pm, sp, box, nbr)[0]) / (2 * h)
        assert abs(fd - F[a, c]) <= 1e-7 * max(scale, abs(F[a, c])) + 1e-11, (a, c, fd, F[a, c])


def test_residual_coefficients_closed_form():
    """Two-layer model with all path weights zero and the latent MLP weights zeroed: x^L = c_old,L x^{L-1}, so
    E(alpha) / E(alpha = 0 reference) = prod_L 1/sqrt(1+alpha_L^2) -- a closed form the oracle's loop must reproduce."""
    hp = _hp(1)
    pos, sp, box = cluster(6, hp.n_species, 5, extent=3.5)
    nbr = O.neighbor_list(pos, box, hp.r_cut)
    m, _ = oracle_model(hp, zero_alpha=True)
    for lat in m.latent:
        for W in lat:
            W.zero_()
    E = O.energy_forces(m, pos, sp, box, nbr)[0]
    hp0 = dataclasses.replace(hp, resid_alpha=(0.0, 0.0))
    m0, _ = oracle_model(hp0, zero_alpha=True)
    for lat in m0.latent:
        for W in lat:
            W.zero_()
    E0 = O.energy_forces(m0, pos, sp, box, nbr)[0]
    want = math.prod(1.0 / math.sqrt(1 + a * a) for a in hp.resid_alpha)
    assert abs(E0) > 1e-6 and E / E0 == pytest.approx(want, rel=1e-12)
