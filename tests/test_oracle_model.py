"""Pins P7-P14 for the oracle's network, energies and forces."""
import math

import numpy as np
import pytest
import torch

from oracle import allegro_oracle as O
from synthetic import CONFIGS
from synthetic.configs import Hparams
from synthetic.weights import blob_num_floats

from oracle_util import cluster, oracle_model, small_system


def _EF(m, pos, sp, box, cutoff=None, **kw):
    nbr = O.neighbor_list(pos, box, cutoff or m.hp.r_cut)
    return O.energy_forces(m, pos, sp, box, nbr, **kw)


# ---- P7: Eq. (2) line 1 == line 2 --------------------------------------------
@pytest.mark.parametrize("ci", [0, 1, 4])
def test_P7_bilinearity(ci):
    hp = CONFIGS[ci].hp
    m, _ = oracle_model(hp)
    pos, sp, box = cluster(7, hp.n_species, 3, extent=4.0)
    ei, ej, es = O.neighbor_list(pos, box, hp.r_cut)
    t = lambda a: torch.from_numpy(a)
    _, parts = m.edge_energies(t(pos), t(sp.astype(np.int64)), t(box), t(ei), t(ej), t(es), return_parts=True)
    n, lmax = hp.n_tensor, hp.l_max
    c_env = 1 / math.sqrt(hp.avg_num_neighbors)
    Y = parts["Y"]
    for L in range(1, hp.n_layers + 1):
        V, T = parts["V"][L - 1], parts["V"][L]
        om = (parts["x"][L - 1] @ m.A[L]).reshape(-1, n, lmax + 1)
        K = m.K[L - 1]
        slow = torch.zeros_like(T)
        for e in range(ei.shape[0]):                      # ordered pair (i, j)
            for k in np.nonzero(ei == ei[e])[0]:          # k in N(i): product first, then sum
                wy = om[k][:, m.env_l] * Y[k][None, :]
                slow[e] += c_env * torch.einsum("abc,na,nb->nc", K, V[e], wy)
        assert torch.abs(slow - T).max() < 1e-12 * max(1.0, float(torch.abs(T).max()))


# ---- P8: symmetries ------------------------------------------------------------------------------
def _rand_O3(rng, improper):
    Q, R = np.linalg.qr(rng.standard_normal((3, 3)))
    Q = Q * np.sign(np.diag(R))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    return -Q if improper else Q


@pytest.mark.parametrize("ci,improper", [(0, False), (1, True), (4, False), (4, True)])
def test_P8_rotation_reflection(ci, improper):
    hp = CONFIGS[ci].hp
    m, _ = oracle_model(hp, mu=[-1.0 - z for z in range(hp.n_species)])
    pos, sp, box = cluster(12, hp.n_species, 11 + ci)
    E0, Ea0, F0 = _EF(m, pos, sp, box)
    R = _rand_O3(np.random.default_rng(ci), improper)
    pos2 = (pos - 50.0) @ R.T + 50.0
    E1, Ea1, F1 = _EF(m, pos2, sp, box)
    scale = np.abs(F0).max()
    assert scale > 1e-6
    assert abs(E1 - E0) < 1e-11 * max(1, abs(E0))
    np.testing.assert_allclose(Ea1, Ea0, atol=1e-11)
    np.testing.assert_allclose(F1, F0 @ R.T, atol=1e-11 * max(1, scale))


def test_P8_translation_permutation_sumF():
    cfg, pos, sp, box = small_system(0, 81)
    hp = cfg.hp
    m, _ = oracle_model(hp, mu=[-1.0, -2.0])
    E0, Ea0, F0 = _EF(m, pos, sp, box)
    assert np.abs(F0.sum(0)).max() < 1e-10 * np.abs(F0).sum()
    # non-lattice translation
    E1, Ea1, F1 = _EF(m, pos + np.array([0.37, -1.91, 5.5]), sp, box)
    assert abs(E1 - E0) < 1e-10
    np.testing.assert_allclose(F1, F0, atol=1e-10)
    # lattice translation of individual atoms (unwrapped inputs): geometry unchanged
    g = np.random.default_rng(0)
    pos2 = pos + g.integers(-2, 3, pos.shape) * box
    E2, Ea2, F2 = _EF(m, pos2, sp, box)
    assert abs(E2 - E0) < 1e-10
    np.testing.assert_allclose(F2, F0, atol=1e-10)
    # permutation
    perm = g.permutation(pos.shape[0])
    E3, Ea3, F3 = _EF(m, pos[perm], sp[perm], box)
    assert abs(E3 - E0) < 1e-10
    np.testing.assert_allclose(F3, F0[perm], atol=1e-10)
    np.testing.assert_allclose(Ea3, Ea0[perm], atol=1e-11)


# ---- P9: strict locality ----------------------------------------------------------
def test_P9_strict_locality():
    cfg, pos, sp, box = small_system(0, 192)
    hp = cfg.hp
    m, _ = oracle_model(hp, mu=[-1.0, -2.0])
    nbr = O.neighbor_list(pos, box, hp.r_cut)
    E0, Ea0, F0 = O.energy_forces(m, pos, sp, box, nbr)
    i = 5
    # an atom k outside r_c of i (minimum image)
    d = pos - pos[i]
    d -= box * np.rint(d / box)
    far = np.nonzero(np.linalg.norm(d, axis=1) > hp.r_cut + 0.5)[0]
    k = int(far[0])
    pos2 = pos.copy()
    pos2[k] += np.array([0.2, -0.1, 0.15])
    nbr2 = O.neighbor_list(pos2, box, hp.r_cut)
    # E-hat_i evaluated from centre i's edges alone, before and after: bit-identical
    _, Ea_i, _ = O.energy_forces(m, pos, sp, box, nbr, centers=np.array([i]))
    _, Ea_i2, _ = O.energy_forces(m, pos2, sp, box, nbr2, centers=np.array([i]))
    assert Ea_i[i] == Ea_i2[i]
    # and the one-centre evaluation equals the full-system value
    assert abs(Ea_i[i] - Ea0[i]) < 1e-12
    # sub-system forces: F_a from centres within r_c of a only
    a = 17
    da = pos - pos[a]
    da -= box * np.rint(da / box)
    near = np.nonzero(np.linalg.norm(da, axis=1) < hp.r_cut)[0]
    _, _, Fsub = O.energy_forces(m, pos, sp, box, nbr, centers=near)
    np.testing.assert_allclose(Fsub[a], F0[a], atol=1e-12)


# ---- P10: continuity at the cutoff ---------------------------------------------------------------
def test_P10_cutoff_continuity():
    hp = CONFIGS[0].hp
    m, _ = oracle_model(hp)
    pos, sp, box = cluster(6, hp.n_species, 2, extent=3.0)
    pos = np.concatenate([pos, pos[:1] + np.array([[hp.r_cut, 0.0, 0.0]])])   # atom 6 exactly at r_c from atom 0
    sp = np.concatenate([sp, sp[:1]])
    out = []
    for dx in (-2e-6, -1e-6, 0.0, 1e-6, 2e-6):
        p = pos.copy(); p[6, 0] += dx
        out.append(_EF(m, p, sp, box))
    # atom 6 also interacts smoothly with the rest of the cluster, so test second differences across
    # r_c: a jump in E (or a kink, i.e. a jump in F) at the cutoff would show up at O(jump), the smooth
    # part only at O(E'' dx^2) ~ 1e-12
    for a, b, c in zip(out[:-2], out[1:-1], out[2:]):
        assert abs(a[0] - 2 * b[0] + c[0]) < 1e-10
        assert np.abs(a[2] - 2 * b[2] + c[2]).max() < 1e-9
    # list-membership change leaves E unchanged: a list built at r_c + skin gives the same E, F
    p = pos.copy(); p[6, 0] -= 0.3
    Ea = _EF(m, p, sp, box)
    Eb = _EF(m, p, sp, box, cutoff=hp.r_cut + 1.0)
    assert Ea[0] == pytest.approx(Eb[0], abs=1e-13)
    np.testing.assert_allclose(Ea[2], Eb[2], atol=1e-13)


# ---- P11: central finite differences -------------------------------------------------------------
@pytest.mark.parametrize("ci", [0, 1, 2, 4])
def test_P11_finite_differences(ci):
    hp = CONFIGS[ci].hp
    m, _ = oracle_model(hp)
    cfg, pos, sp, box = small_system(ci if ci != 2 else 4, 24)
    if ci == 2:
        sp = (np.arange(24) % hp.n_species).astype(np.int32)
    box = box * 1.0
    nbr = O.neighbor_list(pos, box, hp.r_cut + 0.01)
    E0, _, F = O.energy_forces(m, pos, sp, box, nbr)
    h = 1e-4
    g = np.random.default_rng(ci)
    comps = [(a, c) for a in range(24) for c in range(3)]
    if ci in (2, 4):
        comps = [comps[k] for k in g.permutation(len(comps))[:24]]
    scale = np.sqrt((F ** 2).mean())
    assert scale > 1e-8
    for (a, c) in comps:
        pp = pos.copy(); pp[a, c] += h
        pm = pos.copy(); pm[a, c] -= h
        Ep = O.energy_forces(m, pp, sp, box, nbr)[0]
        Em = O.energy_forces(m, pm, sp, box, nbr)[0]
        fd = -(Ep - Em) / (2 * h)
        assert abs(fd - F[a, c]) <= 1e-7 * max(scale, abs(F[a, c])) + 1e-11, (a, c, fd, F[a, c])


# ---- P12: parameter count of the paper's model --------------------------------
def test_P12_parameter_count():
    hp = Hparams(n_species=15, l_max=2, n_layers=2, n_tensor=64, n_bessel=8, poly_p=6, r_cut=4.0,
                 twobody_dims=(128, 256, 512, 1024), latent_dims=(1024, 1024, 1024), edge_dims=(128,),
                 avg_num_neighbors=26.8, resid_alpha=(0.5, 0.5))
    npaths = [len(p) for p in O.layer_paths(2, 2)]
    nfl = blob_num_floats(hp, npaths)
    assert nfl - sum(npaths) == 7_836_544
    total = nfl + 8 * 15 * 15                      # + per-ordered-pair Bessel frequencies (not built: NEXT-1)
    assert abs(total - 7.85e6) / 7.85e6 < 2.5e-3   # "7.85 million weights"
    m, blob = oracle_model(CONFIGS[0].hp)
    assert m.n_weights == blob_num_floats(CONFIGS[0].hp, [2])


# ---- P13 / P14: pair-potential special case, dense layers vs numpy -------------------------------
def _np_silu(z):
    return z / (1 + np.exp(-z))


def _pair_energy(hp, blob, zi, zj, r):
    """Independent numpy evaluation of E_ij(r, Z_i, Z_j) when all path weights are zero."""
    S, NB, d, n = hp.n_species, hp.n_bessel, hp.d, hp.n_tensor
    w = np.frombuffer(blob, dtype="<f4").astype(np.float64)
    o = 0
    def take(fi, fo):
        nonlocal o
        W = w[o:o + fi * fo].reshape(fi, fo); o += fi * fo
        return W
    x = r / hp.r_cut
    u = 1 - 28 * x ** 6 + 48 * x ** 7 - 21 * x ** 8 if x < 1 else 0.0
    h = np.zeros(2 * S + NB)
    h[zi] = 1; h[S + zj] = 1
    for k in range(NB):
        h[2 * S + k] = math.sqrt(2 / hp.r_cut) * math.sin((k + 1) * math.pi * r / hp.r_cut) / r * u
    fi = 2 * S + NB
    for wd in hp.twobody_dims:
        h = _np_silu(h @ take(fi, wd)); fi = wd
    xl = u * h
    nA = n * (hp.l_max + 1)
    o += d * nA
    npaths = [len(p) for p in O.layer_paths(hp.l_max, hp.n_layers)]
    for L in range(hp.n_layers):
        o += d * nA + npaths[L]
        mm = np.concatenate([xl, np.zeros(n)]); fi = d + n
        for wd in hp.latent_dims:
            mm = _np_silu(mm @ take(fi, wd)); fi = wd
        a = hp.resid_alpha[L]
        xl = xl / math.sqrt(1 + a * a) + a / math.sqrt(1 + a * a) * u * mm
    fi = d
    for wd in list(hp.edge_dims) + [1]:
        xl = xl @ take(fi, wd); fi = wd
    return float(xl[0])


@pytest.mark.parametrize("ci", [0, 1])
def test_P13_pair_potential_limit(ci):
    hp = CONFIGS[ci].hp
    m, blob = oracle_model(hp, zero_alpha=True)
    pos, sp, box = cluster(9, hp.n_species, 21)
    ei, ej, es = O.neighbor_list(pos, box, hp.r_cut)
    E, Ea, F = O.energy_forces(m, pos, sp, box, (ei, ej, es))
    Epair = 0.0
    Fpair = np.zeros_like(F)
    for i, j in zip(ei, ej):
        rv = pos[j] - pos[i]
        r = np.linalg.norm(rv)
        Epair += _pair_energy(hp, blob, sp[i], sp[j], r)
        h = 1e-5
        dE = (_pair_energy(hp, blob, sp[i], sp[j], r + h) - _pair_energy(hp, blob, sp[i], sp[j], r - h)) / (2 * h)
        Fpair[i] += dE * rv / r            # g_e parallel to r-hat
        Fpair[j] -= dE * rv / r
    assert abs(E - Epair) < 1e-11 * max(1, abs(Epair))
    np.testing.assert_allclose(F, Fpair, atol=1e-7 * max(1e-3, np.abs(F).max()))


def test_P14_two_body_latent_vs_numpy():
    # with the true alphas, x^0 must still equal the independent numpy two-body chain
    hp = CONFIGS[1].hp
    m, blob = oracle_model(hp)
    pos, sp, box = cluster(5, hp.n_species, 4, extent=3.0)
    ei, ej, es = O.neighbor_list(pos, box, hp.r_cut)
    t = lambda a: torch.from_numpy(a)
    _, parts = m.edge_energies(t(pos), t(sp.astype(np.int64)), t(box), t(ei), t(ej), t(es), return_parts=True)
    w = np.frombuffer(blob, dtype="<f4").astype(np.float64)
    S, NB = hp.n_species, hp.n_bessel
    for e in range(ei.shape[0]):
        r = np.linalg.norm(pos[ej[e]] - pos[ei[e]])
        x = r / hp.r_cut
        u = 1 - 28 * x ** 6 + 48 * x ** 7 - 21 * x ** 8
        h = np.zeros(2 * S + NB); h[sp[ei[e]]] = 1; h[S + sp[ej[e]]] = 1
        h[2 * S:] = [math.sqrt(2 / hp.r_cut) * math.sin(k * math.pi * r / hp.r_cut) / r * u for k in range(1, NB + 1)]
        o, fi = 0, 2 * S + NB
        for wd in hp.twobody_dims:
            h = _np_silu(h @ w[o:o + fi * wd].reshape(fi, wd)); o += fi * wd; fi = wd
        np.testing.assert_allclose(parts["x"][0][e].numpy(), u * h, atol=1e-13)
