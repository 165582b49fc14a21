"""GPU-vs-oracle parity with species-distinct sigma_{Z_i} and layer-distinct resid_alpha (`-m gpu`).

Every other parity test uses sigma = 1 for all species and alpha = 0.5 in all layers, which cannot see a wrong species
index in the three kernels that carry sigma (k_geom_fill -> sig[e], the EPI_LATENT_LAST epilogue, k_energy_parts), a
sigma dropped from the backward, or a per-layer c_old / c_new slip.  The oracle side of the same readings is pinned in
tests/test_oracle_sigma_alpha.py."""
import dataclasses

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import allegro_oracle as O
from synthetic import make_system
from synthetic.configs import scaled_config

from gpu_util import gpu_eval, make_both
from test_gpu_parity import _check_EF, _subsystem_check

ALPHA = {1: (0.8,), 2: (0.3, 0.8), 3: (0.3, 0.8, 0.5)}


def _sig(S):
    return [0.7 + 0.6 * z / max(S - 1, 1) for z in range(S)]


def _cfg(ci, n):
    cfg = scaled_config(ci, n)
    cfg.hp = dataclasses.replace(cfg.hp, resid_alpha=ALPHA[cfg.hp.n_layers])
    return cfg


@pytest.mark.parametrize("ci,n,precision", [(0, 192, 0), (1, 1536, 0), (2, 3000, 0), (4, 1200, 0), (1, 1536, 3), (4, 1200, 3)])
def test_energy_forces_fp32_distinct_sigma_alpha(ci, n, precision):
    cfg = _cfg(ci, n)
    pos, sp, box = make_system(cfg)
    sig = _sig(cfg.hp.n_species)
    model, oracle = make_both(cfg, precision=precision, sigma=sig)
    got, nb = gpu_eval(model, pos, sp, box)
    nbr = O.neighbor_list(pos, box, cfg.hp.r_cut)
    want = O.energy_forces(oracle, pos, sp, box, nbr)
    _check_EF(got, want, n, f"cfg{ci} prec{precision} sigma/alpha distinct")
    # the result must differ from the uniform-sigma one by far more than the tolerance (the case does discriminate)
    _, flat = make_both(cfg, precision=precision, sigma=1.0)
    F1 = O.energy_forces(flat, pos, sp, box, nbr)[2]
    assert np.abs(F1 - want[2]).max() > 1e-2 * np.abs(want[2]).max()


@pytest.mark.parametrize("ci,n", [(0, 192), (1, 1536), (2, 3000), (4, 1200)])
def test_energy_forces_tf32_distinct_sigma_alpha(ci, n):
    cfg = _cfg(ci, n)
    pos, sp, box = make_system(cfg)
    sig = _sig(cfg.hp.n_species)
    model, oracle = make_both(cfg, precision=1, sigma=sig)
    (E, Ea, F), nb = gpu_eval(model, pos, sp, box)
    E0, Ea0, F0 = O.energy_forces(oracle, pos, sp, box, O.neighbor_list(pos, box, cfg.hp.r_cut))
    mu = np.array(cfg.mu())[sp]
    assert abs(E - E0) <= 2e-3 * np.abs(Ea0 - mu).sum()
    assert np.abs(Ea - Ea0).max() <= 2e-3 * np.abs(Ea0 - mu).max()
    assert np.abs(F - F0).max() <= 2e-3 * np.abs(F0).max()
    assert np.linalg.norm(F - F0) <= 2e-3 * np.linalg.norm(F0)


def test_edge_energies_are_sigma_free_and_alpha_aware():
    """allegro_edge_energies returns E_ij before sigma / mu: same values whatever sigma is, and equal to
    the oracle's with layer-distinct alpha."""
    cfg = _cfg(1, 768)
    pos, sp, box = make_system(cfg)
    model, oracle = make_both(cfg, precision=0, sigma=_sig(2))
    p = torch.from_numpy(pos).cuda(); s = torch.from_numpy(sp).cuda()
    nb = model.neighbors(p, box, cfg.hp.r_cut)
    e, ee = model.edge_energies(p, s, box, nb)
    oi, oj, os_ = O.neighbor_list(pos, box, cfg.hp.r_cut)
    t = torch.from_numpy
    want = oracle.edge_energies(t(pos), t(sp.astype(np.int64)), t(box), t(oi), t(oj), t(os_)).numpy()
    np.testing.assert_allclose(ee.cpu().numpy(), want, atol=3e-6)
    Ei = np.zeros(pos.shape[0]); np.add.at(Ei, oi, want)
    sig, mu = np.array(_sig(2)), np.array(cfg.mu())
    assert abs(e.item() - float((sig[sp] * Ei + mu[sp]).sum())) / pos.shape[0] <= 1e-6


@pytest.mark.parametrize("ci,precision", [(2, 1), (4, 0)])
def test_full_size_subsystem_parity_distinct_sigma_alpha(ci, precision):
    S = {2: 5, 4: 4}[ci]
    _subsystem_check(ci, 16, precision, seed=1, sigma=_sig(S), resid_alpha=ALPHA[{2: 2, 4: 3}[ci]])
