"""GPU-vs-oracle parity for the SURVEY.md §8(f) additions (`-m gpu`): trained per-pair Bessel frequencies, ZBL pair
repulsion, energy-only and per-edge-energy outputs, Nose-Hoover NVT steps.  Tolerances as in test_gpu_parity.py."""
import ctypes
import dataclasses
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import allegro_oracle as O
from synthetic import make_system, maxwell_boltzmann
from synthetic.configs import ATOMIC_NUMBERS, WATER_PAIR_CUTOFFS, scaled_config
from synthetic.systems import masses_for

from gpu_util import gpu_eval, make_both, nbr_as_arrays
from test_gpu_parity import F_TOL_REL, _check_EF


def _freq_table(hp, seed):
    """n pi / r_c of each ordered pair, perturbed by up to +-20 % (a stand-in for trained values)."""
    g = np.random.default_rng(seed)
    S, nb = hp.n_species, hp.n_bessel
    rc = np.full((S, S), hp.r_cut) if hp.r_cut_pair is None else np.array(hp.r_cut_pair)
    w = np.arange(1, nb + 1)[None, None, :] * math.pi / rc[:, :, None]
    w = w * (1 + 0.2 * g.uniform(-1, 1, w.shape))
    return tuple(tuple(tuple(float(x) for x in row) for row in mat) for mat in w)


def _cfg(ci, n, **hp_changes):
    cfg = scaled_config(ci, n)
    cfg.hp = dataclasses.replace(cfg.hp, **hp_changes)
    return cfg


def _zn(cfg):
    return tuple(ATOMIC_NUMBERS[s] for s in cfg.species_names) if cfg.kind != "random4" else (1.0, 6.0, 7.0, 8.0)


@pytest.mark.parametrize("ci,n,precision,pair", [(0, 192, 0, False), (1, 1536, 0, True), (1, 1536, 3, True), (2, 3000, 0, False)])
def test_bessel_frequencies(ci, n, precision, pair):
    cfg = _cfg(ci, n)
    if pair:
        cfg.hp = dataclasses.replace(cfg.hp, r_cut_pair=WATER_PAIR_CUTOFFS)
    cfg.hp = dataclasses.replace(cfg.hp, bessel_freq_pair=_freq_table(cfg.hp, 7 + ci))
    pos, sp, box = make_system(cfg)
    model, oracle = make_both(cfg, precision=precision)
    got, _ = gpu_eval(model, pos, sp, box, cutoff=cfg.hp.r_cut + 0.5)
    want = O.energy_forces(oracle, pos, sp, box, O.neighbor_list(pos, box, cfg.hp.r_cut))
    _check_EF(got, want, n, f"bessel freq cfg{ci}")
    # the default table is the untrained basis
    plain = _cfg(ci, n, r_cut_pair=cfg.hp.r_cut_pair)
    model.set_bessel_frequencies(None)
    got0, _ = gpu_eval(model, pos, sp, box)
    _, oracle0 = make_both(plain, precision=precision)
    _check_EF(got0, O.energy_forces(oracle0, pos, sp, box, O.neighbor_list(pos, box, cfg.hp.r_cut)), n, "default basis")


@pytest.mark.parametrize("ci,n,precision,pair", [(0, 192, 0, False), (1, 1536, 0, True), (2, 3000, 0, False),
                                                 (4, 1200, 0, False), (1, 1536, 1, False)])
def test_zbl(ci, n, precision, pair):
    cfg = _cfg(ci, n)
    cfg.hp = dataclasses.replace(cfg.hp, zbl_Z=_zn(cfg), r_cut_pair=WATER_PAIR_CUTOFFS if pair else None)
    pos, sp, box = make_system(cfg)
    model, oracle = make_both(cfg, precision=precision)
    (E, Ea, F), _ = gpu_eval(model, pos, sp, box, cutoff=cfg.hp.r_cut + 0.5)
    nbr = O.neighbor_list(pos, box, cfg.hp.r_cut)
    want = O.energy_forces(oracle, pos, sp, box, nbr)
    # the ZBL part alone, from the oracle without it (same blob): it must be a visible share of E and F
    _, oracle_n = make_both(_cfg(ci, n, r_cut_pair=cfg.hp.r_cut_pair), precision=precision)
    base = O.energy_forces(oracle_n, pos, sp, box, nbr)
    assert abs(want[0] - base[0]) > 1e-3 and np.abs(want[2] - base[2]).max() > 1e-3
    if precision in (0, 3):
        _check_EF((E, Ea, F), want, n, f"zbl cfg{ci}")
    else:
        mu = np.array(cfg.mu())[sp]
        assert abs(E - want[0]) <= 2e-3 * np.abs(want[1] - mu).sum()
        assert np.abs(F - want[2]).max() <= 2e-3 * np.abs(want[2]).max()
    # fp64 term: switching the network's contribution off (compare differences) leaves ZBL to ~1e-12 relative
    model.set_zbl(None)
    (E_n, Ea_n, F_n), _ = gpu_eval(model, pos, sp, box, cutoff=cfg.hp.r_cut + 0.5)
    dz = (Ea - Ea_n) - (want[1] - base[1])
    assert np.abs(dz).max() <= 1e-9 * max(1.0, np.abs(want[1] - base[1]).max())
    dzf = (F - F_n) - (want[2] - base[2])
    assert np.abs(dzf).max() <= 1e-9 * max(1.0, np.abs(want[2] - base[2]).max())


@pytest.mark.parametrize("ci,n,precision", [(0, 192, 0), (1, 1536, 1)])
def test_energy_only_matches_full_evaluation(ci, n, precision):
    cfg = _cfg(ci, n, zbl_Z=(1.0, 8.0))
    pos, sp, box = make_system(cfg)
    model, _ = make_both(cfg, precision=precision)
    p = torch.from_numpy(pos).cuda(); s = torch.from_numpy(sp).cuda()
    nb = model.neighbors(p, box, cfg.hp.r_cut + 0.5)
    e, ea, f = model.compute(p, s, box, nb)
    l0 = model.launches
    e2, ea2, f2 = model.compute(p, s, box, nb, want_forces=False)
    l1 = model.launches
    model.compute(p, s, box, nb)
    l2 = model.launches
    torch.cuda.synchronize()
    assert f2 is None and e2.item() == e.item() and torch.equal(ea, ea2)      # same kernels, same order: bit-exact
    assert (l1 - l0) <= (l2 - l1) - 5                                         # the backward launches are gone
    E_h, Ea_h, F_h = model.compute_host(pos, sp, box, nb)
    assert E_h == e.item()


@pytest.mark.parametrize("ci,n,precision,pair", [(0, 192, 0, False), (1, 1536, 0, True), (4, 1200, 3, False)])
def test_edge_energies(ci, n, precision, pair):
    cfg = _cfg(ci, n, r_cut_pair=WATER_PAIR_CUTOFFS if pair else None)
    pos, sp, box = make_system(cfg)
    model, oracle = make_both(cfg, precision=precision, chunk_edges=20000 if ci == 1 else None)
    p = torch.from_numpy(pos).cuda(); s = torch.from_numpy(sp).cuda()
    nb = model.neighbors(p, box, cfg.hp.r_cut + 0.5)                          # skin list: some candidates are not edges
    e, ee = model.edge_energies(p, s, box, nb)
    e_full, ea, _ = model.compute(p, s, box, nb)
    torch.cuda.synchronize()
    gi, gj, gs = nbr_as_arrays(nb)
    t = torch.from_numpy
    want = oracle.edge_energies(t(pos), t(sp.astype(np.int64)), t(box), t(gi), t(gj), t(gs)).numpy()
    got = ee.cpu().numpy()
    assert got.shape == want.shape
    assert np.array_equal(got == 0.0, want == 0.0) and (want == 0.0).sum() > 0   # dropped candidates: exactly 0
    print(f"[edge energies cfg{ci}] max|dE_ij|={np.abs(got - want).max():.3e} max|E_ij|={np.abs(want).max():.3e}")
    assert np.abs(got - want).max() <= 1e-6
    assert e.item() == e_full.item()
    # E-hat_i = sigma_Z sum_j E_ij + mu_Z from the returned edge energies
    Ei = np.zeros(n); np.add.at(Ei, gi, got)
    assert np.abs(cfg.sigma * Ei + np.array(cfg.mu())[sp] - ea.cpu().numpy()).max() < 1e-9


def test_nvt_steps_match_oracle():
    cfg = _cfg(0, 192, zbl_Z=(1.0, 8.0))
    pos, sp, box = make_system(cfg)
    vel = maxwell_boltzmann(cfg, sp) * 1.3                                    # start off-target so xi moves
    model, oracle = make_both(cfg)
    mass = masses_for(cfg)
    dt, nsteps, t0, tau = 0.5, 6, 300.0, 20.0

    def force_fn(p):
        E, _, F = O.energy_forces(oracle, p, sp, box, O.neighbor_list(p, box, cfg.hp.r_cut))
        return E, F
    p_o, v_o = pos.copy(), vel.copy()
    e_o, f_o = force_fn(p_o)
    xi = eta = 0.0
    for _ in range(nsteps):
        p_o, v_o, f_o, e_o, ek_o, xi, eta = O.nvt_step(force_fn, p_o, v_o, f_o, mass[sp], dt, xi, eta, t0, tau)
    p = torch.from_numpy(pos.copy()).cuda(); v = torch.from_numpy(vel.copy()).cuda()
    s = torch.from_numpy(sp).cuda(); mg = torch.from_numpy(mass).cuda()
    nb = model.neighbors(p, box, cfg.hp.r_cut + 1.0)
    e, _, f = model.compute(p, s, box, nb)
    ek = torch.zeros(1, dtype=torch.float64, device="cuda")
    st = torch.zeros(2, dtype=torch.float64, device="cuda")
    ctr = ctypes.c_int64(0)
    for _ in range(nsteps):
        model.step_nvt(p, v, f, s, mg, box, dt, 3, 1.0, nb, ctr, e, ek, st, t0, tau)
    torch.cuda.synchronize()
    assert ctr.value == nsteps and abs(xi) > 1e-5
    np.testing.assert_allclose(p.cpu().numpy(), p_o, atol=1e-7)
    np.testing.assert_allclose(v.cpu().numpy(), v_o, atol=1e-7)
    xi_g, eta_g = st.cpu().numpy()
    assert abs(xi_g - xi) <= 1e-6 * abs(xi) and abs(eta_g - eta) <= 1e-6 * abs(eta)
    tol_ek = nsteps * dt * F_TOL_REL * np.abs(v_o).sum()
    assert abs(ek.item() - ek_o) < tol_ek
    # the conserved quantity of the two trajectories agrees (its own drift is the integrator's, pinned in
    # tests/test_oracle_next4.py on a harmonic system; here ZBL makes the O-H forces stiff on purpose)
    H = O.nh_conserved(e.item(), ek.item(), xi_g, eta_g, 3 * 192, t0, tau)
    H_o = O.nh_conserved(e_o, ek_o, xi, eta, 3 * 192, t0, tau)
    assert abs(H - H_o) < 192 * 2e-6 + 2 * tol_ek


def test_md_steps_replayed_from_a_cuda_graph_match_the_oracle():
    """14 NVE steps with a rebuild every 6: steps 0, 6, 12 run eagerly (list rebuild), 1, 7, 13 are captured, the others
    are graph replays; the trajectory must still be the oracle's."""
    import os
    cfg = _cfg(0, 192)
    pos, sp, box = make_system(cfg)
    vel = maxwell_boltzmann(cfg, sp)
    model, oracle = make_both(cfg)
    mass = masses_for(cfg)
    dt, nsteps = 0.5, 14

    def force_fn(p):
        E, _, F = O.energy_forces(oracle, p, sp, box, O.neighbor_list(p, box, cfg.hp.r_cut))
        return E, F
    p_o, v_o = pos.copy(), vel.copy()
    e_o, f_o = force_fn(p_o)
    for _ in range(nsteps):
        p_o, v_o, f_o, e_o = O.nve_step(force_fn, p_o, v_o, f_o, mass[sp], dt)
    p = torch.from_numpy(pos.copy()).cuda(); v = torch.from_numpy(vel.copy()).cuda()
    s = torch.from_numpy(sp).cuda(); mg = torch.from_numpy(mass).cuda()
    nb = model.neighbors(p, box, cfg.hp.r_cut + 1.0)
    e, _, f = model.compute(p, s, box, nb)
    ek = torch.zeros(1, dtype=torch.float64, device="cuda")
    ctr = ctypes.c_int64(0)
    per_step = []
    for _ in range(nsteps):
        l0 = model.launches
        model.step_nve(p, v, f, s, mg, box, dt, 6, 1.0, nb, ctr, e, ek)
        per_step.append(model.launches - l0)
    torch.cuda.synchronize()
    if os.environ.get("B200_ALLEGRO_NO_GRAPH"):
        assert model.graph_steps == 0
    else:
        assert model.graph_steps == nsteps - 3, model.graph_steps          # all but the three rebuild steps
        assert len(set(per_step[k] for k in range(nsteps) if k % 6)) == 1   # replayed steps count the same launches
    np.testing.assert_allclose(p.cpu().numpy(), p_o, atol=2e-7)
    np.testing.assert_allclose(v.cpu().numpy(), v_o, atol=2e-7)
    assert abs(e.item() - e_o) / 192 < 2e-6
    # a setter invalidates the captured step: the next step runs eagerly with the new configuration
    g0 = model.graph_steps
    model.set_zbl((1.0, 8.0))
    model.step_nve(p, v, f, s, mg, box, dt, 6, 1.0, nb, ctr, e, ek)       # step 14: no rebuild, but not the captured state
    torch.cuda.synchronize()
    assert model.graph_steps == g0
    e_chk, _, f_chk = model.compute(p, s, box, nb)
    torch.cuda.synchronize()
    assert abs(e_chk.item() - e.item()) < 1e-9 and (f_chk - f).abs().max().item() < 1e-9   # forces include the ZBL term


def test_edge_cases_of_the_new_entry_points():
    """n_local = N is allegro_compute, n_local = 0 evaluates nothing; a centre whose candidates all lie beyond its pair
    cutoffs gets mu_Z (+ ZBL); an isolated system has no edges at all."""
    cfg = _cfg(0, 192, zbl_Z=(1.0, 8.0))
    pos, sp, box = make_system(cfg)
    model, _ = make_both(cfg)
    p = torch.from_numpy(pos).cuda(); s = torch.from_numpy(sp).cuda()
    nb = model.neighbors(p, box, cfg.hp.r_cut + 0.5)
    e, ea, f = model.compute(p, s, box, nb)
    eN, eaN, fN = model.compute_local(p, s, 192, box, nb)
    e0, ea0, f0 = model.compute_local(p, s, 0, box, nb)
    eh, eah, fh = model.compute_local(p, s, 100, box, nb)
    torch.cuda.synchronize()
    assert eN.item() == e.item() and torch.equal(ea, eaN) and (f - fN).abs().max().item() < 1e-12
    assert e0.item() == 0.0 and ea0.abs().max().item() == 0.0 and f0.abs().max().item() == 0.0
    assert torch.equal(eah[:100], ea[:100]) and eah[100:].abs().max().item() == 0.0
    assert abs(eh.item() - ea[:100].sum().item()) < 1e-9
    # tiny pair cutoffs: no edge survives the compaction although every row has candidates
    model.set_pair_cutoffs(((0.2, 0.2), (0.2, 0.2)))
    model.set_zbl(None)
    e1, ea1, f1 = model.compute(p, s, box, nb)
    e_e, ee = model.edge_energies(p, s, box, nb)
    torch.cuda.synchronize()
    mu = np.array(cfg.mu())[sp]
    assert model.last_active_edges() == 0
    assert np.array_equal(ea1.cpu().numpy(), mu) and f1.abs().max().item() == 0.0 and ee.abs().max().item() == 0.0
    # two atoms further apart than the cutoff in a big box: empty list
    model.set_pair_cutoffs(None)
    p2 = torch.tensor([[1.0, 1.0, 1.0], [9.0, 9.0, 9.0]], dtype=torch.float64, device="cuda")
    s2 = torch.tensor([0, 1], dtype=torch.int32, device="cuda")
    nb2 = model.neighbors(p2, [30.0, 30.0, 30.0], cfg.hp.r_cut)
    assert nb2.n_edges == 0
    e2, ea2, f2 = model.compute(p2, s2, [30.0, 30.0, 30.0], nb2)
    e3, ee3 = model.edge_energies(p2, s2, [30.0, 30.0, 30.0], nb2)
    torch.cuda.synchronize()
    assert np.array_equal(ea2.cpu().numpy(), np.array(cfg.mu())) and f2.abs().max().item() == 0.0 and ee3.numel() == 0
