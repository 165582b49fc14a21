"""Pins for the oracle's NEXT-1/NEXT-4 additions: trained per-pair Bessel frequencies
(PAPER.md:222), the ZBL pair repulsion and the Nose-Hoover thermostat; the readings
are listed in DESIGN.md.  Every pin is something other than the oracle's own formula: limits, invariants, brute
force, finite differences, conservation laws."""
import dataclasses
import math

import numpy as np
import torch

from oracle import allegro_oracle as O
from synthetic import CONFIGS

from oracle_util import cluster, oracle_model


def _EF(m, pos, sp, box):
    return O.energy_forces(m, pos, sp, box, O.neighbor_list(pos, box, m.hp.r_cut))


# ---------------------------------------------------------------------------------------------------
# per-pair Bessel frequencies
# ---------------------------------------------------------------------------------------------------
def test_bessel_freq_default_and_quarter_wave():
    r = torch.tensor([0.7, 1.3, 2.9], dtype=torch.float64)
    rc, nb = 4.0, 8
    w0 = (torch.arange(1, nb + 1, dtype=torch.float64) * math.pi / rc).expand(3, nb)
    assert torch.allclose(O.bessel_basis(r, rc, nb, w0), O.bessel_basis(r, rc, nb), rtol=0, atol=1e-15)
    # w r = pi/2 -> sin = 1 -> b = sqrt(2/rc)/r ;  w r = pi -> 0
    w = torch.stack([math.pi / 2 / r, math.pi / r], dim=1)
    b = O.bessel_basis(r, rc, 2, w)
    assert torch.allclose(b[:, 0], math.sqrt(2 / rc) / r, rtol=1e-15)
    assert b[:, 1].abs().max() < 1e-15


def test_pair_freq_table_default_equals_no_table_and_forces_fd():
    hp0 = CONFIGS[0].hp
    S, nb = hp0.n_species, hp0.n_bessel
    default = tuple(tuple(tuple(n * math.pi / hp0.r_cut for n in range(1, nb + 1)) for _ in range(S)) for _ in range(S))
    pos, sp, box = cluster(9, 2, 11, extent=3.5)
    m0, _ = oracle_model(hp0, mu=[-1.0, -2.0])
    m1, _ = oracle_model(dataclasses.replace(hp0, bessel_freq_pair=default), mu=[-1.0, -2.0])
    E0, _, F0 = _EF(m0, pos, sp, box)
    E1, _, F1 = _EF(m1, pos, sp, box)
    assert abs(E0 - E1) < 1e-13 and np.abs(F0 - F1).max() < 1e-13
    # trained (perturbed, ordered: [0][1] != [1][0]) frequencies: a different model whose forces are still -dE/dr
    g = np.random.default_rng(5)
    pert = tuple(tuple(tuple(w * (1 + 0.2 * g.uniform(-1, 1)) for w in row) for row in mat) for mat in default)
    m2, _ = oracle_model(dataclasses.replace(hp0, bessel_freq_pair=pert), mu=[-1.0, -2.0])
    E2, _, F2 = _EF(m2, pos, sp, box)
    assert abs(E2 - E0) > 1e-6
    h = 1e-4
    for a in (0, 5):
        for k in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[a, k] += h
            pm[a, k] -= h
            fd = -(_EF(m2, pp, sp, box)[0] - _EF(m2, pm, sp, box)[0]) / (2 * h)
            assert abs(fd - F2[a, k]) <= 1e-6 * max(1.0, np.abs(F2).max())


# ---------------------------------------------------------------------------------------------------
# ZBL
# ---------------------------------------------------------------------------------------------------
def test_zbl_limits_and_screening_length():
    t = lambda v: torch.tensor([v], dtype=torch.float64)
    # screening coefficients sum to one: phi -> bare Coulomb k_e Z_i Z_j / r as r -> 0
    assert abs(sum(O.ZBL_C) - 1.0) < 1e-12
    r = 1e-7
    phi = O.zbl_pair_energy(t(r), t(6.0), t(8.0), 4.0, 6).item()
    assert abs(phi * r / (O.KE_EV_A * 48.0) - 1.0) < 1e-5
    # k_e = e^2/(4 pi eps0) = alpha * hbar c = 1.973269804e3 eV A / 137.035999
    assert abs(O.KE_EV_A - 1973.269804 / 137.035999084) < 1e-6
    # a_ij = 0.8854 a_0 / (Z_i^0.23 + Z_j^0.23) with the Bohr radius 0.529177 A (the published universal length)
    assert abs(0.46850 / (0.8854 * 0.52917721) - 1.0) < 2e-4
    # repulsive, decreasing, and exactly zero from the cutoff on, C^1-continuously
    rr = torch.linspace(0.3, 3.999, 400, dtype=torch.float64)
    ph = O.zbl_pair_energy(rr, torch.full_like(rr, 1.0), torch.full_like(rr, 8.0), 4.0, 6)
    assert (ph > 0).all() and (ph[1:] < ph[:-1]).all()
    assert O.zbl_pair_energy(t(4.0), t(1.0), t(8.0), 4.0, 6).item() == 0.0
    assert O.zbl_pair_energy(t(4.0 - 1e-5), t(1.0), t(8.0), 4.0, 6).item() < 1e-12


def test_zbl_total_is_sum_over_unordered_pairs_and_forces():
    hp = dataclasses.replace(CONFIGS[0].hp, zbl_Z=(1.0, 8.0))
    pos, sp, box = cluster(10, 2, 21, extent=4.0, dmin=0.7)
    m0, _ = oracle_model(CONFIGS[0].hp, mu=[-1.0, -2.0])
    m1, _ = oracle_model(hp, mu=[-1.0, -2.0])
    E0, Ea0, F0 = _EF(m0, pos, sp, box)
    E1, Ea1, F1 = _EF(m1, pos, sp, box)
    zn = np.array(hp.zbl_Z)
    tot = 0.0
    per_atom = np.zeros(len(sp))
    for i in range(len(sp)):
        for j in range(i + 1, len(sp)):
            r = np.linalg.norm(pos[j] - pos[i])
            if r < hp.r_cut:
                ph = O.zbl_pair_energy(torch.tensor([r]), torch.tensor([zn[sp[i]]]), torch.tensor([zn[sp[j]]]), hp.r_cut, hp.poly_p).item()
                tot += ph
                per_atom[i] += 0.5 * ph
                per_atom[j] += 0.5 * ph
    assert tot > 0 and abs((E1 - E0) - tot) < 1e-10 * tot
    assert np.abs((Ea1 - Ea0) - per_atom).max() < 1e-10 * tot
    assert np.abs(F1.sum(0)).max() < 1e-9
    h = 1e-5
    for a in (0, 3, 9):
        for k in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[a, k] += h
            pm[a, k] -= h
            fd = -(_EF(m1, pp, sp, box)[0] - _EF(m1, pm, sp, box)[0]) / (2 * h)
            assert abs(fd - F1[a, k]) <= 1e-6 * max(1.0, np.abs(F1).max()), (a, k, fd, F1[a, k])


def test_zbl_uses_flat_cutoff_with_pair_cutoffs():
    """An (H centre, O neighbour) pair at 2 A is outside its ordered cutoff 1.25 A but still repels by ZBL."""
    from synthetic.configs import WATER_PAIR_CUTOFFS
    hp = dataclasses.replace(CONFIGS[0].hp, zbl_Z=(1.0, 8.0), r_cut_pair=WATER_PAIR_CUTOFFS)
    hpn = dataclasses.replace(CONFIGS[0].hp, r_cut_pair=WATER_PAIR_CUTOFFS)
    pos = np.array([[50.0, 50.0, 50.0], [52.0, 50.0, 50.0]])
    sp = np.array([0, 1], dtype=np.int32)
    box = np.array([100.0] * 3)
    m1, _ = oracle_model(hp)
    m0, _ = oracle_model(hpn)
    _, Ea1, _ = _EF(m1, pos, sp, box)
    _, Ea0, _ = _EF(m0, pos, sp, box)
    t = lambda v: torch.tensor([v], dtype=torch.float64)
    ph = O.zbl_pair_energy(t(2.0), t(1.0), t(8.0), 4.0, 6).item()
    assert np.allclose(Ea1 - Ea0, [0.5 * ph, 0.5 * ph], rtol=1e-12)


# ---------------------------------------------------------------------------------------------------
# Nose-Hoover
# ---------------------------------------------------------------------------------------------------
def _harmonic(n=24, seed=3):
    g = np.random.default_rng(seed)
    k = g.uniform(0.5, 4.0, (n, 3))                  # eV / A^2, independent oscillators of different frequencies
    x0 = np.zeros((n, 3))
    mass = g.uniform(1.0, 16.0, n)

    def force_fn(pos):
        d = pos - x0
        return float(0.5 * (k * d * d).sum()), -k * d
    pos = g.normal(0, 0.05, (n, 3))
    vel = g.normal(0, 0.01, (n, 3))
    return force_fn, pos, vel, mass


def test_nh_infinite_tau_is_nve_bit_for_bit():
    f, pos, vel, mass = _harmonic()
    e, F = f(pos)
    a = O.nve_step(f, pos, vel, F, mass, 0.5)
    b = O.nvt_step(f, pos, vel, F, mass, 0.5, 0.0, 0.0, 300.0, 1e30)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and abs(b[5]) < 1e-50


def _run(dt, steps, tau=25.0, t0=300.0):
    f, pos, vel, mass = _harmonic()
    e, F = f(pos)
    xi = eta = 0.0
    g = 3 * pos.shape[0]
    H0 = O.nh_conserved(e, O.kinetic_energy(vel, mass), xi, eta, g, t0, tau)
    worst, temps = 0.0, []
    for _ in range(steps):
        pos, vel, F, e, ek, xi, eta = O.nvt_step(f, pos, vel, F, mass, dt, xi, eta, t0, tau)
        worst = max(worst, abs(O.nh_conserved(e, ek, xi, eta, g, t0, tau) - H0))
        temps.append(2 * ek / (g * O.KB_EV))
    return worst, np.array(temps), (pos, vel, F, xi, eta, mass, f)


def test_nh_conserved_quantity_second_order():
    w1, _, _ = _run(0.5, 2000)
    w2, _, _ = _run(0.25, 4000)
    assert w1 < 1e-3 and 3.5 < w1 / w2 < 4.5, (w1, w2)


def test_nh_holds_the_target_temperature():
    # the time average of the kinetic temperature is T0 exactly for Nose-Hoover dynamics (d xi/dt averages to zero)
    _, temps, _ = _run(0.5, 20000, tau=20.0, t0=300.0)
    assert abs(temps[2000:].mean() / 300.0 - 1.0) < 0.02, temps[2000:].mean()


def test_nh_time_reversal():
    f, pos0, vel0, mass = _harmonic()
    e, F = f(pos0)
    pos, vel, xi, eta = pos0.copy(), vel0.copy(), 0.0, 0.0
    for _ in range(200):
        pos, vel, F, e, ek, xi, eta = O.nvt_step(f, pos, vel, F, mass, 0.5, xi, eta, 300.0, 25.0)
    vel, xi = -vel, -xi
    for _ in range(200):
        pos, vel, F, e, ek, xi, eta = O.nvt_step(f, pos, vel, F, mass, 0.5, xi, eta, 300.0, 25.0)
    assert np.abs(pos - pos0).max() < 1e-10 and np.abs(vel + vel0).max() < 1e-10 and abs(xi) < 1e-12
