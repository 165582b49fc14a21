"""Pins P15 (neighbor list) and P16 (NVE integrator) for the oracle."""
import math

import numpy as np

from oracle import allegro_oracle as O
from synthetic import CONFIGS, make_system
from synthetic.configs import scaled_config


def _as_set(nbr):
    i, j, s = nbr
    return set(zip(i.tolist(), j.tolist(), s[:, 0].tolist(), s[:, 1].tolist(), s[:, 2].tolist()))


def test_P15_tree_vs_brute_and_symmetry():
    cfg = scaled_config(1, 384)            # 128 waters, L = 18.6 A > 2 * 5 A: the k-d tree branch
    pos, sp, box = make_system(cfg)
    g = np.random.default_rng(1)
    pos = pos + g.integers(-1, 2, pos.shape) * box     # unwrapped input
    for cutoff in (4.0, 5.0):
        a = O.neighbor_list(pos, box, cutoff)
        b = O.neighbor_list_brute(pos, box, cutoff)
        for x, y in zip(a, b):
            assert np.array_equal(x, y)
        S = _as_set(a)
        assert len(S) == a[0].shape[0]
        for (i, j, sx, sy, sz) in list(S)[:5000]:
            assert (j, i, -sx, -sy, -sz) in S
        # sorted by (i, j, sx, sy, sz)
        key = list(zip(a[0].tolist(), a[1].tolist(), *[a[2][:, k].tolist() for k in range(3)]))
        assert key == sorted(key)
    deg = O.neighbor_list(pos, box, 4.0)[0].shape[0] / pos.shape[0]
    assert abs(deg - 4 / 3 * math.pi * 64 * 0.1 * (128 / 216)) / 15.9 < 0.15       # mean degree -> 26.8


def test_P15_small_box_multiple_images_and_self_images():
    g = np.random.default_rng(3)
    box = np.array([3.0, 3.5, 4.2])
    pos = g.uniform(0, 1, (5, 3)) * box
    i, j, s = O.neighbor_list(pos, box, 4.0)
    assert ((i == j) & (np.abs(s).sum(1) > 0)).any()          # self-images are edges when L < cutoff
    # independent check by explicit image enumeration
    cnt = 0
    for a in range(5):
        for b in range(5):
            for sx in range(-3, 4):
                for sy in range(-3, 4):
                    for sz in range(-3, 4):
                        if a == b and sx == sy == sz == 0:
                            continue
                        d = pos[b] - pos[a] + np.array([sx, sy, sz]) * box
                        cnt += (d @ d) < 16.0
    assert cnt == i.shape[0]


def test_P15_lattice_shift_invariance():
    cfg = scaled_config(0, 192)
    pos, sp, box = make_system(cfg)
    a = O.neighbor_list(pos, box, 4.0)
    k = np.zeros_like(pos); k[7] = [1, -2, 0]; k[100] = [0, 0, 3]
    b = O.neighbor_list(pos + k * box, box, 4.0)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    # shifts change by q_i - q_j, geometry does not
    np.testing.assert_array_equal(b[2], a[2] + k[a[0]].astype(int) - k[a[1]].astype(int))


def test_P16_harmonic_oscillator_and_reversal():
    # 1-D harmonic oscillator through the same integrator routines: velocity Verlet closed form
    k_spring, mass, dt = 2.0, 3.0, 0.5
    m = np.array([mass])

    def force_fn(p):
        return 0.5 * k_spring * float(p[0, 0] ** 2), np.array([[-k_spring * p[0, 0], 0.0, 0.0]])

    pos = np.array([[1.0, 0.0, 0.0]]); vel = np.zeros((1, 3))
    _, F = force_fn(pos)
    w2 = k_spring / mass * O.ACC_CONV
    # exact velocity-Verlet propagator for the oscillator: x_n = cos(n theta), cos theta = 1 - w2 dt^2 / 2
    theta = math.acos(1 - w2 * dt * dt / 2)
    e0 = 0.5 * k_spring + O.kinetic_energy(vel, m)
    p, v, f = pos, vel, F
    for n in range(1, 201):
        p, v, f, ep = O.nve_step(force_fn, p, v, f, m, dt)
        assert abs(p[0, 0] - math.cos(n * theta)) < 1e-10
    etot = ep + O.kinetic_energy(v, m)
    assert abs(etot - e0) < w2 * dt * dt * e0            # bounded O(dt^2) energy error
    # time reversal
    v = -v
    for n in range(200):
        p, v, f, ep = O.nve_step(force_fn, p, v, f, m, dt)
    assert abs(p[0, 0] - 1.0) < 1e-10 and abs(v[0, 0]) < 1e-10


def test_P16_drift_scales_dt2():
    errs = []
    for dt in (0.5, 0.25):
        k_spring, m = 2.0, np.array([3.0])
        f = lambda p: (0.5 * k_spring * float(p[0, 0] ** 2), np.array([[-k_spring * p[0, 0], 0.0, 0.0]]))
        p = np.array([[1.0, 0, 0]]); v = np.zeros((1, 3)); F = f(p)[1]
        worst = 0.0
        for _ in range(int(200 / dt)):
            p, v, F, ep = O.nve_step(f, p, v, F, m, dt)
            worst = max(worst, abs(ep + O.kinetic_energy(v, m) - 1.0))
        errs.append(worst)
    assert 3.5 < errs[0] / errs[1] < 4.5
