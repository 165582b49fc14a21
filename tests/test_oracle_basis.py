"""Pins P1-P3: the oracle's angular and radial basis against closed forms."""
import math

import numpy as np
import torch

from oracle import allegro_oracle as O


def _rand_unit(n, seed=0):
    g = np.random.default_rng(seed)
    v = g.standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def _closed_form_Y(v):
    """SURVEY §8(c) S4 closed forms, l <= 3 (component normalisation, m = -l..l)."""
    x, y, z = v[:, 0], v[:, 1], v[:, 2]
    s = math.sqrt
    cols = [np.ones_like(x),
            s(3) * y, s(3) * z, s(3) * x,
            s(15) * x * y, s(15) * y * z, s(5) / 2 * (3 * z * z - 1), s(15) * x * z, s(15) / 2 * (x * x - y * y),
            s(35 / 8) * y * (3 * x * x - y * y), s(105) * x * y * z, s(21 / 8) * y * (5 * z * z - 1),
            s(7) / 2 * (5 * z ** 3 - 3 * z), s(21 / 8) * x * (5 * z * z - 1), s(105) / 2 * z * (x * x - y * y),
            s(35 / 8) * x * (x * x - 3 * y * y)]
    return np.stack(cols, axis=1)


def test_P1_closed_forms_l_le_3():
    v = _rand_unit(200)
    Y = O.real_sph_harm(torch.from_numpy(v), 3).numpy()
    assert Y.shape == (200, 16)
    np.testing.assert_allclose(Y, _closed_form_Y(v), rtol=0, atol=1e-13)


def test_P1_poles_and_axes():
    v = np.array([[0, 0, 1.0], [0, 0, -1.0], [1.0, 0, 0], [0, 1.0, 0]])
    Y = O.real_sph_harm(torch.from_numpy(v), 3).numpy()
    np.testing.assert_allclose(Y, _closed_form_Y(v), rtol=0, atol=1e-14)


def test_P1_norm_and_parity_to_l6():
    v = _rand_unit(50, 1)
    Y = O.real_sph_harm(torch.from_numpy(v), 6).numpy()
    Ym = O.real_sph_harm(torch.from_numpy(-v), 6).numpy()
    for l in range(7):
        blk = slice(l * l, (l + 1) ** 2)
        np.testing.assert_allclose((Y[:, blk] ** 2).sum(1), 2 * l + 1, rtol=1e-12)
        np.testing.assert_allclose(Ym[:, blk], (-1) ** l * Y[:, blk], atol=1e-12)


def test_P1_orthogonality_on_sphere():
    # (1/4pi) int Y_a Y_b dOmega = delta_ab  (component normalisation), Gauss-Legendre x uniform phi
    nt, nph = 16, 32
    ct, wt = np.polynomial.legendre.leggauss(nt)
    ph = np.arange(nph) * 2 * np.pi / nph
    CT, PH = np.meshgrid(ct, ph, indexing="ij")
    st = np.sqrt(1 - CT ** 2)
    v = np.stack([st * np.cos(PH), st * np.sin(PH), CT], -1).reshape(-1, 3)
    w = (wt[:, None] * np.ones(nph)[None, :] / nph / 2).reshape(-1)
    Y = O.real_sph_harm(torch.from_numpy(v), 4).numpy()
    G = (Y * w[:, None]).T @ Y
    np.testing.assert_allclose(G, np.eye(25), atol=1e-12)


def test_P2_envelope():
    p = 6
    x = torch.tensor([0.0, 1.0, 1.5, 0.3], dtype=torch.float64)
    u = O.poly_cutoff(x, p)
    assert u[0] == 1.0 and u[1] == 0.0 and u[2] == 0.0
    # p = 6 coefficients 28 / 48 / 21
    assert abs(float(u[3]) - (1 - 28 * 0.3 ** 6 + 48 * 0.3 ** 7 - 21 * 0.3 ** 8)) < 1e-15
    # u'(1) = u''(1) = 0 and closed form u'(x) = -(p(p+1)(p+2)/2) x^(p-1) (1-x)^2, via autograd
    xs = torch.linspace(0.05, 0.999, 40, dtype=torch.float64).requires_grad_(True)
    us = O.poly_cutoff(xs, p)
    du, = torch.autograd.grad(us.sum(), xs, create_graph=True)
    want = -(p * (p + 1) * (p + 2) / 2) * xs ** (p - 1) * (1 - xs) ** 2
    np.testing.assert_allclose(du.detach().numpy(), want.detach().numpy(), atol=1e-12)
    x1 = torch.tensor([1.0 - 1e-9], dtype=torch.float64, requires_grad=True)
    d1, = torch.autograd.grad(O.poly_cutoff(x1, p).sum(), x1, create_graph=True)
    d2, = torch.autograd.grad(d1.sum(), x1)
    assert abs(float(d1.detach())) < 1e-12 and abs(float(d2)) < 1e-6


def test_P3_bessel_orthonormal():
    # int_0^rc b_n b_m r^2 dr = delta_nm : fixes the prefactor sqrt(2/rc) (vs 2/rc)
    rc = 4.0
    xg, wg = np.polynomial.legendre.leggauss(200)
    r = 0.5 * rc * (xg + 1)
    w = 0.5 * rc * wg
    b = O.bessel_basis(torch.from_numpy(r), rc, 8).numpy()
    G = (b * (w * r * r)[:, None]).T @ b
    np.testing.assert_allclose(G, np.eye(8), atol=1e-10)
    # value check at one point, n = 3
    assert abs(b[17, 2] - math.sqrt(2 / rc) * math.sin(3 * math.pi * r[17] / rc) / r[17]) < 1e-14
