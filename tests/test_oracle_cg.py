"""Pins P4, P5, P5b, P6: Clebsch-Gordan blocks, paths, fused tensor."""
import itertools
import math

import numpy as np
import pytest
import torch

from oracle import allegro_oracle as O

TRIPLES = [(l1, l2, lo) for l1 in range(4) for l2 in range(4) for lo in range(abs(l1 - l2), min(l1 + l2, 3) + 1)]


def _Y(v, l):
    return O.real_sph_harm(torch.from_numpy(np.atleast_2d(v)), l).numpy()[:, l * l:(l + 1) ** 2]


def _rand_O3(rng, improper):
    A = rng.standard_normal((3, 3))
    Q, R = np.linalg.qr(A)
    Q = Q * np.sign(np.diag(R))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    return -Q if improper else Q


def _wigner_D(R, l, rng):
    """D with Y_l(R v) = D Y_l(v), least squares over random unit vectors."""
    v = rng.standard_normal((60, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    Yv, YRv = _Y(v, l), _Y(v @ R.T, l)
    D, res, *_ = np.linalg.lstsq(Yv, YRv, rcond=None)
    assert np.abs(Yv @ D - YRv).max() < 1e-11
    return D.T


@pytest.mark.parametrize("l1,l2,lo", TRIPLES)
def test_P4_orthonormal(l1, l2, lo):
    C = O.real_cg(l1, l2, lo)
    G = np.einsum("abc,abd->cd", C, C)
    np.testing.assert_allclose(G, np.eye(2 * lo + 1), atol=1e-13)


def test_P4_closed_forms():
    for l in range(4):
        C = O.real_cg(l, 0, l)                      # l x 0 -> l = identity
        np.testing.assert_allclose(C[:, 0, :], np.eye(2 * l + 1), atol=1e-14)
        C = O.real_cg(l, l, 0)                      # l x l -> 0 = delta / sqrt(2l+1)
        np.testing.assert_allclose(C[:, :, 0], np.eye(2 * l + 1) / math.sqrt(2 * l + 1), atol=1e-14)
    # 1 x 1 -> 1 = +- epsilon_abc / sqrt 2 in the (y, z, x) component order (a cross product)
    C = O.real_cg(1, 1, 1)
    eps = np.zeros((3, 3, 3))
    for a, b, c in itertools.permutations(range(3)):
        eps[a, b, c] = np.linalg.det(np.eye(3)[[a, b, c]])
    # component order (y,z,x) is a cyclic permutation of (x,y,z): epsilon is unchanged
    assert np.allclose(C, eps / math.sqrt(2)) or np.allclose(C, -eps / math.sqrt(2))
    # sign rule: first non-zero entry positive
    for (l1, l2, lo) in TRIPLES:
        f = O.real_cg(l1, l2, lo).reshape(-1)
        assert f[np.nonzero(np.abs(f) > 1e-12)[0][0]] > 0


def test_P4_complex_cg_textbook_values():
    # <1 0 1 0|2 0> = sqrt(2/3), <1 1 1 -1|0 0> = 1/sqrt3, <1 1 1 -1|1 0> = 1/sqrt2, <2 0 1 0|1 0> = -sqrt(2/5)
    assert abs(O.su2_cg(1, 0, 1, 0, 2, 0) - math.sqrt(2 / 3)) < 1e-15
    assert abs(O.su2_cg(1, 1, 1, -1, 0, 0) - 1 / math.sqrt(3)) < 1e-15
    assert abs(O.su2_cg(1, 1, 1, -1, 1, 0) - 1 / math.sqrt(2)) < 1e-15
    assert abs(O.su2_cg(2, 0, 1, 0, 1, 0) + math.sqrt(2 / 5)) < 1e-15
    assert abs(O.su2_cg(1, 1, 1, 1, 2, 2) - 1.0) < 1e-15


@pytest.mark.parametrize("improper", [False, True])
def test_P5_equivariance(improper):
    rng = np.random.default_rng(5 + improper)
    R = _rand_O3(rng, improper)
    D = {l: _wigner_D(R, l, rng) for l in range(4)}
    for (l1, l2, lo) in TRIPLES:
        C = O.real_cg(l1, l2, lo)
        x = rng.standard_normal(2 * l1 + 1)
        y = rng.standard_normal(2 * l2 + 1)
        lhs = np.einsum("abc,a,b->c", C, D[l1] @ x, D[l2] @ y)
        rhs = D[lo] @ np.einsum("abc,a,b->c", C, x, y)
        # D from Y carries parity (-1)^l; the CG block maps parities p1 p2 -> must be compared with
        # the output irrep's own parity: for odd l1+l2+lo the output is a pseudo-tensor.
        if improper and (l1 + l2 + lo) % 2 == 1:
            rhs = -rhs
        np.testing.assert_allclose(lhs, rhs, atol=1e-10)


def test_P5b_self_coupling():
    # C(Y_l1(v), Y_l2(v)) = kappa * Y_lo(v), kappa independent of v (even sum) and == 0 (odd sum)
    rng = np.random.default_rng(7)
    v = rng.standard_normal((20, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    for (l1, l2, lo) in TRIPLES:
        C = O.real_cg(l1, l2, lo)
        z = np.einsum("abc,ea,eb->ec", C, _Y(v, l1), _Y(v, l2))
        if (l1 + l2 + lo) % 2 == 1:
            assert np.abs(z).max() < 1e-12
        else:
            Yo = _Y(v, lo)
            kappa = (z * Yo).sum(1) / (Yo * Yo).sum(1)
            np.testing.assert_allclose(z, kappa[:, None] * Yo, atol=1e-12)
            assert np.ptp(kappa) < 1e-12 and abs(kappa[0]) > 1e-3
    # magnitudes from the survey's scratch check (before the sign rule): sqrt3, 1.095445, sqrt2, sqrt3
    def kap(l1, l2, lo):
        C = O.real_cg(l1, l2, lo)
        z = np.einsum("abc,a,b->c", C, _Y(v[0], l1)[0], _Y(v[0], l2)[0])
        Yo = _Y(v[0], lo)[0]
        return abs((z * Yo).sum() / (Yo * Yo).sum())
    assert abs(kap(1, 1, 0) - math.sqrt(3)) < 1e-12
    assert abs(kap(1, 1, 2) - 1.0954451150103321) < 1e-12
    assert abs(kap(2, 1, 1) - math.sqrt(2)) < 1e-12
    assert abs(kap(3, 2, 1) - math.sqrt(3)) < 1e-12


def test_P6_irreps_paths_nnz():
    want = {(1, 1): ([4, 1], [2], [4]),
            (2, 2): ([9, 9, 1], [11, 3], [83, 9]),
            (3, 3): ([16, 31, 16, 1], [34, 34, 4], [611, 611, 16])}
    for (lm, nl), (D, npth, nnz) in want.items():
        S = O.layer_irreps(lm, nl)
        P = O.layer_paths(lm, nl)
        assert [O.irreps_dim(s) for s in S] == D
        assert [len(p) for p in P] == npth
        for s in S:
            assert O.irreps_dim(s) <= 2 * (lm + 1) ** 2
        K = O.fused_cg(lm, nl, [np.ones(len(p)) for p in P])
        assert [int((np.abs(k) > 1e-12).sum()) for k in K] == nnz
        # path rule |l1-l2| <= lo <= l1+l2, p_out = p1 p2
        for L, ps in enumerate(P):
            assert ps == sorted(ps)
            for (i1, l2, io) in ps:
                l1, p1 = S[L][i1]
                lo, po = S[L + 1][io]
                assert abs(l1 - l2) <= lo <= l1 + l2 and po == p1 * (-1) ** l2
    S = O.layer_irreps(3, 3)
    assert S[1] == [(0, 1), (1, -1), (1, 1), (2, 1), (2, -1), (3, -1), (3, 1)]
    assert S[3] == [(0, 1)]
    # last layer: only m1 == m2 entries
    K = O.fused_cg(2, 2, [np.ones(11), np.ones(3)])[1]
    a, b, c = np.nonzero(np.abs(K) > 1e-12)
    assert (a == b).all() and (c == 0).all()
