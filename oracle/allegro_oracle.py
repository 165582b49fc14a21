"""fp64 CPU oracle of the Allegro per-edge energy+force path (arXiv 2304.10061).

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` leg may import this.  It shares no code with the CUDA path
(`paper_2304_10061_b200/`), and neither imports the other.  Plain numpy / PyTorch-CPU float64, written
step by step in the paper's order so it can be checked against the paper by eye.  Readings of points
the paper leaves open are those of SURVEY.md §8(c) (S1..S10), repeated in DESIGN.md.

Forces are *defined* as F_i = -dE/dr_i ("force-only MSE loss", MD use PAPER.md:50) and are
obtained here by reverse-mode differentiation (torch.autograd) of the fp64 energy written below — the
CUDA path carries a hand-derived analytic backward instead, so the two share no derivative code.  The
autograd result is itself pinned by central finite differences (tests/test_oracle_model.py, pin P11).

Pins (tests/test_oracle_*.py, `-m "not gpu"`): closed-form Y_lm (P1), envelope/Bessel identities (P2,
P3), CG closed forms / orthonormality / equivariance / self-coupling (P4, P5, P5b), path counts (P6),
bilinearity Eq. (2) (P7), O(3)/translation/permutation symmetry and sum F = 0 (P8), strict locality
(P9), continuity at r_c (P10), finite differences (P11), parameter count 7.85 M (P12), pair-potential
special case (P13), neighbor lists vs brute force and symmetry (P15), NVE closed form (P16).
Absolute E, F for a given blob: PARITY UNPINNED by the paper (it prints no worked example); pinned
only jointly by P7-P13.
"""
from __future__ import annotations

import math
from fractions import Fraction
from typing import List, Sequence, Tuple

import numpy as np
import torch

F64 = torch.float64


def _zeros(*shape):
    return torch.zeros(*shape, dtype=F64)

ACC_CONV = 9.648533212e-3   # (eV/A/amu) -> A/fs^2          (S10)
KB_EV = 8.617333262e-5      # eV/K


# ----------------------------------------------------------------------------------------------
# S2. radial functions  ("8 Bessel functions and a polynomial cutoff envelope as
#     specified in [9]"; formulas are the SURVEY §8(c) S2 reading)
# ----------------------------------------------------------------------------------------------
def poly_cutoff(x: torch.Tensor, p: int) -> torch.Tensor:
    """u(x) = 1 - (p+1)(p+2)/2 x^p + p(p+2) x^(p+1) - p(p+1)/2 x^(p+2) for x < 1, else 0."""
    u = 1.0 - ((p + 1.0) * (p + 2.0) / 2.0) * x ** p + p * (p + 2.0) * x ** (p + 1) \
        - (p * (p + 1.0) / 2.0) * x ** (p + 2)
    return torch.where(x < 1.0, u, torch.zeros_like(u))


def bessel_basis(r: torch.Tensor, r_cut, n_bessel: int, freq=None) -> torch.Tensor:
    """b_n(r) = sqrt(2/r_c) sin(w_n r) / r, n = 1..N_B, with w_n = n pi / r_c unless `freq` is given.  Returns [..., N_B].
    r_cut: a float, or a tensor of the shape of r (one cutoff per edge: ordered species-pair cutoffs).
    freq: optional tensor [..., N_B] of angular frequencies in 1/Angstrom, one row per edge (the "trainable
    per-ordered-species-pair radial basis" of PAPER.md:222: the trained values of w_n for the edge's pair)."""
    n = torch.arange(1, n_bessel + 1, dtype=torch.float64)
    rc = torch.as_tensor(r_cut, dtype=torch.float64)
    if rc.ndim:
        rc = rc[..., None]
    w = n * math.pi / rc if freq is None else freq
    return torch.sqrt(2.0 / rc) * torch.sin(w * r[..., None]) / r[..., None]


# ----------------------------------------------------------------------------------------------
# NEXT-4. ZBL pair repulsion ("We also add a repulsive Ziegler-Biersack-Littmark (ZBL) term to the
#     potential").  The paper gives no formula; reading: the universal screened-Coulomb form
#         phi_ij(r) = k_e Z_i Z_j / r * Phi(r / a_ij) * u(r / r_c),   a_ij = 0.46850 / (Z_i^0.23 + Z_j^0.23) Angstrom,
#         Phi(x) = 0.18175 e^{-3.19980 x} + 0.50986 e^{-0.94229 x} + 0.28022 e^{-0.40290 x} + 0.02817 e^{-0.20162 x},
#     times the model's own polynomial envelope u at the FLAT cutoff r_c (a pair potential must be symmetric in
#     (i, j), which the ordered pair cutoffs are not), E_ZBL = 1/2 sum over ordered pairs, split evenly between the
#     two atoms, not scaled by sigma_Z.
# ----------------------------------------------------------------------------------------------
KE_EV_A = 14.399645478425668   # e^2 / (4 pi eps0) in eV * Angstrom
ZBL_C = (0.18175, 0.50986, 0.28022, 0.02817)
ZBL_D = (3.19980, 0.94229, 0.40290, 0.20162)


def zbl_pair_energy(r: torch.Tensor, zi: torch.Tensor, zj: torch.Tensor, r_cut: float, p: int) -> torch.Tensor:
    """phi_ij(r) of the reading above, elementwise; zi, zj are atomic numbers (float64)."""
    a = 0.46850 / (zi ** 0.23 + zj ** 0.23)
    x = r / a
    Phi = sum(c * torch.exp(-dd * x) for c, dd in zip(ZBL_C, ZBL_D))
    return KE_EV_A * zi * zj / r * Phi * poly_cutoff(r / r_cut, p)


# ----------------------------------------------------------------------------------------------
# S4. real spherical harmonics, component normalisation (sum_m Y_lm^2 = 2l+1), m = -l..l,
#     no Condon-Shortley sign in the real forms.  Generic l by the associated-Legendre recursion,
#     written in Cartesian form so it is smooth at the poles.
# ----------------------------------------------------------------------------------------------
def real_sph_harm(rhat: torch.Tensor, l_max: int) -> torch.Tensor:
    """rhat [..., 3] unit vectors -> Y [..., (l_max+1)^2], index l*l + (m + l)."""
    x, y, z = rhat[..., 0], rhat[..., 1], rhat[..., 2]
    # A_m + i B_m = (x + i y)^m  ( = sin^m(theta) e^{i m phi} )
    A = [torch.ones_like(x)]
    B = [torch.zeros_like(x)]
    for m in range(1, l_max + 1):
        A.append(x * A[m - 1] - y * B[m - 1])
        B.append(x * B[m - 1] + y * A[m - 1])
    # Q_l^m(z) = P_l^m(z) / sin^m(theta) without Condon-Shortley phase
    Q = {}
    for m in range(0, l_max + 1):
        dfact = 1.0
        for k in range(1, 2 * m, 2):
            dfact *= k                                    # (2m-1)!!
        Q[(m, m)] = dfact * torch.ones_like(z)
        if m + 1 <= l_max:
            Q[(m + 1, m)] = (2 * m + 1) * z * Q[(m, m)]
        for l in range(m + 2, l_max + 1):
            Q[(l, m)] = ((2 * l - 1) * z * Q[(l - 1, m)] - (l + m - 1) * Q[(l - 2, m)]) / (l - m)
    out = []
    for l in range(l_max + 1):
        row = [None] * (2 * l + 1)
        for m in range(0, l + 1):
            N = math.sqrt((2 * l + 1) * math.factorial(l - m) / math.factorial(l + m))
            if m == 0:
                row[l] = N * Q[(l, 0)]
            else:
                row[l + m] = math.sqrt(2.0) * N * Q[(l, m)] * A[m]
                row[l - m] = math.sqrt(2.0) * N * Q[(l, m)] * B[m]
        out.extend(row)
    return torch.stack(out, dim=-1)


# ----------------------------------------------------------------------------------------------
# S5. real Clebsch-Gordan blocks
# ----------------------------------------------------------------------------------------------
def _f(n: int) -> int:
    return math.factorial(n)


def su2_cg(j1: int, m1: int, j2: int, m2: int, j3: int, m3: int) -> float:
    """<j1 m1 j2 m2 | j3 m3>, Condon-Shortley convention, Racah's formula (exact rationals inside
    the square root)."""
    if m1 + m2 != m3 or not (abs(j1 - j2) <= j3 <= j1 + j2):
        return 0.0
    if abs(m1) > j1 or abs(m2) > j2 or abs(m3) > j3:
        return 0.0
    pref = Fraction((2 * j3 + 1) * _f(j3 + j1 - j2) * _f(j3 - j1 + j2) * _f(j1 + j2 - j3), _f(j1 + j2 + j3 + 1))
    pref *= _f(j3 + m3) * _f(j3 - m3) * _f(j1 - m1) * _f(j1 + m1) * _f(j2 - m2) * _f(j2 + m2)
    s = Fraction(0)
    for k in range(0, j1 + j2 - j3 + 1):
        dens = [k, j1 + j2 - j3 - k, j1 - m1 - k, j2 + m2 - k, j3 - j2 + m1 + k, j3 - j1 - m2 + k]
        if min(dens) < 0:
            continue
        den = 1
        for q in dens:
            den *= _f(q)
        s += Fraction((-1) ** k, den)
    return float(s) * math.sqrt(float(pref))


def real_basis_U(l: int) -> np.ndarray:
    """Y^real = U_l Y^complex; rows a = m_real + l, columns m_complex + l."""
    U = np.zeros((2 * l + 1, 2 * l + 1), dtype=np.complex128)
    s2 = 1.0 / math.sqrt(2.0)
    U[l, l] = 1.0
    for m in range(1, l + 1):
        U[l + m, l + m] = (-1) ** m * s2          # m > 0 : ((-1)^m e_m + e_-m)/sqrt2
        U[l + m, l - m] = s2
        U[l - m, l - m] = 1j * s2                 # m < 0 : i (e_-|m| - (-1)^m e_|m|)/sqrt2
        U[l - m, l + m] = -1j * (-1) ** m * s2
    return U


def real_cg(l1: int, l2: int, lo: int) -> np.ndarray:
    """C[a,b,c], orthonormal (sum_ab C[a,b,c] C[a,b,c'] = delta), real; sign fixed so that the first
    entry with |value| > 1e-12 in (a,b,c) lexicographic order is positive."""
    cg = np.zeros((2 * l1 + 1, 2 * l2 + 1, 2 * lo + 1))
    for m1 in range(-l1, l1 + 1):
        for m2 in range(-l2, l2 + 1):
            mo = m1 + m2
            if abs(mo) <= lo:
                cg[m1 + l1, m2 + l2, mo + lo] = su2_cg(l1, m1, l2, m2, lo, mo)
    U1, U2, Uo = real_basis_U(l1), real_basis_U(l2), real_basis_U(lo)
    C = np.einsum("am,bn,co,mno->abc", U1, U2, np.conj(Uo), cg.astype(np.complex128))
    if (l1 + l2 + lo) % 2 == 0:
        assert np.abs(C.imag).max() < 1e-12
        C = C.real.copy()
    else:
        assert np.abs(C.real).max() < 1e-12
        C = C.imag.copy()
    flat = C.reshape(-1)
    nz = np.nonzero(np.abs(flat) > 1e-12)[0]
    if nz.size and flat[nz[0]] < 0:
        C = -C
    C[np.abs(C) < 1e-14] = 0.0
    return C


# ----------------------------------------------------------------------------------------------
# S6. irreps per layer, paths, fused tensor
# ----------------------------------------------------------------------------------------------
Irrep = Tuple[int, int]   # (l, p)


def _sort_irreps(s) -> List[Irrep]:
    # l ascending; for equal l the natural parity (-1)^l first
    return sorted(set(s), key=lambda ir: (ir[0], 0 if ir[1] == (-1) ** ir[0] else 1))


def layer_irreps(l_max: int, n_layers: int) -> List[List[Irrep]]:
    """S_0..S_NL after pruning paths that can never reach the final scalars."""
    env = [(l, (-1) ** l) for l in range(l_max + 1)]
    O = [list(env)]
    for _ in range(n_layers):
        nxt = set()
        for (l1, p1) in O[-1]:
            for (l2, p2) in env:
                for lo in range(abs(l1 - l2), min(l1 + l2, l_max) + 1):
                    nxt.add((lo, p1 * p2))
        O.append(_sort_irreps(nxt))
    S = [None] * (n_layers + 1)
    S[n_layers] = [(0, 1)]
    for L in range(n_layers - 1, -1, -1):
        keep = []
        for (l1, p1) in O[L]:
            ok = False
            for (l2, p2) in env:
                for (lo, po) in S[L + 1]:
                    if abs(l1 - l2) <= lo <= l1 + l2 and po == p1 * p2:
                        ok = True
            if ok:
                keep.append((l1, p1))
        S[L] = _sort_irreps(keep)
    return S


def layer_paths(l_max: int, n_layers: int) -> List[List[Tuple[int, int, int]]]:
    """paths[L-1] = [(index of irrep1 in S_{L-1}, l2, index of irrep_o in S_L)], canonical order."""
    S = layer_irreps(l_max, n_layers)
    out = []
    for L in range(1, n_layers + 1):
        ps = []
        for i1, (l1, p1) in enumerate(S[L - 1]):
            for l2 in range(l_max + 1):
                p2 = (-1) ** l2
                for io, (lo, po) in enumerate(S[L]):
                    if abs(l1 - l2) <= lo <= l1 + l2 and po == p1 * p2:
                        ps.append((i1, l2, io))
        out.append(ps)
    return out


def path_fan(l_max: int, n_layers: int) -> List[List[int]]:
    """For each path, the number of paths of its layer sharing its output irrep (alpha scale)."""
    out = []
    for ps in layer_paths(l_max, n_layers):
        cnt = {}
        for (_, _, io) in ps:
            cnt[io] = cnt.get(io, 0) + 1
        out.append([cnt[io] for (_, _, io) in ps])
    return out


def irreps_dim(irreps: Sequence[Irrep]) -> int:
    return sum(2 * l + 1 for l, _ in irreps)


def irreps_offsets(irreps: Sequence[Irrep]) -> List[int]:
    off, o = [], 0
    for l, _ in irreps:
        off.append(o)
        o += 2 * l + 1
    return off


def fused_cg(l_max: int, n_layers: int, alphas: Sequence[np.ndarray]) -> List[np.ndarray]:
    """K^L[a,b,c] = sum_paths alpha_path * C_path placed at the path's blocks (Fig. 3).
    a over S_{L-1} layout, b over the full environment layout (l_max+1)^2, c over S_L layout."""
    S = layer_irreps(l_max, n_layers)
    paths = layer_paths(l_max, n_layers)
    Ks = []
    for L in range(1, n_layers + 1):
        off1, offo = irreps_offsets(S[L - 1]), irreps_offsets(S[L])
        K = np.zeros((irreps_dim(S[L - 1]), (l_max + 1) ** 2, irreps_dim(S[L])))
        for alpha, (i1, l2, io) in zip(alphas[L - 1], paths[L - 1]):
            l1, lo = S[L - 1][i1][0], S[L][io][0]
            C = real_cg(l1, l2, lo)
            K[off1[i1]:off1[i1] + 2 * l1 + 1, l2 * l2:l2 * l2 + 2 * l2 + 1, offo[io]:offo[io] + 2 * lo + 1] \
                += float(alpha) * C
        Ks.append(K)
    return Ks


# ----------------------------------------------------------------------------------------------
# S1. neighbor list
# ----------------------------------------------------------------------------------------------
def _canonical_accept(pos, box, i, j, s, cutoff):
    # dx = (x_j - x_i) + s_x L_x ; d2 = (dx*dx + dy*dy) + dz*dz   in fp64, this association, no FMA
    dx = (pos[j, 0] - pos[i, 0]) + s[:, 0] * box[0]
    dy = (pos[j, 1] - pos[i, 1]) + s[:, 1] * box[1]
    dz = (pos[j, 2] - pos[i, 2]) + s[:, 2] * box[2]
    d2 = (dx * dx + dy * dy) + dz * dz
    return d2 < cutoff * cutoff


def _sorted_edges(i, j, s):
    order = np.lexsort((s[:, 2], s[:, 1], s[:, 0], j, i))
    return i[order].astype(np.int64), j[order].astype(np.int64), s[order].astype(np.int64)


def neighbor_list_brute(pos: np.ndarray, box: np.ndarray, cutoff: float):
    """All (i, j, s) with (i != j or s != 0) and d2 < cutoff^2, sorted by (i, j, sx, sy, sz).
    Brute force over all i, j and s in [-m, m]^3."""
    pos = np.asarray(pos, dtype=np.float64)
    box = np.asarray(box, dtype=np.float64)
    N = pos.shape[0]
    off = int(np.ceil(np.abs(np.floor(pos / box)).max())) + 1 if N else 0
    m = [int(math.ceil(cutoff / box[k])) + off for k in range(3)]
    ii, jj = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    ii, jj = ii.reshape(-1), jj.reshape(-1)
    I, J, Sh = [], [], []
    for sx in range(-m[0], m[0] + 1):
        for sy in range(-m[1], m[1] + 1):
            for sz in range(-m[2], m[2] + 1):
                s = np.broadcast_to(np.array([sx, sy, sz], dtype=np.float64), (ii.size, 3))
                ok = _canonical_accept(pos, box, ii, jj, s, cutoff)
                if sx == 0 and sy == 0 and sz == 0:
                    ok &= ii != jj
                if ok.any():
                    I.append(ii[ok]); J.append(jj[ok])
                    Sh.append(np.broadcast_to(np.array([sx, sy, sz]), (int(ok.sum()), 3)).copy())
    if not I:
        z = np.zeros(0, dtype=np.int64)
        return z, z, np.zeros((0, 3), dtype=np.int64)
    return _sorted_edges(np.concatenate(I), np.concatenate(J), np.concatenate(Sh))


def neighbor_list(pos: np.ndarray, box: np.ndarray, cutoff: float):
    """Same set as `neighbor_list_brute`.  For boxes wider than 2*cutoff candidates come from a
    periodic k-d tree (scipy; candidate generation only) and the accept test is the canonical one."""
    pos = np.asarray(pos, dtype=np.float64)
    box = np.asarray(box, dtype=np.float64)
    if pos.shape[0] <= 64 or box.min() <= 2.0 * cutoff * (1 + 1e-6) + 1e-6:
        return neighbor_list_brute(pos, box, cutoff)
    from scipy.spatial import cKDTree
    q = np.floor(pos / box)
    w = pos - q * box
    w = np.where(w >= box, w - box, w)
    w = np.where(w < 0, w + box, w)
    q = np.rint((pos - w) / box)
    tree = cKDTree(w, boxsize=box)
    pairs = tree.query_pairs(cutoff * (1 + 1e-9) + 1e-9, output_type="ndarray")
    i = np.concatenate([pairs[:, 0], pairs[:, 1]])
    j = np.concatenate([pairs[:, 1], pairs[:, 0]])
    t = -np.rint((w[j] - w[i]) / box)              # nearest image in the wrapped frame
    s = t - q[j] + q[i]                            # shift relative to the positions as given
    ok = _canonical_accept(pos, box, i, j, s, cutoff)
    return _sorted_edges(i[ok], j[ok], s[ok])


# ----------------------------------------------------------------------------------------------
# model
# ----------------------------------------------------------------------------------------------
def silu(z: torch.Tensor) -> torch.Tensor:
    return z / (1.0 + torch.exp(-z))


class OracleModel:
    """Weights parsed from the flat blob (SURVEY §8(b) blob layout), promoted fp32 -> fp64."""

    def __init__(self, hp, blob: bytes):
        self.hp = hp
        S, NB, d, n, lmax, NL = hp.n_species, hp.n_bessel, hp.d, hp.n_tensor, hp.l_max, hp.n_layers
        assert hp.latent_dims[-1] == d
        self.irreps = layer_irreps(lmax, NL)
        self.paths = layer_paths(lmax, NL)
        nA = n * (lmax + 1)
        nfl = 0
        f32 = np.frombuffer(blob, dtype="<f4", count=(len(blob) - 16 * S) // 4)

        def take(fi, fo):
            nonlocal nfl
            w = f32[nfl:nfl + fi * fo].astype(np.float64).reshape(fi, fo)
            nfl += fi * fo
            return torch.from_numpy(w.copy())

        self.twobody = []
        fi = 2 * S + NB
        for wdt in hp.twobody_dims:
            self.twobody.append(take(fi, wdt)); fi = wdt
        self.A = [take(d, nA)]
        self.alpha, self.latent = [], []
        for L in range(NL):
            self.A.append(take(d, nA))
            npth = len(self.paths[L])
            self.alpha.append(f32[nfl:nfl + npth].astype(np.float64).copy()); nfl += npth
            lat, fi = [], d + n
            for wdt in hp.latent_dims:
                lat.append(take(fi, wdt)); fi = wdt
            self.latent.append(lat)
        self.edge, fi = [], d
        for wdt in list(hp.edge_dims) + [1]:
            self.edge.append(take(fi, wdt)); fi = wdt
        tail = nfl * 4
        tail += (-tail) % 8
        assert len(blob) == tail + 16 * S, (len(blob), tail + 16 * S)
        sm = np.frombuffer(blob, dtype="<f8", offset=tail, count=2 * S)
        self.sigma = torch.from_numpy(sm[:S].copy())
        self.mu = torch.from_numpy(sm[S:].copy())
        self.n_weights = nfl
        self.K = [torch.from_numpy(k) for k in fused_cg(lmax, NL, self.alpha)]
        # index maps: layout position -> l, for the environment (all l <= l_max, natural parity)
        self.env_l = torch.tensor([l for l in range(lmax + 1) for _ in range(2 * l + 1)])
        # V^0 layout = S_0 irreps (each natural): position -> l and -> position in Y
        self.v0_l = torch.tensor([l for (l, _) in self.irreps[0] for _ in range(2 * l + 1)])
        self.v0_y = torch.tensor([l * l + k for (l, _) in self.irreps[0] for k in range(2 * l + 1)])

    # -- S2..S8 ---------------------------------------------------------------------------------
    def edge_energies(self, pos: torch.Tensor, species: torch.Tensor, box: torch.Tensor,
                      ei: torch.Tensor, ej: torch.Tensor, es: torch.Tensor,
                      return_parts: bool = False):
        """Per-edge energies E_e for the given edge list (every edge of every centre present must
        be listed: the environment sum runs over the listed edges of each centre).  Edges with
        r >= r_c contribute exactly zero."""
        hp = self.hp
        n, lmax, NL, d = hp.n_tensor, hp.l_max, hp.n_layers, hp.d
        rvec = pos[ej] - pos[ei] + es.to(torch.float64) * box                  # S1 convention
        r = torch.sqrt((rvec * rvec).sum(-1))
        # cutoff of each ordered pair (i centre, j neighbour): r_c, or r_c[Z_i][Z_j] with ordered species-pair
        # cutoffs (NEXT-1 reading in DESIGN.md: the pair's own cutoff enters the edge
        # criterion, the envelope argument x = r / r_c[Z_i][Z_j] and the Bessel functions)
        pair = getattr(hp, "r_cut_pair", None)
        if pair is None:
            rc = torch.full_like(r, hp.r_cut)
        else:
            rc = torch.tensor(pair, dtype=torch.float64)[species[ei], species[ej]]
        keep = r < rc                                                          # skin lists (S9 last line)
        full_E = r.shape[0]
        idx = torch.nonzero(keep).reshape(-1)
        ei, ej, rvec, r, rc = ei[idx], ej[idx], rvec[idx], r[idx], rc[idx]
        E = r.shape[0]
        cent, ec = torch.unique(ei, return_inverse=True)      # local centre numbering for the env sum
        n_cent = cent.shape[0]
        x = r / rc
        u = poly_cutoff(x, hp.poly_p)                                           # S2
        fq = getattr(hp, "bessel_freq_pair", None)                              # [S][S][N_B] or None
        fq = None if fq is None else torch.tensor(fq, dtype=torch.float64)[species[ei], species[ej]]
        B = bessel_basis(r, rc, hp.n_bessel, fq) * u[:, None]
        onehot = torch.eye(hp.n_species, dtype=torch.float64)
        h = torch.cat([onehot[species[ei]], onehot[species[ej]], B], dim=1)     # S3
        for W in self.twobody:
            h = silu(h @ W)
        xl = u[:, None] * h                                                     # x^0
        Y = real_sph_harm(rvec / r[:, None], lmax)                              # S4
        w0 = (xl @ self.A[0]).reshape(E, n, lmax + 1)
        V = w0[:, :, self.v0_l] * Y[:, None, self.v0_y]                         # V^0
        c_env = 1.0 / math.sqrt(hp.avg_num_neighbors)
        parts = {"x": [xl], "V": [V], "Gamma": [], "Y": Y, "u": u, "B": B, "idx": idx, "cent": cent}
        for L in range(1, NL + 1):                                              # S7
            om = (xl @ self.A[L]).reshape(E, n, lmax + 1)
            wy = om[:, :, self.env_l] * Y[:, None, :]
            Gam = c_env * _zeros(n_cent, n, (lmax + 1) ** 2).index_add(0, ec, wy)   # Eq. (2) line 2
            T = torch.einsum("abc,ena,enb->enc", self.K[L - 1], V, Gam[ec])
            s = T[:, :, 0]                                                      # the (0,+1) block
            m = torch.cat([xl, s], dim=1)
            for W in self.latent[L - 1]:
                m = silu(m @ W)
            a = hp.resid_alpha[L - 1]
            c_old, c_new = 1.0 / math.sqrt(1 + a * a), a / math.sqrt(1 + a * a)
            xl = c_old * xl + c_new * u[:, None] * m
            V = T
            parts["x"].append(xl); parts["V"].append(V); parts["Gamma"].append(Gam)
        Ee = xl                                                                 # S8
        for W in self.edge:
            Ee = Ee @ W
        out = _zeros(full_E).index_add(0, idx, Ee[:, 0])
        if return_parts:
            return out, parts
        return out

    def atom_energies(self, pos, species, box, ei, ej, es, centers=None):
        """E-hat_i = sigma_{Z_i} sum_j E_ij + mu_{Z_i}.  `centers`: optional
        boolean mask [N]; only those atoms' energies are summed in the returned total."""
        N = pos.shape[0]
        Ee = self.edge_energies(pos, species, box, ei, ej, es)
        Ei = _zeros(N).index_add(0, ei, Ee)
        Ehat = self.sigma[species] * Ei + self.mu[species]
        zn = getattr(self.hp, "zbl_Z", None)
        if zn is not None:                                                     # NEXT-4: ZBL, 1/2 phi_ij to the centre
            zn = torch.tensor(zn, dtype=torch.float64)
            rvec = pos[ej] - pos[ei] + es.to(torch.float64) * box
            r = torch.sqrt((rvec * rvec).sum(-1))
            phi = zbl_pair_energy(r, zn[species[ei]], zn[species[ej]], self.hp.r_cut, self.hp.poly_p)
            Ehat = Ehat + _zeros(N).index_add(0, ei, 0.5 * phi)
        if centers is not None:
            Ehat = Ehat * centers
        return Ehat


def energy_forces(model: OracleModel, pos: np.ndarray, species: np.ndarray, box: np.ndarray,
                  nbr, chunk_edges: int = 150_000, centers: np.ndarray | None = None):
    """E (float), E-hat_i f64[N], F f64[N,3] = -dE/dr.  Centres are processed in contiguous chunks
    (strict locality: E-hat_i needs only the edges of centre i) to bound autograd memory.
    `centers`: optional index array — only those centres are evaluated (sub-system parity, SURVEY
    §8(d)); E-hat of the others is returned as 0 and F is -d(sum_{c in centers} E-hat_c)/dr."""
    ei_np, ej_np, es_np = nbr
    N = pos.shape[0]
    sp = torch.from_numpy(np.asarray(species, dtype=np.int64))
    bx = torch.from_numpy(np.asarray(box, dtype=np.float64))
    p = torch.from_numpy(np.asarray(pos, dtype=np.float64).copy()).requires_grad_(True)
    row_ptr = np.searchsorted(ei_np, np.arange(N + 1))
    if centers is None:
        todo = np.arange(N)
    else:
        todo = np.sort(np.asarray(centers))
    Eatom = np.zeros(N)
    F = np.zeros((N, 3))
    k = 0
    while k < todo.size:
        k1, ne = k, 0
        while k1 < todo.size and (ne == 0 or ne + row_ptr[todo[k1] + 1] - row_ptr[todo[k1]] <= chunk_edges):
            ne += row_ptr[todo[k1] + 1] - row_ptr[todo[k1]]
            k1 += 1
        cs = todo[k:k1]
        sel = np.concatenate([np.arange(row_ptr[c], row_ptr[c + 1]) for c in cs]) if cs.size else np.zeros(0, int)
        mask = _zeros(N)
        mask[torch.from_numpy(cs)] = 1.0
        Ehat = model.atom_energies(p, sp, bx, torch.from_numpy(ei_np[sel]), torch.from_numpy(ej_np[sel]),
                                   torch.from_numpy(es_np[sel]), centers=mask)
        Etot = Ehat.sum()
        g, = torch.autograd.grad(Etot, p)
        F -= g.numpy()
        Eatom += Ehat.detach().numpy()
        k = k1
    return float(Eatom.sum()), Eatom, F


# ----------------------------------------------------------------------------------------------
# S10. velocity-Verlet NVE step
# ----------------------------------------------------------------------------------------------
def nve_half_kick(vel, force, mass_per_atom, dt_fs):
    return vel + (0.5 * dt_fs) * (force / mass_per_atom[:, None]) * ACC_CONV


def nve_drift(pos, vel, dt_fs):
    return pos + dt_fs * vel


def kinetic_energy(vel, mass_per_atom):
    return float((0.5 * mass_per_atom[:, None] * vel * vel).sum() / ACC_CONV)


def nve_step(force_fn, pos, vel, force, mass_per_atom, dt_fs):
    """v += dt/2 a; r += dt v; F = force_fn(r); v += dt/2 a.  Positions are never wrapped.
    Returns pos, vel, force, e_pot."""
    vel = nve_half_kick(vel, force, mass_per_atom, dt_fs)
    pos = nve_drift(pos, vel, dt_fs)
    e_pot, force = force_fn(pos)
    vel = nve_half_kick(vel, force, mass_per_atom, dt_fs)
    return pos, vel, force, e_pot


# ----------------------------------------------------------------------------------------------
# NEXT-4. thermostatted MD ("stable temperature around thermostat setting of 300K"; the paper does not
#     name the thermostat).  Reading: one Nose-Hoover thermostat variable xi (1/fs) of relaxation time
#     tau, Q = g k_B T0 tau^2, g = 3N degrees of freedom, integrated by the symmetric Trotter splitting
#         [thermostat dt/2] [velocity-Verlet NVE step dt] [thermostat dt/2],
#     thermostat half step:  xi += dt/4 * G(K);  v *= s = exp(-xi dt/2) (K *= s^2);  xi += dt/4 * G(K),
#     G(K) = (2 K - g k_B T0) / Q.   Conserved: K + E_pot + Q xi^2 / 2 + g k_B T0 eta,  d(eta)/dt = xi.
# ----------------------------------------------------------------------------------------------
def nh_half_step(vel, xi, eta, e_kin, n_dof, t0_K, tau_fs, dt_fs):
    """One thermostat half step.  Returns vel, xi, eta, e_kin (all after the half step)."""
    gkt = n_dof * KB_EV * t0_K
    Q = gkt * tau_fs * tau_fs
    xi = xi + 0.25 * dt_fs * (2.0 * e_kin - gkt) / Q
    s = math.exp(-xi * 0.5 * dt_fs)
    eta = eta + xi * 0.5 * dt_fs
    vel = vel * s
    e_kin = e_kin * s * s
    xi = xi + 0.25 * dt_fs * (2.0 * e_kin - gkt) / Q
    return vel, xi, eta, e_kin


def nvt_step(force_fn, pos, vel, force, mass_per_atom, dt_fs, xi, eta, t0_K, tau_fs):
    """Nose-Hoover NVT step of the reading above.  Returns pos, vel, force, e_pot, e_kin, xi, eta."""
    g = 3 * pos.shape[0]
    vel, xi, eta, _ = nh_half_step(vel, xi, eta, kinetic_energy(vel, mass_per_atom), g, t0_K, tau_fs, dt_fs)
    pos, vel, force, e_pot = nve_step(force_fn, pos, vel, force, mass_per_atom, dt_fs)
    vel, xi, eta, e_kin = nh_half_step(vel, xi, eta, kinetic_energy(vel, mass_per_atom), g, t0_K, tau_fs, dt_fs)
    return pos, vel, force, e_pot, e_kin, xi, eta


def nh_conserved(e_pot, e_kin, xi, eta, n_dof, t0_K, tau_fs):
    gkt = n_dof * KB_EV * t0_K
    return e_pot + e_kin + 0.5 * gkt * tau_fs * tau_fs * xi * xi + gkt * eta
