"""Seeded synthetic atomic systems (SURVEY.md §8(d) recipes; stand-ins for the paper's water boxes,
PAPER.md:258, and solvated biomolecules, PAPER.md:194 — the paper's structure files are not available).

No method arithmetic here: positions, species, box, velocities only.  numpy Generator(PCG64(seed)).
"""
from __future__ import annotations

import math
from typing import Dict, Tuple

import numpy as np

from .configs import Config, MASSES_AMU

_OH = 0.9572                       # A
_HOH = math.radians(104.52)
KB_EV = 8.617333262e-5             # eV/K
ACC_CONV = 9.648533212e-3          # (eV/A/amu) -> A/fs^2


def _random_rotations(rng: np.random.Generator, n: int) -> np.ndarray:
    """Uniform random rotation matrices from unit quaternions (4 normals)."""
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def _waters_at(rng: np.random.Generator, o_pos: np.ndarray) -> np.ndarray:
    """O,H,H triples: jitter O by uniform +-0.3 A, H at 0.9572 A / 104.52 deg, random orientation."""
    n = o_pos.shape[0]
    o = o_pos + rng.uniform(-0.3, 0.3, size=(n, 3))
    h1 = np.array([_OH * math.sin(_HOH / 2), 0.0, _OH * math.cos(_HOH / 2)])
    h2 = np.array([-_OH * math.sin(_HOH / 2), 0.0, _OH * math.cos(_HOH / 2)])
    R = _random_rotations(rng, n)
    out = np.empty((n, 3, 3))
    out[:, 0] = o
    out[:, 1] = o + R @ h1
    out[:, 2] = o + R @ h2
    return out.reshape(3 * n, 3)


def _grid_sites(M: int, spacing: float) -> np.ndarray:
    g = (np.arange(M) + 0.5) * spacing
    return np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)


def _min_dist_points(rng, n, sampler, dmin, box=None):
    """Sequential rejection: accept a proposal iff farther than dmin from every accepted point
    (periodic if `box` given).  Hash grid of cell size dmin."""
    cells: Dict[Tuple[int, int, int], list] = {}
    pts = np.empty((n, 3))
    k = 0
    ncell = None if box is None else max(1, int(box / dmin))
    csz = dmin if box is None else box / ncell
    d2min = dmin * dmin
    while k < n:
        prop = sampler(rng, max(1024, (n - k) * 2))
        for p in prop:
            c = (int(p[0] // csz), int(p[1] // csz), int(p[2] // csz))
            ok = True
            for dx in (-1, 0, 1):
                for dy in (-1, 0, 1):
                    for dz in (-1, 0, 1):
                        cc = (c[0] + dx, c[1] + dy, c[2] + dz)
                        if ncell is not None:
                            cc = (cc[0] % ncell, cc[1] % ncell, cc[2] % ncell)
                        lst = cells.get(cc)
                        if not lst:
                            continue
                        for q in lst:
                            d = pts[q] - p
                            if box is not None:
                                d -= box * np.round(d / box)
                            if d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < d2min:
                                ok = False
                                break
                        if not ok:
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if ok:
                pts[k] = p
                cells.setdefault(c if ncell is None else (c[0] % ncell, c[1] % ncell, c[2] % ncell), []).append(k)
                k += 1
                if k == n:
                    break
    return pts


def make_system(cfg: Config):
    """Returns (pos f64[N,3], species i32[N], box f64[3])."""
    rng = np.random.Generator(np.random.PCG64(cfg.pos_seed))
    N = cfg.n_atoms
    names = cfg.species_names
    if cfg.kind == "water":
        assert N % 3 == 0
        nw = N // 3
        spacing = (3.0 / cfg.density) ** (1.0 / 3.0)
        M = int(math.ceil(nw ** (1.0 / 3.0) - 1e-9))
        sites = _grid_sites(M, spacing)
        if nw < M ** 3:
            sites = sites[np.sort(rng.permutation(M ** 3)[:nw])]
        pos = _waters_at(rng, sites)
        sp = np.tile(np.array([names.index("O"), names.index("H"), names.index("H")], dtype=np.int32), nw)
        L = M * spacing
        return pos, sp, np.array([L, L, L])
    if cfg.kind == "solvated":
        spacing = (3.0 / cfg.density) ** (1.0 / 3.0)
        nw = int(round(0.7 * N)) // 3
        nb = N - 3 * nw
        rho_b = 0.12
        Rb = (3.0 * nb / (4.0 * math.pi * rho_b)) ** (1.0 / 3.0)
        M = 2
        while True:
            L = M * spacing
            sites = _grid_sites(M, spacing)
            far = np.linalg.norm(sites - L / 2, axis=1) > Rb + 1.5
            if far.sum() >= nw and L / 2 > Rb + 1.5:
                break
            M += 1
        elig = np.nonzero(far)[0]
        chosen = np.sort(elig[rng.permutation(elig.size)[:nw]])
        wpos = _waters_at(rng, sites[chosen])
        wsp = np.tile(np.array([names.index("O"), names.index("H"), names.index("H")], dtype=np.int32), nw)

        def sphere_sampler(r, m):
            v = r.uniform(-Rb, Rb, size=(int(m * 2.2) + 16, 3))
            v = v[np.einsum("ij,ij->i", v, v) <= Rb * Rb]
            return v + L / 2

        bpos = _min_dist_points(rng, nb, sphere_sampler, 1.0)
        probs = {"H": 0.50, "C": 0.32, "N": 0.09, "O": 0.08, "S": 0.01}
        bsp = rng.choice(len(names), size=nb, p=[probs[s] for s in names]).astype(np.int32)
        pos = np.concatenate([bpos, wpos], axis=0)
        sp = np.concatenate([bsp, wsp])
        return pos, sp, np.array([L, L, L])
    if cfg.kind == "random4":
        L = (N / cfg.density) ** (1.0 / 3.0)

        def box_sampler(r, m):
            return r.uniform(0.0, L, size=(m, 3))

        pos = _min_dist_points(rng, N, box_sampler, 1.0, box=L)
        sp = rng.integers(0, len(names), size=N).astype(np.int32)
        return pos, sp, np.array([L, L, L])
    raise ValueError(cfg.kind)


def masses_for(cfg: Config) -> np.ndarray:
    return np.array([MASSES_AMU[s] for s in cfg.species_names])


def maxwell_boltzmann(cfg: Config, species: np.ndarray) -> np.ndarray:
    """Velocities (A/fs) ~ N(0, kB T / m) per component, centre-of-mass velocity removed, no rescale."""
    rng = np.random.Generator(np.random.PCG64(cfg.vel_seed))
    m = masses_for(cfg)[species]
    sd = np.sqrt(KB_EV * cfg.temperature / m * ACC_CONV)
    v = rng.standard_normal((species.shape[0], 3)) * sd[:, None]
    v -= (m[:, None] * v).sum(0) / m.sum()
    return v
