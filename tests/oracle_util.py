"""Helpers for oracle tests: small systems + oracle model construction (oracle side only)."""
import dataclasses

import numpy as np

from oracle import allegro_oracle as O
from synthetic import CONFIGS, make_blob, make_system
from synthetic.configs import scaled_config


def oracle_model(hp, sigma=1.0, mu=None, seed=0, zero_alpha=False):
    fan = O.path_fan(hp.l_max, hp.n_layers)
    S = hp.n_species
    sig = list(sigma) if np.ndim(sigma) else [sigma] * S          # scalar: one value for every species; else per species
    assert len(sig) == S
    blob = make_blob(hp, fan, sig, mu if mu is not None else [0.0] * S, seed)
    m = O.OracleModel(hp, blob)
    if zero_alpha:
        m.alpha = [a * 0 for a in m.alpha]
        import torch
        m.K = [torch.from_numpy(k) for k in O.fused_cg(hp.l_max, hp.n_layers, m.alpha)]
    return m, blob


def small_system(cfg_index, n_atoms):
    cfg = scaled_config(cfg_index, n_atoms)
    pos, sp, box = make_system(cfg)
    return cfg, pos, sp, box


def cluster(n, n_species, seed, extent=5.0, dmin=0.9):
    """Non-periodic-like cluster in a huge box (no images within range)."""
    g = np.random.default_rng(seed)
    pts = []
    while len(pts) < n:
        p = g.uniform(-extent / 2, extent / 2, 3)
        if all(np.linalg.norm(p - q) > dmin for q in pts):
            pts.append(p)
    pos = np.array(pts) + 50.0
    sp = g.integers(0, n_species, n).astype(np.int32)
    return pos, sp, np.array([100.0, 100.0, 100.0])
