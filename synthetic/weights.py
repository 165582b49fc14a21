"""Seeded flat weight blob (SURVEY.md §8(b) "Blob layout"; the weights stand in for the paper's trained
SPICE model, which is not available).

Layout, little-endian fp32 unless noted, dense layers stored [fan_in][fan_out] row-major:
  two-body layers (fan_in0 = 2*S + n_bessel)
  A^0                                  [d][n_tensor*(l_max+1)], column = n*(l_max+1)+l
  for L = 1..n_layers:  A^L, alpha^L[n_paths_L], latent layers (fan_in0 = d + n_tensor)
  edge layers (d -> edge_dims... -> 1)
  zero padding to a multiple of 8 bytes
  sigma[S], mu[S]                      fp64

The number of tensor-product paths per layer (and, for the alpha scale, how many paths share each
path's output irrep) is method logic, so it is passed IN by the caller (from `oracle/` in oracle
tests, from the C library's `allegro_path_info` on the product side) — this file draws numbers only.
"""
from __future__ import annotations

from typing import List, Sequence

import numpy as np

from .configs import Hparams


def _layer_shapes(hp: Hparams, n_paths: Sequence[int]):
    S, NB, d, n = hp.n_species, hp.n_bessel, hp.d, hp.n_tensor
    nA = n * (hp.l_max + 1)
    shapes = []
    fi = 2 * S + NB
    for w in hp.twobody_dims:
        shapes.append(("dense", fi, w)); fi = w
    shapes.append(("dense", d, nA))
    for L in range(hp.n_layers):
        shapes.append(("dense", d, nA))
        shapes.append(("alpha", n_paths[L], L))
        fi = d + n
        for w in hp.latent_dims:
            shapes.append(("dense", fi, w)); fi = w
    fi = d
    for w in list(hp.edge_dims) + [1]:
        shapes.append(("dense", fi, w)); fi = w
    return shapes


def blob_num_floats(hp: Hparams, n_paths: Sequence[int]) -> int:
    tot = 0
    for s in _layer_shapes(hp, n_paths):
        tot += s[1] * s[2] if s[0] == "dense" else s[1]
    return tot


def make_blob(hp: Hparams, path_fan: List[List[int]], sigma: Sequence[float], mu: Sequence[float],
              seed: int = 0) -> bytes:
    """path_fan[L][p] = number of layer-(L+1) paths sharing path p's output irrep (canonical order).
    Xavier-normal dense weights N(0, 2/(fan_in+fan_out)); alpha_p ~ N(0, 1/path_fan)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    parts = []
    for s in _layer_shapes(hp, [len(p) for p in path_fan]):
        if s[0] == "dense":
            _, fi, fo = s
            w = rng.standard_normal((fi, fo)) * np.sqrt(2.0 / (fi + fo))
        else:
            fan = np.asarray(path_fan[s[2]], dtype=np.float64)
            w = rng.standard_normal(fan.shape[0]) / np.sqrt(fan)
        parts.append(np.ascontiguousarray(w, dtype="<f4").tobytes())
    raw = b"".join(parts)
    if len(raw) % 8:
        raw += b"\0" * (8 - len(raw) % 8)
    raw += np.asarray(sigma, dtype="<f8").tobytes() + np.asarray(mu, dtype="<f8").tobytes()
    return raw
