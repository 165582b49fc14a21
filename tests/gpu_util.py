"""Helpers for GPU parity tests: build the product model and the oracle from the same seeded blob."""
import numpy as np

import paper_2304_10061_b200 as P
from oracle import allegro_oracle as O
from synthetic import make_blob


def make_both(cfg, precision=0, sigma=None, chunk_edges=None, tensor_track=0):
    hp = cfg.hp
    chp = P.hparams_from(hp, precision)
    fan_gpu = P.path_fan(chp)                       # product side: from the C library
    fan_or = O.path_fan(hp.l_max, hp.n_layers)      # oracle side: its own enumeration
    assert fan_gpu == fan_or
    s = cfg.sigma if sigma is None else sigma
    sig = list(s) if np.ndim(s) else [s] * hp.n_species           # scalar: same for every species; else per species
    assert len(sig) == hp.n_species
    blob = make_blob(hp, fan_gpu, sig, cfg.mu(), cfg.weight_seed)
    model = P.Allegro(chp, blob, chunk_edges=chunk_edges)
    if tensor_track:
        model.set_tensor_track(tensor_track)          # 1: per-edge product kernels instead of the per-centre contraction
    if getattr(hp, "r_cut_pair", None) is not None:
        model.set_pair_cutoffs(hp.r_cut_pair)
    if getattr(hp, "bessel_freq_pair", None) is not None:
        model.set_bessel_frequencies(hp.bessel_freq_pair)
    if getattr(hp, "zbl_Z", None) is not None:
        model.set_zbl(hp.zbl_Z)
    oracle = O.OracleModel(hp, blob)
    return model, oracle


def gpu_eval(model, pos, sp, box, cutoff=None):
    import torch
    p = torch.from_numpy(np.ascontiguousarray(pos)).cuda()
    s = torch.from_numpy(np.ascontiguousarray(sp, dtype=np.int32)).cuda()
    nb = model.neighbors(p, box, cutoff or model.hp.r_cut)
    e, ea, f = model.compute(p, s, box, nb)
    torch.cuda.synchronize()
    out = float(e.item()), ea.cpu().numpy(), f.cpu().numpy()
    return out, nb


def nbr_as_arrays(nb):
    rp, j, s = nb.to_host()
    i = np.repeat(np.arange(rp.shape[0] - 1), np.diff(rp))
    return i.astype(np.int64), j.astype(np.int64), s.astype(np.int64)
