"""16-bit operand MLP modes through the C ABI (`-m gpu`): precision 4 = IEEE fp16, precision 2 = bfloat16 storage of every
tensor that only the MLP GEMMs and their epilogues touch (include/b200_allegro.h: allegro_hparams::precision).

fp16 has TF32's 10 explicit mantissa bits, so precision 4 is held to the TF32 tolerance of BASELINE.json's north_star
(2e-3 relative on E and F, read as in test_gpu_parity.test_energy_forces_tf32).  bfloat16 has 7: its unit round-off is 8x
TF32's and the mode does NOT meet 2e-3 (DESIGN.md section 9 lists the measured errors); it is tested against 8 x 2e-3 and is
documented as outside the north_star tolerance."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2304_10061_b200 as P
from oracle import allegro_oracle as O
from synthetic import make_system
from synthetic.configs import scaled_config

from gpu_util import gpu_eval, make_both
from test_gpu_parity import _subsystem_check, _variant

TOL = {4: 2e-3, 2: 1.6e-2}


def _errors(cfg, precision, **kw):
    pos, sp, box = make_system(cfg)
    model, oracle = make_both(cfg, precision=precision, **kw)
    (E, Ea, F), nb = gpu_eval(model, pos, sp, box)
    E0, Ea0, F0 = O.energy_forces(oracle, pos, sp, box, O.neighbor_list(pos, box, cfg.hp.r_cut))
    mu = np.array(cfg.mu())[sp]
    relE = abs(E - E0) / np.abs(Ea0 - mu).sum()
    relEa = np.abs(Ea - Ea0).max() / np.abs(Ea0 - mu).max()
    relF_max = np.abs(F - F0).max() / np.abs(F0).max()
    relF_l2 = np.linalg.norm(F - F0) / np.linalg.norm(F0)
    assert np.isfinite(F).all() and np.isfinite(Ea).all()
    assert abs(F.sum(0)).max() < 1e-6 * np.abs(F).sum()             # Newton's third law holds in every precision mode
    return relE, relEa, relF_max, relF_l2


@pytest.mark.parametrize("precision", [4, 2])
@pytest.mark.parametrize("ci,n", [(1, 1536), (2, 3000), (4, 1200)])
def test_energy_forces_16bit(ci, n, precision):
    relE, relEa, relF_max, relF_l2 = _errors(scaled_config(ci, n), precision)
    print(f"[{'fp16' if precision == 4 else 'bf16'} cfg{ci}] relE={relE:.3e} relE_i={relEa:.3e} relF: max/max={relF_max:.3e} l2={relF_l2:.3e}")
    tol = TOL[precision]
    assert relE <= tol and relEa <= tol and relF_max <= tol and relF_l2 <= tol


@pytest.mark.parametrize("ci", [2, 4])
def test_full_size_subsystem_parity_fp16(ci):
    """bench.py's launch configuration (default chunking, skin list) at the full size, sampled centres and probe atoms."""
    _subsystem_check(ci, 24, 4)


# shapes the 16-bit modes accept besides the configs: narrow l_max = 3 models with three and two layers, a second latent
# layer, one layer, a per-species sigma and non-default residual weights (c_old / c_new enter the fused epilogues)
SHAPES_16 = {
    "lmax3_three_layers_n32": (4, 600, dict(n_tensor=32, resid_alpha=(0.3, 0.5, 0.7), twobody_dims=(32, 64), latent_dims=(64,))),
    "lmax1_two_layers_n32": (0, 384, dict(n_layers=2, n_tensor=32, resid_alpha=(0.5, 0.5), twobody_dims=(32, 64), latent_dims=(64,))),
    "two_latent_layers": (1, 768, dict(twobody_dims=(32, 64), latent_dims=(64, 64), edge_dims=(32, 16))),
    "one_layer": (1, 768, dict(n_layers=1, resid_alpha=(0.5,), twobody_dims=(32, 64), latent_dims=(64,))),
}


@pytest.mark.parametrize("name", sorted(SHAPES_16))
def test_other_shapes_fp16(name):
    base, n, changes = SHAPES_16[name]
    cfg = _variant(base, n, **changes)
    sigma = [0.7 + 0.3 * z for z in range(cfg.hp.n_species)]
    relE, relEa, relF_max, relF_l2 = _errors(cfg, 4, sigma=sigma)
    print(f"[fp16 {name}] relE={relE:.3e} relE_i={relEa:.3e} relF: max/max={relF_max:.3e} l2={relF_l2:.3e}")
    assert relE <= 2e-3 and relF_max <= 2e-3 and relF_l2 <= 2e-3


def test_chunking_invariance_fp16():
    """Chunk boundaries (ragged last chunk, one chunk of a few hundred edges) do not change the result beyond fp64 summation
    order: every per-edge value is computed the same way whatever chunk it lands in."""
    cfg = scaled_config(1, 1536)
    pos, sp, box = make_system(cfg)
    ref = None
    for ce in (None, 20000, 7777):
        model, _ = make_both(cfg, precision=4, chunk_edges=ce)
        (E, Ea, F), _ = gpu_eval(model, pos, sp, box, cutoff=cfg.hp.r_cut + 0.5)
        if ref is None:
            ref = (E, Ea, F)
            continue
        assert abs(E - ref[0]) <= 1e-9 * np.abs(ref[1]).sum()
        assert np.abs(Ea - ref[1]).max() <= 1e-9 * np.abs(ref[1]).max()
        assert np.abs(F - ref[2]).max() <= 1e-9 * np.abs(ref[2]).max()


def test_16bit_modes_refuse_what_they_do_not_cover():
    """The 16-bit modes exist only on the per-centre-contracted tensor track with the K-concatenated x-bar GEMM: the per-edge
    product kernels (allegro_set_tensor_track(1)) and shapes outside the contraction are refused with
    ALLEGRO_ERR_UNIMPLEMENTED at the first compute, never run in another precision."""
    cfg = scaled_config(1, 768)
    pos, sp, box = make_system(cfg)
    model, _ = make_both(cfg, precision=4, tensor_track=1)
    with pytest.raises(P.AllegroError) as ei:
        gpu_eval(model, pos, sp, box)
    assert ei.value.code == -7 and "16-bit" in str(ei.value)
    # l_max = 2 with three layers: the middle layers carry pseudo-irreps, outside the contracted track's generated patterns
    # (csrc/tpc_kernels.cu: tpc_eligible); the TF32 / fp32 modes run it on the generic kernels (test_gpu_parity.VARIANTS)
    cfg3 = _variant(1, 768, n_layers=3, resid_alpha=(0.5,) * 3, twobody_dims=(32, 64), latent_dims=(64,))
    model3, _ = make_both(cfg3, precision=2)
    with pytest.raises(P.AllegroError) as ei:
        gpu_eval(model3, pos, sp, box)
    assert ei.value.code == -7
