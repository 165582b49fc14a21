"""Run-to-run reproducibility of the CUDA path (SURVEY.md section 5 "run-to-run determinism check"; `-m gpu`).

Every reduction that feeds the energies runs in a fixed order (segmented per-centre sums, partial buffers written with
plain stores and summed in order, fixed-order fp64 tree sums), so E and the per-atom energies must be BIT-identical
from run to run.  Forces are accumulated into f64[N,3] with fp64 atomicAdd (F_i += g_e, F_j -= g_e; the list need not be
symmetric under ordered pair cutoffs, so there is no reverse-edge gather): the order of the additions varies, the values
must agree to fp64 round-off."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from synthetic import make_system
from synthetic.configs import scaled_config

from gpu_util import gpu_eval, make_both


@pytest.mark.parametrize("ci,n,precision", [(1, 3072, 1), (1, 3072, 0), (4, 1200, 1), (2, 3000, 1), (2, 3000, 4), (4, 1200, 2)])
def test_run_to_run(ci, n, precision):
    cfg = scaled_config(ci, n)
    pos, sp, box = make_system(cfg)
    model, _ = make_both(cfg, precision=precision, chunk_edges=20000)      # several chunks, ragged tail
    runs = [gpu_eval(model, pos, sp, box, cutoff=cfg.hp.r_cut + 0.5)[0] for _ in range(4)]
    model2, _ = make_both(cfg, precision=precision, chunk_edges=20000)     # a second model from the same blob
    runs.append(gpu_eval(model2, pos, sp, box, cutoff=cfg.hp.r_cut + 0.5)[0])
    E0, Ea0, F0 = runs[0]
    fmax = np.abs(F0).max()
    for E, Ea, F in runs[1:]:
        assert E == E0                                   # bit-identical
        assert np.array_equal(Ea, Ea0)                   # bit-identical per-atom energies
        assert np.abs(F - F0).max() <= 1e-12 * fmax      # fp64 atomics: order-dependent round-off only


@pytest.mark.parametrize("ci,n,precision", [(2, 20000, 1), (2, 20000, 4), (4, 6000, 1), (1, 12288, 2), (2, 20000, 0), (4, 6000, 0)])
def test_cta_pairs_match_single_cta_tiles(ci, n, precision):
    """allegro_set_gemm_pairs: the MLP GEMMs on CTA pairs (cta_group::2, 256-row tiles, the default for large launches) and on
    single CTAs (128-row tiles) accumulate over K in the same order, so energies are bit-identical and forces agree to the
    round-off of their fp64 atomics.  Sizes chosen so that every launch is large enough for the pair path (ragged last tiles,
    odd numbers of 128-row blocks included: 20,000 / 6,000 atoms give chunk sizes that are not multiples of 256)."""
    cfg = scaled_config(ci, n)
    pos, sp, box = make_system(cfg)
    out = []
    for pairs in (False, True):
        model, _ = make_both(cfg, precision=precision, chunk_edges=150001)
        model.set_gemm_pairs(pairs)
        out.append(gpu_eval(model, pos, sp, box, cutoff=cfg.hp.r_cut + 0.5)[0])
    (E0, Ea0, F0), (E1, Ea1, F1) = out
    assert E0 == E1
    assert np.array_equal(Ea0, Ea1)
    assert np.abs(F0 - F1).max() <= 1e-12 * np.abs(F0).max()
