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
