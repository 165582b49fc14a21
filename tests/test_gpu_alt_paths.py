"""The library keeps older / alternative kernels behind environment switches.  They are
read once per process, so each case runs a small parity check in a fresh interpreter: energy + forces of a
reduced config against the fp64 oracle, with the same tolerances as the default path."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import sys, numpy as np
sys.path.insert(0, {root!r}); sys.path.insert(0, {root!r} + "/tests")
from oracle import allegro_oracle as O
from synthetic import make_system
from synthetic.configs import scaled_config
from gpu_util import make_both, gpu_eval
ci, n, precision = {ci}, {n}, {precision}
cfg = scaled_config(ci, n)
pos, sp, box = make_system(cfg)
model, oracle = make_both(cfg, precision=precision)
(E, Ea, F), nb = gpu_eval(model, pos, sp, box)
E0, Ea0, F0 = O.energy_forces(oracle, pos, sp, box, O.neighbor_list(pos, box, cfg.hp.r_cut))
mu = np.array(cfg.mu())[sp]
if precision in (0, 3):
    assert abs(E - E0) / n <= 1e-6, abs(E - E0) / n
    assert np.abs(F - F0).max() <= 1e-5 * max(1.0, float(np.sqrt((F0 ** 2).mean()))), np.abs(F - F0).max()
else:
    assert abs(E - E0) <= 2e-3 * np.abs(Ea0 - mu).sum()
    assert np.abs(F - F0).max() <= 2e-3 * np.abs(F0).max()
print("ok", abs(E - E0) / n, np.abs(F - F0).max())
"""

CASES = [
    ("tp_old_cfg1", {"B200_ALLEGRO_TP_OLD": "1"}, 1, 1536, 0),          # first-generation tensor-track kernels
    ("tp_old_cfg4", {"B200_ALLEGRO_TP_OLD": "1"}, 4, 1200, 0),
    ("no_prep_cfg1", {"B200_ALLEGRO_NO_PREP": "1"}, 1, 1536, 0),        # separate k_bwd_prep pass
    ("no_prep_tf32", {"B200_ALLEGRO_NO_PREP": "1"}, 1, 1536, 1),
    ("tp_mreg_cfg1", {"B200_ALLEGRO_TP_MREG": "1"}, 1, 1536, 0),        # 9x9x9 backward with M in registers
    ("tp3_bwd2_cfg4", {"B200_ALLEGRO_TP3_BWD": "2"}, 4, 1200, 0),       # lane-split l_max = 3 backward, 4 blocks
    ("tp3_bwd3_cfg4", {"B200_ALLEGRO_TP3_BWD": "3"}, 4, 1200, 0),       # ... 8 blocks
    ("fp32_simt_env", {"B200_ALLEGRO_FP32_SIMT": "1"}, 1, 1536, 0),
    ("tp3_no_mma_tf32_cfg4", {"B200_ALLEGRO_TP3_NO_MMA": "1"}, 4, 1200, 1),   # FFMA forward for l_max = 3 in TF32 mode
    ("no_kcat_cfg1", {"B200_ALLEGRO_NO_KCAT": "1"}, 1, 1536, 0),        # separate dX-latent and x-bar GEMMs
    ("no_kcat_tf32_cfg4", {"B200_ALLEGRO_NO_KCAT": "1"}, 4, 1200, 1),
    ("no_sweep_cfg1", {"B200_ALLEGRO_SWEEP": "0"}, 1, 1536, 1),         # every kernel walks the edges forward
    ("no_sweep_cfg4", {"B200_ALLEGRO_SWEEP": "0"}, 4, 1200, 0),
    ("no_kcat_no_prep", {"B200_ALLEGRO_NO_KCAT": "1", "B200_ALLEGRO_NO_PREP": "1"}, 2, 3000, 0),
]


@pytest.mark.gpu
@pytest.mark.parametrize("name,env,ci,n,precision", CASES, ids=[c[0] for c in CASES])
def test_alternative_kernel_paths(name, env, ci, n, precision):
    e = dict(os.environ)
    e.update(env)
    r = subprocess.run([sys.executable, "-c", SCRIPT.format(root=ROOT, ci=ci, n=n, precision=precision)],
                       env=e, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert r.stdout.strip().startswith("ok")
