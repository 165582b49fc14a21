"""`-m gpu`: the deferred-error channel of the asynchronous calls (allegro_status), the halo kernels of the spatial
decomposition against the torch expressions they replace, and the peak probes bench.py uses as roofline denominators."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2304_10061_b200 as P
from synthetic import make_system
from synthetic.configs import scaled_config

from gpu_util import make_both


def test_status_surfaces_coincident_atoms_and_bad_species():
    cfg = scaled_config(0, 192)
    model, _ = make_both(cfg)
    box = np.array([20.0, 20.0, 20.0])
    pos = torch.tensor([[1.0, 1.0, 1.0], [1.0, 1.0, 1.0], [2.0, 1.0, 1.0]], dtype=torch.float64).cuda()
    sp = torch.tensor([0, 1, 0], dtype=torch.int32).cuda()
    nb = model.neighbors(pos, box, 4.0)
    model.compute(pos, sp, box, nb)                     # device-pointer call: returns after enqueueing, no error yet
    with pytest.raises(P.AllegroError) as ei:
        model.status()
    assert ei.value.code == -5                          # ALLEGRO_ERR_NONFINITE: r = 0
    model.status()                                      # the flag was cleared
    # species outside [0, n_species): flagged, and no table is read out of bounds (look-ups clamp)
    pos2, sp2, box2 = make_system(cfg)
    p2 = torch.from_numpy(pos2).cuda()
    bad = sp2.copy(); bad[7] = 5; bad[11] = -3
    nb2 = model.neighbors(p2, box2, cfg.hp.r_cut)
    e, ea, f = model.compute(p2, torch.from_numpy(bad).cuda(), box2, nb2)
    with pytest.raises(P.AllegroError) as ei:
        model.status()
    assert ei.value.code == -8                          # ALLEGRO_ERR_BAD_ARG
    assert torch.isfinite(f).all()
    # and a clean evaluation afterwards reports nothing
    model.compute(p2, torch.from_numpy(sp2).cuda(), box2, nb2)
    model.status()


def test_halo_kernels_match_torch_expressions():
    cfg = scaled_config(1, 1536)
    pos, sp, box = make_system(cfg)
    model, _ = make_both(cfg)
    g = np.random.default_rng(5)
    p = torch.from_numpy(pos).cuda(); s = torch.from_numpy(sp).cuda()
    k = 700
    idx = torch.from_numpy(g.integers(0, pos.shape[0], k)).cuda()                      # duplicates on purpose
    shift = torch.from_numpy(g.integers(-1, 2, (k, 3)) * box).cuda().contiguous()
    rows = model.halo_pack(p, s, idx, shift)
    want = torch.cat([p[idx] + shift, s[idx].to(torch.float64)[:, None]], dim=1)
    assert torch.equal(rows, want)
    origin = np.array([-3.0, 1.5, 0.25])
    pos_all, sp_all = model.halo_assemble(p, s, rows, origin)
    o = torch.from_numpy(origin).cuda()
    assert torch.equal(pos_all, torch.cat([p, rows[:, :3]], dim=0) - o)
    assert torch.equal(sp_all, torch.cat([s, s[idx]], dim=0))
    f_all = torch.from_numpy(g.standard_normal((pos.shape[0] + k, 3))).cuda()
    ret = torch.from_numpy(g.standard_normal((k, 3))).cuda()
    out = model.halo_accumulate(f_all, pos.shape[0], idx, ret)
    ref = f_all[: pos.shape[0]].clone(); ref.index_add_(0, idx, ret)
    assert torch.allclose(out, ref, rtol=0, atol=1e-12)
    # empty messages
    z = torch.zeros(0, dtype=torch.int64, device="cuda")
    assert model.halo_pack(p, s, z, torch.zeros((0, 3), dtype=torch.float64, device="cuda")).shape == (0, 4)


def test_peak_probes_are_plausible():
    cfg = scaled_config(0, 192)
    model, _ = make_both(cfg)
    pk = model.probe_peaks(0.2)
    assert 30.0 < pk["ffma"]["burst"] < 90.0            # 148 SMs x 128 lanes x 2 x 1.965 GHz = 74.4 TFLOP/s
    assert 500.0 < pk["tf32_mma"]["burst"] < 1300.0     # nominal dense TF32 ~1.1 PFLOP/s


def test_profile_groups_with_nvtx_ranges():
    """allegro_profile_enable bit mask: 1 = CUDA-event timing per kernel group, 2 = NVTX range per group.  The ranges are host-side
    markers (visible to a profiler only); here: both bits on, the result is unchanged and the group timers still fill."""
    cfg = scaled_config(1, 768)
    pos, sp, box = make_system(cfg)
    model, _ = make_both(cfg, precision=1)
    p = torch.from_numpy(pos).cuda(); s = torch.from_numpy(sp.astype(np.int32)).cuda()
    nb = model.neighbors(p, box, cfg.hp.r_cut)
    e0, _, f0 = model.compute(p, s, box, nb)
    model.profile_enable(True, nvtx=True)
    e1, _, f1 = model.compute(p, s, box, nb)
    ms, n = model.profile_read("gemm")
    model.profile_enable(False)
    assert n > 0 and ms > 0.0
    assert float(e0.item()) == float(e1.item())
    assert (f0 - f1).abs().max().item() <= 1e-12 * f0.abs().max().item()
