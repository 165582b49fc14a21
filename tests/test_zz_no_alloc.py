"""allegro_kinetic_energy_noalloc (include/b200_allegro.h, csrc/noalloc.cu): the kinetic-energy reduction with its scratch in
a fixed __device__ array instead of a cudaMalloc'ed buffer (`-m gpu`).  The file name sorts last on purpose: the
run is `pytest -x`, and a failure here must not hide any other test.

Checked against the existing allegro_kinetic_energy on two calls in a row with different inputs (the second call finds the
first call's values in the shared scratch and must not see them), against the numpy definition, and that the call refuses a
size beyond its fixed maximum and leaves the device's free memory unchanged."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2304_10061_b200 as P
from synthetic import make_system, maxwell_boltzmann
from synthetic.configs import scaled_config
from synthetic.systems import masses_for

from gpu_util import make_both

ACC_CONV = 9.648533212e-3          # eV / (amu A^2 fs^-2), the constant of the velocity-Verlet step


def _inputs(cfg, seed, n_atoms):
    """Seeded velocities of the config's Maxwell-Boltzmann recipe (synthetic/systems.py), a different draw per `seed`."""
    import dataclasses
    _, sp, _ = make_system(cfg)
    sp = np.resize(sp, n_atoms).astype(np.int32)
    c = dataclasses.replace(cfg, vel_seed=cfg.vel_seed + seed, temperature=300.0 + 50.0 * seed)
    return maxwell_boltzmann(c, sp), sp, masses_for(cfg)


def test_kinetic_energy_noalloc_matches_existing_path_twice():
    cfg = scaled_config(1, 1536)
    model, _ = make_both(cfg, precision=1)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    # consecutive calls with different sizes and velocities: the later calls find the earlier calls' values in the shared
    # scratch (entries [1536, 40000) stay stale during the second call) and must not read them
    for k, (seed, n_atoms) in enumerate(((1, 40000), (2, 1536), (3, 40000))):
        vel, sp, mass = _inputs(cfg, seed, n_atoms)
        v = torch.from_numpy(vel).cuda()
        s = torch.from_numpy(sp).cuda()
        mk = torch.from_numpy(mass).cuda()
        want = float(model.kinetic_energy(v, s, mk).item())              # existing path (cudaMalloc'ed scratch)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        model.kinetic_energy_noalloc(v, s, mk, out)
        torch.cuda.synchronize()
        if k > 0:     # (the first call on a device may load the library's CUDA module lazily; later calls change nothing)
            assert torch.cuda.mem_get_info()[0] == free_before            # no device allocation by the call
        got = float(out.item())
        ref = float((0.5 * mass[sp] * (vel ** 2).sum(1)).sum() / ACC_CONV)
        # same arithmetic in the same order as the existing path; asserted at the fp64 round-off level that
        # tests/test_gpu_determinism.py allows for order-dependent sums (1e-12 relative)
        assert abs(got - want) <= 1e-12 * abs(want), (seed, got, want)
        assert abs(got - ref) <= 1e-12 * abs(ref), (seed, got, ref)


def test_kinetic_energy_noalloc_limits():
    cfg = scaled_config(1, 768)
    model, _ = make_both(cfg, precision=1)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    lib = P.load_library()
    nmax = 1048576                                                       # ALLEGRO_KINETIC_NOALLOC_MAX_ATOMS
    mass = torch.from_numpy(masses_for(cfg)).cuda()
    # at the maximum: accepted and correct
    g = torch.Generator(device="cuda").manual_seed(5)
    v = torch.randn(nmax, 3, dtype=torch.float64, device="cuda", generator=g) * 1e-2
    s = torch.zeros(nmax, dtype=torch.int32, device="cuda")
    got = float(model.kinetic_energy_noalloc(v, s, mass, out).item())
    want = float(model.kinetic_energy(v, s, mass).item())
    assert abs(got - want) <= 1e-12 * abs(want)
    # one atom more: refused with ALLEGRO_ERR_CAPACITY and a message that names the limit; `out` untouched
    out.fill_(-1.0)
    rc = lib.allegro_kinetic_energy_noalloc(model._h, v.data_ptr(), s.data_ptr(), mass.data_ptr(), nmax + 1, out.data_ptr())
    assert rc == -4
    assert b"1048576" in lib.allegro_last_error(model._h)
    torch.cuda.synchronize()
    assert float(out.item()) == -1.0
    # zero atoms: 0 eV
    assert lib.allegro_kinetic_energy_noalloc(model._h, v.data_ptr(), s.data_ptr(), mass.data_ptr(), 0, out.data_ptr()) == 0
    torch.cuda.synchronize()
    assert float(out.item()) == 0.0
