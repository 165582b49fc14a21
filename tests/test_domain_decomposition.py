"""NEXT-3: spatial domain decomposition with halo forward / reverse exchange.

CPU (`-m "not gpu"`): world_size-2 and -4 gloo runs of the real exchange code (`Domain.energy_forces` over
`TorchComm`), with the fp64 oracle standing in for the CUDA library as the per-domain evaluator; the assembled energy and
forces must be those of the undivided system.  GPU (`-m gpu`): 2 and 8 domains evaluated one after the other on the
one GPU through `allegro_compute_local`, the messages routed by hand, against the single-domain GPU result and the
oracle."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from oracle import allegro_oracle as O
from synthetic import make_system
from synthetic.configs import scaled_config

HALO = 4.6


def _oracle_for(cfg):
    from oracle_util import oracle_model
    m, _ = oracle_model(cfg.hp, sigma=cfg.sigma, mu=cfg.mu(), seed=cfg.weight_seed)
    return m


def _oracle_evaluator(oracle, r_cut):
    def compute_local(pos_all, sp_all, n_local, box_local):
        p, s = pos_all.numpy(), sp_all.numpy()
        nbr = O.neighbor_list(p, np.asarray(box_local), r_cut)
        _, Ea, F = O.energy_forces(oracle, p, s, np.asarray(box_local), nbr, centers=np.arange(n_local))
        return torch.tensor(Ea[:n_local].sum(), dtype=torch.float64), torch.from_numpy(F)
    return compute_local


def _worker(rank, world, port, grid, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.set_num_threads(2)
    from paper_2304_10061_b200.domain import Domain, DomainGrid, TorchComm
    cfg = scaled_config(0, 192)
    pos, sp, box = make_system(cfg)
    pos = pos + np.array([3.3, -20.1, 7.7])                 # unwrapped input: the decomposition wraps
    oracle = _oracle_for(cfg)
    g = DomainGrid(box, grid)
    dom = Domain(g, rank, HALO, cfg.hp.r_cut, compute_local=_oracle_evaluator(oracle, cfg.hp.r_cut))
    gid = dom.take_owned(torch.from_numpy(pos), torch.from_numpy(sp))
    comm = TorchComm()
    e, f = dom.energy_forces(comm)
    # move every atom a little (< halo - r_cut) and evaluate again WITHOUT rebuilding the ghost lists
    disp = np.random.default_rng(7).uniform(-0.25, 0.25, pos.shape)
    dom.pos = dom.pos + torch.from_numpy(disp)[gid]
    e2, f2 = dom.energy_forces(comm, rebuild=False)
    # migrate after a large collective displacement and evaluate once more
    dom.pos = dom.pos + torch.tensor([5.0, 0.0, 0.0], dtype=torch.float64)
    dom.migrate(comm)
    e3, f3 = dom.energy_forces(comm)
    out[rank] = (gid.numpy(), e.item(), f.numpy(), e2.item(), f2.numpy(), dom.gid.numpy(), e3.item(), f3.numpy(),
                 sum(dom.send_counts), dom.pos.shape[0])
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,grid,port", [(2, (2, 1, 1), 29551), (4, (2, 2, 1), 29552)])
def test_halo_exchange_reproduces_the_undivided_system_gloo(world, grid, port):
    cfg = scaled_config(0, 192)
    pos, sp, box = make_system(cfg)
    oracle = _oracle_for(cfg)
    E0, _, F0 = O.energy_forces(oracle, pos, sp, box, O.neighbor_list(pos, box, cfg.hp.r_cut))
    disp = np.random.default_rng(7).uniform(-0.25, 0.25, pos.shape)
    E1, _, F1 = O.energy_forces(oracle, pos + disp, sp, box, O.neighbor_list(pos + disp, box, cfg.hp.r_cut))
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, grid, out), nprocs=world, join=True)
    F, F2, F3 = np.zeros_like(F0), np.zeros_like(F0), np.zeros_like(F0)
    seen, seen3, n_ghost = [], [], 0
    for r in range(world):
        gid, e, f, e2, f2, gid3, e3, f3, ng, nloc = out[r]
        F[gid], F2[gid], F3[gid3] = f, f2, f3
        seen += gid.tolist(); seen3 += gid3.tolist(); n_ghost += ng
        assert abs(e - E0) < 1e-9 * max(1.0, abs(E0)) and abs(e2 - E1) < 1e-9 * max(1.0, abs(E1))
        assert abs(e3 - E1) < 1e-9 * max(1.0, abs(E1))          # a rigid translation leaves E and F unchanged
    assert sorted(seen) == list(range(192)) and sorted(seen3) == list(range(192)) and n_ghost > 192
    assert np.abs(F - F0).max() < 1e-10 and np.abs(F2 - F1).max() < 1e-10 and np.abs(F3 - F1).max() < 1e-10


def test_grid_geometry_and_ghost_lists():
    from paper_2304_10061_b200.domain import Domain, DomainGrid, auto_grid
    assert auto_grid(8, (10.0, 10.0, 10.0)) == (2, 2, 2) and auto_grid(4, (40.0, 10.0, 10.0)) == (4, 1, 1)
    g = DomainGrid((12.0, 9.0, 6.0), (2, 3, 1))
    assert g.n_ranks == 6 and g.coords(5) == (1, 2, 0)
    lo, hi = g.bounds(5)
    assert np.allclose(lo, [6.0, 6.0, 0.0]) and np.allclose(hi, [12.0, 9.0, 6.0])
    gen = torch.Generator().manual_seed(3)
    pos = (torch.rand((500, 3), generator=gen, dtype=torch.float64) - 0.3) * torch.tensor([30.0, 20.0, 15.0], dtype=torch.float64)
    w = g.wrap(pos)
    assert (w >= 0).all() and (w < torch.tensor([12.0, 9.0, 6.0])).all()
    own = g.owner(w)
    assert own.min() >= 0 and own.max() < 6
    # brute-force ghost set of one domain: every image within halo of the cell, except the atoms themselves
    halo, r = 2.5, 3
    doms = [Domain(g, k, halo, 2.0, compute_local=lambda *a: None) for k in range(6)]
    sp = torch.zeros(500, dtype=torch.int32)
    for d in doms:
        d.take_owned(pos, sp)
        d.build_send_lists()
    lo, hi = g.bounds(r)
    want = 0
    for s in np.ndindex(3, 3, 3):
        sv = (np.array(s) - 1) * g.box
        p = w.numpy() + sv
        inside = np.all((p >= lo - halo) & (p < hi + halo), axis=1)
        if tuple(np.array(s) - 1) == (0, 0, 0):
            inside &= own.numpy() != r
        want += int(inside.sum())
    got = sum(d.send_counts[r] for d in doms)
    assert got == want and want > 0


# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("ci,n,grid,precision", [(0, 192, (2, 1, 1), 0), (1, 1536, (2, 2, 2), 0), (1, 1536, (2, 2, 2), 1),
                                                 (2, 3000, (2, 2, 1), 0)])
def test_domains_on_one_gpu_match_the_single_domain_result(ci, n, grid, precision):
    from gpu_util import gpu_eval, make_both
    from paper_2304_10061_b200.domain import Domain, DomainGrid
    import dataclasses
    cfg = scaled_config(ci, n)
    from synthetic.configs import ATOMIC_NUMBERS
    cfg.hp = dataclasses.replace(cfg.hp, zbl_Z=tuple(ATOMIC_NUMBERS[s] for s in cfg.species_names))
    pos, sp, box = make_system(cfg)
    model, oracle = make_both(cfg, precision=precision)
    (E1, Ea1, F1), _ = gpu_eval(model, pos, sp, box)
    g = DomainGrid(box, grid)
    P, S = torch.from_numpy(pos).cuda(), torch.from_numpy(sp).cuda()
    doms = [Domain(g, r, cfg.hp.r_cut + 0.6, cfg.hp.r_cut, model=model) for r in range(g.n_ranks)]
    gids = [d.take_owned(P, S) for d in doms]
    for d in doms:
        d.build_send_lists()
    # forward exchange by hand: rows packed by destination
    packs = [d.pack_forward() for d in doms]
    offs = [np.concatenate([[0], np.cumsum(d.send_counts)]) for d in doms]
    E, F = 0.0, torch.zeros_like(P)
    f_alls, n_locals = [], []
    for r, d in enumerate(doms):
        ghosts = torch.cat([packs[s][offs[s][r]:offs[s][r + 1]] for s in range(g.n_ranks)])
        pos_all, sp_all, n_local, box_local = d.local_system(ghosts)
        d._nbr = None
        e, f_all = d.compute_local(pos_all, sp_all, n_local, box_local)
        E += e.item(); f_alls.append(f_all); n_locals.append(n_local)
    # reverse exchange by hand: domain r holds the ghosts of source s in the order s sent them
    for s, d in enumerate(doms):
        back = []
        for r in range(g.n_ranks):
            start = n_locals[r] + sum(doms[q].send_counts[r] for q in range(s))
            back.append(f_alls[r][start:start + d.send_counts[r]])
        F[gids[s]] = d.finish(f_alls[s], torch.cat(back))
    torch.cuda.synchronize()
    F = F.cpu().numpy()
    fs = max(1.0, float(np.sqrt((F1 ** 2).mean())))
    print(f"[domains cfg{ci} grid={grid} prec={precision}] |dE|/N={abs(E - E1) / n:.3e} max|dF|={np.abs(F - F1).max():.3e}")
    if precision == 0:
        assert abs(E - E1) / n <= 2e-6 and np.abs(F - F1).max() <= 2e-5 * fs          # two fp32-mode evaluations apart
        E0, _, F0 = O.energy_forces(oracle, pos, sp, box, O.neighbor_list(pos, box, cfg.hp.r_cut))
        assert abs(E - E0) / n <= 1e-6 and np.abs(F - F0).max() <= 1e-5 * fs
    else:
        assert np.abs(F - F1).max() <= 2e-3 * np.abs(F1).max()


@pytest.mark.gpu
def test_decomposed_md_over_nccl_world1_matches_the_plain_step():
    """`bench.py --decompose` at one rank: the single domain exchanges its periodic images with itself through the real
    NCCL all_to_all_single path (migration at every rebuild included); after 8 MD steps the energies must be those of
    the plain allegro_step_nve run."""
    import json
    import subprocess
    outs = []
    for extra in (["--decompose"], ["--no-cpu-baseline", "--repeats", "1", "--no-peak-probe"]):   # both: 3 + 5 steps
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "0", "--steps", "5", "--warmup", "3"] + extra,
                           capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-3000:]
        outs.append(json.loads(r.stdout.strip().splitlines()[-1]))
    dec, std = outs
    assert dec["scaling"] == "strong" and dec["config"]["ghost_atoms_max"] > 0 and dec["gpu_launches"] > 0
    assert abs(dec["e_pot"] - std["e_pot"]) < 192 * 2e-6 and abs(dec["e_kin"] - std["e_kin"]) < 1e-4
