"""Spatial domain decomposition of the energy+force evaluation over the GPUs of one node (SURVEY.md section 8(e),
NEXT-3; the paper: one rank per GPU over LAMMPS's spatial decomposition).

Strict locality (E-hat_i needs only the atoms within r_c of i) makes the path shard by space: every
rank owns the atoms of one cell of a px x py x pz grid over the periodic box, evaluates E-hat_i and -dE/dr for its own
centres with `allegro_compute_local`, and two neighbour-wise exchanges per evaluation connect the domains:

  forward  : the positions of the atoms within `halo` of a domain face go to that domain as GHOSTS (with the periodic
             image shift applied; a domain that spans the box in some direction receives images of its own atoms),
  reverse  : the forces the domain accumulated on its ghosts go back to their owners and are added there,

plus one scalar all-reduce for the total energy.  Both exchanges are `all_to_all_single` calls with split sizes (NCCL over
NVLink on GPUs; gloo in the CPU tests), the same index lists serving both directions.  Everything here is plumbing
(index lists, packing, torch.distributed); the arithmetic of the path runs in the CUDA library.  The class is driven in
phases (`pack` / `unpack` / `local_system` / `finish`) so that the tests can also route the messages by hand between
several domains inside one process (one GPU)."""
from __future__ import annotations

import itertools
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np
import torch


class DomainGrid:
    """px x py x pz cells over the periodic box [0, L); rank = (ix * py + iy) * pz + iz."""

    def __init__(self, box: Sequence[float], grid: Sequence[int]):
        self.box = np.asarray(box, dtype=np.float64)
        self.grid = tuple(int(g) for g in grid)
        assert len(self.grid) == 3 and all(g >= 1 for g in self.grid)
        self.n_ranks = self.grid[0] * self.grid[1] * self.grid[2]
        self.cell = self.box / np.asarray(self.grid, dtype=np.float64)

    def coords(self, rank: int) -> Tuple[int, int, int]:
        px, py, pz = self.grid
        return rank // (py * pz), (rank // pz) % py, rank % pz

    def bounds(self, rank: int) -> Tuple[np.ndarray, np.ndarray]:
        c = np.asarray(self.coords(rank), dtype=np.float64)
        return c * self.cell, (c + 1.0) * self.cell

    def wrap(self, pos: torch.Tensor) -> torch.Tensor:
        L = torch.as_tensor(self.box, dtype=pos.dtype, device=pos.device)
        w = pos - torch.floor(pos / L) * L
        return torch.where(w >= L, w - L, w)            # pos = -1e-17 -> w = L after rounding

    def owner(self, pos_wrapped: torch.Tensor) -> torch.Tensor:
        cell = torch.as_tensor(self.cell, dtype=pos_wrapped.dtype, device=pos_wrapped.device)
        g = torch.as_tensor(self.grid, dtype=torch.int64, device=pos_wrapped.device)
        idx = torch.minimum(torch.floor(pos_wrapped / cell).to(torch.int64), g - 1).clamp_(min=0)
        return (idx[:, 0] * self.grid[1] + idx[:, 1]) * self.grid[2] + idx[:, 2]


def auto_grid(n_ranks: int, box: Sequence[float]) -> Tuple[int, int, int]:
    """Factorisation of n_ranks into px*py*pz with the most cubic cells (smallest halo surface)."""
    best, best_s = (n_ranks, 1, 1), None
    for px in range(1, n_ranks + 1):
        if n_ranks % px:
            continue
        for py in range(1, n_ranks // px + 1):
            if (n_ranks // px) % py:
                continue
            pz = n_ranks // px // py
            c = [box[0] / px, box[1] / py, box[2] / pz]
            s = c[0] * c[1] + c[1] * c[2] + c[0] * c[2]
            if best_s is None or s < best_s - 1e-12:
                best, best_s = (px, py, pz), s
    return best


class TorchComm:
    """torch.distributed plumbing: variable all-to-all of row blocks (all_to_all_single with split sizes, which both
    NCCL and gloo implement) and a sum all-reduce."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def exchange_counts(self, counts: List[int], device) -> List[int]:
        s = torch.tensor(counts, dtype=torch.int64, device=device)
        r = torch.empty_like(s)
        self.dist.all_to_all_single(r, s, group=self.group)
        return [int(x) for x in r.tolist()]

    def all_to_all_rows(self, send: torch.Tensor, send_counts: List[int], recv_counts: List[int]) -> torch.Tensor:
        """send: [sum(send_counts), C] rows grouped by destination -> [sum(recv_counts), C] rows grouped by source."""
        out = torch.empty((sum(recv_counts),) + tuple(send.shape[1:]), dtype=send.dtype, device=send.device)
        self.dist.all_to_all_single(out, send.contiguous(), output_split_sizes=recv_counts, input_split_sizes=send_counts,
                                    group=self.group)
        return out

    def all_reduce_sum(self, t: torch.Tensor) -> torch.Tensor:
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return t


class Domain:
    """One rank's share of the system: its own atoms, the ghost send lists, the two exchanges.

    compute_local(pos_all f64[n,3], species_all i32[n], n_local, box_local[3]) -> (e_local f64 scalar tensor,
    force_all f64[n,3]) evaluates the local centres; the default binds `Allegro.neighbors` + `Allegro.compute_local`
    (CUDA; there is no CPU fallback); the multi-process CPU tests inject their own evaluator."""

    def __init__(self, grid: DomainGrid, rank: int, halo: float, r_cut: float, model=None,
                 compute_local: Optional[Callable] = None):
        assert halo >= r_cut > 0
        assert all(grid.box[k] >= halo for k in range(3)), "box edge shorter than the halo: images beyond +-1 needed"
        self.grid, self.rank, self.halo, self.r_cut = grid, rank, float(halo), float(r_cut)
        self.lo, self.hi = grid.bounds(rank)
        self.model = model
        self._nbr = None
        self.compute_local = compute_local or self._compute_with_library
        self.pos = self.species = self.gid = None
        self.send_idx = self.send_shift = None
        self.send_counts: List[int] = []
        self.recv_counts: List[int] = []

    # ---- ownership ------------------------------------------------------------------------------------------
    def take_owned(self, pos_global: torch.Tensor, species_global: torch.Tensor):
        """Setup from arrays every rank holds (e.g. read from one file): keep the atoms of this domain.  Returns the
        global ids kept.  pos is stored wrapped into the box."""
        w = self.grid.wrap(pos_global)
        mine = torch.nonzero(self.grid.owner(w) == self.rank).reshape(-1)
        self.gid = mine
        self.pos = w[mine].contiguous()
        self.species = species_global[mine].contiguous()
        return mine

    def migrate(self, comm: "TorchComm", extra: Optional[torch.Tensor] = None):
        """Re-partition after the atoms moved: every atom goes to the domain whose cell holds its wrapped position
        (with its species, global id and the rows of `extra`, e.g. velocities).  Call before build_send_lists when an
        atom may have left its cell by more than halo - r_cut.  Returns the migrated `extra`."""
        w = self.grid.wrap(self.pos)
        dest = self.grid.owner(w)
        order = torch.argsort(dest, stable=True)
        counts = torch.bincount(dest, minlength=self.grid.n_ranks).tolist()
        cols = [w, self.species.to(w.dtype)[:, None], self.gid.to(w.dtype)[:, None]]
        if extra is not None:
            cols.append(extra.reshape(extra.shape[0], -1).to(w.dtype))
        rows = torch.cat(cols, dim=1)[order]
        rc = comm.exchange_counts([int(c) for c in counts], w.device)
        got = comm.all_to_all_rows(rows, [int(c) for c in counts], rc)
        self.pos = got[:, :3].contiguous()
        self.species = got[:, 3].round().to(self.species.dtype).contiguous()
        self.gid = got[:, 4].round().to(torch.int64).contiguous()
        self.send_idx = None
        return got[:, 5:].contiguous() if extra is not None else None

    # ---- ghost lists (rebuilt whenever atoms may have moved by more than halo - r_cut) ---------------------------
    def build_send_lists(self):
        """For every destination domain d: which (own atom, image shift) pairs lie within `halo` of d.  The atom itself
        (shift 0) in its own domain is not a ghost."""
        pos, L = self.pos, self.grid.box
        dev = pos.device
        idx_d, shift_d = [], []
        for d in range(self.grid.n_ranks):
            lo, hi = self.grid.bounds(d)
            lo_t = torch.as_tensor(lo - self.halo, dtype=pos.dtype, device=dev)
            hi_t = torch.as_tensor(hi + self.halo, dtype=pos.dtype, device=dev)
            ii, ss = [], []
            for s in itertools.product((-1, 0, 1), repeat=3):
                if d == self.rank and s == (0, 0, 0):
                    continue
                sv = torch.as_tensor(np.asarray(s, dtype=np.float64) * L, dtype=pos.dtype, device=dev)
                # an image can only reach d's expanded cell if the shifted DOMAIN overlaps it: cheap reject
                if np.any(self.lo + np.asarray(s) * L >= hi + self.halo) or np.any(self.hi + np.asarray(s) * L <= lo - self.halo):
                    continue
                p = pos + sv
                m = ((p >= lo_t) & (p < hi_t)).all(dim=1)
                k = torch.nonzero(m).reshape(-1)
                if k.numel():
                    ii.append(k)
                    ss.append(sv.expand(k.numel(), 3))
            idx_d.append(torch.cat(ii) if ii else torch.zeros(0, dtype=torch.int64, device=dev))
            shift_d.append(torch.cat(ss) if ss else torch.zeros((0, 3), dtype=pos.dtype, device=dev))
        self.send_counts = [int(x.numel()) for x in idx_d]
        self.send_idx = torch.cat(idx_d)
        self.send_shift = torch.cat(shift_d)
        self._nbr_dirty = True     # new ghost set: rebuild the list INTO the existing handle (buffers are reused, nothing leaks)
        return self.send_counts

    # ---- forward exchange ----------------------------------------------------------------------------------------
    def pack_forward(self) -> torch.Tensor:
        """Rows [x, y, z, species] of the ghosts this rank provides, grouped by destination."""
        if self._on_device():          # one library kernel (allegro_halo_pack) instead of gather + add + cast + cat
            return self.model.halo_pack(self.pos, self.species, self.send_idx, self.send_shift)
        p = self.pos[self.send_idx] + self.send_shift
        return torch.cat([p, self.species[self.send_idx].to(p.dtype)[:, None]], dim=1)

    def _on_device(self) -> bool:
        """The per-atom halo work runs in the library's kernels whenever the domain's arrays are CUDA tensors and a model is
        bound; the torch expressions below are the same operations for the CPU (gloo) tests of the exchange logic."""
        return self.model is not None and self.pos.is_cuda and self.species.dtype == torch.int32

    def local_system(self, ghosts: torch.Tensor):
        """Local atoms followed by the received ghosts, in a frame whose periodic box cannot connect opposite faces."""
        n_local = self.pos.shape[0]
        if self._on_device():          # allegro_halo_assemble: concatenate, shift into the local frame, cast the species
            origin_h = self.lo - self.halo
            pos_all, sp_all = self.model.halo_assemble(self.pos, self.species, ghosts.contiguous(), origin_h)
            return pos_all, sp_all, n_local, (self.hi - self.lo) + 3.0 * self.halo + 1.0
        pos_all = torch.cat([self.pos, ghosts[:, :3]], dim=0)
        sp_all = torch.cat([self.species, ghosts[:, 3].round().to(self.species.dtype)], dim=0)
        origin = torch.as_tensor(self.lo - self.halo, dtype=pos_all.dtype, device=pos_all.device)
        ext = (self.hi - self.lo) + 2.0 * self.halo
        box_local = ext + self.halo + 1.0            # > extent + cutoff: no pair is found through the boundary
        return (pos_all - origin).contiguous(), sp_all.contiguous(), n_local, box_local

    def _compute_with_library(self, pos_all, sp_all, n_local, box_local):
        if self.model is None:
            raise RuntimeError("Domain needs an Allegro model (CUDA): there is no CPU fallback")
        # the list is rebuilt with the ghost lists (build_send_lists) and reused in between (Verlet skin = halo - r_cut)
        if self._nbr is None or getattr(self, "_nbr_dirty", True) or self._nbr_n != pos_all.shape[0]:
            self._nbr = self.model.neighbors(pos_all, box_local, self.halo, reuse=self._nbr)
            self._nbr_n = pos_all.shape[0]
            self._nbr_dirty = False
        e, _, f = self.model.compute_local(pos_all, sp_all, n_local, box_local, self._nbr)
        return e, f

    # ---- reverse exchange ------------------------------------------------------------------------------------------
    def finish(self, f_all: torch.Tensor, returned: torch.Tensor) -> torch.Tensor:
        """Local part of the forces plus what the other domains accumulated on the ghosts this rank provided."""
        if self._on_device() and f_all.is_cuda:          # allegro_halo_accumulate
            return self.model.halo_accumulate(f_all.contiguous(), self.pos.shape[0], self.send_idx, returned.contiguous())
        f = f_all[: self.pos.shape[0]].clone()
        if returned.numel():
            f.index_add_(0, self.send_idx, returned)
        return f

    # ---- one velocity-Verlet NVE step of this domain's atoms (kicks and drift by the library's kernels) ---------------
    def nve_step(self, comm: "TorchComm", vel: torch.Tensor, force: torch.Tensor, mass: torch.Tensor, dt_fs: float,
                 rebuild: bool):
        """v += dt/2 a; r += dt v; [migrate + new ghost lists if rebuild]; halo exchange + forces; v += dt/2 a.
        vel / force belong to this rank's atoms and come back re-ordered when atoms migrated.  Returns
        (e_pot all-reduced f64[1], vel, force)."""
        self.model.nve_kick(self.pos, vel, force, self.species, mass, dt_fs, True)
        if rebuild:
            vel = self.migrate(comm, vel).reshape(-1, 3).contiguous()
        e, force = self.energy_forces(comm, rebuild=rebuild)
        force = force.contiguous()
        self.model.nve_kick(self.pos, vel, force, self.species, mass, dt_fs, False)
        return e, vel, force

    # ---- the whole evaluation over a communicator ----------------------------------------------------------------------
    def energy_forces(self, comm: TorchComm, rebuild: bool = True):
        """Total energy (all-reduced, f64 tensor [1]) and the forces on this rank's atoms."""
        if rebuild or self.send_idx is None:
            self.build_send_lists()
            self.recv_counts = comm.exchange_counts(self.send_counts, self.pos.device)
        ghosts = comm.all_to_all_rows(self.pack_forward(), self.send_counts, self.recv_counts)
        pos_all, sp_all, n_local, box_local = self.local_system(ghosts)
        e_local, f_all = self.compute_local(pos_all, sp_all, n_local, box_local)
        returned = comm.all_to_all_rows(f_all[n_local:].contiguous(), self.recv_counts, self.send_counts)
        e = comm.all_reduce_sum(e_local.reshape(1).clone())
        return e, self.finish(f_all, returned)
