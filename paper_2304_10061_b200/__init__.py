"""paper_2304_10061_b200 — thin Python binding of libb200allegro.so (include/b200_allegro.h).

Argument marshalling only: every step of the hot path runs in the library's CUDA kernels.  PyTorch is
used for device memory (tensors, caching allocator hook), streams and nothing else.  There is no CPU
fallback: if the shared library is missing or no CUDA device is present, calls fail loudly.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

from .build import build as build_library, lib_path

__all__ = ["Hparams", "Allegro", "NeighborList", "AllegroError", "load_library", "hparams_from"]

_I32x8 = C.c_int32 * 8
_F64x8 = C.c_double * 8


class Hparams(C.Structure):
    """Mirror of `allegro_hparams` (include/b200_allegro.h)."""
    _fields_ = [
        ("n_species", C.c_int32), ("l_max", C.c_int32), ("n_layers", C.c_int32), ("n_tensor", C.c_int32),
        ("n_bessel", C.c_int32), ("poly_p", C.c_int32),
        ("r_cut", C.c_double),
        ("n_twobody", C.c_int32), ("twobody_dims", _I32x8),
        ("n_latent", C.c_int32), ("latent_dims", _I32x8),
        ("n_edge", C.c_int32), ("edge_dims", _I32x8),
        ("avg_num_neighbors", C.c_double),
        ("resid_alpha", _F64x8),
        ("precision", C.c_int32),
        ("max_atoms", C.c_int64), ("max_edges", C.c_int64),
    ]


def hparams_from(hp, precision: int = 0) -> Hparams:
    """Build the C struct from any object with the attribute names of synthetic.configs.Hparams."""
    h = Hparams()
    h.n_species, h.l_max, h.n_layers, h.n_tensor = hp.n_species, hp.l_max, hp.n_layers, hp.n_tensor
    h.n_bessel, h.poly_p, h.r_cut = hp.n_bessel, hp.poly_p, hp.r_cut
    h.n_twobody = len(hp.twobody_dims)
    h.n_latent = len(hp.latent_dims)
    h.n_edge = len(hp.edge_dims)
    for k, v in enumerate(hp.twobody_dims):
        h.twobody_dims[k] = v
    for k, v in enumerate(hp.latent_dims):
        h.latent_dims[k] = v
    for k, v in enumerate(hp.edge_dims):
        h.edge_dims[k] = v
    h.avg_num_neighbors = hp.avg_num_neighbors
    for k, v in enumerate(hp.resid_alpha):
        h.resid_alpha[k] = v
    h.precision = precision
    h.max_atoms = 0
    h.max_edges = 0
    return h


class AllegroError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libb200allegro error {code}: {msg}")
        self.code = code


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)
_lib = None

EXPORTS = [
    "allegro_blob_size", "allegro_path_info", "allegro_create", "allegro_destroy", "allegro_set_stream",
    "allegro_set_allocator", "allegro_set_chunk_edges", "allegro_neighbors", "allegro_neighbors_host",
    "allegro_nbr_info", "allegro_nbr_copy_host", "allegro_nbr_free", "allegro_compute", "allegro_compute_host",
    "allegro_step_nve", "allegro_step_nve_host", "allegro_profile_enable", "allegro_profile_read",
    "allegro_launch_count", "allegro_last_active_edges", "allegro_set_debug", "allegro_set_pair_cutoffs", "allegro_debug_tensor",
    "allegro_set_bessel_frequencies", "allegro_set_zbl", "allegro_edge_energies", "allegro_step_nvt", "allegro_graph_steps", "allegro_compute_local",
    "allegro_nve_kick", "allegro_kinetic_energy", "allegro_kinetic_energy_noalloc", "allegro_status", "allegro_probe_ffma", "allegro_probe_tf32", "allegro_halo_pack", "allegro_halo_assemble", "allegro_halo_accumulate", "allegro_set_tensor_track", "allegro_set_gemm_pairs",
    "allegro_last_error",
]


def load_library(path: Optional[str] = None) -> C.CDLL:
    """dlopen the in-tree libb200allegro.so.  Raises (never falls back) if it is missing."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or lib_path()
    if not os.path.exists(p):
        raise FileNotFoundError(
            f"{p} not found: run `python -m paper_2304_10061_b200.build` (or __graft_entry__.build()). "
            "There is no CPU fallback for the Allegro hot path.")
    lib = C.CDLL(p)
    vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int32
    P = C.POINTER
    lib.allegro_blob_size.argtypes = [P(Hparams), P(C.c_size_t)]
    lib.allegro_path_info.argtypes = [P(Hparams), i32, P(i32), P(i32), P(i32)]
    lib.allegro_create.argtypes = [P(Hparams), vp, C.c_size_t, P(vp)]
    lib.allegro_destroy.argtypes = [vp]
    lib.allegro_set_stream.argtypes = [vp, vp]
    lib.allegro_set_allocator.argtypes = [vp, _ALLOC_FN, _FREE_FN, vp]
    lib.allegro_set_chunk_edges.argtypes = [vp, i64]
    lib.allegro_set_debug.argtypes = [vp, C.c_int]
    lib.allegro_set_pair_cutoffs.argtypes = [vp, vp]
    lib.allegro_neighbors.argtypes = [vp, vp, i64, P(C.c_double), C.c_double, P(vp)]
    lib.allegro_neighbors_host.argtypes = [vp, vp, i64, P(C.c_double), C.c_double, P(vp)]
    lib.allegro_nbr_info.argtypes = [vp, P(i64), P(i64), P(vp), P(vp), P(vp)]
    lib.allegro_nbr_copy_host.argtypes = [vp, vp, vp, vp, vp]
    lib.allegro_nbr_free.argtypes = [vp, vp]
    lib.allegro_compute.argtypes = [vp, vp, vp, i64, P(C.c_double), vp, vp, vp, vp]
    lib.allegro_compute_host.argtypes = [vp, vp, vp, i64, P(C.c_double), vp, vp, vp, vp]
    lib.allegro_step_nve.argtypes = [vp, vp, vp, vp, vp, vp, i64, P(C.c_double), C.c_double, i32, C.c_double, P(vp),
                                     P(i64), vp, vp]
    lib.allegro_step_nve_host.argtypes = lib.allegro_step_nve.argtypes
    lib.allegro_step_nvt.argtypes = lib.allegro_step_nve.argtypes + [vp, C.c_double, C.c_double]
    lib.allegro_nve_kick.argtypes = [vp, vp, vp, vp, vp, vp, i64, C.c_double, i32]
    lib.allegro_kinetic_energy.argtypes = [vp, vp, vp, vp, i64, vp]
    lib.allegro_kinetic_energy_noalloc.argtypes = [vp, vp, vp, vp, i64, vp]
    lib.allegro_compute_local.argtypes = [vp, vp, vp, i64, i64, P(C.c_double), vp, vp, vp, vp]
    lib.allegro_edge_energies.argtypes = [vp, vp, vp, i64, P(C.c_double), vp, vp, vp]
    lib.allegro_set_bessel_frequencies.argtypes = [vp, vp]
    lib.allegro_set_zbl.argtypes = [vp, vp]
    lib.allegro_profile_enable.argtypes = [vp, i32]
    lib.allegro_profile_read.argtypes = [vp, C.c_char_p, P(C.c_double), P(i64)]
    lib.allegro_launch_count.argtypes = [vp, P(i64)]
    lib.allegro_graph_steps.argtypes = [vp, P(i64)]
    lib.allegro_last_active_edges.argtypes = [vp, P(i64)]
    lib.allegro_debug_tensor.argtypes = [vp, C.c_char_p, vp, P(i64)]
    lib.allegro_status.argtypes = [vp]
    lib.allegro_set_tensor_track.argtypes = [vp, i32]
    lib.allegro_set_gemm_pairs.argtypes = [vp, i32]
    lib.allegro_halo_pack.argtypes = [vp, vp, vp, vp, vp, i64, vp]
    lib.allegro_halo_assemble.argtypes = [vp, vp, vp, i64, vp, i64, P(C.c_double), vp, vp]
    lib.allegro_halo_accumulate.argtypes = [vp, vp, i64, vp, vp, i64, vp]
    lib.allegro_probe_ffma.argtypes = [vp, C.c_double, P(C.c_double), P(C.c_double)]
    lib.allegro_probe_tf32.argtypes = [vp, C.c_double, P(C.c_double), P(C.c_double)]
    lib.allegro_last_error.argtypes = [vp]
    lib.allegro_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name != "allegro_last_error":
            getattr(lib, name).restype = C.c_int
    if path is None:
        _lib = lib
    return lib


def _box3(box) -> C.Array:
    return (C.c_double * 3)(float(box[0]), float(box[1]), float(box[2]))


def path_fan(hp: Hparams):
    """Per layer, per path (canonical order): number of paths sharing the path's output irrep
    (`allegro_path_info`).  Used by the synthetic blob writer for the alpha scale."""
    lib = load_library()
    out = []
    for L in range(1, hp.n_layers + 1):
        n = C.c_int32(0)
        rc = lib.allegro_path_info(C.byref(hp), L, C.byref(n), None, None)
        if rc:
            raise AllegroError(rc, lib.allegro_last_error(None).decode())
        fan = (C.c_int32 * n.value)()
        lib.allegro_path_info(C.byref(hp), L, C.byref(n), fan, None)
        out.append(list(fan))
    return out


def layer_dims(hp: Hparams):
    lib = load_library()
    dims = []
    for L in range(1, hp.n_layers + 1):
        n = C.c_int32(0)
        dd = (C.c_int32 * 2)()
        rc = lib.allegro_path_info(C.byref(hp), L, C.byref(n), None, dd)
        if rc:
            raise AllegroError(rc, lib.allegro_last_error(None).decode())
        if L == 1:
            dims.append(dd[0])
        dims.append(dd[1])
    return dims


class NeighborList:
    """Opaque handle to a device CSR list (allegro_nbr)."""

    def __init__(self, model: "Allegro"):
        self._model = model
        self._h = C.c_void_p(None)

    @property
    def n_edges(self) -> int:
        ne = C.c_int64(0)
        self._model._lib.allegro_nbr_info(self._h, None, C.byref(ne), None, None, None)
        return ne.value

    def to_host(self):
        """(row_ptr int64[N+1], j int32[E], shift int8[E,3]) as numpy arrays."""
        import numpy as np
        na, ne = C.c_int64(0), C.c_int64(0)
        self._model._lib.allegro_nbr_info(self._h, C.byref(na), C.byref(ne), None, None, None)
        rp = np.empty(na.value + 1, dtype=np.int64)
        j = np.empty(ne.value, dtype=np.int32)
        s = np.empty((ne.value, 3), dtype=np.int8)
        self._model._check(self._model._lib.allegro_nbr_copy_host(
            self._model._h, self._h, rp.ctypes.data, j.ctypes.data, s.ctypes.data))
        return rp, j, s

    def free(self):
        # the list's buffers came from the model's allocator: free only while the model is alive (allegro_destroy does
        # not own lists; a list that outlives its model is abandoned to the allocator's own teardown)
        if self._h and self._model._h:
            self._model._lib.allegro_nbr_free(self._model._h, self._h)
        self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Allegro:
    """allegro_model handle.  Tensors are torch CUDA tensors (float64 positions/forces, int32 species)."""

    def __init__(self, hp: Hparams, blob: bytes, use_torch_allocator: bool = True, chunk_edges: Optional[int] = None):
        import torch
        if not torch.cuda.is_available():
            raise AllegroError(-6, "no CUDA device: the Allegro hot path has no CPU fallback")
        self._torch = torch
        self._lib = load_library()
        self.hp = hp
        self._h = C.c_void_p(None)
        buf = C.create_string_buffer(blob, len(blob))
        rc = self._lib.allegro_create(C.byref(hp), buf, len(blob), C.byref(self._h))
        if rc:
            raise AllegroError(rc, self._lib.allegro_last_error(None).decode())
        self._keep = []
        if use_torch_allocator:
            dev = torch.cuda.current_device()

            alloc_fn, delete_fn, stream_fn = (torch.cuda.caching_allocator_alloc, torch.cuda.caching_allocator_delete,
                                              torch.cuda.current_stream)

            def _alloc(nbytes, _user):
                return alloc_fn(int(nbytes), dev, stream_fn(dev))

            def _free(ptr, _user):
                # bound at creation: at interpreter shutdown the torch.cuda module attributes may already be gone
                try:
                    delete_fn(ptr)
                except Exception:
                    pass

            a, f = _ALLOC_FN(_alloc), _FREE_FN(_free)
            self._keep += [a, f]
            self._check(self._lib.allegro_set_allocator(self._h, a, f, None))
        if chunk_edges:
            self._check(self._lib.allegro_set_chunk_edges(self._h, int(chunk_edges)))
        self._sync_stream()

    # -- plumbing ---------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc:
            raise AllegroError(rc, self._lib.allegro_last_error(self._h).decode())

    def _sync_stream(self):
        s = self._torch.cuda.current_stream().cuda_stream
        self._lib.allegro_set_stream(self._h, C.c_void_p(s))

    def close(self):
        if self._h:
            self._lib.allegro_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launches(self) -> int:
        v = C.c_int64(0)
        self._lib.allegro_launch_count(self._h, C.byref(v))
        return v.value

    @property
    def graph_steps(self) -> int:
        """Number of MD steps served by a CUDA-graph launch so far (-1: capture failed and was switched off)."""
        v = C.c_int64(0)
        self._check(self._lib.allegro_graph_steps(self._h, C.byref(v)))
        return v.value

    def set_tensor_track(self, mode: int) -> None:
        """allegro_set_tensor_track: 0 contracted per centre (default), 1 per-edge products (before the first compute)."""
        self._check(self._lib.allegro_set_tensor_track(self._h, int(mode)))

    def status(self) -> None:
        """allegro_status: synchronise the model's stream and raise what the device-pointer calls since the last check
        flagged (coincident atoms -> ALLEGRO_ERR_NONFINITE, species out of range -> ALLEGRO_ERR_BAD_ARG)."""
        self._check(self._lib.allegro_status(self._h))

    def probe_peaks(self, sustain_s: float = 2.0) -> dict:
        """allegro_probe_ffma / allegro_probe_tf32 -> TFLOP/s, burst and sustained (roofline denominators of bench.py)."""
        self._sync_stream()
        out = {}
        for name, fn in (("ffma", self._lib.allegro_probe_ffma), ("tf32_mma", self._lib.allegro_probe_tf32)):
            b, s = C.c_double(0), C.c_double(0)
            self._check(fn(self._h, float(sustain_s), C.byref(b), C.byref(s)))
            out[name] = {"burst": b.value, "sustained": s.value}
        return out

    # -- NEXT-3 halo kernels (domain.py) ------------------------------------------------------------------
    def halo_pack(self, pos, species, idx, shift):
        """allegro_halo_pack -> f64[n_send, 4] rows [x, y, z, species] of the ghosts this rank provides."""
        t = self._torch
        self._sync_stream()
        k = int(idx.shape[0])
        out = t.empty((k, 4), dtype=t.float64, device=pos.device)
        self._check(self._lib.allegro_halo_pack(self._h, pos.data_ptr(), species.data_ptr(), idx.data_ptr(), shift.data_ptr(), k,
                                                out.data_ptr()))
        return out

    def halo_assemble(self, pos, species, ghost_rows, origin):
        """allegro_halo_assemble -> (pos_all f64[n_local + n_ghost, 3] in the local frame, species_all int32)."""
        t = self._torch
        self._sync_stream()
        nl, ng = int(pos.shape[0]), int(ghost_rows.shape[0])
        pos_all = t.empty((nl + ng, 3), dtype=t.float64, device=pos.device)
        sp_all = t.empty(nl + ng, dtype=t.int32, device=pos.device)
        self._check(self._lib.allegro_halo_assemble(self._h, pos.data_ptr(), species.data_ptr(), nl, ghost_rows.data_ptr(), ng,
                                                    _box3(origin), pos_all.data_ptr(), sp_all.data_ptr()))
        return pos_all, sp_all

    def halo_accumulate(self, force_all, n_local, idx, returned):
        """allegro_halo_accumulate -> f64[n_local, 3]: local forces + what came back for the ghosts this rank provided."""
        t = self._torch
        self._sync_stream()
        out = t.empty((n_local, 3), dtype=t.float64, device=force_all.device)
        self._check(self._lib.allegro_halo_accumulate(self._h, force_all.data_ptr(), int(n_local), idx.data_ptr(), returned.data_ptr(),
                                                      int(idx.shape[0]), out.data_ptr()))
        return out

    def last_active_edges(self) -> int:
        v = C.c_int64(0)
        self._check(self._lib.allegro_last_active_edges(self._h, C.byref(v)))
        return v.value

    # -- the four calls of the boundary -----------------------------------------------------------
    def neighbors(self, pos, box: Sequence[float], cutoff: float, reuse: Optional[NeighborList] = None) -> NeighborList:
        """allegro_neighbors: pos = CUDA float64 [N,3]."""
        assert pos.is_cuda and pos.dtype == self._torch.float64 and pos.is_contiguous()
        self._sync_stream()
        nb = reuse or NeighborList(self)
        self._check(self._lib.allegro_neighbors(self._h, pos.data_ptr(), pos.shape[0], _box3(box), float(cutoff),
                                                C.byref(nb._h)))
        return nb

    def compute(self, pos, species, box: Sequence[float], nbr: NeighborList, want_atom_energies: bool = True,
                want_forces: bool = True):
        """allegro_compute -> (e_total f64[1], e_atom f64[N] | None, force f64[N,3] | None) CUDA tensors.
        want_forces=False: energy-only evaluation (no backward pass)."""
        t = self._torch
        assert pos.is_cuda and pos.dtype == t.float64 and pos.is_contiguous()
        assert species.is_cuda and species.dtype == t.int32 and species.is_contiguous()
        self._sync_stream()
        N = pos.shape[0]
        e = t.empty(1, dtype=t.float64, device=pos.device)
        ea = t.empty(N, dtype=t.float64, device=pos.device) if want_atom_energies else None
        f = t.empty((N, 3), dtype=t.float64, device=pos.device) if want_forces else None
        self._check(self._lib.allegro_compute(self._h, pos.data_ptr(), species.data_ptr(), N, _box3(box), nbr._h,
                                              e.data_ptr(), ea.data_ptr() if ea is not None else None,
                                              f.data_ptr() if f is not None else None))
        return e, ea, f

    def compute_local(self, pos, species, n_local: int, box: Sequence[float], nbr: NeighborList):
        """allegro_compute_local: atoms [0, n_local) are centres, the rest ghosts -> (e_total, e_atom, force) CUDA."""
        t = self._torch
        assert pos.is_cuda and pos.dtype == t.float64 and pos.is_contiguous()
        assert species.is_cuda and species.dtype == t.int32 and species.is_contiguous()
        self._sync_stream()
        N = pos.shape[0]
        e = t.empty(1, dtype=t.float64, device=pos.device)
        ea = t.empty(N, dtype=t.float64, device=pos.device)
        f = t.empty((N, 3), dtype=t.float64, device=pos.device)
        self._check(self._lib.allegro_compute_local(self._h, pos.data_ptr(), species.data_ptr(), N, int(n_local), _box3(box),
                                                    nbr._h, e.data_ptr(), ea.data_ptr(), f.data_ptr()))
        return e, ea, f

    def edge_energies(self, pos, species, box: Sequence[float], nbr: NeighborList):
        """allegro_edge_energies -> (e_total f64[1], e_edge f64[nbr.n_edges]) CUDA tensors, list order."""
        t = self._torch
        assert pos.is_cuda and pos.dtype == t.float64 and pos.is_contiguous()
        assert species.is_cuda and species.dtype == t.int32 and species.is_contiguous()
        self._sync_stream()
        e = t.empty(1, dtype=t.float64, device=pos.device)
        ee = t.zeros(max(nbr.n_edges, 1), dtype=t.float64, device=pos.device)
        self._check(self._lib.allegro_edge_energies(self._h, pos.data_ptr(), species.data_ptr(), pos.shape[0], _box3(box),
                                                    nbr._h, e.data_ptr(), ee.data_ptr()))
        return e, ee[:nbr.n_edges]

    def compute_into(self, pos, species, box3, nbr: NeighborList, e, ea, f):
        """allegro_compute into preallocated tensors (no allocation: bench inner loop)."""
        self._check(self._lib.allegro_compute(self._h, pos.data_ptr(), species.data_ptr(), pos.shape[0], box3, nbr._h,
                                              e.data_ptr(), ea.data_ptr() if ea is not None else None, f.data_ptr()))

    def neighbors_host(self, pos_np, box, cutoff, reuse: Optional[NeighborList] = None) -> NeighborList:
        import numpy as np
        pos_np = np.ascontiguousarray(pos_np, dtype=np.float64)
        self._sync_stream()
        nb = reuse or NeighborList(self)
        self._check(self._lib.allegro_neighbors_host(self._h, pos_np.ctypes.data, pos_np.shape[0], _box3(box),
                                                     float(cutoff), C.byref(nb._h)))
        return nb

    def compute_host(self, pos_np, species_np, box, nbr: NeighborList):
        """allegro_compute_host: numpy in, numpy out; H2D/D2H copies happen inside the library."""
        import numpy as np
        pos_np = np.ascontiguousarray(pos_np, dtype=np.float64)
        species_np = np.ascontiguousarray(species_np, dtype=np.int32)
        N = pos_np.shape[0]
        e = np.zeros(1)
        ea = np.zeros(N)
        f = np.zeros((N, 3))
        self._sync_stream()
        self._check(self._lib.allegro_compute_host(self._h, pos_np.ctypes.data, species_np.ctypes.data, N, _box3(box),
                                                   nbr._h, e.ctypes.data, ea.ctypes.data, f.ctypes.data))
        return float(e[0]), ea, f

    def step_nve(self, pos, vel, force, species, mass, box, dt_fs: float, rebuild_every: int, skin: float,
                 nbr: NeighborList, step_counter: C.c_int64, e_pot, e_kin):
        """allegro_step_nve; pos/vel/force updated in place; nbr rebuilt when due."""
        self._check(self._lib.allegro_step_nve(self._h, pos.data_ptr(), vel.data_ptr(), force.data_ptr(),
                                               species.data_ptr(), mass.data_ptr(), pos.shape[0], _box3(box),
                                               float(dt_fs), int(rebuild_every), float(skin), C.byref(nbr._h),
                                               C.byref(step_counter), e_pot.data_ptr(), e_kin.data_ptr()))

    def nve_kick(self, pos, vel, force, species, mass, dt_fs: float, drift: bool):
        """allegro_nve_kick: half kick (and drift) in place on CUDA tensors."""
        self._sync_stream()
        self._check(self._lib.allegro_nve_kick(self._h, pos.data_ptr(), vel.data_ptr(), force.data_ptr(), species.data_ptr(),
                                               mass.data_ptr(), vel.shape[0], float(dt_fs), 1 if drift else 0))

    def kinetic_energy(self, vel, species, mass):
        """allegro_kinetic_energy -> CUDA float64 [1] (eV)."""
        self._sync_stream()
        ek = self._torch.empty(1, dtype=self._torch.float64, device=vel.device)
        self._check(self._lib.allegro_kinetic_energy(self._h, vel.data_ptr(), species.data_ptr(), mass.data_ptr(),
                                                     vel.shape[0], ek.data_ptr()))
        return ek

    def kinetic_energy_noalloc(self, vel, species, mass, out):
        """allegro_kinetic_energy_noalloc: writes e_kin (eV) into `out` (CUDA float64 [1], the caller's); allocates nothing."""
        self._sync_stream()
        self._check(self._lib.allegro_kinetic_energy_noalloc(self._h, vel.data_ptr(), species.data_ptr(), mass.data_ptr(),
                                                             vel.shape[0], out.data_ptr()))
        return out

    def step_nvt(self, pos, vel, force, species, mass, box, dt_fs: float, rebuild_every: int, skin: float,
                 nbr: NeighborList, step_counter: C.c_int64, e_pot, e_kin, nh_state, t0_K: float, tau_fs: float):
        """allegro_step_nvt (Nose-Hoover); nh_state = CUDA float64 [2] = {xi, eta}, updated in place."""
        assert nh_state.is_cuda and nh_state.dtype == self._torch.float64 and nh_state.numel() == 2
        self._check(self._lib.allegro_step_nvt(self._h, pos.data_ptr(), vel.data_ptr(), force.data_ptr(),
                                               species.data_ptr(), mass.data_ptr(), pos.shape[0], _box3(box),
                                               float(dt_fs), int(rebuild_every), float(skin), C.byref(nbr._h),
                                               C.byref(step_counter), e_pot.data_ptr(), e_kin.data_ptr(),
                                               nh_state.data_ptr(), float(t0_K), float(tau_fs)))

    def step_nve_host(self, pos, vel, force, species, mass, box, dt_fs, rebuild_every, skin, nbr, step_counter,
                      e_pot, e_kin):
        """allegro_step_nve_host: all arrays are HOST buffers (numpy arrays or pinned CPU torch tensors)."""
        ptr = lambda a: a.ctypes.data if hasattr(a, "ctypes") else a.data_ptr()
        self._check(self._lib.allegro_step_nve_host(self._h, ptr(pos), ptr(vel), ptr(force), ptr(species), ptr(mass),
                                                    pos.shape[0], _box3(box), float(dt_fs), int(rebuild_every),
                                                    float(skin), C.byref(nbr._h), C.byref(step_counter), ptr(e_pot),
                                                    ptr(e_kin)))

    def set_gemm_pairs(self, pairs: bool):
        """allegro_set_gemm_pairs: MLP GEMMs on CTA pairs (256-row tiles, the default for large launches) or on single CTAs."""
        self._check(self._lib.allegro_set_gemm_pairs(self._h, 1 if pairs else 0))

    def profile_enable(self, on, nvtx: bool = False):
        """allegro_profile_enable: CUDA-event timing per kernel group (`on`) and / or NVTX ranges per group (`nvtx`)."""
        self._check(self._lib.allegro_profile_enable(self._h, (1 if on else 0) | (2 if nvtx else 0)))

    def profile_read(self, name: str):
        ms, n = C.c_double(0), C.c_int64(0)
        self._check(self._lib.allegro_profile_read(self._h, name.encode(), C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def set_pair_cutoffs(self, rc_pair):
        """Ordered species-pair cutoffs rc_pair[Z_centre][Z_neighbour]; None = flat r_cut."""
        import numpy as np
        if rc_pair is None:
            self._check(self._lib.allegro_set_pair_cutoffs(self._h, None))
            return
        a = np.ascontiguousarray(rc_pair, dtype=np.float64)
        assert a.shape == (self.hp.n_species, self.hp.n_species)
        self._check(self._lib.allegro_set_pair_cutoffs(self._h, a.ctypes.data))

    def set_bessel_frequencies(self, freq):
        """Trained Bessel angular frequencies freq[Z_centre][Z_neighbour][n] in 1/A; None = n pi / r_c."""
        import numpy as np
        if freq is None:
            self._check(self._lib.allegro_set_bessel_frequencies(self._h, None))
            return
        a = np.ascontiguousarray(freq, dtype=np.float64)
        assert a.shape == (self.hp.n_species, self.hp.n_species, self.hp.n_bessel)
        self._check(self._lib.allegro_set_bessel_frequencies(self._h, a.ctypes.data))

    def set_zbl(self, atomic_numbers):
        """ZBL pair repulsion with these atomic numbers per species; None = off."""
        import numpy as np
        if atomic_numbers is None:
            self._check(self._lib.allegro_set_zbl(self._h, None))
            return
        a = np.ascontiguousarray(atomic_numbers, dtype=np.float64)
        assert a.shape == (self.hp.n_species,)
        self._check(self._lib.allegro_set_zbl(self._h, a.ctypes.data))

    def set_debug(self, on: bool = True):
        """Keep every tensor debug_tensor() can name (tests only)."""
        self._check(self._lib.allegro_set_debug(self._h, 1 if on else 0))

    def debug_tensor(self, name: str, max_floats: int = 1 << 26):
        import numpy as np
        out = np.empty(max_floats, dtype=np.float32)
        n = C.c_int64(max_floats)
        self._check(self._lib.allegro_debug_tensor(self._h, name.encode(), out.ctypes.data, C.byref(n)))
        return out[:n.value].copy()
