#!/usr/bin/env python
"""bench.py — atom-steps/s of the Allegro energy+force hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path: one velocity-Verlet NVE step
through the C ABI (`allegro_step_nve`): half-kick + drift, neighbor rebuild when due (every
`rebuild_every` steps at r_c + skin), active-edge compaction + edge basis, two-body MLP, Allegro layers,
edge energies, fp64 sums, analytic backward, force scatter, half-kick, kinetic energy.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--precision 1] [--impl ours|reference]

Default workload = config 3 (1,000,000 atoms, the largest single-GPU config of BASELINE.json); --config 0..4 selects the others.

N > 1: launched by torchrun, one rank per GPU.  The path does not shard in this build (north_star: one
GPU, no collectives) -> "replicas only": every rank runs an independent replica of the same workload;
value = sum of atom-steps over ranks / max-over-ranks device time.
"""
from __future__ import annotations

import argparse
import ctypes
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

FFMA_LANES_PER_SM = 128          # B200_PROFILING.md / blackwell guide: 4 SMSP x 32 fp32 FMA lanes
TF32_OVER_BF16 = 0.5             # nominal dense ratio (B200_PROFILING.md table: 1.1 vs 2.25 PFLOP/s); fallback only


def gemm_alg_bytes_per_edge(hp):
    """ALGORITHMIC HBM bytes per active edge of the MLP group: "minimum bytes if only layer-boundary
    tensors touch HBM: x^0 .. x^NL written once + read for the backward" = (NL + 1) * d * 4 B * 2."""
    return 8.0 * (hp.n_layers + 1) * hp.twobody_dims[-1]


def gemm_macs_per_edge(hp):
    """Algorithmic MACs per ACTIVE edge of the GEMM kernel group, forward + backward (dX only)."""
    d, n, nA = hp.twobody_dims[-1], hp.n_tensor, hp.n_tensor * (hp.l_max + 1)
    tb = sum(a * b for a, b in zip(hp.twobody_dims[:-1], hp.twobody_dims[1:]))
    lat = (d + n) * hp.latent_dims[0] + sum(a * b for a, b in zip(hp.latent_dims[:-1], hp.latent_dims[1:]))
    fwd = tb + d * 2 * nA + hp.n_layers * lat + (hp.n_layers - 1) * d * nA
    bwd = tb + hp.n_layers * lat + 2 * nA * d + (hp.n_layers - 1) * nA * d
    return fwd + bwd


def gemm_impl_bytes_per_edge(hp, kcat=True):
    """IMPLEMENTATION HBM bytes per ACTIVE edge of the GEMM kernel group (fp32 storage) -- what this build's own launch
    list moves, NOT the algorithmic minimum (gemm_alg_bytes_per_edge): every launch reads its A
    operand once and writes its outputs once; aux operands of the fused epilogues are read once.  Weights are
    L2-resident and not counted.  Mirrors the launch list of csrc/compute.cu::run_chunk (default path: last latent
    layer fused with the energy / z-bar epilogue, z-bar prep stage fused into the x-bar GEMMs, and -- kcat, the tensor-core
    modes -- the x-bar part of the first latent layer's dX folded into the x-bar GEMM by K-concatenation)."""
    d, n, nA, NL = hp.twobody_dims[-1], hp.n_tensor, hp.n_tensor * (hp.l_max + 1), hp.n_layers
    tb, lat = list(hp.twobody_dims), list(hp.latent_dims)
    parts = 12.0 * ((d + 31) // 32) / 4.0             # fp64 energy + fp32 u-bar partial per 32 columns, in floats
    fl = 0.0
    for k in range(1, len(tb)):                       # two-body forward: A, C (activation), out2 (pre-activation)
        fl += tb[k - 1] + 2 * tb[k]
    fl += d + 2 * nA                                  # [w0 | omega1]
    for L in range(1, NL + 1):
        for k in range(len(lat)):
            K = d + n if k == 0 else lat[k - 1]
            last = k == len(lat) - 1
            if last and L == NL:
                fl += K + lat[k] + d + parts          # A, z-bar out, residual x^{L-1} read, row partials (x^{NL} not stored)
            else:
                fl += K + 2 * lat[k] + (d if last else 0)
        if L < NL:
            fl += d + nA
    for L in range(NL, 0, -1):                        # backward
        for k in range(len(lat) - 1, 0, -1):
            fl += lat[k] + 2 * lat[k - 1]             # A, aux z, C
        Kx = 2 * nA if L == 1 else nA
        if kcat:
            # s-bar GEMM: A = z-bar, C = s-bar only; then ONE x-bar GEMM over the concatenated K axis [z-bar | omega-bar]
            # (+ prep stage): A, aux1 unless rank-1, z of the MLP below, z-bar out, u-bar partials, C = x-bar (not for L = 1)
            fl += lat[0] + n
            fl += (lat[0] + Kx) + (0 if L == NL else d) + d + d + parts / 3.0 + (d if L > 1 else 0)
        else:
            fl += lat[0] + (d + n)                    # dX of the first latent layer -> [x-bar part | s-bar]
            # x-bar GEMM + prep stage: A, aux2 (+ aux1 unless rank-1), z of the MLP below, z-bar out, u-bar partials,
            # C = x-bar (not stored for L = 1)
            fl += Kx + d + (0 if L == NL else d) + d + d + parts / 3.0 + (d if L > 1 else 0)
    for k in range(len(tb) - 1, 0, -1):
        fl += tb[k] + 2 * tb[k - 1]
    return 4.0 * fl


def tp_bytes_per_edge(hp):
    """HBM bytes per ACTIVE edge the tensor-track kernels have to move (fp32 storage; Y rows and per-centre quantities not
    counted).  Default kernels (tensor track contracted per centre, csrc/tpc_impl.cuh): only the per-edge scalars-by-l and
    scalar blocks exist -- forward, per layer: omega^L (nl n) + w0 (nl n) read, s^L (n) written; backward, per layer:
    s-bar^L (n) + w0 (nl n) read, omega^L (nl n) read, omega-bar^L (nl n) written; layer 1 also reads the other layers'
    s-bar and writes w0-bar (nl n).  SURVEY.md section 8(d)'s figure for the per-edge product formulation (V read + T write,
    2,304 + 2,304 B at config 2 layer 1) is what these kernels no longer move; it is reported as `survey_bytes_per_edge`."""
    n, nl, NL = hp.n_tensor, hp.l_max + 1, hp.n_layers
    fwd = NL * n * (2 * nl + 1)
    bwd = NL * n * (1 + 3 * nl) + n * ((NL - 1) + nl)
    return {"tp_fwd": 4.0 * fwd, "tp_bwd": 4.0 * bwd}


def tp_survey_bytes_per_edge(hp):
    """SURVEY.md section 8(d) figure for the tensor product as a per-edge product (V^{L-1} read + T^L written per layer, forward;
    omega, V, V-bar, s-bar in and V-bar, omega-bar out, backward): what the round-1 kernels moved."""
    n, nl = hp.n_tensor, hp.l_max + 1
    D = {(1, 1): [4, 1], (2, 2): [9, 9, 1], (3, 3): [16, 31, 16, 1]}.get((hp.l_max, hp.n_layers))
    if D is None:
        return {"tp_fwd": 0.0, "tp_bwd": 0.0}
    fwd = bwd = 0.0
    for L in range(1, hp.n_layers + 1):
        din, dout = D[L - 1], D[L]
        vin = nl if L == 1 else din
        tout = dout if L < hp.n_layers else 0
        fwd += n * (nl + vin + tout + 1)
        bwd += n * (nl + vin + tout + 1 + vin + nl)
    return {"tp_fwd": 4.0 * fwd, "tp_bwd": 4.0 * bwd}


DTYPE = {0: "f32 (3xtf32)", 1: "tf32", 2: "bf16 operands (fp32 accumulate)", 3: "f32", 4: "fp16 operands (fp32 accumulate)"}


def tp_flops_per_edge(hp):
    """Algorithmic flops per ACTIVE edge of the tensor product: forward 3 nnz n per layer (K^L applied as
    listed, 2 multiplies + 1 add per non-zero and channel), backward twice that (V-bar and Gamma-bar)."""
    nnz = {(1, 1): [4], (2, 2): [83, 9], (3, 3): [611, 611, 16]}.get((hp.l_max, hp.n_layers))
    if nnz is None:
        return {"tp_fwd": 0.0, "tp_bwd": 0.0}
    f = 3.0 * sum(nnz) * hp.n_tensor
    return {"tp_fwd": f, "tp_bwd": 2.0 * f}


def tf32_matmul_peak(dev, n=8192, sustain_s=4.0):
    """MEASURED_PEAKS.json's procedure with TF32 allowed: torch.matmul fp32 n^3 (cuBLAS TF32 tensor cores), best of 10
    (burst) and back to back for `sustain_s` seconds (sustained).  A library call used as a yardstick only."""
    import torch
    old = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = True
    try:
        a = torch.randn(n, n, device=dev); b = torch.randn(n, n, device=dev); c = torch.empty(n, n, device=dev)
        for _ in range(3):
            torch.matmul(a, b, out=c)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        best = 1e30
        for _ in range(10):
            e0.record(); torch.matmul(a, b, out=c); e1.record(); torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        reps = int(sustain_s * 1e3 / best) + 1
        e0.record()
        for _ in range(reps):
            torch.matmul(a, b, out=c)
        e1.record(); torch.cuda.synchronize()
        fl = 2.0 * n ** 3
        return {"burst": fl / (best * 1e-3) / 1e12, "sustained": fl * reps / (e0.elapsed_time(e1) * 1e-3) / 1e12}
    finally:
        torch.backends.cuda.matmul.allow_tf32 = old


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        super().__init__(daemon=True)
        self.gpu, self.samples, self.stop_flag = gpu_index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.samples.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(s[0]) for s in self.samples)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(s[2 + k].lower().startswith("active") for s in self.samples)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.samples[0][1]), "reasons": reasons,
                "samples": len(sm)}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return {"hbm_gbs": j["hbm_gbs"], "bf16_burst": j["bf16_tflops"], "bf16_sustained": j["bf16_tflops_sustained"],
                "sm_max_mhz": j.get("sm_max_mhz", 1965.0), "src": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "sm_max_mhz": 1965.0, "src": "fallback"}


def aggregate_over_ranks(ms_local, atoms_local, steps, dist=None, device="cpu"):
    """Whole-job throughput for N independent replicas ("replicas only"): units summed over ranks divided by
    the MAX over ranks of the device time.  Returns (atom-steps/s, max ms)."""
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    a = torch.tensor([float(atoms_local)], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(a, op=dist.ReduceOp.SUM)
    return float(a.item()) * steps / (float(t.item()) * 1e-3), float(t.item())


def oracle_sample(cfg, pos, sp, box, n_centers):
    """Energy + forces of `n_centers` contiguous centres by the fp64 oracle (cpu_baseline / reference arm)."""
    import torch
    from oracle import allegro_oracle as O
    from synthetic import make_blob
    hp = cfg.hp
    blob = make_blob(hp, O.path_fan(hp.l_max, hp.n_layers), [cfg.sigma] * hp.n_species, cfg.mu(), cfg.weight_seed)
    om = O.OracleModel(hp, blob)
    nbr = O.neighbor_list(pos, box, hp.r_cut)
    centers = np.arange(min(n_centers, pos.shape[0]))

    def run():
        t0 = time.perf_counter()
        O.energy_forces(om, pos, sp, box, nbr, centers=centers)
        return time.perf_counter() - t0
    return run, centers.size, torch.get_num_threads()


def run_decomposed(args, cfg, model, p, v, s, mass, box, dist, dev, rank, world, local_rank, K, W, metric, unit, workload):
    """NEXT-3: the same NVE step with ONE system split over the ranks by spatial domains
    (paper_2304_10061_b200/domain.py): halo forward / reverse exchange over NCCL all_to_all_single, migration at every
    list rebuild, energy all-reduce.  Strong scaling: value = total atoms x steps / max-over-ranks time."""
    import torch
    from paper_2304_10061_b200.domain import Domain, DomainGrid, TorchComm, auto_grid
    N = p.shape[0]
    grid = auto_grid(world, box)
    dom = Domain(DomainGrid(box, grid), rank, cfg.hp.r_cut + cfg.skin, cfg.hp.r_cut, model=model)
    gid = dom.take_owned(p, s)
    vel = v[gid].contiguous()
    comm = TorchComm()
    e, f = dom.energy_forces(comm)
    f = f.contiguous()
    state = {"vel": vel, "f": f, "e": e, "k": 0}

    def step():
        rebuild = state["k"] % cfg.rebuild_every == 0
        state["e"], state["vel"], state["f"] = dom.nve_step(comm, state["vel"], state["f"], mass, cfg.dt_fs, rebuild)
        state["k"] += 1

    for _ in range(W):
        step()
    dist.barrier(); torch.cuda.synchronize()
    l0 = model.launches
    sampler = ClockSampler(local_rank); sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist.barrier(); torch.cuda.synchronize()
    ev0.record()
    for _ in range(K):
        step()
    ev1.record()
    dist.barrier(); torch.cuda.synchronize()
    sampler.stop_flag = True
    ms = ev0.elapsed_time(ev1)
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    cnt = torch.tensor([float(dom.pos.shape[0]), float(sum(dom.recv_counts))], dtype=torch.float64, device=dev)
    cmax = cnt.clone(); dist.all_reduce(cmax, op=dist.ReduceOp.MAX)
    dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    ek = model.kinetic_energy(state["vel"], dom.species, mass)
    dist.all_reduce(ek, op=dist.ReduceOp.SUM)
    if rank == 0:
        print(json.dumps({
            "metric": metric, "value": N * K / (ms_max * 1e-3), "unit": unit, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": DTYPE[args.precision], "data": "synthetic",
            "config": {"workload": workload, "n_atoms": N, "precision_mode": args.precision, "dt_fs": cfg.dt_fs,
                       "rebuild_every": cfg.rebuild_every, "skin": cfg.skin,
                       "parallelism": f"spatial decomposition {grid[0]}x{grid[1]}x{grid[2]}, halo {cfg.hp.r_cut + cfg.skin} A",
                       "local_atoms_max": int(cmax[0].item()), "ghost_atoms_max": int(cmax[1].item()),
                       "ghost_atoms_total": int(cnt[1].item())},
            "timesteps_per_s": K / (ms_max * 1e-3), "ns_per_day": K / (ms_max * 1e-3) * cfg.dt_fs * 0.0864,
            "e_pot": float(state["e"].item()), "e_kin": float(ek.item()),
            "gpu_launches": model.launches - l0, "clocks": sampler.summary()}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    # default = the contract line: config 3 (1 M atoms, the largest single-GPU config of BASELINE.json), 3 repeats of K steps
    # after W warm-up steps; the timed region is seconds long, so nvidia-smi clock samples are plentiful
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--repeats", type=int, default=3, help="timed repeats of K steps each; the median is reported")
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--precision", type=int, default=1, choices=[0, 1, 2, 3, 4],
                    help="0 fp32 (3xTF32 on tensor cores), 1 TF32 tensor cores (the paper's scheme, the contract line), 3 fp32 FFMA, "
                         "2 / 4 bf16 / fp16 operand storage for the MLPs (fp32 accumulate)")
    ap.add_argument("--no-peak-probe", action="store_true", help="skip the TF32 / FFMA peak measurements (~10 s)")
    ap.add_argument("--drift-steps", type=int, default=0,
                    help="also run this many NVE steps from the initial state and report the drift of E_pot + E_kin "
                         "(SURVEY.md section 8(d): config 1, 100 steps at 0.5 fs)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--gemm-pairs", type=int, default=1, choices=[0, 1],
                    help="MLP GEMMs on CTA pairs (tcgen05 cta_group::2, the default) or on single CTAs: allegro_set_gemm_pairs")
    ap.add_argument("--nvtx", action="store_true",
                    help="NVTX range per kernel group around the library's launches (for `ncu --nvtx --nvtx-include \"gemm/\"`)")
    ap.add_argument("--no-extra-modes", action="store_true",
                    help="skip the fp16-operand sub-record that the default (TF32, one GPU) run appends (~10 s)")
    ap.add_argument("--chunk-edges", type=int, default=0, help="override the per-chunk edge budget (0 = library default)")
    ap.add_argument("--decompose", action="store_true",
                    help="NEXT-3: ONE system split over the N GPUs by spatial domains with halo exchange (strong scaling) "
                         "instead of N replicas; at N = 1 the single domain exchanges its periodic images with itself")
    ap.add_argument("--pair-cutoffs", default="none", choices=["none", "water"],
                    help="ordered species-pair cutoffs (PAPER.md:172-182, :222); 'water' = the paper's H/O values, configs 0-1 only")
    args = ap.parse_args()
    K, W = args.steps, max(args.warmup, 3)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from synthetic import CONFIGS, make_blob, make_system, maxwell_boltzmann
    from synthetic.systems import masses_for
    cfg = CONFIGS[args.config]
    workload = f"config{cfg.index}:{cfg.name}"
    if args.pair_cutoffs == "water":
        import dataclasses
        from synthetic.configs import WATER_PAIR_CUTOFFS
        assert cfg.index in (0, 1), "the water pair cutoffs need the (H, O) species of configs 0-1"
        cfg = dataclasses.replace(cfg, hp=dataclasses.replace(cfg.hp, r_cut_pair=WATER_PAIR_CUTOFFS))
        workload += " + ordered species-pair cutoffs (H-H 3.0, H-O 1.25, O-H 3.0, O-O 4.0)"
    metric, unit = "atom-steps/s (energy+forces, 1 B200)", "atom-steps/s"

    # ---------------------------------------------------------------- reference arm = the oracle on host cores
    if args.impl == "reference":
        if rank != 0:
            return
        pos, sp, box = make_system(cfg)
        n_c = {0: 192, 1: 3072, 2: 512, 3: 512, 4: 256}[cfg.index]
        run, n_c, cores = oracle_sample(cfg, pos, sp, box, n_c)
        for _ in range(W):
            run()
        t = sum(run() for _ in range(K))
        val = n_c * K / t
        print(json.dumps({
            "impl": "reference", "metric": metric, "value": val, "unit": unit, "n_gpus": args.gpus, "steps": K,
            "warmup": W, "ms_per_step": 1e3 * t / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload, "n_atoms": int(pos.shape[0]), "sample": f"{n_c} contiguous centres per step"},
            "cpu_baseline": {"value": val, "unit": unit, "cores": cores, "kind": "oracle",
                             "sample": f"energy+forces of {n_c} centres (all their edges) of {workload}, per step"},
            "e2e": {"value": val, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return

    # ---------------------------------------------------------------- our arm
    import torch
    import paper_2304_10061_b200 as P
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: the hot path has no CPU fallback"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1 or args.decompose:
        import torch.distributed as dist
        if world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29577")
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", local_rank))
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    pos, sp, box = make_system(cfg)
    vel = maxwell_boltzmann(cfg, sp)
    N = pos.shape[0]
    chp = P.hparams_from(cfg.hp, args.precision)
    blob = make_blob(cfg.hp, P.path_fan(chp), [cfg.sigma] * cfg.hp.n_species, cfg.mu(), cfg.weight_seed)
    model = P.Allegro(chp, blob, chunk_edges=args.chunk_edges) if args.chunk_edges else P.Allegro(chp, blob)
    if cfg.hp.r_cut_pair is not None:
        model.set_pair_cutoffs(cfg.hp.r_cut_pair)
    if not args.gemm_pairs:
        model.set_gemm_pairs(False)
    if args.nvtx:
        model.profile_enable(False, nvtx=True)
    dev = torch.device("cuda", local_rank)
    p = torch.from_numpy(pos.copy()).to(dev); v = torch.from_numpy(vel.copy()).to(dev)
    s = torch.from_numpy(sp).to(dev); mass = torch.from_numpy(masses_for(cfg)).to(dev)
    if args.decompose:
        run_decomposed(args, cfg, model, p, v, s, mass, box, dist, dev, rank, world, local_rank, K, W, metric, unit, workload)
        dist.destroy_process_group()
        return
    nb = model.neighbors(p, box, cfg.hp.r_cut + cfg.skin)
    e, _, f = model.compute(p, s, box, nb, want_atom_energies=False)
    ek = torch.zeros(1, dtype=torch.float64, device=dev)
    ctr = ctypes.c_int64(0)

    drift = None
    if args.drift_steps > 0:
        # NVE energy conservation from the initial state (the paper's stability claim, needs trained weights; with
        # the seeded weights this checks that forces are the gradient of the energy the integrator sees)
        p0, v0, f0 = p.clone(), v.clone(), f.clone()
        c0 = ctypes.c_int64(0)
        ek0 = model.kinetic_energy(v0, s, mass)
        series = [float(e.item()) + float(ek0.item())]
        kin = [float(ek0.item())]
        for _ in range(args.drift_steps):
            model.step_nve(p0, v0, f0, s, mass, box, cfg.dt_fs, cfg.rebuild_every, cfg.skin, nb, c0, e, ek)
            series.append(float(e.item()) + float(ek.item())); kin.append(float(ek.item()))
        a = np.asarray(series)
        drift = {"steps": args.drift_steps, "dt_fs": cfg.dt_fs, "e_tot_first": a[0], "e_tot_last": a[-1],
                 "drift_per_atom_eV": (a[-1] - a[0]) / N, "max_dev_per_atom_eV": float(np.abs(a - a[0]).max()) / N,
                 "rms_fluct_per_atom_eV": float(a.std()) / N, "e_kin_first": kin[0], "e_kin_last": kin[-1],
                 "e_kin_per_atom_eV": kin[0] / N}
        nb = model.neighbors(p, box, cfg.hp.r_cut + cfg.skin, reuse=nb)
        e, _, f = model.compute(p, s, box, nb, want_atom_energies=False)

    def step():
        model.step_nve(p, v, f, s, mass, box, cfg.dt_fs, cfg.rebuild_every, cfg.skin, nb, ctr, e, ek)

    for _ in range(W):
        step()
    barrier()
    sampler = ClockSampler(local_rank); sampler.start()
    # R repeats of EXACTLY K steps, each bracketed by barrier + synchronize and timed with CUDA events on the launching
    # stream; the reported region is the MEDIAN repeat ("median of >= 3 repeats")
    reps = []
    for _ in range(max(args.repeats, 1)):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = model.launches
        barrier()
        ev0.record()
        for _ in range(K):
            step()
        ev1.record()
        barrier()
        reps.append((ev0.elapsed_time(ev1), model.launches - l0))
    sampler.stop_flag = True
    model.status()                                     # deferred device-side errors (coincident atoms, bad species)
    ms, launches = sorted(reps)[len(reps) // 2]
    n_active = model.last_active_edges()
    e_pot, e_kin = float(e.item()), float(ek.item())
    value, ms_max = aggregate_over_ranks(ms, N, K, dist, dev)

    # ---- e2e: the same step through the C ABI with HOST (pinned) buffers, copies inside the timed region
    hp_ = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    ph, vh, fh = hp_(p.cpu().numpy()), hp_(v.cpu().numpy()), hp_(f.cpu().numpy())
    sh, mh = hp_(sp), hp_(masses_for(cfg))
    eh, ekh = torch.zeros(1, dtype=torch.float64).pin_memory(), torch.zeros(1, dtype=torch.float64).pin_memory()
    for _ in range(2):
        model.step_nve_host(ph, vh, fh, sh, mh, box, cfg.dt_fs, cfg.rebuild_every, cfg.skin, nb, ctr, eh, ekh)
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        model.step_nve_host(ph, vh, fh, sh, mh, box, cfg.dt_fs, cfg.rebuild_every, cfg.skin, nb, ctr, eh, ekh)
    torch.cuda.synchronize()
    e2e_val, _ = aggregate_over_ranks((time.perf_counter() - t0) * 1e3, N, K, dist, dev)
    h2d = 3 * N * 24 + N * 4 + cfg.hp.n_species * 8
    d2h = 3 * N * 24 + 16

    # ---- allegro_compute alone and allegro_neighbors alone, outside the timed region above
    # the e2e loop above advanced its own host copy of the system and rebuilt `nb` there: rebuild the list for the
    # device-resident positions `p` before timing single calls (a list from other positions has fewer active edges)
    nb = model.neighbors(p, box, cfg.hp.r_cut + cfg.skin, reuse=nb)
    def _ev_ms(fn, reps):
        fn(); torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ts = []
        for _ in range(reps):
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return sorted(ts)[len(ts) // 2]
    compute_ms = _ev_ms(lambda: model.compute(p, s, box, nb, want_atom_energies=False), 3)
    energy_only_ms = _ev_ms(lambda: model.compute(p, s, box, nb, want_atom_energies=False, want_forces=False), 3)
    neighbors_ms = _ev_ms(lambda: model.neighbors(p, box, cfg.hp.r_cut + cfg.skin, reuse=nb), 3)

    # ---- roofline of the dominant kernel group: one more pass of K steps with per-group CUDA events on the launching stream
    groups = ["gemm", "tp_fwd", "tp_bwd", "geom", "twobody0", "energy", "bwd_elem", "edge_bwd", "neighbors", "nve"]
    tp_bytes = tp_bytes_per_edge(cfg.hp)
    model.profile_enable(True, nvtx=args.nvtx)
    for _ in range(K):
        model.step_nve(p, v, f, s, mass, box, cfg.dt_fs, cfg.rebuild_every, cfg.skin, nb, ctr, e, ek)
    prof = {g: model.profile_read(g) for g in groups}
    model.profile_enable(False, nvtx=args.nvtx)
    tot_prof = sum(t for t, _ in prof.values())
    pk = peaks()
    gemm_ms, gemm_n = prof["gemm"]
    long_region = ms_max * 1e-3 > 2.0                  # seconds-long timed region runs under the power cap -> sustained peaks
    which = "sustained" if long_region else "burst"

    # measured peaks that MEASURED_PEAKS.json does not hold
    probes = None
    if not args.no_peak_probe:
        probes = model.probe_peaks(2.0)                # the library's own FFMA and tcgen05 kind::tf32 issue-rate probes
        probes["tf32_matmul_8192"] = tf32_matmul_peak(dev)   # MEASURED_PEAKS.json's procedure with TF32 allowed (cuBLAS)
    macs = gemm_macs_per_edge(cfg.hp)
    flops_per_step = 2.0 * macs * n_active
    gemm_tflops = flops_per_step * K / (gemm_ms * 1e-3) / 1e12 if gemm_ms > 0 else 0.0
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    if args.precision == 3:
        bound = "alu"
        if probes:
            peak = probes["ffma"][which]
            peak_note = (f"fp32 FFMA probe (allegro_probe_ffma), {which}: burst {probes['ffma']['burst']:.1f} / sustained "
                         f"{probes['ffma']['sustained']:.1f} TFLOP/s; unit-count figure {nsm} SMs x {FFMA_LANES_PER_SM} lanes x 2 x "
                         f"{pk['sm_max_mhz']} MHz = {nsm * FFMA_LANES_PER_SM * 2 * pk['sm_max_mhz'] * 1e6 / 1e12:.1f}")
        else:
            peak = nsm * FFMA_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
            peak_note = f"{nsm} SMs x {FFMA_LANES_PER_SM} FFMA lanes x 2 x {pk['sm_max_mhz']} MHz (not probed)"
    elif args.precision in (2, 4):
        bound = "tensor"
        peak = pk["bf16_sustained"] if long_region else pk["bf16_burst"]
        peak_note = f"16-bit dense matmul {which} {peak} TFLOP/s (MEASURED_PEAKS.json, {pk['src']}; fp16 and bf16 share the rate)"
    else:
        bound = "tensor"
        div = 3.0 if args.precision == 0 else 1.0      # 3xTF32: three TF32 MMAs per algorithmic MAC
        if probes:
            tm = probes["tf32_matmul_8192"]
            peak = tm[which] / div
            peak_note = (f"TF32 8192^3 torch.matmul (cuBLAS, allow_tf32), measured in this run the way MEASURED_PEAKS.json measures "
                         f"bf16: burst {tm['burst']:.1f} / sustained {tm['sustained']:.1f} TFLOP/s, {which} used (timed region "
                         f"{ms_max * 1e-3:.2f} s); tcgen05 kind::tf32 issue-rate probe {probes['tf32_mma']['burst']:.1f} / "
                         f"{probes['tf32_mma']['sustained']:.1f}; bf16 {pk['bf16_burst']} / {pk['bf16_sustained']} ({pk['src']})"
                         + (" ; / 3 for 3xTF32 split operands" if div > 1 else ""))
        else:
            base = pk["bf16_sustained"] if long_region else pk["bf16_burst"]
            peak = base * TF32_OVER_BF16 / div
            peak_note = f"FALLBACK (no probe): bf16 {which} {base} TF/s ({pk['src']}) x nominal tf32/bf16 ratio {TF32_OVER_BF16}" + (" / 3" if div > 1 else "")
    # K-concatenated x-bar GEMM: tensor-core modes with a 32-multiple first latent width
    kcat = args.precision != 3 and cfg.hp.latent_dims[0] % 32 == 0
    alg_b, impl_b = gemm_alg_bytes_per_edge(cfg.hp), gemm_impl_bytes_per_edge(cfg.hp, kcat)
    secs = gemm_ms * 1e-3
    alg_gbs = alg_b * n_active * K / secs / 1e9 if gemm_ms > 0 else 0.0
    impl_gbs = impl_b * n_active * K / secs / 1e9 if gemm_ms > 0 else 0.0
    f_compute, f_hbm = gemm_tflops / peak, alg_gbs / pk["hbm_gbs"]
    comp = {"bound": bound, "achieved": gemm_tflops, "peak": peak, "unit": "TFLOP/s", "frac": f_compute, "peak_note": peak_note,
            "algorithmic_flops_per_edge": 2.0 * macs}
    hbm = {"bound": "hbm", "achieved": alg_gbs, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": f_hbm,
           "peak_note": f"copy bandwidth ({pk['src']}); algorithmic bytes = 8 (NL+1) d = {alg_b:.0f} B per active edge "
                        f"(SURVEY.md 8(d): x^0..x^NL written once + read once for the backward)"}
    top = hbm if f_hbm > f_compute else comp           # a kernel's fraction = max(bytes / t / HBM, flops / t / peak)
    traffic = traffic_src = None
    tpath = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if os.path.exists(tpath):   # dram__bytes_read + write per GEMM launch from the committed ncu --set full capture
        tj = json.load(open(tpath)).get(f"config{cfg.index}_precision{args.precision}")
        if tj:
            traffic, traffic_src = tj["gemm_dram_bytes_per_launch"], tj.get("source")
    kname = {0: "MLP GEMM group (fwd+bwd), k_gemm_tf32<.., SPLIT> (3xTF32)", 1: "MLP GEMM group (fwd+bwd), k_gemm_tf32",
             2: "MLP GEMM group (fwd+bwd), k_gemm_tf32<.., H16> (bf16 operands)", 3: "MLP GEMM group (fwd+bwd), k_gemm_simt",
             4: "MLP GEMM group (fwd+bwd), k_gemm_tf32<.., H16> (fp16 operands)"}[args.precision]
    per_launch = K / max(gemm_n, 1)
    roofline = {"bound": top["bound"], "kernel": kname,
                "achieved": top["achieved"], "peak": top["peak"], "unit": top["unit"], "frac": top["frac"],
                "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_bytes_per_launch": alg_b * n_active * per_launch,
                "algorithmic_flops_per_launch": flops_per_step * per_launch,
                "peak_note": top["peak_note"], "compute_roofline": comp, "hbm_roofline": hbm,
                # what this build's launch list actually moves (every A operand, aux operand and output once): NOT algorithmic
                "implementation_bytes_per_edge": impl_b, "implementation_hbm_gbs": impl_gbs,
                "implementation_hbm_frac": impl_gbs / pk["hbm_gbs"],
                "launches_per_step": gemm_n / K, "avg_launch_ms": gemm_ms / max(gemm_n, 1),
                "share_of_step": gemm_ms / tot_prof if tot_prof else None,
                "groups_ms_per_step": {g: round(t / K, 4) for g, (t, _) in prof.items()},
                "measured_peaks_tflops": probes,
                # the tensor-track kernels against the HBM roofline (north_star: gather/tensor-product/scatter >= 50 %)
                "tensor_track_hbm": {k: {"achieved": tp_bytes[k] * n_active * K / (prof[k][0] * 1e-3) / 1e9 if prof[k][0] > 0 else 0.0,
                                         "peak": pk["hbm_gbs"], "unit": "GB/s",
                                         "frac": (tp_bytes[k] * n_active * K / (prof[k][0] * 1e-3) / 1e9 / pk["hbm_gbs"]) if prof[k][0] > 0 else 0.0,
                                         "algorithmic_bytes_per_edge": tp_bytes[k],
                                         "survey_bytes_per_edge": tp_survey_bytes_per_edge(cfg.hp)[k]} for k in ("tp_fwd", "tp_bwd")}}
    if probes and cfg.hp.l_max == 3:
        # config 4: the tensor product is bound by the fp32 pipes, not HBM: report it against the FFMA probe too
        fl = tp_flops_per_edge(cfg.hp)
        roofline["tensor_track_alu"] = {k: {"achieved": fl[k] * n_active * K / (prof[k][0] * 1e-3) / 1e12 if prof[k][0] > 0 else 0.0,
                                            "peak": probes["ffma"][which], "unit": "TFLOP/s",
                                            "frac": (fl[k] * n_active * K / (prof[k][0] * 1e-3) / 1e12 / probes["ffma"][which]) if prof[k][0] > 0 else 0.0,
                                            "algorithmic_flops_per_edge": fl[k]} for k in ("tp_fwd", "tp_bwd")}

    out = {
        "metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": DTYPE[args.precision], "data": "synthetic",
        "config": {"workload": workload, "n_atoms": N, "active_edges": n_active, "candidate_edges": nb.n_edges,
                   "precision_mode": args.precision, "dt_fs": cfg.dt_fs, "rebuild_every": cfg.rebuild_every, "skin": cfg.skin,
                   "l2": "per-step working set (edge activations, several GB) is far larger than the 126 MB L2",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "timesteps_per_s": K / (ms_max * 1e-3), "ns_per_day": K / (ms_max * 1e-3) * cfg.dt_fs * 0.0864,
        "repeats_ms_per_step": [round(t / K, 4) for t, _ in reps], "repeat_reported": "median",
        "e_pot": e_pot, "e_kin": e_kin,
        # medians of 3 calls, CUDA events: energy+forces alone, energy only (no backward), list build alone
        "compute_only_ms": compute_ms, "energy_only_ms": energy_only_ms, "neighbors_only_ms": neighbors_ms,
        "gpu_launches": launches,
        "clocks": sampler.summary(),
        "e2e": {"value": e2e_val, "unit": unit, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "roofline": roofline,
    }
    if drift is not None:
        out["nve_drift"] = drift
    if rank == 0 and world == 1 and args.precision == 1 and not args.no_extra_modes and not args.decompose:
        # The same K steps in the fp16-operand MLP mode (precision 4: 16-bit storage of the MLP-only tensors, fp32 accumulate,
        # inside north_star's 2e-3 tolerance, tests/test_gpu_16bit.py) as a sub-record; the line above stays the TF32 one.
        try:
            del model, nb
            chp4 = P.hparams_from(cfg.hp, 4)
            m4 = P.Allegro(chp4, blob, chunk_edges=args.chunk_edges) if args.chunk_edges else P.Allegro(chp4, blob)
            if cfg.hp.r_cut_pair is not None:
                m4.set_pair_cutoffs(cfg.hp.r_cut_pair)
            p4 = torch.from_numpy(pos.copy()).to(dev); v4 = torch.from_numpy(vel.copy()).to(dev)
            nb4 = m4.neighbors(p4, box, cfg.hp.r_cut + cfg.skin)
            e4, _, f4 = m4.compute(p4, s, box, nb4, want_atom_energies=False)
            ek4 = torch.zeros(1, dtype=torch.float64, device=dev); c4 = ctypes.c_int64(0)
            for _ in range(W):
                m4.step_nve(p4, v4, f4, s, mass, box, cfg.dt_fs, cfg.rebuild_every, cfg.skin, nb4, c4, e4, ek4)
            torch.cuda.synchronize()
            smp = ClockSampler(local_rank); smp.start()
            a4, b4 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l4 = m4.launches
            a4.record()
            for _ in range(K):
                m4.step_nve(p4, v4, f4, s, mass, box, cfg.dt_fs, cfg.rebuild_every, cfg.skin, nb4, c4, e4, ek4)
            b4.record(); torch.cuda.synchronize()
            smp.stop_flag = True
            m4.status()
            ms4 = a4.elapsed_time(b4)
            out["extra_modes"] = {"fp16_operands": {
                "precision_mode": 4, "dtype": DTYPE[4], "steps": K, "warmup": W, "ms_per_step": ms4 / K,
                "value": N * K / (ms4 * 1e-3), "unit": unit, "gpu_launches": m4.launches - l4, "e_pot": float(e4.item()),
                "clocks": smp.summary(),
                "note": "same workload and step as the line; extra mode, not the paper's F32-activation / TF32-matmul scheme"}}
            del m4
        except P.AllegroError as ex:
            out["extra_modes"] = {"fp16_operands": {"unavailable": str(ex)}}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_all, n_one = {0: (192, 192), 1: (3072, 768), 2: (512, 128), 3: (512, 128), 4: (256, 64)}[cfg.index]
        import torch as _t
        ncores = _t.get_num_threads()

        def timed(n_c, budget):
            run, n_c, _ = oracle_sample(cfg, pos, sp, box, n_c)
            run()
            reps_, tt = 0, 0.0
            while tt < budget and reps_ < 200:
                tt += run(); reps_ += 1
            return n_c * reps_ / tt, n_c, reps_, tt
        v_all, nc_all, r_all, t_all = timed(n_all, 8.0)
        _t.set_num_threads(1)
        v_one, nc_one, r_one, t_one = timed(n_one, 8.0)
        _t.set_num_threads(ncores)
        out["cpu_baseline"] = {"value": v_all, "unit": unit, "cores": ncores, "kind": "oracle",
                               "sample": f"energy+forces of {nc_all} contiguous centres (all their edges) of {workload}, "
                                         f"{r_all} repeats, {t_all:.1f} s",
                               "one_thread": {"value": v_one, "unit": unit, "cores": 1,
                                              "sample": f"{nc_one} contiguous centres, {r_one} repeats, {t_one:.1f} s"}}
    if rank == 0:
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
