"""N > 1 path of bench.py ("replicas only"): world_size-2 gloo run on CPU of the rank
aggregation (sum of units over ranks / max over ranks of the time) and of the reference arm's rank gating."""
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    import bench
    ms_local = 10.0 if rank == 0 else 12.5          # rank 1 is the slow one
    val, ms_max = bench.aggregate_over_ranks(ms_local, 1000 * (rank + 1), 5, dist, "cpu")
    dist.barrier()
    out[rank] = (val, ms_max)
    dist.destroy_process_group()


def test_replica_aggregation_world2_gloo():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29531, out), nprocs=2, join=True)
    for r in (0, 1):
        val, ms_max = out[r]
        assert ms_max == 12.5
        assert abs(val - (1000 + 2000) * 5 / 12.5e-3) < 1e-6


def test_single_rank_aggregation_is_plain_ratio():
    sys.path.insert(0, ROOT)
    import bench
    val, ms = bench.aggregate_over_ranks(4.0, 12288, 10)
    assert ms == 4.0 and abs(val - 12288 * 10 / 4e-3) < 1e-6


def test_reference_arm_nonzero_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "0",
                        "--steps", "1", "--warmup", "1"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
