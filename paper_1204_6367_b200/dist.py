"""Multi-GPU plumbing: one process per GPU, projections sharded across ranks.

Projections are independent (each image depends only on the read-only volume
and tables), so the path shards with NO data-path
collective: every rank holds a replica of the volume and projects its own
gantry angles.  The only collectives are the harness's: a barrier around the
timed region, MAX of the elapsed time and SUM of the work counters.
Host logic only; works with the gloo backend on CPU (tests/test_dist_gloo.py).
"""
import os

import numpy as np


def world_from_env():
    """(rank, local_rank, world_size) from the torchrun environment."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init_process_group(backend):
    """Join the job torchrun started (MASTER_ADDR/MASTER_PORT from the env).
    Returns (rank, local_rank, world_size); a no-op for world_size 1."""
    rank, local_rank, world = world_from_env()
    if world > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29500")
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def strided_shard(n_total, world_size, rank):
    """Indices rank owns out of n_total projections: rank, rank + world, ...
    Interleaving keeps every rank's mix of gantry angles (hence of path
    lengths) the same, so ranks finish together."""
    if not (0 <= rank < world_size):
        raise ValueError("rank out of range")
    return np.arange(rank, n_total, world_size, dtype=np.int64)


def scan_angles(n_total):
    """n_total gantry angles evenly spaced over 2 pi, end point excluded
    (reading Q16)."""
    return 2.0 * np.pi * np.arange(n_total, dtype=np.float64) / n_total


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def _reduce(value, op_name, device=None):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return value
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return float(t.item())


def max_over_ranks(value, device=None):
    return _reduce(value, "MAX", device)


def sum_over_ranks(value, device=None):
    return _reduce(value, "SUM", device)
