"""Multi-GPU host logic ("every ray is independent"): one process per GPU, no
data-path collective.  bench.py --gpus N runs N replicas of the workload (weak scaling); a caller that wants
one image from N GPUs shards the pixel list with shard_pixels() and renders each shard with
Ipole.make_pixels().  The only exchange is the max-over-ranks of the device time (and, for a sharded image,
a gather of the Stokes planes), done with torch.distributed on whatever backend the job was started with
(nccl on GPUs; gloo in the CPU tests).  No arithmetic of the imaging method lives here.
"""
import numpy as np


def shard_pixels(n_pixels, rank, world):
    """Interleaved shard rank::world of the flat pixel indices 0..n_pixels-1 (int64).  Interleaving spreads
    the long photon-ring rays evenly over ranks; the shards partition the image exactly."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world %d" % (rank, world))
    return np.arange(rank, n_pixels, world, dtype=np.int64)


def max_over_ranks(value, device="cpu"):
    """max of a python float over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank, seconds_max, world):
    """whole-job rate: units of all ranks / the slowest rank's time"""
    return world * units_per_rank / seconds_max


def scatter_shard(full, shard, rank, world):
    """write a rank's shard values into a flat full-image array (host-side assembly of a sharded image)"""
    full[rank::world] = shard
    return full
