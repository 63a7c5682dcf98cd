"""Host logic of the N > 1 path on CPU: world_size 2 over gloo (rays shard by pixel, no
data-path collective; the only exchange is the max-over-ranks of the timing)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2302_02733_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = [12.5, 19.25][rank]
        worst = replicas.max_over_ranks(ms)
        pix = replicas.shard_pixels(37, rank, world)
        # stand-in for a rendered shard: the pixel index itself, gathered on every rank
        mine = torch.from_numpy(pix.astype(np.float64))
        sizes = [len(replicas.shard_pixels(37, r, world)) for r in range(world)]
        parts = [torch.empty(s, dtype=torch.float64) for s in sizes]
        for r in range(world):  # shards differ in length by one: broadcast each from its owner
            dist.broadcast(mine if r == rank else parts[r], src=r)
        parts[rank] = mine
        full = np.full(37, -1.0)
        for r in range(world):
            replicas.scatter_shard(full, parts[r].numpy(), r, world)
        out.put((rank, worst, full.tolist(), replicas.job_throughput(1000, worst * 1e-3, world)))
    finally:
        dist.destroy_process_group()


def test_shards_partition_the_image():
    for n in (0, 1, 7, 1024):
        for world in (1, 2, 3, 8):
            parts = [replicas.shard_pixels(n, r, world) for r in range(world)]
            allp = np.sort(np.concatenate(parts))
            assert allp.dtype == np.int64 and np.array_equal(allp, np.arange(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.job_throughput(10, 2.0, 4) == 20.0


def test_world_size_two_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, worst, full, rate in res:
        assert worst == 19.25                       # both ranks agree on the slowest rank's time
        assert full == list(map(float, range(37)))  # the two shards assemble the whole image, nothing twice
        assert rate == 2 * 1000 / 19.25e-3
