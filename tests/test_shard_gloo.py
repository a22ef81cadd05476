"""The N > 1 host logic (restart sharding, max-over-ranks timing, the final all-gather) on CPU: world size 2, gloo."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_06656_b200 import shard


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        t = shard.max_over_ranks(10.0 + 5.0 * rank)
        best = torch.tensor([3, 7 + rank, 2, 8] if rank == 0 else [8, 1, 8, 0], dtype=torch.int32)
        allc, top = shard.gather_best(best)
        X0 = shard.rank_start_points(2606066560, 1, rank, (4, 6))
        out.put((rank, t, allc.tolist(), top, float(X0.sum())))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
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
    (r0, t0, c0, top0, s0), (r1, t1, c1, top1, s1) = res
    assert t0 == t1 == 15.0                                   # the slowest rank's time, on every rank
    assert c0 == c1 == [[3, 7, 2, 8], [8, 1, 8, 0]]           # every rank sees every rank's counts
    assert top0 == top1 == (0, 3, 8)                          # earliest (rank, restart) among the ties at 8
    assert s0 != s1                                           # ranks draw different start points


def test_restart_ranges_partition_the_batch():
    for B in (1, 7, 64, 1000, 4096):
        for world in (1, 2, 3, 8):
            edges = [shard.restart_range(B, world, r) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == B
            assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1


def test_single_process_paths():
    allc, top = shard.gather_best(torch.tensor([1, 5, 5], dtype=torch.int32))
    assert allc.tolist() == [[1, 5, 5]] and top == (0, 1, 5)
    assert shard.max_over_ranks(2.5) == 2.5
    a = shard.rank_start_points(1, 0, 0, (2, 3)); b = shard.rank_start_points(1, 0, 0, (2, 3))
    assert np.array_equal(a, b) and a.dtype == np.float32 and np.all(np.abs(a) <= 1)
