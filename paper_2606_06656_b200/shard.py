"""Multi-GPU plumbing of the sharded job: restarts are independent
(PAPER.md L164, L182), so the batch is partitioned across ranks, the problem is replicated, and nothing is exchanged
inside the PGD loop.  One exchange at the end: the best satisfied counts of every rank.  torch.distributed only
(NCCL on GPUs, gloo in the CPU tests); none of the method's arithmetic lives here."""
from __future__ import annotations

import numpy as np


def restart_range(B: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous share [b0, b1) of B restarts owned by `rank` (strong scaling: sizes differ by at most one)."""
    q, r = divmod(int(B), int(world))
    b0 = rank * q + min(rank, r)
    return b0, b0 + q + (1 if rank < r else 0)


def rank_start_points(base_seed: int, cfg: int, rank: int, shape) -> np.ndarray:
    """Weak scaling: every rank draws its own X0 ~ U[-1,1] (fp32) for the same instance."""
    rng = np.random.Generator(np.random.PCG64(int(base_seed) + 1000 * (int(rank) + 1) + int(cfg)))
    return rng.uniform(-1.0, 1.0, size=shape).astype(np.float32)


def max_over_ranks(value: float, device=None) -> float:
    """Device time of the job = the slowest rank's."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_best(best_sat):
    """All-gather of the per-restart best counts (int32 [B_local], equal length on every rank).
    Returns (counts [world, B_local] tensor, (rank, restart, count) of the overall best; earliest rank/restart on ties)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size() if dist.is_initialized() else 1
    if world == 1:
        allc = best_sat.unsqueeze(0)
    else:
        parts = [torch.empty_like(best_sat) for _ in range(world)]
        dist.all_gather(parts, best_sat)
        allc = torch.stack(parts)
    flat = allc.reshape(-1).cpu()
    top = int(flat.max().item()) if flat.numel() else 0
    idx = int((flat == top).nonzero()[0].item()) if flat.numel() else 0
    B = allc.shape[1]
    return allc, (idx // B, idx % B, top)
