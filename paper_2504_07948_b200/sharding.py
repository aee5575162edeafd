"""Host-side logic for running one crowd per GPU.

Walkers are independent units ("evaluated independently across thousands of processing
units"), so the hot path shards over walkers with NO data-path collective: rank r owns global walkers
[r*W, (r+1)*W) -- weak scaling, per-GPU work fixed -- and its RNG streams are keyed on the global walker
id, so a sharded run reproduces exactly what one big crowd would do (reading A20).  The only
communication is the reduction of scalars for reporting (max of the elapsed time, sums of counts and
energies)."""
from __future__ import annotations

import os


def dist_env():
    """(rank, local_rank, world_size) from the torchrun environment (single process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")))


def walker_slice(walkers_per_gpu: int, rank: int):
    """Global walker ids owned by `rank` under weak scaling."""
    if walkers_per_gpu < 1 or rank < 0:
        raise ValueError("walkers_per_gpu >= 1 and rank >= 0 required")
    return rank * walkers_per_gpu, (rank + 1) * walkers_per_gpu


def reduce_report(elapsed_ms: float, n_moves: int, e_sum: float, e_sq_sum: float, n_walkers: int, backend_device="cpu"):
    """All-reduce the per-rank scalars: MAX of time, SUM of the rest.  Works without torch.distributed
    (single process) and with any backend (gloo on CPU, nccl on GPU)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return dict(elapsed_ms=elapsed_ms, n_moves=n_moves, e_sum=e_sum, e_sq_sum=e_sq_sum, n_walkers=n_walkers)
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=backend_device)
    s = torch.tensor([float(n_moves), e_sum, e_sq_sum, float(n_walkers)], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(s, op=dist.ReduceOp.SUM)
    s = s.cpu()
    return dict(elapsed_ms=float(t.item()), n_moves=int(round(s[0].item())), e_sum=float(s[1]), e_sq_sum=float(s[2]),
                n_walkers=int(round(s[3].item())))
