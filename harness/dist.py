"""Multi-process plumbing for ``bench.py --gpus N`` (the pass does not shard — every rank is an
independent serving replica running the same deterministic pass on its own queue; no data-path collective).

Only the barrier and the max-over-ranks / sum-over-ranks of the timing scalars go through torch.distributed
(NCCL on the GPU box, gloo in the CPU tests)."""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def init(backend: str):
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    if dist.is_initialized():
        dist.barrier()


def aggregate(units: float, elapsed_ms: float, device="cpu"):
    """Whole-job figures of a replicated run: (sum of units over ranks, max of elapsed time over ranks)."""
    if not dist.is_initialized():
        return float(units), float(elapsed_ms)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()), float(t.item())


def throughput(units: float, elapsed_ms: float, device="cpu") -> float:
    """units/s of the whole job = all ranks' units / the slowest rank's time."""
    u, t = aggregate(units, elapsed_ms, device)
    return u / (t * 1e-3) if t > 0 else 0.0


def finalize():
    if dist.is_initialized():
        dist.destroy_process_group()
