"""Multi-GPU plumbing: replicas only.

BASELINE.json:north_star rules out sharding and inter-GPU collectives for this path ("every domain lives on one
GPU"), so `bench.py --gpus N` runs N independent replicas: rank k solves its own right-hand side (source stream k
of the workload's seed) against the same gauge field on its own GPU.  torch.distributed is used only for the
barrier and the max-over-ranks reduction of the device-measured time; no tensor of the data path crosses ranks.
The same functions run on the gloo backend (CPU tensors), which is how tests/test_replicas.py covers them.
"""
from __future__ import annotations

import os


def env_rank():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when launched directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def source_streams(rank: int, world: int, n_rhs: int = 1):
    """Right-hand-side streams of one replica: n_rhs consecutive streams, disjoint over ranks."""
    if not 0 <= rank < world or n_rhs < 1:
        raise ValueError("source_streams: bad rank/world/n_rhs")
    return list(range(rank * n_rhs, (rank + 1) * n_rhs))


def init(backend: str, device=None):
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    if dist.is_initialized():
        return
    if device is not None:
        dist.init_process_group(backend, device_id=device)
    else:
        dist.init_process_group(backend)


def barrier(world: int, cuda: bool):
    import torch
    import torch.distributed as dist
    if world > 1:
        dist.barrier()
    if cuda:
        torch.cuda.synchronize()


def max_over_ranks(x: float, world: int, device="cpu") -> float:
    """Every rank gets the maximum of x over the ranks (the job takes as long as its slowest replica)."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_summary(ms_per_step_local: float, solves_per_step_local: int, world: int, device="cpu") -> dict:
    """Whole-job numbers of a weak-scaling replica run: the step time is the slowest rank's, the work is the sum."""
    ms = max_over_ranks(ms_per_step_local, world, device)
    return {"ms_per_step": ms, "solves_per_step": solves_per_step_local * world,
            "solves_per_s": solves_per_step_local * world / (ms * 1e-3) if ms > 0 else 0.0}


def shutdown(world: int):
    import torch.distributed as dist
    if world > 1 and dist.is_initialized():
        dist.destroy_process_group()
