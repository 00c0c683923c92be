"""Multi-GPU plumbing for the splice: **replicas only** (DESIGN.md "Measurement, multi-GPU").

The path has no exchange step: layers, requests and tensor-parallel ranks (the MLA latent cache is replicated
under TP; PAPER.md:350, :732 use SGLang TP=4 for model serving only) are independent given the small host plan.
So N GPUs run N independent replicas of the workload, one process per GPU, and no data-path collective exists.
What is left for `torch.distributed` is the measurement contract: a barrier on both sides of the timed region,
the MAX over ranks of the per-step time, and whole-job throughput = all ranks' bytes / that time.  These helpers
take the device explicitly so that the same code runs under `gloo` on CPU (tests) and `nccl` on GPUs (bench.py).
"""
from __future__ import annotations

import os


def env_rank():
    """(rank, world_size, local_rank) as torchrun exports them; (0, 1, 0) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str, device=None):
    """Join the process group when WORLD_SIZE > 1 (rendezvous on 127.0.0.1 unless the launcher says otherwise)."""
    rank, world, local = env_rank()
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if not dist.is_initialized():
            kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
            dist.init_process_group(backend, rank=rank, world_size=world, **kw)
    return rank, world, local


def barrier(world: int, device=None):
    """dist.barrier() (N > 1) followed by a device synchronise when `device` is a CUDA device."""
    import torch
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    if device is not None and torch.device(device).type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(x: float, world: int, device="cpu") -> float:
    """The slowest rank's figure: a step of the job is done when every replica has finished it."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, world: int, device="cpu") -> float:
    """Units processed by the whole job (each replica reports its own)."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput_gbs(bytes_this_rank: int, ms_this_rank: float, world: int, device="cpu"):
    """Whole-job GB/s = bytes all ranks processed / max-over-ranks step time.  Returns (GB/s, ms)."""
    ms = max_over_ranks(ms_this_rank, world, device)
    total = sum_over_ranks(float(bytes_this_rank), world, device)
    return total / (ms * 1e-3) / 1e9, ms


def finish(world: int):
    if world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.barrier()
            dist.destroy_process_group()
