"""Multi-GPU plumbing of bench.py: the hot path does not shard (SURVEY.md section 8(e):
"replicas only"), so N GPUs run N independent trajectories.  The only inter-rank traffic is the
timing protocol: a barrier on both sides of the timed region and the MAX over ranks of the
device-measured time.  No collective touches the data path.  Backend "nccl" on the GPU box,
"gloo" in the CPU tests (tests/test_replicas.py)."""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def world():
    return int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0"))


def init(backend: str = "nccl", device=None):
    """Join the process group when launched under torchrun (WORLD_SIZE > 1); no-op otherwise."""
    n, _, _ = world()
    if n > 1 and not dist.is_initialized():
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=device)
        else:
            dist.init_process_group(backend)
    return n


def barrier(device=None):
    if dist.is_initialized():
        dist.barrier()
    if device is not None and torch.device(device).type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(value: float, device=None) -> float:
    """MAX over ranks of a host scalar (the per-rank device-timed milliseconds)."""
    if not dist.is_initialized():
        return float(value)
    dev = device if (device is not None and dist.get_backend() == "nccl") else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: float, ms_max: float, n_ranks: int) -> float:
    """Whole-job throughput: every rank processed `units_per_rank` units in (at most) ms_max."""
    return n_ranks * units_per_rank / (ms_max * 1e-3)


def finish():
    if dist.is_initialized():
        dist.destroy_process_group()
