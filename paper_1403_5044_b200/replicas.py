"""Plumbing for `bench.py --gpus N`: the path does not shard ("replicas only"), so
N ranks run N independent replicas and exchange nothing on the data path.  torch.distributed
is used for the bracketing barrier and the max-over-ranks of the device time only.  Works
with backend "nccl" (one rank per GPU) and "gloo" (CPU tests, world_size 2)."""
from __future__ import annotations

import os

_state = {"on": False, "device": None}


def world() -> int:
    return int(os.environ.get("WORLD_SIZE", "1"))


def init(backend: str = "nccl", device: int | None = None) -> bool:
    """Join the process group if launched by torchrun (WORLD_SIZE > 1); no-op otherwise."""
    if world() <= 1:
        return False
    import torch.distributed as dist
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend)
    _state["on"] = True
    _state["device"] = device if backend == "nccl" else None
    return True


def _tensor(x: float):
    import torch
    dev = f"cuda:{_state['device']}" if _state["device"] is not None else "cpu"
    return torch.tensor([float(x)], dtype=torch.float64, device=dev)


def barrier() -> None:
    if _state["on"]:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(x: float) -> float:
    """The slowest rank's time: what a whole-job throughput divides by."""
    if not _state["on"]:
        return float(x)
    import torch.distributed as dist
    t = _tensor(x)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float) -> float:
    if not _state["on"]:
        return float(x)
    import torch.distributed as dist
    t = _tensor(x)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_per_rank: float, local_ms: float) -> float:
    """Whole-job units/s of N independent replicas: sum of units / max of time."""
    return sum_over_ranks(units_per_rank) / (max_over_ranks(local_ms) * 1e-3)


def finalize() -> None:
    if _state["on"]:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
        _state["on"] = False
