"""Rank logic of the multi-GPU run: REPLICAS ONLY.

The path is defined on one GPU with no sharding (BASELINE.json north_star), so N GPUs run N
independent replicas: every rank encrypts its own message under its own key, there is no data-path
collective, and `torch.distributed` carries only the barrier and the max-over-ranks of the device
time.  This module holds that host logic so that it can be tested with the `gloo` backend on CPU;
it contains none of the method's arithmetic and does not load the CUDA library.
"""
from __future__ import annotations

import os
from typing import Tuple


def rank_env() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def replica_key(key: bytes, rank: int) -> bytes:
    """Rank r's key: the config's key with every byte XORed by r (rank 0 keeps the config's key), so
    that the replicas are independent messages and not N copies of one."""
    return bytes(b ^ (rank & 0xFF) for b in key) if rank else bytes(key)


def replica_seed(seed: int, rank: int) -> int:
    return seed + rank


def init(backend: str, device=None) -> int:
    """Initialises the default process group when WORLD_SIZE > 1; returns the world size."""
    _, _, world = rank_env()
    if world > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            kw = {"device_id": device} if device is not None else {}
            dist.init_process_group(backend, **kw)
    return world


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    """The slowest rank's figure (a time): every multi-GPU number is the max over ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_gbs(bytes_per_rank_per_step: int, steps: int, slowest_ms: float, world: int) -> float:
    """Whole-job throughput: the bytes all ranks processed divided by the slowest rank's time."""
    return world * steps * bytes_per_rank_per_step / (slowest_ms * 1e-3) / 1e9


def finish() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
