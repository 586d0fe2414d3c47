"""Multi-GPU plumbing for the decode-attention path: REPLICAS ONLY.

The path has no exchange step on one node: every sequence's pages live on the GPU that owns the
sequence (partition "by sequence"), so N GPUs run N independent replicas of the
step and the only communication is the benchmark's own barrier and max-over-ranks of the device
time.  One process per GPU, ``torch.distributed`` (NCCL on GPUs, gloo in the CPU tests).

Nothing here touches the attention arithmetic.
"""
from __future__ import annotations

import os
from typing import List, Sequence, Tuple

import torch
import torch.distributed as dist


def world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str) -> Tuple[int, int, int]:
    """Join the process group when launched under torchrun (WORLD_SIZE > 1); no-op otherwise."""
    rank, local_rank, ws = world()
    if ws > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        kw = {}
        if backend == "nccl":
            kw["device_id"] = torch.device("cuda", local_rank)
        dist.init_process_group(backend=backend, rank=rank, world_size=ws, **kw)
    return rank, local_rank, ws


def barrier() -> None:
    if dist.is_initialized():
        dist.barrier()


def max_over_ranks(x: float, device="cpu") -> float:
    """MAX all-reduce of one scalar (the timed region's device milliseconds)."""
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, device="cpu") -> float:
    """SUM all-reduce of one scalar (units of work all ranks processed)."""
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def shard_sequences(seq_lens: Sequence[int], world_size: int) -> List[List[int]]:
    """Partition sequence indices over ranks "by sequence" (whole sequences, no exchange):
    longest-first greedy onto the least-loaded rank, ties to the lowest rank — a pure function of
    seq_lens, so every rank computes the same assignment without talking."""
    order = sorted(range(len(seq_lens)), key=lambda i: (-int(seq_lens[i]), i))
    load = [0] * world_size
    out: List[List[int]] = [[] for _ in range(world_size)]
    for i in order:
        r = min(range(world_size), key=lambda j: (load[j], j))
        out[r].append(i)
        load[r] += int(seq_lens[i])
    for r in range(world_size):
        out[r].sort()
    return out


def finalize() -> None:
    if dist.is_initialized():
        dist.destroy_process_group()
