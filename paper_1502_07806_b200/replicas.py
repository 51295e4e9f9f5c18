"""Multi-GPU plumbing shared by both N>1 modes of bench.py: process-group setup, barrier,
MAX-over-ranks timing, whole-job aggregation.

Default for N>1 is the SHARDED solve (paper_1502_07806_b200/sharded.py): one eigenproblem split
over the ranks with all-gathers around step 4.  `bench.py --replicas` is the other mode: rank r solves its own matrix
of the same config -- one per k-point / spin channel / SCF replica in the paper's setting ("a sequence of
eigenvalue problems") -- with no data-path collective; the only communication is the barrier and the max-over-ranks of
the timings.  This module holds that host logic so it can be tested on CPU with the gloo backend.
"""
from __future__ import annotations

import os


def env_world():
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def replica_seed_offset(rank: int) -> int:
    """Rank r draws an independent matrix of the same config: pfsm_inputs.problem(k, seed_offset=r) seeds it with
    config seed + 1000 r."""
    return rank


def init(backend: str, world: int, rank: int, device=None):
    import torch.distributed as dist
    if world == 1 or dist.is_initialized():
        return
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29511")
    kw = {}
    if device is not None and backend == "nccl":
        kw["device_id"] = device
    dist.init_process_group(backend, world_size=world, rank=rank, **kw)


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(x: float, world: int, device="cpu") -> float:
    """Timing rule: every multi-GPU number is the MAX over ranks of the device-measured time."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_ok(flag: bool, world: int, device="cpu") -> bool:
    """True iff every rank's solve reported info == 0."""
    if world == 1:
        return bool(flag)
    import torch
    import torch.distributed as dist
    t = torch.tensor([0.0 if flag else 1.0], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item()) == 0.0


def aggregate_tflops(flops_per_solve: float, solves_per_rank: int, world: int, max_total_ms: float) -> float:
    """Whole-job throughput: all ranks' algorithmic flops over the slowest rank's time (weak scaling)."""
    return world * solves_per_rank * flops_per_solve / (max_total_ms * 1e-3) * 1e-12


def finalize(world: int):
    if world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
