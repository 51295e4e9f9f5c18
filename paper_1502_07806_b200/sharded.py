"""One PFSM solve sharded over the ranks of a torch.distributed group.

The paper distributes slices over nodes and all-gathers.  Here rank g owns the slices
[g P/G, (g+1) P/G) = rows [g N/G, (g+1) N/G) of the row-major V (columns of the column-major V).  The compute
phases run in libpfsm (pfsm_shard_phase); this module only sequences them with the all-gathers between:

    phase 1  steps 2-3 on the own rows                 -> all-gather V rows          (8 N^2 / G bytes per rank)
    phase 2  own block row of G = V V^T                -> all-gather G rows
    phase 3  Cholesky (replicated) + own rows of the triangular solve  -> all-gather rows of V^T R^-1
    phase 4  step 5 on the own rows                    -> all-gather lambda, residuals

With the NCCL backend the gathers run GPU to GPU over NVLink/NVSwitch on the solve's stream; with gloo (CPU tests,
or several ranks time-sharing one GPU) they are staged through host memory.  Flop split per rank: steps 2, 3, 5 and
the Gram / triangular-solve parts of step 4 scale 1/G; the N^3/3 Cholesky is replicated (2 % of the flops).
"""
from __future__ import annotations


def _all_gather_rows(t, world: int, rank: int, group=None, force: bool = False):
    """In-place all-gather of a tensor split into `world` equal row blocks (dim 0); this rank's block is valid.
    force: run the collective even for world == 1 (a test executes the NCCL branch on a one-GPU box that way)."""
    import torch
    import torch.distributed as dist
    if world == 1 and not force:
        return
    chunks = list(t.chunk(world, dim=0))
    assert len(chunks) == world and all(c.shape == chunks[0].shape for c in chunks)
    if dist.get_backend(group) == "nccl":
        # in place, GPU to GPU: rank g's block already sits at its position in the output (ncclAllGather's in-place
        # form), no staging copy; ordered after the solve's stream (torch's NCCL stream waits on the current stream)
        assert t.is_contiguous()
        dist.all_gather_into_tensor(t, chunks[rank], group=group)
        return
    host = [torch.empty(chunks[0].shape, dtype=t.dtype) for _ in range(world)]
    dist.all_gather(host, chunks[rank].cpu(), group=group)
    for k, c in enumerate(chunks):
        if k != rank:
            c.copy_(host[k])


def solve_sharded(h, A, Vr, lam, group=None, mark=None):
    """Collective: every rank calls it with its own handle (already `set_shard(rank, world)`), the replicated A, and
    full-size Vr (N, N) / lam (N,) buffers.  On return every rank holds the complete V, lambda and residuals.
    mark(label), if given, is called at the start and after every phase / gather (bench.py records CUDA events there)."""
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    mark = mark or (lambda label: None)
    mark("start")
    h.shard_phase(1, A, Vr, None)
    mark("phase1_steps2_3")
    _all_gather_rows(Vr, world, rank, group)
    mark("gather_V")
    h.shard_phase(2, None, Vr, None)
    mark("phase2_gram_rows")
    _all_gather_rows(h.shard_buffer(0), world, rank, group)
    mark("gather_G")
    h.shard_phase(3, None, Vr, None)
    mark("phase3_cholesky_trsm_rows")
    _all_gather_rows(h.shard_buffer(1), world, rank, group)
    mark("gather_VRinv")
    h.shard_phase(4, A, Vr, lam)
    mark("phase4_step5_rows")
    _all_gather_rows(lam, world, rank, group)
    _all_gather_rows(h.residuals_view(), world, rank, group)
    mark("gather_lambda_resid")
