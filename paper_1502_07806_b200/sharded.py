"""One PFSM solve sharded over the ranks of a torch.distributed group.

The paper distributes slices over nodes and all-gathers.  Here rank g owns the slices
[g P/G, (g+1) P/G) = rows [g N/G, (g+1) N/G) of the row-major V (columns of the column-major V).  The compute
phases run in libpfsm (pfsm_shard_phase); this module only sequences them with the all-gathers between:

    phase 1  steps 2-3 on the own rows                 -> all-gather V rows          (8 N^2 / G bytes per rank)
    phase 2  own block row of G = V V^T                -> all-gather G rows
    phase 3  Cholesky (replicated) + own rows of the triangular solve  -> all-gather rows of V^T R^-1
    phase 4  step 5 on the own rows                    -> all-gather lambda, residuals

With the NCCL backend the gathers run GPU to GPU over NVLink/NVSwitch on the solve's stream; with gloo (CPU tests,
or several ranks time-sharing one GPU) they are staged through host memory.

PEER-WRITE MODE (setup_peers, then solve_sharded(..., peers=...)): no gathers at all.  Each rank maps the other ranks' V, G,
V^T R^-1, lambda and residual buffers through CUDA IPC once; from then on the GEMM epilogues of phases 1-3 store every
finished tile into all ranks' buffers (peer memory over NVLink / NVSwitch, overlapped with the product tile by tile) and
only a barrier separates the phases.  Same results as the gather mode, bit for bit.  Flop split per rank: steps 2, 3, 5 and
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


class Peers:
    """The other ranks' buffers of one sharded solve, mapped into this process (see setup_peers)."""

    def __init__(self, bases, group):
        self.bases = bases       # IPC mappings to close
        self.group = group
        self.token = None        # 1-element CUDA tensor for the stream-ordered NCCL barrier

    def close(self):
        from . import ipc_close
        for b in self.bases:
            ipc_close(b)
        self.bases = []


def setup_peers(h, Vr, lam, group=None):
    """Collective, once per (handle, Vr, lam): exchanges CUDA IPC handles of the five exchanged buffers (V, G, V^T R^-1,
    lambda, residuals), maps the other ranks' copies and registers them with the handle (pfsm_set_shard_peers).  Vr and lam
    must be the tensors later passed to solve_sharded.  Returns a Peers object (keep it alive; close() unmaps)."""
    import torch.distributed as dist
    from . import ipc_export, ipc_open
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    mine = [ipc_export(t) for t in (Vr, h.shard_buffer(0), h.shard_buffer(1), lam, h.residuals_view())]
    everyone = [None] * world
    dist.all_gather_object(everyone, mine, group=group)
    bases = []
    opened = {}                 # one mapping per (rank, allocation): several buffers may live in one allocation
    for which in range(5):
        ptrs = []
        for r in range(world):
            if r == rank:
                continue
            handle, off = everyone[r][which]
            key = (r, handle)
            if key not in opened:
                base, _ = ipc_open(handle, 0)
                opened[key] = base
                bases.append(base)
            ptrs.append(opened[key] + off)
        h.set_shard_peers(which, ptrs)
    return Peers(bases, group)


def _phase_barrier(peers):
    """All ranks' work of the phase (their peer stores included) is complete before anyone goes on.  NCCL: a one-element
    all-reduce on the solve's stream (stream-ordered, no host synchronization); gloo: device synchronize + host barrier."""
    import torch
    import torch.distributed as dist
    if dist.get_backend(peers.group) == "nccl":
        if peers.token is None:
            peers.token = torch.zeros(1, device="cuda")
        dist.all_reduce(peers.token, group=peers.group)
    else:
        if torch.cuda.is_available():
            torch.cuda.synchronize()
        dist.barrier(group=peers.group)


def solve_sharded_peer_writes(h, A, Vr, lam, peers, mark=None):
    """The sharded solve in peer-write mode: four compute phases, a barrier after each, no gather.  Collective."""
    mark = mark or (lambda label: None)
    mark("start")
    for phase, label in ((1, "phase1_steps2_3"), (2, "phase2_gram_rows"), (3, "phase3_cholesky_trsm_rows"),
                         (4, "phase4_step5_rows")):
        h.shard_phase(phase, A if phase in (1, 4) else None, Vr, lam if phase == 4 else None)
        mark(label)
        _phase_barrier(peers)
        mark("barrier_after_phase%d" % phase)
