"""World-size-2 CPU tests (gloo) of the N>1 paths' host logic.  Replica mode (bench.py --replicas): ranks draw
distinct matrices, timings are reduced with MAX over ranks, the whole-job value aggregates all ranks' flops, failure
on any rank is seen by all.  Sharded mode (bench.py's N>1 default): the in-place all-gather of row
blocks, and the whole solve_sharded sequence driven end to end with a recording fake handle."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank),
                      LOCAL_RANK=str(rank))
    import oracle
    import pfsm_inputs as gen
    from paper_1502_07806_b200 import replicas
    assert replicas.env_world() == (world, rank, rank)
    replicas.init("gloo", world, rank)
    p = gen.problem(0, seed_offset=replicas.replica_seed_offset(rank))
    c = p.cfg
    # stand-in for the GPU solve on this CPU-only box: the oracle solves this rank's replica
    r = oracle.pfsm(p.A, c.P, c.window, c.iters, p.alpha)
    fake_ms = 10.0 * (rank + 1)                      # rank 1 is the slow one
    replicas.barrier(world)
    tmax = replicas.max_over_ranks(fake_ms, world)
    ok_all = replicas.all_ok(r["info"] == 0, world)
    ok_mixed = replicas.all_ok(rank != 1, world)      # rank 1 "fails": every rank must see it
    val = replicas.aggregate_tflops(1e12, 1, world, tmax)
    q.put((rank, float(p.A[0, 1]), float(r["lam"].sum()), tmax, ok_all, ok_mixed, val))
    replicas.finalize(world)


def test_two_rank_replicas_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, a0, s0, t0, ok0, mixed0, v0), (r1, a1, s1, t1, ok1, mixed1, v1) = res
    assert (r0, r1) == (0, 1)
    assert a0 != a1 and s0 != s1                      # independent replicas (different seeds)
    assert t0 == t1 == 20.0                           # MAX over ranks, identical on every rank
    assert ok0 and ok1 and not mixed0 and not mixed1
    assert v0 == v1 and abs(v0 - 2 * 1e12 / 20e-3 * 1e-12) < 1e-9   # both ranks' flops over the slowest time


def test_single_rank_is_a_no_op():
    from paper_1502_07806_b200 import replicas
    assert replicas.max_over_ranks(3.5, 1) == 3.5
    assert replicas.all_ok(True, 1) and not replicas.all_ok(False, 1)
    assert np.isclose(replicas.aggregate_tflops(2e12, 3, 1, 1000.0), 6.0)


def _gather_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank))
    import torch
    import torch.distributed as dist
    from paper_1502_07806_b200 import sharded
    dist.init_process_group("gloo", world_size=world, rank=rank)
    N = 8
    t = torch.full((N, N), float("nan"), dtype=torch.float64)
    rows = N // world
    t[rank * rows:(rank + 1) * rows] = float(rank + 1)      # only the own row block is valid
    sharded._all_gather_rows(t, world, rank)
    v = torch.full((N,), float("nan"), dtype=torch.float64)
    v[rank * rows:(rank + 1) * rows] = float(10 * (rank + 1))
    sharded._all_gather_rows(v, world, rank)
    q.put((rank, t.tolist(), v.tolist()))
    dist.destroy_process_group()


def test_sharded_all_gather_of_row_blocks_gloo():
    """Host logic of the sharded solve (f3): the in-place all-gather of equal row blocks, world size 2, CPU."""
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gather_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want_t = [[1.0] * 8] * 4 + [[2.0] * 8] * 4
    want_v = [10.0] * 4 + [20.0] * 4
    for rank, t, v in res:
        assert t == want_t and v == want_v


class _RecordingHandle:
    """Stands in for pfsm.Handle on a CPU-only box: records the phase order and, like the library, leaves only the OWN
    row block of each phase's output valid (everything else NaN), so a missing or misplaced all-gather shows up."""

    def __init__(self, N, rank, world):
        import torch
        self.N, self.rank, self.world = N, rank, world
        self.calls = []
        self.bufs = [torch.full((N, N), float("nan"), dtype=torch.float64) for _ in range(2)]
        self.resid = torch.full((N,), float("nan"), dtype=torch.float64)

    def _own(self):
        rows = self.N // self.world
        return slice(self.rank * rows, (self.rank + 1) * rows)

    def shard_phase(self, phase, A, Vr, lam, stream=None):
        import torch
        own = self._own()
        self.calls.append((phase, A is not None, lam is not None))
        if phase == 1:
            Vr[own] = 100.0 + self.rank                       # steps 2-3 on the own rows
        elif phase == 2:
            assert not torch.isnan(Vr).any(), "phase 2 needs every rank's rows of V (all-gather 1 missing)"
            self.bufs[0][own] = 200.0 + self.rank             # own block row of G
        elif phase == 3:
            assert not torch.isnan(self.bufs[0]).any(), "phase 3 needs all of G (all-gather 2 missing)"
            self.bufs[1][own] = 300.0 + self.rank             # own rows of the triangular solve
        elif phase == 4:
            assert not torch.isnan(self.bufs[1]).any(), "phase 4 needs all of V^T R^-1 (all-gather 3 missing)"
            Vr[:] = self.bufs[1].T                            # the library transposes the gathered buffer into V
            lam[own] = 400.0 + self.rank
            self.resid[own] = 500.0 + self.rank

    def shard_buffer(self, which):
        return self.bufs[which]

    def residuals_view(self):
        return self.resid


def _sharded_sequence_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank))
    import torch
    import torch.distributed as dist
    from paper_1502_07806_b200 import sharded
    dist.init_process_group("gloo", world_size=world, rank=rank)
    N = 8
    h = _RecordingHandle(N, rank, world)
    A = torch.zeros((N, N), dtype=torch.float64)
    Vr = torch.full((N, N), float("nan"), dtype=torch.float64)
    lam = torch.full((N,), float("nan"), dtype=torch.float64)
    sharded.solve_sharded(h, A, Vr, lam)
    q.put((rank, h.calls, Vr.tolist(), lam.tolist(), h.resid.tolist(), h.bufs[0].tolist()))
    dist.destroy_process_group()


def test_sharded_solve_sequencing_gloo():
    """solve_sharded end to end on CPU with a recording fake handle, world size 2: phases run 1-2-3-4 with A passed
    only where the library reads it (phases 1 and 4) and lambda only in phase 4; after each phase exactly the buffer
    that phase produced is gathered, so every rank ends with the complete V, lambda, residuals."""
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_sharded_sequence_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want_lam = [400.0] * 4 + [401.0] * 4
    want_res = [500.0] * 4 + [501.0] * 4
    want_G = [[200.0] * 8] * 4 + [[201.0] * 8] * 4
    want_V = np.array([[300.0] * 8] * 4 + [[301.0] * 8] * 4).T.tolist()
    for rank, calls, V, lam, resid, G in res:
        assert calls == [(1, True, False), (2, False, False), (3, False, False), (4, True, True)]
        assert lam == want_lam and resid == want_res and G == want_G and V == want_V


class _PeerWritingHandle:
    """Stands in for pfsm.Handle in PEER-WRITE mode on a CPU-only box.  The ranks' buffers are shared-memory tensors, so a
    phase can do what the library's PEER epilogues do: store its own row block into EVERY rank's copy.  Before it works,
    each phase asserts that all ranks' rows of the previous phase have arrived in its OWN copy -- which only holds if
    solve_sharded_peer_writes puts a barrier after every phase."""

    def __init__(self, rank, world, bufs):
        self.rank, self.world, self.bufs = rank, world, bufs      # bufs[name][r] = rank r's copy (shared memory)
        self.calls = []

    def _own(self, n):
        rows = n // self.world
        return slice(self.rank * rows, (self.rank + 1) * rows)

    def _write_all(self, name, value):
        for r in range(self.world):
            t = self.bufs[name][r]
            t[self._own(t.shape[0])] = value

    def shard_phase(self, phase, A, Vr, lam, stream=None):
        import time

        import torch
        mine = {k: v[self.rank] for k, v in self.bufs.items()}
        self.calls.append((phase, A is not None, lam is not None))
        if self.rank == 1:
            time.sleep(0.2)                                        # a slow rank: without barriers the fast one would run ahead
        if phase == 1:
            self._write_all("V", 100.0 + self.rank)
        elif phase == 2:
            assert not torch.isnan(mine["V"]).any(), "phase 2 started before every rank's rows of V had arrived"
            self._write_all("G", 200.0 + self.rank)
        elif phase == 3:
            assert not torch.isnan(mine["G"]).any(), "phase 3 started before every rank's rows of G had arrived"
            self._write_all("O", 300.0 + self.rank)
        elif phase == 4:
            assert not torch.isnan(mine["O"]).any(), "phase 4 started before every rank's rows of V^T R^-1 had arrived"
            self._write_all("lam", 400.0 + self.rank)


def _peer_sequence_worker(rank, world, port, bufs, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank))
    import torch
    import torch.distributed as dist
    from paper_1502_07806_b200 import sharded
    dist.init_process_group("gloo", world_size=world, rank=rank)
    h = _PeerWritingHandle(rank, world, bufs)
    peers = sharded.Peers([], None)
    A = torch.zeros((8, 8), dtype=torch.float64)
    labels = []
    sharded.solve_sharded_peer_writes(h, A, bufs["V"][rank], bufs["lam"][rank], peers, mark=labels.append)
    # after the last barrier every rank's lambda is complete in every copy
    q.put((rank, h.calls, labels, bufs["lam"][rank].tolist()))
    dist.destroy_process_group()


def test_peer_write_solve_sequencing_gloo():
    """solve_sharded_peer_writes end to end on CPU, world size 2: phases 1-4 in order, A only where the library reads it, a
    barrier after EVERY phase (a slow rank's stores have landed before the fast rank's next phase reads them; the one after
    phase 4 makes lambda complete everywhere before the call returns)."""
    import torch
    world, N = 2, 8
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    bufs = {name: [torch.full(shape, float("nan"), dtype=torch.float64).share_memory_() for _ in range(world)]
            for name, shape in (("V", (N, N)), ("G", (N, N)), ("O", (N, N)), ("lam", (N,)))}
    procs = [ctx.Process(target=_peer_sequence_worker, args=(r, world, port, bufs, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want_labels = ["start"]
    for k, name in ((1, "phase1_steps2_3"), (2, "phase2_gram_rows"), (3, "phase3_cholesky_trsm_rows"), (4, "phase4_step5_rows")):
        want_labels += [name, "barrier_after_phase%d" % k]
    for rank, calls, labels, lam in res:
        assert calls == [(1, True, False), (2, False, False), (3, False, False), (4, True, True)]
        assert labels == want_labels
        assert lam == [400.0] * 4 + [401.0] * 4
