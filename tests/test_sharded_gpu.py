"""f3: one solve sharded over 2 ranks.  The box has one GPU, so the two ranks are two processes time-sharing it and
the all-gathers go through the gloo backend (host staging); no kernel of one rank waits on the other.  The result
must equal the single-rank solve."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, N, P, w, iters, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank))
    import torch
    import torch.distributed as dist

    import paper_1502_07806_b200 as pfsm
    import pfsm_inputs as gen
    from paper_1502_07806_b200 import sharded
    dist.init_process_group("gloo", world_size=world, rank=rank)
    torch.cuda.set_device(0)
    p = gen.small_problem(N, 1e-3, 16.0, seed=4242)
    h = pfsm.Handle(N, P, w, iters, p.alpha)
    h.set_shard(rank, world)
    dA = torch.from_numpy(p.A).cuda()
    dV = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    dl = torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")
    sharded.solve_sharded(h, dA, dV, dl)
    torch.cuda.synchronize()
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), lam=dl.cpu().numpy(), V=dV.cpu().numpy(),
             res=h.residuals().cpu().numpy(), info=h.info())
    h.destroy()
    dist.destroy_process_group()


@pytest.mark.parametrize("N,P,w,iters", [(512, 4, 16, 2), (768, 6, 24, 3)])
def test_two_rank_sharded_solve_equals_single_rank(tmp_path, N, P, w, iters):
    import torch

    import oracle
    import paper_1502_07806_b200 as pfsm
    import pfsm_inputs as gen
    world = 2
    ctx = mp.get_context("spawn")
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, N, P, w, iters, str(tmp_path))) for r in range(world)]
    for pr in procs:
        pr.start()
    for pr in procs:
        pr.join(timeout=300)
        assert pr.exitcode == 0
    p = gen.small_problem(N, 1e-3, 16.0, seed=4242)
    h = pfsm.Handle(N, P, w, iters, p.alpha)
    dA = torch.from_numpy(p.A).cuda()
    dV = torch.empty((N, N), dtype=torch.float64, device="cuda")
    dl = torch.empty((N,), dtype=torch.float64, device="cuda")
    h.solve(dA, dV, dl)
    ref_l, ref_V, ref_r = dl.cpu().numpy(), dV.cpu().numpy(), h.residuals().cpu().numpy()
    assert h.info() == 0
    h.destroy()
    o = oracle.pfsm(p.A, P, w, iters, p.alpha)
    nF = p.normF
    for r in range(world):
        d = np.load(os.path.join(str(tmp_path), f"rank{r}.npz"))
        assert int(d["info"]) == 0
        # every rank ends with the complete result, equal to the single-rank solve to rounding
        assert np.abs(d["lam"] - ref_l).max() < 1e-13
        assert np.abs(d["V"] - ref_V).max() < 1e-12
        assert np.abs(d["res"] - ref_r).max() < 1e-13
        # and within the parity gates of the oracle
        assert np.abs(d["lam"] - o["lam"]).max() <= 1e-10 * nF
        assert np.abs(d["V"] @ d["V"].T - np.eye(N)).max() <= 1e-12 * N


def _nccl_worker(port, out_path):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE="1", RANK="0")
    import torch
    import torch.distributed as dist
    from paper_1502_07806_b200 import sharded
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", world_size=1, rank=0, device_id=torch.device("cuda", 0))
    t = torch.arange(64, dtype=torch.float64, device="cuda").reshape(8, 8).contiguous()
    want = t.clone()
    sharded._all_gather_rows(t, 1, 0, force=True)          # in-place all_gather_into_tensor on the solve's stream
    v = torch.arange(8, dtype=torch.float64, device="cuda")
    sharded._all_gather_rows(v, 1, 0, force=True)
    torch.cuda.synchronize()
    ok = bool(torch.equal(t, want)) and bool(torch.equal(v, torch.arange(8, dtype=torch.float64, device="cuda")))
    open(out_path, "w").write("ok" if ok else "mismatch")
    dist.destroy_process_group()


def test_nccl_branch_of_the_row_gather_executes(tmp_path):
    """The box has one GPU, so the NCCL branch of sharded._all_gather_rows (in-place ncclAllGather through
    all_gather_into_tensor) can only run with world size 1: that still executes the call the multi-GPU bench makes
    (argument layout, contiguity, in-place form accepted by the backend) and must leave the buffer unchanged."""
    ctx = mp.get_context("spawn")
    out = str(tmp_path / "nccl.txt")
    pr = ctx.Process(target=_nccl_worker, args=(_free_port(), out))
    pr.start()
    pr.join(timeout=300)
    assert pr.exitcode == 0
    assert open(out).read() == "ok"


def test_bench_n_gt_1_path_dry_run_on_one_gpu():
    """`python bench.py --gpus 2` starts its own two ranks (torchrun re-exec) and runs the SHARDED solve, the N>1 default.
    The box has one GPU, so --share-gpu lets the ranks time-share it with host-staged (gloo) gathers: a dry run that
    executes the whole N>1 bench path -- self-launch, phase/gather events, e2e leg, max-over-ranks, the JSON line -- and
    must reproduce the single-GPU quality numbers.  Not a scaling number, and the line says so."""
    import json
    import subprocess
    common = ["--config", "0", "--steps", "2", "--no-syevd", "--no-calibrate", "--cpu-cols", "0"]
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--share-gpu", *common],
                         capture_output=True, text=True, timeout=600, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "strong" and "dry_run" in line
    assert "sharded over 2 ranks" in line["config"]["parallelism"]
    assert set(line["step_ms"]) >= {"phase1_steps2_3", "gather_V", "phase2_gram_rows", "gather_G",
                                    "phase3_cholesky_trsm_rows", "gather_VRinv", "phase4_step5_rows"}
    one = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *common], capture_output=True, text=True,
                         timeout=600, env=env)
    assert one.returncode == 0, one.stderr[-2000:]
    ref = json.loads(one.stdout.strip().splitlines()[-1])
    # the same run in peer-write mode (GEMM epilogues store into the other rank's buffers through CUDA IPC; barriers, no gathers)
    pw = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--share-gpu", "--peer-writes", *common],
                        capture_output=True, text=True, timeout=600, env=env)
    assert pw.returncode == 0, pw.stderr[-2000:]
    pwl = json.loads(pw.stdout.strip().splitlines()[-1])
    assert "peer-write mode" in pwl["config"]["parallelism"] and "barrier_after_phase3" in pwl["step_ms"]
    assert pwl["quality"] == line["quality"]                 # bit-for-bit the gather mode's result
    assert line["quality"]["info"] == 0 and ref["quality"]["info"] == 0
    assert abs(line["quality"]["max_residual"] - ref["quality"]["max_residual"]) < 1e-12
    assert line["quality"]["orthogonality_max"] <= 1e-12 * 256
    # without --share-gpu a rank without a GPU of its own is an error, not a silent single-rank run
    bad = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", *common], capture_output=True,
                         text=True, timeout=600, env=env)
    import torch
    if torch.cuda.device_count() < 2:
        assert bad.returncode != 0 and "has no GPU of its own" in bad.stderr


def _peer_worker(rank, world, port, N, P, w, iters, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank))
    import torch
    import torch.distributed as dist

    import paper_1502_07806_b200 as pfsm
    import pfsm_inputs as gen
    from paper_1502_07806_b200 import sharded
    dist.init_process_group("gloo", world_size=world, rank=rank)
    torch.cuda.set_device(0)
    p = gen.small_problem(N, 1e-3, 16.0, seed=4242)
    h = pfsm.Handle(N, P, w, iters, p.alpha)
    h.set_shard(rank, world)
    dA = torch.from_numpy(p.A).cuda()
    dV = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    dl = torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")
    peers = sharded.setup_peers(h, dV, dl)                 # CUDA IPC: the other process's buffers, mapped here
    for rep in range(2):                                   # twice: the second solve starts on top of the first one's buffers
        sharded.solve_sharded_peer_writes(h, dA, dV, dl, peers)
    torch.cuda.synchronize()
    np.savez(os.path.join(out_dir, f"peer{rank}.npz"), lam=dl.cpu().numpy(), V=dV.cpu().numpy(),
             res=h.residuals().cpu().numpy(), info=h.info())
    dist.barrier()
    peers.close()
    h.destroy()
    dist.destroy_process_group()


@pytest.mark.parametrize("N,P,w,iters", [(512, 4, 16, 2), (768, 6, 24, 3), (512, 4, 16, 0)])
def test_peer_write_mode_equals_gather_mode(tmp_path, N, P, w, iters):
    """Peer-write mode of the sharded solve: the GEMM epilogues store every finished tile into the other rank's buffers
    (mapped through CUDA IPC) and only barriers separate the phases.  Two processes time-share the one GPU -- IPC works
    between processes on one device, and no kernel of one rank waits on the other (phases are separated by a device
    synchronize + host barrier) -- so the whole mechanism (handle export / open, peer registration, the PEER epilogues of
    the UPDATE / Gram / panel GEMMs, the copy kernel for lambda and residuals, and for iters = 0 the start vectors) runs
    here exactly as it would across NVLink.  Must equal the gather mode bit for bit, on every rank."""
    world = 2
    ctx = mp.get_context("spawn")
    for target, port in ((_worker, _free_port()), (_peer_worker, _free_port())):
        procs = [ctx.Process(target=target, args=(r, world, port, N, P, w, iters, str(tmp_path))) for r in range(world)]
        for pr in procs:
            pr.start()
        for pr in procs:
            pr.join(timeout=300)
            assert pr.exitcode == 0
    for r in range(world):
        g = np.load(os.path.join(str(tmp_path), f"rank{r}.npz"))      # gather mode (host-staged gloo gathers)
        q = np.load(os.path.join(str(tmp_path), f"peer{r}.npz"))      # peer-write mode
        assert int(g["info"]) == 0 and int(q["info"]) == 0
        assert np.array_equal(q["lam"], g["lam"]) and np.array_equal(q["V"], g["V"]) and np.array_equal(q["res"], g["res"])
        assert not np.isnan(q["V"]).any() and not np.isnan(q["lam"]).any()
