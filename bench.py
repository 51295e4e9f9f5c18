#!/usr/bin/env python
"""bench.py -- one PFSM solve per step on synthetic matrices shaped like the paper's workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path (batched submatrix
eigensolves, folded-spectrum iterations, Cholesky-QR orthonormalization, Rayleigh quotients) over one
N x N matrix.  The metric is BASELINE.json's: ms per solve and sustained FP64 TFLOP/s, where the flops are
the ALGORITHMIC ones of SURVEY.md section 8(d):  F = (4 iters + 7/3) N^3 + 2 N^2 M.
Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FP64_NOMINAL_RATIO = 45.0 / 2250.0  # guide's nominal B200 FP64-tensor : bf16-tensor dense peaks
# dram__bytes_read.sum + dram__bytes_write.sum per full-k gemm_tn_kernel launch.  NOT measured in this run: ncu cannot
# run inside a timed bench, so the figure is copied from a committed `ncu --set full` capture of the same kernel at the
# same config (config index -> (bytes, file)); configs without a capture report null.
NCU_TRAFFIC_PER_GEMM_LAUNCH = {4: (8.126e9 + 0.528e9, "profiles/r02_ncu_full_gemm.md")}


def algorithmic_flops(N: int, M: int, iters: int) -> dict:
    f3 = 2.0 * N * N * M + (2 * iters - 1) * 2.0 * N ** 3 if iters > 0 else 0.0
    f4 = 7.0 * N ** 3 / 3.0
    f5 = 2.0 * N ** 3 + 5.0 * N * N
    return {"step3": f3, "step4": f4, "step5": f5, "total": f3 + f4 + f5}


def measured_peaks() -> dict:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "_source": "fallback"}


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons of one GPU while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, line in self.rows:
            if not (t0 - 0.05 <= t <= t1 + 0.05):
                continue
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples inside the timed region"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def oracle_sample(cfg_index: int, ncols: int, reps: int, warmup: int, min_seconds: float = 0.0, max_reps: int = 8):
    """Times the oracle, as it stands, on a bounded sample of config `cfg_index`: slice P/2's submatrix
    eigensolve (O2), then Eq. 11 (O3), Gram-Schmidt (O4) and the Rayleigh quotients (O5) for `ncols` of its eigenvectors.
    Returns (seconds per sample (list), flops per sample, description, threads)."""
    import numpy as np

    import oracle
    import pfsm_inputs as gen
    p = gen.problem(cfg_index)
    c = p.cfg
    N, m = c.N, c.m
    ncols = min(ncols, m)
    M, g0, lo, off = oracle.partition(N, c.P, c.window)
    s = c.P // 2
    times = []
    rep = -1
    while True:
        rep += 1
        if rep >= warmup + reps and (sum(times) >= min_seconds or len(times) >= max_reps):
            break
        t0 = time.perf_counter()
        B = p.A[lo[s]:lo[s] + M, lo[s]:lo[s] + M]
        mu, Y, _ = oracle.jacobi_eig(B)
        V0 = np.zeros((N, N))
        eps = np.zeros(N)
        c0, c1 = int(g0[s]), int(g0[s]) + ncols
        V0[c0:c1, lo[s]:lo[s] + M] = Y[:, off[s]:off[s] + ncols].T
        eps[c0:c1] = mu[off[s]:off[s] + ncols]
        V3 = oracle.step3(p.A, V0, eps, c.iters, p.alpha, c0, c1)
        Q, info = oracle.step4_mgs(V3[c0:c1])          # Gram-Schmidt among the sampled vectors (O4 on a subset)
        assert info == 0
        V3[c0:c1] = Q
        oracle.step5(p.A, V3, c0, c1)
        dt = time.perf_counter() - t0
        if rep >= warmup:
            times.append(dt)
    # algorithmic flops of the sample (same counting rule as the GPU line; step 2 excluded; step 4 = Gram-Schmidt of
    # ncols vectors of length N)
    flops = ncols * (2.0 * N * M + (2 * c.iters - 1) * 2.0 * N * N) + 2.0 * N * ncols * ncols + ncols * 2.0 * N * N
    desc = (f"config {cfg_index} (N={N}): slice {s}'s {M}x{M} Jacobi eigensolve, {c.iters} folded-spectrum iterations, "
            f"Gram-Schmidt and Rayleigh quotients for {ncols} of its {m} eigenvectors (steps O2-O5 on a subset)")
    return times, flops, desc, oracle.num_threads()


def whole_oracle_record(k: int, total_flops: float):
    """Wall time of ONE whole oracle solve (O1-O5, every eigenvector) of config k, recorded by
    tests/golden/make_golden_large.py when it wrote the config's golden file -- on the BUILD box, not on this host, so
    it is context beside the sampled figure, with its thread count.  None when the config has no such record."""
    path = os.path.join(ROOT, "tests", "golden", f"config{k}_oracle.txt")
    if not os.path.exists(path):
        return None
    rec = {}
    for ln in open(path):
        f = ln.split()
        if len(f) == 2 and f[0] in ("oracle_wall_s", "oracle_threads"):
            rec[f[0]] = float(f[1])
    if "oracle_wall_s" not in rec:
        return None
    return {"wall_s": rec["oracle_wall_s"], "threads": int(rec.get("oracle_threads", 0)),
            "tflops": total_flops / rec["oracle_wall_s"] * 1e-12,
            "where": "build box (recorded in tests/golden/config%d_oracle.txt), not this host" % k}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    k = args.config
    import pfsm_inputs as gen
    c = gen.config(k)
    times, flops, desc, threads = oracle_sample(k, args.cpu_cols if args.cpu_cols > 0 else 128, args.steps, args.warmup)
    total = sum(times)
    value = flops * len(times) / total * 1e-12
    line = {
        "impl": "reference",
        "metric": "PFSM solve sustained FP64 TFLOP/s (algorithmic flops / solve time)",
        "value": value, "unit": "TFLOP/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(c, args.gpus),
        "cpu_baseline": {"value": value, "unit": "TFLOP/s", "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def workload_config(c, n_gpus: int, sharded: bool = False, opts=None, peer_writes: bool = False) -> dict:
    origin = f"BASELINE.json configs[{c.index}]" if c.index <= 4 else "extra (SURVEY 8(f) f4)"
    return {"workload": f"{origin}: {c.name}, synthetic A = D + E",
            "N": c.N, "P": c.P, "window": c.window, "M": c.M, "iters": c.iters,
            "alpha": "0.5/max|d|^2", "replicas": 1 if sharded else n_gpus, "options": opts or "defaults (product path)",
            "parallelism": ((f"one solve sharded over {n_gpus} ranks (slices -> ranks; peer-write mode: GEMM epilogues store into the "
                             "other ranks' buffers, barriers between the 4 phases)" if peer_writes else
                             f"one solve sharded over {n_gpus} ranks (slices -> ranks, 4 all-gathers around step 4)") if sharded
                            else ("single GPU" if n_gpus == 1 else f"replicas x{n_gpus} (independent solves, no collective)")),
            "l2_policy": f"inputs larger than L2 (A, V, W are {8 * c.N * c.N / 2**20:.0f} MiB each vs 126 MB L2)"
            if 8 * c.N * c.N > 126e6 else "L2 flushed between timed iterations (256 MiB write)"}


def run_ours(args):
    import numpy as np
    import torch

    import paper_1502_07806_b200 as pfsm
    import pfsm_inputs as gen
    from paper_1502_07806_b200 import replicas

    world, rank, local_rank = replicas.env_world()
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; launch with torchrun --nproc-per-node "
                         f"{args.gpus}, or without WORLD_SIZE set (bench.py then starts the ranks itself)")
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the PFSM path has no CPU fallback")
    ndev = torch.cuda.device_count()
    if local_rank >= ndev and not args.share_gpu:
        raise SystemExit(f"bench.py: rank {rank} has no GPU of its own ({ndev} visible, --gpus {args.gpus}); "
                         "--share-gpu runs the N>1 code path with ranks time-sharing the GPUs (a dry run, not a scaling number)")
    dev_index = local_rank % ndev
    torch.cuda.set_device(dev_index)
    # NCCL needs one GPU per rank; the dry run stages its collectives through the host (gloo), so no kernel of one rank
    # ever waits on another rank's kernel
    backend = "gloo" if args.share_gpu else "nccl"
    coll_dev = "cpu" if backend == "gloo" else "cuda"
    replicas.init(backend, world, rank, torch.device("cuda", dev_index))
    n_gpus = world

    k = args.config
    # N > 1 default: ONE solve sharded over the ranks (strong scaling, all-gathers around step 4);
    # --replicas: rank r solves an independent matrix of the same config (weak scaling, no data-path collective)
    sharded_mode = world > 1 and not args.replicas
    prob = gen.problem(k, seed_offset=0 if sharded_mode else replicas.replica_seed_offset(rank))
    c = prob.cfg
    N = c.N
    flops = algorithmic_flops(N, c.M, c.iters)
    opts = {}
    for kv in args.option:
        key, _, val = kv.partition("=")
        opts[key] = int(val)
    h = pfsm.Handle(N, c.P, c.window, c.iters, prob.alpha, options=opts)
    if sharded_mode:
        from paper_1502_07806_b200 import sharded
        h.set_shard(rank, world)

    peers = None   # --peer-writes: the other ranks' buffers mapped through CUDA IPC (set up below, once dV / dl exist)

    def run_sharded(mark=None):
        if peers is not None:
            sharded.solve_sharded_peer_writes(h, dA, dV, dl, peers, mark=mark)
        else:
            sharded.solve_sharded(h, dA, dV, dl, mark=mark)

    def solve_once():
        if sharded_mode:
            run_sharded()
        else:
            h.solve(dA, dV, dl)

    stream = torch.cuda.current_stream()
    A_host = torch.from_numpy(prob.A).pin_memory()
    V_host = torch.empty((N, N), dtype=torch.float64).pin_memory()
    lam_host = torch.empty((N,), dtype=torch.float64).pin_memory()
    dA = A_host.cuda()
    dV = torch.empty((N, N), dtype=torch.float64, device="cuda")
    dl = torch.empty((N,), dtype=torch.float64, device="cuda")
    if sharded_mode and args.peer_writes:
        peers = sharded.setup_peers(h, dV, dl)
    flush = None
    if 8 * N * N <= 126e6:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        torch.cuda.synchronize()
        replicas.barrier(world)
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        return replicas.max_over_ranks(x, world, coll_dev)

    # ---- device-resident leg: K solves, CUDA events on the launching stream ----
    for _ in range(args.warmup):
        solve_once()
    barrier()
    assert replicas.all_ok(h.info() == 0, world, coll_dev), "PFSM reported a numerical breakdown on a bench matrix"
    sampler = ClockSampler(dev_index)
    sampler.start()
    time.sleep(0.3)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t_wall0 = time.time()
    # headline loop: the product launch sequence, step timing OFF (events between the steps would un-chain the Gram
    # product of step 4 from the last step-3 GEMM)
    for i in range(args.steps):
        if flush is not None:
            flush.fill_(i & 0xFF)
        ev[i][0].record(stream)
        solve_once()
        ev[i][1].record(stream)
    barrier()
    solve_ms = [a.elapsed_time(b) for a, b in ev]
    # second pass of the same K solves with the library's per-step events on: step times and the dominant kernel's
    # average launch duration (still inside the clock-sampled region, not part of `value`)
    step_ms = np.zeros(4)
    timed_ms = []
    phase_ms = {}
    if sharded_mode:
        marks = []

        def mark(label):
            e = torch.cuda.Event(enable_timing=True)
            e.record(stream)
            marks.append((label, e))
        for i in range(args.steps):
            run_sharded(mark=mark)
        torch.cuda.synchronize()
        per = len(marks) // args.steps
        for i in range(args.steps):
            seg = marks[i * per:(i + 1) * per]
            for (la, ea), (lb, eb) in zip(seg[:-1], seg[1:]):
                phase_ms[lb] = phase_ms.get(lb, 0.0) + ea.elapsed_time(eb) / args.steps
        phase_ms = {kk: max_over_ranks(v) for kk, v in phase_ms.items()}
    else:
        h.enable_step_timing(True)
        for i in range(args.steps):
            if flush is not None:
                flush.fill_(i & 0xFF)
            ev[i][0].record(stream)
            solve_once()
            ev[i][1].record(stream)
            ev[i][1].synchronize()
            step_ms += np.array(h.step_ms())
            timed_ms.append(ev[i][0].elapsed_time(ev[i][1]))
        h.enable_step_timing(False)
        step_ms /= args.steps
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1)
    total_ms = max_over_ranks(float(sum(solve_ms)))
    ms_per_step = total_ms / args.steps
    value = replicas.aggregate_tflops(flops["total"], args.steps, 1 if sharded_mode else world, total_ms)

    # ---- end-to-end leg: host buffers, copies inside the timed region.  One GPU / replicas: pfsm_solve_host (the
    # library overlaps the copies with steps 2 and 5).  Sharded: every rank uploads the replicated A, runs the sharded
    # solve and reads the complete V and lambda back.
    def e2e_once():
        if sharded_mode:
            dA.copy_(A_host, non_blocking=True)
            run_sharded()
            V_host.copy_(dV, non_blocking=True)
            lam_host.copy_(dl, non_blocking=True)
        else:
            h.solve_host(A_host, V_host, lam_host)

    e2e_steps = max(1, min(args.steps, 3))
    e2e_once()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(e2e_steps):
        e2e_once()
    e1.record(stream)
    barrier()
    e2e_ms = max_over_ranks(e0.elapsed_time(e1)) / e2e_steps
    e2e_value = replicas.aggregate_tflops(flops["total"], 1, 1 if sharded_mode else world, e2e_ms)
    lam = lam_host.numpy().copy()
    Vh = V_host.numpy()

    # ---- quality numbers of the result (BASELINE metric: "max residual/orthogonality") ----
    resid = h.residuals().cpu().numpy()
    dVt = torch.from_numpy(Vh).cuda()
    orth = float((dVt @ dVt.T - torch.eye(N, dtype=torch.float64, device="cuda")).abs().max().item())
    del dVt
    quality = {"max_residual": float(resid.max()), "orthogonality_max": orth,
               "trace_error": float(abs(lam.sum() - np.trace(prob.A))), "info": h.info(),
               "step2_jacobi_sweeps": h.step2_sweeps()}

    if rank != 0:
        replicas.finalize(world)
        return 0

    # ---- roofline of the dominant kernel (gemm_tn_kernel in step 3), live CUDA-event times ----
    # peak = the FP64 tensor (DMMA) issue rate measured in THIS run by the library's register-only probe: MEASURED_PEAKS.json
    # holds no FP64 figure, and the rule "bf16 measured x nominal ratio" (kept as proxy_*) cannot bound this pipe -- it is
    # scaled from a power-capped bf16 run at ~1.26 GHz while FP64 holds the full SM clock.
    peaks = measured_peaks()
    n_launch3 = 2 * c.iters
    if sharded_mode:
        gemm_ms = phase_ms["phase1_steps2_3"] / max(1, n_launch3)
        flops_per_launch = flops["step3"] / max(1, n_launch3) / world
    else:
        gemm_ms = step_ms[1] / max(1, n_launch3)
        flops_per_launch = flops["step3"] / max(1, n_launch3)
    achieved = flops_per_launch / (gemm_ms * 1e-3) * 1e-12 if n_launch3 and gemm_ms > 0 else 0.0
    probe_peak = pfsm.probe_fp64_peak(0)
    proxy_peak = peaks["bf16_tflops_sustained"] * FP64_NOMINAL_RATIO
    sms = torch.cuda.get_device_properties(dev_index).multi_processor_count
    clk_ghz = (clocks.get("sm_max_mhz") or 0.0) * 1e-3
    pipe_peak = sms * 64 * 2 * clk_ghz * 1e-3   # SMs x 64 FP64 FMA/clk/SM x 2 flop x max SM clock
    traffic = NCU_TRAFFIC_PER_GEMM_LAUNCH.get(k) if not sharded_mode else None
    roofline = {
        "bound": "tensor", "kernel": "gemm_tn_kernel (step 3, FP64 DMMA)", "achieved": achieved, "peak": probe_peak,
        "unit": "TFLOP/s", "frac": achieved / probe_peak if probe_peak > 0 else None,
        "traffic": traffic[0] if traffic else None,
        "traffic_source": (f"ncu --set full capture {traffic[1]} (same kernel, same config; NOT measured in this run)"
                           if traffic else "null: no committed ncu capture for this config / mode"),
        "algorithmic_bytes_per_launch": 32.0 * N * N,
        "peak_source": "FP64 DMMA issue-rate probe (pfsm_probe_fp64_peak, register-only mma.sync m8n8k4 f64 on every SM) "
                       "measured in this run; MEASURED_PEAKS.json has no FP64 entry",
        "fp64_pipe_peak_tflops": pipe_peak, "fp64_pipe_peak_rule": f"{sms} SMs x 64 FMA/clk x 2 x {clk_ghz:.3f} GHz",
        "frac_of_fp64_pipe": achieved / pipe_peak if pipe_peak > 0 else None,
        "proxy_peak": proxy_peak, "frac_vs_proxy": achieved / proxy_peak,
        "proxy_peak_rule": f"{peaks['_source']} bf16_tflops_sustained x nominal FP64:bf16 ratio 45/2250 (under-states the "
                           "FP64 pipe: secondary figure)",
        "avg_launch_ms": gemm_ms, "launches_per_step": n_launch3, "flops_per_launch": flops_per_launch,
        "note": ("achieved = algorithmic step-3 flops per launch / average launch time from the library's per-step CUDA "
                 "events, taken in a second pass of the same K solves; the headline `value` loop runs with step timing "
                 "off (the product launch sequence: step 4's Gram product chained to the last step-3 GEMM)"
                 if not sharded_mode else
                 "sharded: achieved = this rank's share of the step-3 flops / phase-1 time (phase 1 also holds step 2)"),
    }
    extra = {}
    if args.calibrate:
        extra["fp64_dmma_issue_peak_tflops"] = probe_peak
        extra["fp64_dfma_issue_peak_tflops"] = pfsm.probe_fp64_peak(1)
        a = torch.randn(8192, 8192, dtype=torch.float64, device="cuda")
        for _ in range(2):
            a @ a
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record()
        for _ in range(3):
            a @ a
        s1.record()
        torch.cuda.synchronize()
        extra["cublas_dgemm_8192_tflops"] = 3 * 2 * 8192.0 ** 3 / (s0.elapsed_time(s1) * 1e-3) * 1e-12
        del a
        roofline["frac_of_cublas_dgemm"] = achieved / extra["cublas_dgemm_8192_tflops"]
    if args.syevd:
        # comparison only, never the product: cuSOLVER dense syevd on the same matrix in the same run
        torch.linalg.eigh(dA[:256, :256].contiguous())
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record()
        w_ex, _ = torch.linalg.eigh(dA)
        s1.record()
        torch.cuda.synchronize()
        extra["cusolver_syevd_ms"] = s0.elapsed_time(s1)
        extra["max_abs_lambda_minus_syevd"] = float(np.abs(np.sort(lam) - w_ex.cpu().numpy()).max())

    if args.generalized:
        # row G (BASELINE configs[4] "also generalized form"): A x = lambda S x, S = I + 1e-4 perturbation, reduced by
        # Cholesky(S) inside pfsm_solve_generalized; reported beside the standard solve, not part of `value`
        pg = gen.problem(k, generalized=True, seed_offset=0 if sharded_mode else replicas.replica_seed_offset(rank))
        dS = torch.from_numpy(pg.S).cuda()
        dX = torch.empty((N, N), dtype=torch.float64, device="cuda")
        dlg = torch.empty((N,), dtype=torch.float64, device="cuda")
        for _ in range(2):
            h.solve_generalized(dA, dS, dX, dlg)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(stream)
        for _ in range(3):
            h.solve_generalized(dA, dS, dX, dlg)
        g1.record(stream)
        torch.cuda.synchronize()
        xsx = dX @ dS @ dX.T
        extra["generalized"] = {"ms_per_solve": g0.elapsed_time(g1) / 3, "info": h.info(),
                                "XtSX_minus_I_max": float((xsx - torch.eye(N, dtype=torch.float64, device="cuda")).abs().max().item()),
                                "max_residual": float(h.residuals().max().item())}
        del dS, dX, xsx

    # the sample is repeated until ~12 s of CPU work have been timed (at most 8 times), so a fast host still gives
    # a stable figure; the value is flops over the total time of the repeats
    if args.cpu_cols > 0 and world == 1:
        cpu_times, cpu_flops, cpu_desc, threads = oracle_sample(k, args.cpu_cols, 1, 0, min_seconds=args.cpu_seconds)
        cpu_value = cpu_flops * len(cpu_times) / sum(cpu_times) * 1e-12
        cpu_desc += f", repeated {len(cpu_times)}x"
    else:  # --cpu-cols 0: skipped (the 2048 x 2048 CPU Jacobi of config 6 alone takes minutes)
        import oracle
        cpu_times, cpu_value, threads = [0.0], None, oracle.num_threads()
        cpu_desc = ("skipped: the CPU-oracle leg runs at N=1 only (torchrun also pins OMP_NUM_THREADS=1 per rank)" if world > 1
                    else "skipped (--cpu-cols 0)")

    whole = whole_oracle_record(k, flops["total"])
    line = {
        "metric": "PFSM solve sustained FP64 TFLOP/s (algorithmic flops / solve time)",
        "value": value, "unit": "TFLOP/s", "n_gpus": n_gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if sharded_mode else "weak",
        "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": workload_config(c, n_gpus, sharded_mode, opts, peers is not None),
        "solve_ms": {"median": float(np.median(solve_ms)), "best": float(min(solve_ms))},
        "step_ms": ({"step2_submatrix_eig": step_ms[0], "step3_folded_spectrum": step_ms[1],
                     "step4_cholesky_qr": step_ms[2], "step5_rayleigh": step_ms[3],
                     "solve_with_step_events_median": float(np.median(timed_ms))} if not sharded_mode else phase_ms),
        "algorithmic_flops": flops, "quality": quality, "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "TFLOP/s", "ms_per_step": e2e_ms,
                # the lower block triangle of A (256-row blocks; A = A^T, mirrored on the device), plus the P diagonal
                # blocks sent ahead for step 2 (not when they are as large as A: wide windows)
                "h2d_bytes_per_step": (8 * N * N if sharded_mode else
                                       8 * sum(min(256, N - r0) * min(N, r0 + 256) for r0 in range(0, N, 256))
                                       + (8 * c.P * c.M * c.M if (c.M <= 160 or 2 * c.P * c.M * c.M <= N * N) else 0)),
                "d2h_bytes_per_step": 8 * N * N + 8 * N},
        "gpu_launches": int(args.steps * h.launches_per_solve()),
        "roofline": roofline,
        "cpu_baseline": {"value": cpu_value, "unit": "TFLOP/s", "cores": threads, "kind": "oracle",
                         "sample": cpu_desc, "seconds": sum(cpu_times), "whole_oracle_solve": whole},
        "workspace_bytes": h.workspace_bytes(),
    }
    if args.share_gpu:
        line["dry_run"] = (f"{world} ranks time-shared {min(world, ndev)} GPU(s), collectives staged through the host (gloo): "
                           "exercises the N>1 code path, NOT a scaling number")
    line.update(extra)
    print(json.dumps(line))
    replicas.finalize(world)
    return 0


def self_launch(args) -> int:
    """`python bench.py --gpus N` without a launcher: start the N ranks under torchrun exactly as the driver would
    (one process per GPU, NCCL over NVLink), and pass its exit code on.  The ranks see WORLD_SIZE and run the bench."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")          # rank / transport lines stay on stderr so a driver can count ranks
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index (default 4: N=8192); extra cases: 5 = Cu256-shaped N=1664, 6 = config 4 shape at gamma = 0.25 (M = 2048)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-cols", type=int, default=128, help="eigenvectors in the oracle sample that both the cpu_baseline leg and --impl reference time (0 = skip the CPU leg)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="repeat the cpu_baseline sample until this much CPU time is timed (max 8 repeats)")
    ap.add_argument("--replicas", action="store_true",
                    help="N>1: independent replicas (rank r solves its own matrix; weak scaling, no collective) instead of "
                         "the default, ONE solve sharded over the ranks (strong scaling)")
    ap.add_argument("--sharded", action="store_true", help="accepted for compatibility: sharding is the N>1 default")
    ap.add_argument("--peer-writes", action="store_true",
                    help="N>1 sharded solve in peer-write mode: GEMM epilogues store their tiles into the other ranks' buffers "
                         "(CUDA IPC peer memory over NVLink), barriers instead of all-gathers")
    ap.add_argument("--share-gpu", action="store_true",
                    help="dry run of the N>1 path on fewer GPUs than ranks: ranks time-share the GPUs, gloo instead of NCCL; "
                         "the line is marked dry_run and is not a scaling number")
    ap.add_argument("--generalized", action="store_true",
                    help="also time pfsm_solve_generalized on the config's matrix with S = I + 1e-4 perturbation (row G)")
    ap.add_argument("--option", action="append", default=[], metavar="KEY=INT",
                    help="pfsm_set_option setting for A/B measurements (include/pfsm.h lists the keys); default: product path")
    ap.add_argument("--no-syevd", dest="syevd", action="store_false")
    ap.add_argument("--no-calibrate", dest="calibrate", action="store_false")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return self_launch(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
