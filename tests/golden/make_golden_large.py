"""Writes tests/golden/config{3,4}_oracle.txt (+ config{3,4}_oracle_vectors.npz): the FULL oracle run of
BASELINE.json configs[3] and configs[4] (the headline bench config), every index.

Calls only pfsm_inputs (the seeded generator) and oracle/.  The paper (arXiv 1502.07806) prints no worked numerical
example, so these are the ORACLE's own outputs, not paper values: they let the GPU suite apply the north_star gates
(|dlambda| <= 1e-10 ||A||_F, |dr| <= 1e-9 ||A||_F, |deps| <= 1e-12 ||A||_F; PAPER.md:83-96 for the steps) to all N
eigenpairs of the two configs whose oracle run takes minutes, without running it inside the test.

Text file: header lines `key value`, then N lines `lambda_i resid_i eps_i` written with repr() (round-trips exactly).
The .npz holds a few whole eigenvectors (rows of Vr after step 4) for a sign-aligned vector comparison.
Run from the repo root:  python tests/golden/make_golden_large.py [3] [4]
"""
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import oracle  # noqa: E402
import pfsm_inputs as gen  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def sampled_vector_indices(N: int, m: int):
    """Eigenvector indices kept whole: both ends, a slice boundary, the middle."""
    return sorted({0, m - 1, m, N // 2 - 1, N // 2, N - m, N - 1})


def write_config(k: int) -> None:
    p = gen.problem(k)
    c = p.cfg
    t0 = time.perf_counter()
    r = oracle.pfsm(p.A, c.P, c.window, c.iters, p.alpha)
    wall = time.perf_counter() - t0
    assert r["info"] == 0
    Vr = r["Vr"]
    ortho = 0.0
    for i0 in range(0, c.N, 1024):               # ||V^T V - I||_max in row blocks (numpy product: a measurement only)
        blk = Vr[i0:i0 + 1024] @ Vr.T
        blk[np.arange(blk.shape[0]), i0 + np.arange(blk.shape[0])] -= 1.0
        ortho = max(ortho, float(np.abs(blk).max()))
    out = os.path.join(HERE, f"config{k}_oracle.txt")
    with open(out, "w") as f:
        f.write(f"# full oracle run of BASELINE.json configs[{k}] (N={c.N}, P={c.P}, window={c.window}, iters={c.iters})\n")
        f.write("# written by tests/golden/make_golden_large.py from oracle/ + pfsm_inputs/ only; not a paper value\n")
        f.write(f"N {c.N}\n")
        f.write(f"alpha {p.alpha!r}\n")
        f.write(f"normF {p.normF!r}\n")
        f.write(f"ortho_max {ortho!r}\n")
        f.write(f"sum_lambda {float(r['lam'].sum())!r}\n")
        f.write(f"oracle_wall_s {wall!r}\n")
        f.write(f"oracle_threads {oracle.num_threads()}\n")
        f.write("# lambda_i resid_i eps_i\n")
        for i in range(c.N):
            f.write(f"{float(r['lam'][i])!r} {float(r['resid'][i])!r} {float(r['eps'][i])!r}\n")
    idx = np.array(sampled_vector_indices(c.N, c.m), dtype=np.int64)
    np.savez(os.path.join(HERE, f"config{k}_oracle_vectors.npz"), idx=idx, Vr=Vr[idx])
    print(f"config {k}: {wall:.1f} s on {oracle.num_threads()} threads, ortho {ortho:.3e}, "
          f"max resid {r['resid'].max():.3e} -> {out}", flush=True)


if __name__ == "__main__":
    for k in ([int(a) for a in sys.argv[1:]] or [3, 4]):
        write_config(k)
