"""Writes tests/golden/config0_oracle.txt.  Calls only pfsm_inputs (the seeded generator) and oracle/.

The paper (arXiv 1502.07806) prints no worked numerical example, so there is no paper-cited fixture;
this file freezes the ORACLE's own summary values for BASELINE.json configs[0] so that a later change
to the oracle's arithmetic is noticed (and must be justified in its commit message).
Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import oracle  # noqa: E402
import pfsm_inputs as gen  # noqa: E402

p = gen.problem(0)
c = p.cfg
r = oracle.pfsm(p.A, c.P, c.window, c.iters, p.alpha)
assert r["info"] == 0
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config0_oracle.txt")
with open(out, "w") as f:
    f.write("# oracle summary for BASELINE.json configs[0] (N=256, P=4, window=16, iters=3, alpha=0.5/max|d|^2)\n")
    f.write("# written by tests/golden/make_golden.py from oracle/ only; not a paper value (the paper prints none)\n")
    f.write(f"alpha {p.alpha!r}\n")
    f.write(f"normF {p.normF!r}\n")
    f.write(f"sum_lambda {float(r['lam'].sum())!r}\n")
    f.write(f"lambda_0 {float(r['lam'][0])!r}\n")
    f.write(f"lambda_255 {float(r['lam'][-1])!r}\n")
    f.write(f"max_resid {float(r['resid'].max())!r}\n")
print(open(out).read())
