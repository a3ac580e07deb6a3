"""Writes tests/golden/cfg2_trajectory.txt: <m>(t) of BASELINE.json configs[1] at the ten 0.1 ns marks, computed by the
ORACLE alone (oracle/ + the seeded input generators; nothing from the CUDA library).

Procedure (PAPER.md:487-489 for the shape of the problem): the 128 x 32 x 1 permalloy strip,
m0 = (1, 0.1, 0.1) normalised + 1e-3 seeded noise; relax with alpha = 0.5 by adaptive DOPRI5 (tol 1e-6, first trial step
1e-13 s) until max|dm/dt| < 1e7 rad/s; then alpha = 0.02, H_ext = (-19.6, 3.4, 0) mT / mu0, t = 0, and adaptive DOPRI5
(tol 1e-6, first trial step 1e-13 s at every mark, last step of each leg clipped to the mark) to 1 ns.

Run from the repository root:  python tests/golden/make_cfg2_trajectory.py      (about ten minutes on 8 cores)
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle                                             # noqa: E402
from paper_2406_16064_b200 import workloads as wl          # noqa: E402  (seeded inputs only)


def main():
    w = wl.cfg2()
    w.alpha = 0.5
    o = oracle.Oracle(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz)
    wl.apply(o, w)
    Ms = w.Ms_array()
    m = np.ascontiguousarray(w.m0 * (Ms > 0))
    tol = 1e-6
    n_relax, md = o.relax(m, tol, 1e7, 200000, 1e-13)
    assert md < 1e7
    o.set_alpha(0.02)
    o.set_H_ext(*wl.CFG2_FIELD)
    o.set_time(0.0)
    live = Ms > 0
    lines = ["# <m> of configs[1] (128 x 32 x 1 strip) at t = k * 0.1 ns, k = 0..10, from the oracle alone.",
             "# Written by tests/golden/make_cfg2_trajectory.py (see its docstring for the procedure); do not edit.",
             f"relax_steps = {n_relax}",
             "m_0 = " + " ".join(f"{m[c][live].mean():.15e}" for c in range(3))]
    total = 0
    for k in range(1, 11):
        t_end = k * 1e-10
        dt = 1e-13
        while o.time() < t_end * (1 - 1e-12):
            dt = min(dt, t_end - o.time())
            ok, err, dn, _ = o.step(m, dt, tol)
            dt = dn
            total += 1
        lines.append(f"m_{k} = " + " ".join(f"{m[c][live].mean():.15e}" for c in range(3)))
        print(lines[-1], flush=True)
    lines.append(f"run_attempts = {total}")
    with open(os.path.join(ROOT, "tests", "golden", "cfg2_trajectory.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
