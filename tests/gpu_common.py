"""Shared helpers of the GPU parity tests: build an oracle and an mm Sim from the same Workload."""
import numpy as np

import oracle
from paper_2406_16064_b200 import workloads as wl


def make_pair(w, prec, demag=None, oracle_demag=None):
    from paper_2406_16064_b200 import Sim
    o = oracle.Oracle(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz)
    wl.apply(o, w, with_demag=demag)
    if oracle_demag is not None:
        o.set_demag(oracle_demag)
    s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=prec)
    wl.apply(s, w, with_demag=demag)
    return o, s


def masked_m(w):
    Ms = w.Ms_array()
    return np.ascontiguousarray(w.m0 * (Ms > 0))


def to_np(t):
    return t.detach().cpu().numpy().astype(np.float64)


def avg_m(m, Ms):
    live = Ms > 0
    return np.array([m[c][live].mean() for c in range(3)])
