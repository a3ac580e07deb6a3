"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic: it only draws seeded random numbers,
builds masks and packs parameters.  It is the one module both the oracle-side tests and
the CUDA binding's tests/bench import (neither the oracle nor the CUDA path imports it).

Arrays: m is float64 [3, nz, ny, nx] (x fastest, SoA), Ms is float64 [nz, ny, nx].
"""
from dataclasses import dataclass, field

import numpy as np

MU0 = 4e-7 * np.pi
DMI_NONE, DMI_BULK, DMI_INTERFACIAL, DMI_D2D = 0, 1, 2, 3
RK4, DOPRI5, CAYLEY_RK4 = 0, 1, 2


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    Ms: object                      # float or ndarray [nz, ny, nx]
    A: float = 0.0
    D: float = 0.0
    dmi_kind: int = DMI_NONE
    Ku: float = 0.0
    axis: tuple = (0.0, 0.0, 1.0)
    H_ext: tuple = (0.0, 0.0, 0.0)
    alpha: float = 0.5
    gamma: float = 2.211e5
    integrator: int = DOPRI5
    demag: bool = True
    dt: float = 1e-14
    m0: np.ndarray = field(default=None, repr=False)
    seed: int = 0
    Kc: float = 0.0                 # cubic anisotropy constant (Eq. 33)
    A_cell: object = field(default=None, repr=False)       # ndarray [nz, ny, nx] or None: cell-based A
    D_cell: object = field(default=None, repr=False)       # ndarray [nz, ny, nx] or None: cell-based D
    H_ext_cell: object = field(default=None, repr=False)   # ndarray [3, nz, ny, nx] or None: per-cell external field

    @property
    def N(self):
        return self.nx * self.ny * self.nz

    @property
    def Ms_max(self):
        return float(np.max(self.Ms))

    def Ms_array(self):
        if np.isscalar(self.Ms):
            return np.full((self.nz, self.ny, self.nx), float(self.Ms))
        return np.asarray(self.Ms, dtype=np.float64)


def random_unit(seed, nx, ny, nz):
    """Normal 3-vector per cell, normalised (BASELINE.json config 1 wording)."""
    rng = np.random.default_rng(seed)
    v = rng.standard_normal((3, nz, ny, nx))
    v /= np.sqrt((v * v).sum(axis=0, keepdims=True))
    return v


def random_mask(seed, nx, ny, nz, fill=0.8):
    rng = np.random.default_rng(seed)
    return (rng.random((nz, ny, nx)) < fill).astype(np.float64)


def cell_params(w, seed, kind=None, Kc=0.0, zero_fraction=0.1):
    """Cell-based material constants in the structure of a granular / multilayer sample ("cell-based",
    :120, :175): A_i and D_i = the workload's uniform values x a seeded factor in [0.5, 1.5], piecewise constant on
    4 x 4 x 2 grains with a sharp interface at mid-x (factor x 0.5 on the right half); D_i = 0 in a seeded fraction
    of the cells (bond value 0 towards them); a per-cell external field = uniform value + a seeded smooth gradient +
    noise.  Draws random numbers only; the bond arithmetic lives in the oracle and in the library."""
    rng = np.random.default_rng(seed)
    gx, gy, gz = -(-w.nx // 4), -(-w.ny // 4), -(-w.nz // 2)
    grain = rng.uniform(0.5, 1.5, (2, gz, gy, gx))
    up = [np.repeat(np.repeat(np.repeat(g, 2, axis=0), 4, axis=1), 4, axis=2)[:w.nz, :w.ny, :w.nx] for g in grain]
    half = np.where(np.arange(w.nx) >= w.nx // 2, 0.5, 1.0)[None, None, :]
    A0 = w.A if w.A != 0.0 else 1.3e-11
    D0 = w.D if w.D != 0.0 else 1.5e-3
    w.A_cell = A0 * up[0] * half
    w.D_cell = D0 * up[1] * (rng.random((w.nz, w.ny, w.nx)) >= zero_fraction)
    if kind is not None:
        w.dmi_kind = kind
    x = (np.arange(w.nx) + 0.5) / w.nx
    H = np.empty((3, w.nz, w.ny, w.nx))
    for c in range(3):
        H[c] = w.H_ext[c] + 2e4 * (x[None, None, :] - 0.5) * (c + 1) + 1e3 * rng.standard_normal((w.nz, w.ny, w.nx))
    w.H_ext_cell = H
    w.Kc = Kc
    return w


def apply(sim, w, with_demag=None):
    """Push a Workload's parameters into any object with the mm_*/mo_* setter names."""
    sim.set_Ms(w.Ms if np.isscalar(w.Ms) else w.Ms_array())
    sim.set_A(w.A)
    sim.set_D(w.D, w.dmi_kind)
    sim.set_Ku(w.Ku)
    sim.set_axis(*w.axis)
    sim.set_H_ext(*w.H_ext)
    if w.Kc != 0.0:
        sim.set_Kc(w.Kc)
    if w.A_cell is not None:
        sim.set_A_cell(np.ascontiguousarray(w.A_cell, dtype=np.float64))
    if w.D_cell is not None:
        sim.set_D_cell(np.ascontiguousarray(w.D_cell, dtype=np.float64), w.dmi_kind)
    if w.H_ext_cell is not None:
        sim.set_H_ext_cell(np.ascontiguousarray(w.H_ext_cell, dtype=np.float64))
    sim.set_alpha(w.alpha)
    sim.set_gamma(w.gamma)
    sim.set_integrator(w.integrator)
    demag = w.demag if with_demag is None else with_demag
    sim.set_demag(1 if demag else 0)
    if demag:
        sim.init_demag()
    return sim


def cfg1():
    """Tiny film 16x16x1, 2 nm cubes, fp64, RK4 dt=1e-14 (configs[0])."""
    w = Workload("cfg1_tiny_film_16x16x1", 16, 16, 1, 2e-9, 2e-9, 2e-9, Ms=8.0e5, A=1.3e-11, alpha=0.5,
                 gamma=2.211e5, H_ext=(0.0, 0.0, 1e5), integrator=RK4, dt=1e-14, seed=1001)
    w.m0 = random_unit(1001, 16, 16, 1)
    return w


def cfg2():
    """Permalloy strip 128x32x1 of 3.90625 x 3.90625 x 3 nm (configs[1]); the geometry of the paper's
    §VIII.E run with BASELINE.json's own initial tilt."""
    nx, ny, nz = 128, 32, 1
    rng = np.random.default_rng(1002)
    m = np.empty((3, nz, ny, nx))
    m[0], m[1], m[2] = 1.0, 0.1, 0.1
    m /= np.sqrt((m * m).sum(axis=0, keepdims=True))
    m += 1e-3 * rng.standard_normal(m.shape)
    m /= np.sqrt((m * m).sum(axis=0, keepdims=True))
    w = Workload("cfg2_strip_128x32x1", nx, ny, nz, 3.90625e-9, 3.90625e-9, 3e-9, Ms=8.0e5, A=1.3e-11,
                 alpha=0.02, integrator=DOPRI5, dt=2e-14, seed=1002)
    w.m0 = m
    return w


CFG2_FIELD = (-19.6e-3 / MU0, 3.4e-3 / MU0, 0.0)      # (-19.6, 3.4, 0) mT / mu0 in A/m


def cfg3(n=256):
    """Skyrmion disk n x n x 1 of 2x2x1 nm (configs[2] at n=256): Ms inside radius 200 nm (scaled with n),
    reversed core of radius 20 nm, 1e-3 seeded noise (R14)."""
    nx = ny = n
    dx = dy = 2e-9
    scale = n / 256.0
    cx, cy, Rd, Rc = 256e-9 * scale, 256e-9 * scale, 200e-9 * scale, 20e-9 * scale
    xc = (np.arange(nx) + 0.5) * dx
    yc = (np.arange(ny) + 0.5) * dy
    X, Y = np.meshgrid(xc, yc, indexing="xy")
    r2 = (X - cx) ** 2 + (Y - cy) ** 2
    inside = (r2 <= Rd * Rd)
    Ms = np.where(inside, 5.8e5, 0.0)[None, :, :]
    rng = np.random.default_rng(1003)
    m = np.zeros((3, 1, ny, nx))
    m[2, 0] = np.where(r2 < Rc * Rc, -1.0, 1.0)
    m += 1e-3 * rng.standard_normal(m.shape)
    m /= np.sqrt((m * m).sum(axis=0, keepdims=True))
    m *= inside[None, None, :, :]
    w = Workload(f"cfg3_skyrmion_disk_{n}x{n}x1", nx, ny, 1, dx, dy, 1e-9, Ms=Ms, A=1.5e-11, D=3.0e-3,
                 dmi_kind=DMI_INTERFACIAL, Ku=8.0e5, axis=(0.0, 0.0, 1.0), alpha=0.3, integrator=DOPRI5,
                 dt=2e-14, seed=1003)
    w.m0 = m
    return w


def cfg4(nx=512, ny=512, nz=16, with_m=True):
    """3-D slab nx x ny x nz of 2.5 nm cubes (configs[3] at 512x512x16); DOPRI5 fixed dt=5e-14."""
    w = Workload(f"cfg4_slab_{nx}x{ny}x{nz}", nx, ny, nz, 2.5e-9, 2.5e-9, 2.5e-9, Ms=8.6e5, A=1.3e-11,
                 D=1.5e-3, dmi_kind=DMI_BULK, Ku=5e4, axis=(1.0, 0.0, 0.0), alpha=0.1,
                 H_ext=(0.0, 0.0, 5e4), integrator=DOPRI5, dt=5e-14, seed=1004)
    if with_m:
        w.m0 = random_unit(1004, nx, ny, nz)
    return w


def cfg5(n, with_m=True):
    """Throughput-sweep film n x n x 1 of 4 nm cubes (configs[4]); demag + exchange + Zeeman."""
    seed = 2000 + int(round(np.log2(n)))
    w = Workload(f"cfg5_film_{n}x{n}x1", n, n, 1, 4e-9, 4e-9, 4e-9, Ms=8e5, A=1.3e-11, alpha=0.02,
                 H_ext=(0.0, 0.0, 1e4), integrator=DOPRI5, dt=2e-14, seed=seed)
    if with_m:
        w.m0 = random_unit(seed, n, n, 1)
    return w
