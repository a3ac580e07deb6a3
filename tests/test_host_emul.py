"""CPU check of the CUDA kernel bodies' index arithmetic: tests/host_emul/emul.cpp compiles the
__host__ __device__ bodies of the convolution passes with g++ and runs all CTAs sequentially.
The result is compared with the oracle.  (The GPU parity tests proper are tests/test_gpu_*.py.)"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

import oracle
from paper_2406_16064_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "host_emul", "emul.cpp")
LIB = os.path.join(ROOT, "tests", "host_emul", "libemul.so")
MU0 = 4e-7 * np.pi
_dp = C.POINTER(C.c_double)


@pytest.fixture(scope="module")
def emul():
    deps = [SRC] + [os.path.join(ROOT, "paper_2406_16064_b200", "csrc", f) for f in ("mm_fft.cuh", "mm_kernels.cuh", "mm_kernels2.cuh", "mm_passAC.cuh", "mm_passB7.cuh", "mm_passB3.cuh", "mm_passB4.cuh", "mm_llg.cuh")]
    if not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(d) for d in deps):
        subprocess.run(["g++", "-O1", "-std=c++17", "-fPIC", "-shared", "-o", LIB, SRC], check=True)
    L = C.CDLL(LIB)
    L.emul_demag.argtypes = [C.c_int] * 8 + [_dp] * 4
    L.emul_local.argtypes = [C.c_int] * 3 + [_dp, C.c_int, C.c_int, _dp, _dp, _dp, C.c_int, _dp]
    L.emul_local2.argtypes = [C.c_int] * 3 + [_dp, C.c_int, C.c_int, _dp, _dp, _dp, _dp, _dp, C.c_int, _dp]
    return L


def khat_full(o, nx, ny, nz):
    """Real part of the DFT of the wrapped oracle tensor, natural order [6, pz, py, px]."""
    px, py, pz = 2 * nx, 2 * ny, (2 * nz if nz > 1 else 1)
    K = np.zeros((6, pz, py, px))
    odd = {3: (1, 1, 0), 4: (1, 0, 1), 5: (0, 1, 1)}
    for c in range(6):
        T = o.demag_kernel(c)
        ox, oy, oz = odd.get(c, (0, 0, 0))
        for sz in ((1, -1) if nz > 1 else (1,)):
            for sy in (1, -1):
                for sx in (1, -1):
                    sgn = (sx if ox else 1) * (sy if oy else 1) * (sz if oz else 1)
                    kk = np.arange(nz) if sz > 0 else (pz - np.arange(1, nz))
                    jj = np.arange(ny) if sy > 0 else (py - np.arange(1, ny))
                    ii = np.arange(nx) if sx > 0 else (px - np.arange(1, nx))
                    src = T[(slice(None) if sz > 0 else slice(1, None)), :, :][:, (slice(None) if sy > 0 else slice(1, None)), :][:, :, (slice(None) if sx > 0 else slice(1, None))]
                    K[c][np.ix_(kk, jj, ii)] = sgn * src
    F = np.fft.fftn(K, axes=(1, 2, 3))
    assert np.abs(F.imag).max() < 1e-12 * np.abs(F.real).max()
    return np.ascontiguousarray(F.real)


@pytest.mark.parametrize("shape,cfg", [((16, 16, 1), (2, 8, 4)), ((32, 8, 1), (1, 8, 2)), ((8, 16, 4), (1, 4, 2)),
                                       ((16, 8, 2), (2, 8, 8)), ((64, 4, 8), (1, 16, 1)), ((4, 2, 1), (1, 8, 1)),
                                       ((32, 16, 1), (4, 8, 8)), ((64, 32, 2), (2, 8, 4)), ((32, 64, 16), (1, 8, 8)),
                                       ((128, 128, 1), (2, 8, 2)), ((256, 16, 4), (1, 8, 1)), ((32, 32, 32), (1, 8, 4))])
@pytest.mark.parametrize("prec64", [1, 0])
@pytest.mark.parametrize("ver", [1, 2, 3, 5, 42, 44])
def test_demag_passes_match_oracle(emul, shape, cfg, prec64, ver):
    nx, ny, nz = shape
    G, CH, TC = cfg
    cell = (2e-9, 1.5e-9, 3e-9)
    Ms = 8e5 * wl.random_mask(21, nx, ny, nz, 0.8)
    m = np.ascontiguousarray(wl.random_unit(22, nx, ny, nz) * (Ms > 0))
    o = oracle.Oracle(nx, ny, nz, *cell)
    o.set_Ms(Ms)
    o.init_demag()
    Href = o.field_terms(m, oracle.TERM_DEMAG)
    K = khat_full(o, nx, ny, nz)
    Hd = np.zeros(3 * nx * ny * nz)
    Msf = np.ascontiguousarray(Ms.reshape(-1))
    emul.emul_demag(ver, prec64, nx, ny, nz, G, CH, TC, K.ctypes.data_as(_dp), Msf.ctypes.data_as(_dp),
                    m.ctypes.data_as(_dp), Hd.ctypes.data_as(_dp))
    Hd = Hd.reshape(3, nz, ny, nx) * (Ms > 0)
    tol = 1e-12 if prec64 else 2e-5
    assert np.abs(Hd - Href).max() / 8e5 < tol


@pytest.mark.parametrize("kind", [wl.DMI_BULK, wl.DMI_INTERFACIAL])
def test_local_field_and_torque_match_oracle(emul, kind):
    nx, ny, nz = 8, 4, 4
    w = wl.cfg4(nx, ny, nz)
    w.dmi_kind = kind
    w.Ms = 8.6e5 * wl.random_mask(31, nx, ny, nz, 0.8)
    o = oracle.Oracle(nx, ny, nz, w.dx, w.dy, w.dz)
    wl.apply(o, w, with_demag=False)
    m = np.ascontiguousarray(w.m0 * (w.Ms > 0))
    d = (w.dx, w.dy, w.dz)
    u = np.array(w.axis) / np.linalg.norm(w.axis)
    gp = w.gamma / (1 + w.alpha**2)
    par = np.array([2 * w.A / (MU0 * x * x) for x in d] + [w.D / (MU0 * x) for x in d] + [2 * w.Ku / MU0] + list(u)
                   + list(w.H_ext) + [gp, w.alpha * gp])
    out = np.zeros(3 * w.N)
    Msf = np.ascontiguousarray(w.Ms.reshape(-1))
    for torque, ref in ((0, o.effective_field(m)), (1, o.llg_rhs(m))):
        emul.emul_local(nx, ny, nz, par.ctypes.data_as(_dp), kind, 15, Msf.ctypes.data_as(_dp), m.ctypes.data_as(_dp),
                        None, torque, out.ctypes.data_as(_dp))
        assert np.abs(out.reshape(ref.shape) - ref).max() <= 1e-12 * np.abs(ref).max()


@pytest.mark.parametrize("use", ["A", "D", "AD", "H", "Kc", "all"])
@pytest.mark.parametrize("kind", [wl.DMI_BULK, wl.DMI_INTERFACIAL, wl.DMI_D2D])
def test_cell_based_local_field_matches_oracle(emul, kind, use):
    """the library's per-cell arithmetic with cell-based A / D (harmonic-mean bonds),
    the D2d table, cubic anisotropy (Eq. 33) and a per-cell external field, compiled for the host, against the oracle."""
    nx, ny, nz = 8, 6, 4
    w = wl.cfg4(nx, ny, nz)
    w.Ms = 8.6e5 * wl.random_mask(33, nx, ny, nz, 0.8)
    wl.cell_params(w, 77, kind=kind, Kc=-3e4)
    if use in ("D", "H", "Kc"):
        w.A_cell = None
    if use in ("A", "H", "Kc"):
        w.D_cell = None
    if use not in ("H", "all"):
        w.H_ext_cell = None
    if use not in ("Kc", "all"):
        w.Kc = 0.0
    o = oracle.Oracle(nx, ny, nz, w.dx, w.dy, w.dz)
    wl.apply(o, w, with_demag=False)
    m = np.ascontiguousarray(w.m0 * (w.Ms > 0))
    d = (w.dx, w.dy, w.dz)
    u = np.array(w.axis) / np.linalg.norm(w.axis)
    gp = w.gamma / (1 + w.alpha**2)
    par = np.array([2 * (1.0 if w.A_cell is not None else w.A) / (MU0 * x * x) for x in d]
                   + [(1.0 if w.D_cell is not None else w.D) / (MU0 * x) for x in d] + [2 * w.Ku / MU0] + list(u)
                   + list(w.H_ext) + [gp, w.alpha * gp, 4 * w.Kc / MU0])
    out = np.zeros(3 * w.N)
    Msf = np.ascontiguousarray(w.Ms.reshape(-1))
    ptr = lambda a: None if a is None else np.ascontiguousarray(a).ctypes.data_as(_dp)
    arrs = [None if a is None else np.ascontiguousarray(a, dtype=np.float64) for a in (w.A_cell, w.D_cell, w.H_ext_cell)]
    for torque, ref in ((0, o.effective_field(m)), (1, o.llg_rhs(m))):
        emul.emul_local2(nx, ny, nz, par.ctypes.data_as(_dp), kind, 15 | 32, Msf.ctypes.data_as(_dp), m.ctypes.data_as(_dp),
                         ptr(arrs[0]), ptr(arrs[1]), ptr(arrs[2]), torque, out.ctypes.data_as(_dp))
        assert np.abs(out.reshape(ref.shape) - ref).max() <= 1e-12 * np.abs(ref).max()


@pytest.mark.parametrize("prec64", [0, 1])
@pytest.mark.parametrize("shape", [(16, 16, 1), (8, 32, 2), (32, 64, 1), (8, 128, 2), (4, 256, 1), (4, 512, 1), (4, 512, 2), (16, 64, 4), (4, 1024, 1), (4, 1024, 2)])
def test_specialised_pass_B_matches_oracle(emul, shape, prec64):
    """mm_passB7.cuh (compile-time ny; fp32 with TC = 4, fp64 with TC = 2): every instantiated ny, films and 3-D."""
    nx, ny, nz = shape
    cell = (2e-9, 1.5e-9, 3e-9)
    Ms = 8e5 * wl.random_mask(23, nx, ny, nz, 0.8)
    m = np.ascontiguousarray(wl.random_unit(24, nx, ny, nz) * (Ms > 0))
    o = oracle.Oracle(nx, ny, nz, *cell)
    o.set_Ms(Ms)
    o.init_demag()
    Href = o.field_terms(m, oracle.TERM_DEMAG)
    K = khat_full(o, nx, ny, nz)
    Hd = np.zeros(3 * nx * ny * nz)
    Msf = np.ascontiguousarray(Ms.reshape(-1))
    for tc in ((2,) if prec64 else (4, 2)):      # fp32 also with 2-column tiles (the library's ny = 512 / 1024 form)
        emul.emul_demag(7, prec64, nx, ny, nz, 1, 8, tc, K.ctypes.data_as(_dp), Msf.ctypes.data_as(_dp), m.ctypes.data_as(_dp),
                        Hd.ctypes.data_as(_dp))
        H2 = Hd.reshape(3, nz, ny, nx) * (Ms > 0)
        assert np.abs(H2 - Href).max() / 8e5 < (1e-12 if prec64 else 2e-5)
