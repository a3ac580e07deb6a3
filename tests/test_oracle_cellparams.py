"""Pins for the oracle's SURVEY 8(f)2 terms: cell-based A and D with harmonic means, the D2d DMI
table, cubic anisotropy (Eq. 33-34) and a per-cell external field (Eq. 35)."""
import numpy as np
import pytest

import oracle
from paper_2406_16064_b200 import workloads as wl

MU0 = 4e-7 * np.pi
Ms = 8e5


def chain(n, d=2e-9):
    o = oracle.Oracle(n, 1, 1, d, d, d)
    o.set_Ms(Ms); o.set_demag(0)
    return o


def test_harmonic_mean_exchange_hand_values():
    """4-cell chain, A = (A1, A1, A2, A2): the bond across the interface carries A12 = 2 A1 A2/(A1 + A2)."""
    A1, A2, d = 1.0e-11, 3.0e-11, 2e-9
    o = chain(4, d)
    o.set_A_cell(np.array([A1, A1, A2, A2]))
    th = np.array([0.0, 0.3, 0.9, 1.0])
    m = np.zeros((3, 1, 1, 4)); m[0, 0, 0] = np.cos(th); m[1, 0, 0] = np.sin(th)
    H = o.field_terms(m, oracle.TERM_EXCHANGE).reshape(3, 4)
    mm = m.reshape(3, 4)
    A12 = 2 * A1 * A2 / (A1 + A2)
    c = 2.0 / (MU0 * Ms * d * d)
    ref1 = c * (A1 * (mm[:, 0] - mm[:, 1]) + A12 * (mm[:, 2] - mm[:, 1]))
    ref2 = c * (A12 * (mm[:, 1] - mm[:, 2]) + A2 * (mm[:, 3] - mm[:, 2]))
    assert np.allclose(H[:, 1], ref1, rtol=1e-14) and np.allclose(H[:, 2], ref2, rtol=1e-14)
    assert np.isclose(A12, 1.5e-11)


def test_cell_arrays_reduce_to_the_uniform_constants():
    nx, ny, nz = 6, 5, 3
    w = wl.cfg4(8, 8, 2)
    mask = wl.random_mask(3, nx, ny, nz, 0.8)
    m = np.ascontiguousarray(wl.random_unit(4, nx, ny, nz) * mask)
    for kind in (oracle.DMI_BULK, oracle.DMI_INTERFACIAL, oracle.DMI_D2D):
        o = oracle.Oracle(nx, ny, nz, 2e-9, 1.5e-9, 3e-9)
        o.set_Ms(Ms * mask); o.set_demag(0); o.set_A(1.3e-11); o.set_D(1.5e-3, kind); o.set_H_ext(1e4, -2e4, 3e4)
        Href = o.effective_field(m)
        o.set_A(0.0); o.set_D(0.0, kind); o.set_H_ext(0, 0, 0)
        o.set_A_cell(np.full((nz, ny, nx), 1.3e-11)); o.set_D_cell(np.full((nz, ny, nx), 1.5e-3), kind)
        Hc = np.zeros((3, nz, ny, nx)); Hc[0], Hc[1], Hc[2] = 1e4, -2e4, 3e4
        o.set_H_ext_cell(Hc)
        assert np.allclose(o.effective_field(m), Href, rtol=0, atol=1e-9 * np.abs(Href).max())


def test_symmetric_bonds_exert_no_net_torque_and_vanishing_A_decouples():
    """A_ij = A_ji (harmonic mean): sum_i Ms_i m_i x H_ex,i = 0.  A region with A = 0 is decoupled (A_ij = 0)."""
    nx, ny, nz = 6, 4, 3
    rng = np.random.default_rng(8)
    Acell = 1e-11 * (0.5 + rng.random((nz, ny, nx)))
    Acell[:, :, 3:] *= 0.0
    Acell[:, :, 4:] = 2e-11
    m = np.ascontiguousarray(wl.random_unit(9, nx, ny, nz))
    o = oracle.Oracle(nx, ny, nz, 2e-9, 2e-9, 2e-9)
    o.set_Ms(Ms); o.set_demag(0); o.set_A_cell(Acell)
    H = o.field_terms(m, oracle.TERM_EXCHANGE)
    tq = np.cross(m.reshape(3, -1).T, H.reshape(3, -1).T).sum(axis=0)
    assert np.abs(tq).max() <= 1e-12 * np.abs(H).max() * m[0].size
    assert np.all(H[:, :, :, 3] == 0.0)            # the A = 0 plane feels nothing ...
    m2 = m.copy(); m2[:, :, :, 3] = wl.random_unit(10, 1, ny, nz).reshape(3, nz, ny)
    H2 = o.field_terms(m2, oracle.TERM_EXCHANGE)
    assert np.array_equal(H2[:, :, :, :3], H[:, :, :, :3]) and np.array_equal(H2[:, :, :, 4:], H[:, :, :, 4:])   # ... and nobody feels it


def test_d2d_helices_closed_form():
    """Eq. 14 / the D2d row of PAPER.md:175 on two helices (derived from Eq. 15 with e_ij = {e_x,-e_x,-e_y,e_y}):
    m = (0, cos qx, sin qx) and m = (cos qy, 0, sin qy) both give interior H = -(2 D sin(q d)/(mu0 Ms d)) m."""
    D, d, q, n = 2e-3, 2e-9, 2 * np.pi / 32e-9, 32
    x = (np.arange(n) + 0.5) * d
    for axis in (0, 1):
        shape = (n, 4, 1) if axis == 0 else (4, n, 1)
        o = oracle.Oracle(*shape, d, d, d)
        o.set_Ms(Ms); o.set_demag(0); o.set_D(D, oracle.DMI_D2D)
        m = np.zeros((3, 1, shape[1], shape[0]))
        ph = (q * x)[None, :] if axis == 0 else (q * x)[:, None]
        if axis == 0:
            m[1, 0] = np.cos(ph); m[2, 0] = np.sin(ph)
        else:
            m[0, 0] = np.cos(ph); m[2, 0] = np.sin(ph)
        H = o.field_terms(m, oracle.TERM_DMI)
        ref = -(2 * D * np.sin(q * d) / (MU0 * Ms * d)) * m
        inner = (slice(None), 0, slice(1, 3), slice(1, n - 1)) if axis == 0 else (slice(None), 0, slice(1, n - 1), slice(1, 3))
        assert np.allclose(H[inner], ref[inner], rtol=1e-12, atol=1e-9 * np.abs(ref).max())


def test_d2d_matches_eq14_by_central_differences():
    nx, ny, d, D = 12, 10, 1e-9, 1e-3
    X, Y = np.meshgrid((np.arange(nx) + 0.5) * d, (np.arange(ny) + 0.5) * d, indexing="xy")
    th, ph = 0.4 + 3e7 * X + 2e7 * Y, 1.1 - 2.5e7 * X + 4e7 * Y
    m = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)])[:, None, :, :]
    o = oracle.Oracle(nx, ny, 1, d, d, d)
    o.set_Ms(Ms); o.set_demag(0); o.set_D(D, oracle.DMI_D2D)
    H = o.field_terms(np.ascontiguousarray(m), oracle.TERM_DMI)[:, 0]
    mm = m[:, 0]
    dmx = (mm[:, 1:-1, 2:] - mm[:, 1:-1, :-2]) / (2 * d)
    dmy = (mm[:, 2:, 1:-1] - mm[:, :-2, 1:-1]) / (2 * d)
    ex, ey = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    cr = lambda e, v: np.stack([e[1] * v[2] - e[2] * v[1], e[2] * v[0] - e[0] * v[2], e[0] * v[1] - e[1] * v[0]])
    ref = -(2 * D / (MU0 * Ms)) * (cr(ey, dmy) - cr(ex, dmx))          # Eq. 14
    assert np.allclose(H[:, 1:-1, 1:-1], ref, rtol=1e-12, atol=1e-9 * np.abs(ref).max())


def test_cubic_anisotropy_field_and_energy():
    Kc = 4.5e4
    o = oracle.Oracle(1, 1, 1, 2e-9, 2e-9, 2e-9)
    o.set_Ms(Ms); o.set_demag(0); o.set_Kc(Kc)
    V = 8e-27
    for v in ([1.0, 0, 0], [1.0, 1.0, 1.0], [0.2, -0.5, 0.7]):
        u = np.array(v) / np.linalg.norm(v)
        m = u.reshape(3, 1, 1, 1).copy()
        H = o.field_terms(m, oracle.TERM_CUBIC).reshape(3)
        assert np.allclose(H, -4 * Kc / (MU0 * Ms) * u**3, rtol=1e-14)           # -(1/(mu0 Ms)) d/dm of Eq. 33
        E, terms = o.energy(m)
        assert np.isclose(E, Kc * V * (u**4).sum(), rtol=1e-13) and np.isclose(terms[3], E)
        # Eq. 34: the same energy up to the constant Kc V
        assert np.isclose(E - Kc * V, -2 * Kc * V * (u[0]**2 * u[1]**2 + u[1]**2 * u[2]**2 + u[2]**2 * u[0]**2), rtol=1e-12)
    # <111> is the easy direction for Kc > 0, <100> the hard one
    e100 = o.energy(np.array([1.0, 0, 0]).reshape(3, 1, 1, 1))[0]
    e111 = o.energy((np.ones(3) / np.sqrt(3)).reshape(3, 1, 1, 1))[0]
    assert np.isclose(e111, e100 / 3)
    # the field is the energy gradient: dE = -mu0 Ms V H . dm for a tangential dm
    u = np.array([0.2, -0.5, 0.7]); u /= np.linalg.norm(u)
    t = np.cross(u, [0, 0, 1.0]); t /= np.linalg.norm(t)
    eps = 1e-6
    up, um = u + eps * t, u - eps * t
    up /= np.linalg.norm(up); um /= np.linalg.norm(um)
    dE = (o.energy(up.reshape(3, 1, 1, 1).copy())[0] - o.energy(um.reshape(3, 1, 1, 1).copy())[0]) / (2 * eps)
    H = o.field_terms(u.reshape(3, 1, 1, 1).copy(), oracle.TERM_CUBIC).reshape(3)
    assert np.isclose(dE, -MU0 * Ms * V * (H @ t), rtol=1e-6)


def test_per_cell_external_field_and_zeeman_energy():
    nx, ny, nz = 4, 3, 2
    rng = np.random.default_rng(12)
    Hc = 1e5 * rng.standard_normal((3, nz, ny, nx))
    mask = wl.random_mask(13, nx, ny, nz, 0.8)
    m = np.ascontiguousarray(wl.random_unit(14, nx, ny, nz) * mask)
    o = oracle.Oracle(nx, ny, nz, 1e-9, 2e-9, 3e-9)
    o.set_Ms(Ms * mask); o.set_demag(0); o.set_H_ext(7e4, 0, 0); o.set_H_ext_cell(Hc)
    H = o.field_terms(m, oracle.TERM_ZEEMAN)
    assert np.array_equal(H, Hc * mask)                     # Eq. 35: the field itself; zero where Ms = 0
    E, terms = o.energy(m)
    assert np.isclose(terms[4], -MU0 * 6e-27 * Ms * (mask * (m * Hc).sum(axis=0)).sum(), rtol=1e-13)
    o.set_H_ext_cell(None)                                  # back to the uniform value
    assert np.allclose(o.field_terms(m, oracle.TERM_ZEEMAN)[0], 7e4 * mask)
