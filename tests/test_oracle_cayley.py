"""Pins of the oracle's Cayley-transform integrator (Eq. 43-49): the transform itself
against the rotation it approximates and against its closed vector form, exact conservation of |m|, 4th-order
convergence on Eq. 53, the paper's Fig. 4 statement (better than classical RK4 + projection at small damping), and
agreement with the projected integrators on a coupled mesh."""
import numpy as np
import pytest
from scipy.linalg import expm

import oracle
from paper_2406_16064_b200 import workloads as wl

GAMMA = 2.211e5


def skew(v):
    return np.array([[0, -v[2], v[1]], [v[2], 0, -v[0]], [-v[1], v[0], 0]])       # Eq. 45


def test_cayley_transform_is_eq_47():
    rng = np.random.default_rng(5)
    for scale in (1e-3, 0.3, 2.0):
        w = scale * rng.standard_normal(3)
        m0 = rng.standard_normal(3)
        m0 /= np.linalg.norm(m0)
        got = oracle.cayley_apply(w, m0)
        O = skew(w)
        Q = np.linalg.solve(np.eye(3) - 0.5 * O, np.eye(3) + 0.5 * O)             # Eq. 47 with a library solve
        assert np.allclose(got, Q @ m0, rtol=1e-13, atol=1e-15)
        assert abs(np.linalg.norm(got) - 1) < 1e-14                                # Q is a rotation
        assert np.allclose(Q.T @ Q, np.eye(3), atol=1e-14) and abs(np.linalg.det(Q) - 1) < 1e-13
        # closed vector form: Q m = m + (w x m + w x (w x m) / 2) / (1 + |w|^2 / 4)
        vec = m0 + (np.cross(w, m0) + 0.5 * np.cross(w, np.cross(w, m0))) / (1 + 0.25 * w @ w)
        assert np.allclose(got, vec, rtol=1e-13, atol=1e-15)
        # rotation axis w, angle 2 atan(|w| / 2): equals exp(skew w) up to |w|^3 / 12
        th = 2 * np.arctan(0.5 * np.linalg.norm(w))
        R = expm(skew(w / np.linalg.norm(w) * th))
        assert np.allclose(got, R @ m0, rtol=1e-12, atol=1e-14)
    w = 1e-2 * np.array([1.0, -2.0, 0.5])
    assert np.abs(oracle.cayley_apply(w, [1, 0, 0]) - expm(skew(w)) @ [1, 0, 0]).max() < np.linalg.norm(w) ** 3 / 12 * 1.01


def eq53(t, alpha, Hz):
    gp = GAMMA / (1 + alpha**2)
    return np.array([np.cos(gp * Hz * t) / np.cosh(alpha * gp * Hz * t), np.sin(gp * Hz * t) / np.cosh(alpha * gp * Hz * t),
                     np.tanh(alpha * gp * Hz * t)])


def run_macrospin(integrator, alpha, dt, T, Hz=1e5):
    o = oracle.Oracle(1, 1, 1, 1e-9, 1e-9, 1e-9)
    o.set_Ms(8e5)
    o.set_demag(oracle.DEMAG_OFF)
    o.set_alpha(alpha)
    o.set_gamma(GAMMA)
    o.set_H_ext(0, 0, Hz)
    o.set_integrator(integrator)
    m = np.ascontiguousarray(np.array([1.0, 0, 0]).reshape(3, 1, 1, 1))
    n = int(round(T / dt))
    for _ in range(n):
        o.step(m, dt)
    return m.reshape(3), o.time()


def test_cayley_rk4_keeps_the_modulus_and_has_order_4():
    """Eq. 53, Fig. 3 parameters: |m| = 1 to rounding WITHOUT projection; error falls 16x per halving."""
    errs = []
    for dt in (8e-12, 4e-12, 2e-12):
        m, t = run_macrospin(oracle.CAYLEY_RK4, 0.5, dt, 4e-10)
        assert abs(np.linalg.norm(m) - 1) < 1e-14
        assert np.isclose(t, 4e-10, rtol=1e-12)
        errs.append(np.abs(m - eq53(4e-10, 0.5, 1e5)).max())
    for a, b in zip(errs, errs[1:]):
        assert 3.7 < np.log2(a / b) < 4.3, errs


def test_fig4_cayley_beats_projected_rk4_at_small_damping():
    """PAPER.md:425-427 (Fig. 4): alpha = 0.05, t = 1 ns, absolute error |m_an - m|: "The Cayley transform version
    performs much better than the projection method for the classical Runge-Kutta scheme"."""
    ref = eq53(1e-9, 0.05, 1e5)
    for dt in (1e-11, 5e-12):
        mc, _ = run_macrospin(oracle.CAYLEY_RK4, 0.05, dt, 1e-9)
        mp, _ = run_macrospin(oracle.RK4, 0.05, dt, 1e-9)
        ec, ep = np.linalg.norm(mc - ref), np.linalg.norm(mp - ref)
        assert ec < 0.5 * ep, (dt, ec, ep)


def test_cayley_matches_projected_integrators_on_a_coupled_mesh():
    """All terms on (exchange, DMI, anisotropy, Zeeman, demag, mask) plus both torque extensions: Cayley-RK4 and
    DOPRI5 + projection converge to the same trajectory; vacuum cells untouched; time advances."""
    nx, ny, nz = 8, 8, 2
    w = wl.cfg4(nx, ny, nz)
    w.Ms = 8.6e5 * wl.random_mask(12, nx, ny, nz, 0.85)
    ms = []
    for integ, dt, n in ((oracle.CAYLEY_RK4, 1e-14, 100), (oracle.DOPRI5, 1e-14, 100), (oracle.CAYLEY_RK4, 2e-14, 50)):
        o = oracle.Oracle(nx, ny, nz, w.dx, w.dy, w.dz)
        wl.apply(o, w)
        o.set_integrator(integ)
        o.set_zhang_li(80.0, 0.0, -30.0, 0.2)
        o.set_slonczewski(2e9, 5e8, 0, 1, 1)
        m = np.ascontiguousarray(w.m0 * (w.Ms > 0))
        for _ in range(n):
            ok, err, dn, md = o.step(m, dt)
            assert ok and err == 0.0 or integ == oracle.DOPRI5
        assert np.isclose(o.time(), 1e-12, rtol=1e-12)
        assert np.all(m[:, w.Ms == 0] == 0)
        ms.append(m)
    assert np.abs(np.sqrt((ms[0] * ms[0]).sum(axis=0))[w.Ms > 0] - 1).max() < 1e-13
    e_fine = np.abs(ms[0] - ms[1]).max()
    e_coarse = np.abs(ms[2] - ms[1]).max()
    assert e_fine < 1e-7 and e_coarse < 16 * 1.3 * max(e_fine, 1e-10) + 1e-8, (e_fine, e_coarse)


def test_cayley_max_dmdt_is_the_llg_rate():
    nx, ny, nz = 8, 4, 2
    w = wl.cfg4(nx, ny, nz)
    o = oracle.Oracle(nx, ny, nz, w.dx, w.dy, w.dz)
    wl.apply(o, w, with_demag=False)
    m = np.ascontiguousarray(w.m0)
    k = o.llg_rhs(m)
    o.set_integrator(oracle.CAYLEY_RK4)
    ok, err, dn, md = o.step(m.copy(), 1e-15)
    assert np.isclose(md, np.sqrt((k * k).sum(axis=0)).max(), rtol=1e-12)
