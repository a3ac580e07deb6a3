"""Pins for the oracle's steepest-descent / Barzilai-Borwein minimiser (oracle/mo.c: mo_sd_update, mo_minimize;
PAPER.md:376-393, Eq. 50-52).  What the paper and the mathematics fix: the explicit update (Eq. 51) solves the implicit
one (Eq. 50) and preserves |m|; a small step moves along -m x (m x H) and lowers the energy; the fixed point is the
energy minimum that LLG relaxation reaches; the Stoner-Wohlfarth switching field of Listing 2; Eq. 52 on a hand case;
"much more efficient" than plain steepest descent."""
import numpy as np
import pytest

import oracle
from paper_2406_16064_b200 import workloads as wl

MU0 = 4e-7 * np.pi


def small_problem(kind=wl.DMI_BULK, seed=7, shape=(8, 8, 2)):
    nx, ny, nz = shape
    w = wl.cfg4(nx, ny, nz)
    w.dmi_kind = kind
    w.Ms = 8.6e5 * wl.random_mask(seed, nx, ny, nz, 0.85)
    o = oracle.Oracle(nx, ny, nz, w.dx, w.dy, w.dz)
    wl.apply(o, w)
    m = np.ascontiguousarray(w.m0 * (w.Ms > 0))
    return w, o, m


@pytest.mark.parametrize("tau", [1e-9, 1e-6, 3e-5, 1e-3])
def test_eq51_solves_eq50_and_preserves_modulus(tau):
    w, o, m = small_problem()
    H = o.effective_field(m)
    m1 = m.copy()
    o.sd_update(m1, H, tau)
    live = w.Ms > 0
    n1 = np.sqrt((m1 * m1).sum(axis=0))
    assert np.abs(n1[live] - 1).max() < 4e-16                       # Eq. 50: m_{k+1}^2 = m_k^2, for ANY tau
    assert np.array_equal(m1[:, ~live], m[:, ~live])
    # residual of the implicit form, Eq. 50:  m' - m + tau (m + m')/2 x (m x H) = 0
    a, b, h = m.reshape(3, -1).T, m1.reshape(3, -1).T, H.reshape(3, -1).T
    res = b - a + tau * np.cross(0.5 * (a + b), np.cross(a, h))
    assert np.abs(res).max() <= 1e-14 * max(1.0, tau * np.abs(h).max())


def test_small_step_follows_damping_direction_and_lowers_energy():
    w, o, m = small_problem(kind=wl.DMI_INTERFACIAL)
    H = o.effective_field(m)
    tau = 1e-12
    m1 = m.copy()
    o.sd_update(m1, H, tau)
    a, h = m.reshape(3, -1).T, H.reshape(3, -1).T
    g = np.cross(a, np.cross(a, h))
    d = (m1 - m).reshape(3, -1).T / tau
    assert np.abs(d + g).max() <= 1e-4 * np.abs(g).max()              # m' = m - tau m x (m x H) + O(tau^2)
    m2 = m.copy()
    o.sd_update(m2, H, 2e-8)
    assert o.energy(m2)[0] < o.energy(m)[0]


def test_eq52_on_a_hand_case():
    """Two updates of a 2-cell system: the tau of the second update must be tau^1 = s.s / s.y (k = 1 is odd) with
    s = m_1 - m_0 and y = g_1 - g_0, sums over both cells; the third uses tau^2 = s.y / y.y."""
    o = oracle.Oracle(2, 1, 1, 2e-9, 2e-9, 2e-9)
    o.set_Ms(8e5); o.set_A(1.3e-11); o.set_Ku(5e4); o.set_axis(0, 0, 1); o.set_H_ext(2e4, 0, 1e4); o.set_demag(0)
    m0 = np.array([[0.6, 0.0], [0.0, 0.8], [0.8, 0.6]]).reshape(3, 1, 1, 2).copy()

    def gof(m):
        a, h = m.reshape(3, -1).T, o.effective_field(m).reshape(3, -1).T
        return np.cross(a, np.cross(a, h))

    tau0 = 1e-7
    ms = [m0.copy()]
    taus = [tau0]
    for k in range(1, 3):
        m = ms[-1].copy()
        o.sd_update(m, o.effective_field(m), taus[-1])
        ms.append(m)
        s = (ms[k] - ms[k - 1]).reshape(3, -1).T
        y = gof(ms[k]) - gof(ms[k - 1])
        taus.append(abs((s * s).sum() / (s * y).sum()) if k % 2 == 1 else abs((s * y).sum() / (y * y).sum()))
    for nsteps in (2, 3):
        m = m0.copy()
        n, _, tau_last = o.minimize(m, tau0, 1e-14, 1.0, 0.0, nsteps)
        assert n == nsteps and np.isclose(tau_last, taus[nsteps - 1], rtol=1e-12)
    assert np.abs(m - (lambda mm: (o.sd_update(mm, o.effective_field(mm), taus[2]), mm)[1])(ms[2].copy())).max() < 1e-15


def test_clamp_reading_on_the_hand_case():
    """DESIGN.md R16 (the paper prints no bounds): |tau| is clamped to [tau_min, tau_max].  Same 2-cell system as above:
    the Barzilai-Borwein value of the second update is computed by hand; with tau_max below it (tau_min above it) the
    update must use exactly the bound, and the resulting m is Eq. 51 with that bound."""
    o = oracle.Oracle(2, 1, 1, 2e-9, 2e-9, 2e-9)
    o.set_Ms(8e5); o.set_A(1.3e-11); o.set_Ku(5e4); o.set_axis(0, 0, 1); o.set_H_ext(2e4, 0, 1e4); o.set_demag(0)
    m0 = np.array([[0.6, 0.0], [0.0, 0.8], [0.8, 0.6]]).reshape(3, 1, 1, 2).copy()
    tau0 = 1e-7

    def gof(m):
        a, h = m.reshape(3, -1).T, o.effective_field(m).reshape(3, -1).T
        return np.cross(a, np.cross(a, h))

    m1 = m0.copy()
    o.sd_update(m1, o.effective_field(m1), tau0)
    sv, yv = (m1 - m0).reshape(3, -1).T, gof(m1) - gof(m0)
    bb = abs((sv * sv).sum() / (sv * yv).sum())
    for lo, hi, expect in ((1e-14, bb / 3, bb / 3), (3 * bb, 1.0, 3 * bb), (bb / 2, 2 * bb, bb)):
        m = m0.copy()
        n, _, tau_last = o.minimize(m, tau0, lo, hi, 0.0, 2)
        assert n == 2 and np.isclose(tau_last, expect, rtol=1e-12), (tau_last, expect)
        ref = m1.copy()
        o.sd_update(ref, o.effective_field(ref), expect)
        assert np.abs(m - ref).max() < 1e-15


def test_fallback_reading_when_the_quotient_is_undefined():
    """DESIGN.md R16: a vanishing or non-finite Barzilai-Borwein quotient falls back to tau0.  At an exact equilibrium
    (m parallel to H in every cell: g = 0) nothing moves, s = y = 0 and both quotients of Eq. 52 are 0/0; with the stop
    criterion off the iteration must carry on with tau0 and leave m finite and untouched."""
    o = oracle.Oracle(2, 1, 1, 2e-9, 2e-9, 2e-9)
    o.set_Ms(8e5); o.set_A(1.3e-11); o.set_Ku(5e4); o.set_axis(0, 0, 1); o.set_H_ext(0, 0, 1e4); o.set_demag(0)
    m = np.zeros((3, 1, 1, 2))
    m[2] = 1.0
    n, maxg, tau_last = o.minimize(m, 3e-8, 1e-14, 1.0, 0.0, 4)
    assert n == 4 and maxg == 0.0 and tau_last == 3e-8
    assert np.array_equal(m[2], np.ones((1, 1, 2))) and np.all(m[:2] == 0)


@pytest.mark.parametrize("kind", [wl.DMI_BULK, wl.DMI_INTERFACIAL])
def test_minimiser_and_llg_relaxation_reach_the_same_minimum(kind):
    w, o, m = small_problem(kind=kind, shape=(4, 4, 2))
    E0 = o.energy(m)[0]
    ma = m.copy()
    n, maxg, _ = o.minimize(ma, 1e-8, 1e-12, 1e-4, 1e-2, 5000)
    assert n < 5000 and maxg < 1e-2
    mb = m.copy()
    o.set_alpha(1.0)
    ns, md = o.relax(mb, 1e-6, 1e7, 4000, 1e-14)      # the adaptive controller's noise floor at tol 1e-6 is ~3e6 rad/s
    assert md < 1e7
    Ea, Eb = o.energy(ma)[0], o.energy(mb)[0]
    assert Ea < E0 and Ea <= Eb and abs(Ea - Eb) <= 2e-6 * abs(Eb)
    assert np.abs(ma - mb).max() < 2e-3
    live = w.Ms > 0
    assert np.abs(np.sqrt((ma * ma).sum(axis=0))[live] - 1).max() < 1e-12      # no projection anywhere, Eq. 50 keeps |m|


def test_bb_steps_beat_a_fixed_step():
    """"much more efficient".  The same stop criterion with tau pinned to the best fixed value the
    problem tolerates needs several times more updates than the Barzilai-Borwein sequence."""
    w, o, m = small_problem(shape=(4, 4, 2))
    ma = m.copy()
    n_bb, g_bb, _ = o.minimize(ma, 1e-8, 1e-12, 1e-4, 1.0, 20000)
    best = None
    for tau in (2e-8, 5e-8, 1e-7, 2e-7):
        mb = m.copy()
        n_fx, g_fx, _ = o.minimize(mb, tau, tau, tau, 1.0, 20000)
        if g_fx < 1.0 and np.isfinite(g_fx):
            best = n_fx if best is None else min(best, n_fx)
    assert g_bb < 1.0 and best is not None and n_bb * 2 < best, (n_bb, best)


def test_stoner_wohlfarth_switching_field_with_the_minimiser():
    """Listing 2 with the minimiser as the driver: easy axis (1,1,0), field along -x; coherent
    rotation switches at H_K/2 = Ku/(mu0 Ms) for a 45 degree easy axis."""
    Ms, Ku = 8e5, 5e4
    Hsw = Ku / (MU0 * Ms)

    def minimised(Hx):
        o = oracle.Oracle(1, 1, 1, 4e-9, 4e-9, 4e-9)
        o.set_Ms(Ms); o.set_Ku(Ku); o.set_axis(1, 1, 0); o.set_demag(0); o.set_H_ext(Hx, 0, 0)
        m = (np.array([1.0, 1.0, 1e-3]) / np.linalg.norm([1.0, 1.0, 1e-3])).reshape(3, 1, 1, 1).copy()
        n, g, _ = o.minimize(m, 1e-6, 1e-10, 1e-3, 1e-4, 100000)
        assert g < 1e-4
        return m.reshape(3)

    m_lo, m_hi = minimised(-0.90 * Hsw), minimised(-1.10 * Hsw)
    assert m_lo[0] > 0 or m_lo[1] > 0.5
    assert m_hi[0] < -0.5 and m_hi[1] < 0.0
