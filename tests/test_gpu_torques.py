"""GPU parity for SURVEY.md 8(f)3 and 8(f)4: Zhang-Li and Slonczewski / SOT torques, the thermal
field with its device Philox generator (Eq. 41-42), and the Cayley-transform RK4 integrator (Eq. 43-49) — libmm.so
through the C ABI against the oracle, element by element, plus the closed forms Eq. 53 / Eq. 54 on the GPU itself."""
import numpy as np
import pytest

import oracle
from gpu_common import avg_m, make_pair, masked_m, to_np
from paper_2406_16064_b200 import workloads as wl

pytestmark = pytest.mark.gpu
F32, F64 = 0, 1
GAMMA = 2.211e5


def problem(nx, ny, nz, mask=True, demag=True, kind=wl.DMI_BULK):
    w = wl.cfg4(nx, ny, nz)
    w.dmi_kind = kind
    if mask:
        w.Ms = 8.6e5 * wl.random_mask(93, nx, ny, nz, 0.85)
    w.demag = demag
    return w


def both(o, s, name, *args):
    getattr(o, name)(*args)
    getattr(s, name)(*args)


@pytest.mark.parametrize("prec", [F64, F32])
def test_thermal_field_matches_oracle(prec):
    """Same Philox counter / key / Box-Muller on both sides: xi of Eq. 42 cell by cell, for two steps and two dt."""
    w = problem(64, 16, 4, demag=False)
    o, s = make_pair(w, prec)
    both(o, s, "set_temperature", 300.0, 0x1234567887654321)
    for dt, step in ((5e-14, 0), (2e-14, 7), (1e-13, (1 << 40) + 3)):
        ref = o.thermal_field(dt, step)
        got = to_np(s.thermal_field(dt, step))
        assert np.abs(got - ref).max() <= (1e-12 if prec == F64 else 2e-7) * np.abs(ref).max()
        assert np.all(got[:, w.Ms_array() == 0] == 0)
    both(o, s, "set_temperature", 0.0, 1)
    assert np.all(to_np(s.thermal_field(5e-14, 0)) == 0)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("shape,demag", [((32, 16, 4), True), ((64, 32, 1), True), ((1, 16, 4), False), ((2, 8, 8), False)])
@pytest.mark.parametrize("which", ["zhang_li", "slonczewski", "both"])
def test_rhs_with_torque_extensions(shape, demag, which, prec):
    w = problem(*shape, demag=demag)
    o, s = make_pair(w, prec)
    if which in ("zhang_li", "both"):
        both(o, s, "set_zhang_li", 120.0, -40.0, 75.0, 0.3)
    if which in ("slonczewski", "both"):
        both(o, s, "set_slonczewski", 3e9, -1.2e9, 1.0, 2.0, -2.0)
    m = masked_m(w)
    dm = s.to_device(m)
    kref = o.llg_rhs(m)
    k = to_np(s.llg_rhs(dm))
    assert np.abs(k - kref).max() <= (1e-9 if prec == F64 else 2e-4) * np.abs(kref).max()
    assert np.all(k[:, w.Ms_array() == 0] == 0)
    # the effective field itself does not contain the torque terms
    assert np.abs(to_np(s.effective_field(dm)) - o.effective_field(m)).max() / w.Ms_max <= (1e-10 if prec == F64 else 2e-4)
    # switching the terms off restores the plain path bit for bit
    s.set_zhang_li(0, 0, 0, 0); s.set_slonczewski(0, 0, 0, 0, 1)
    s2 = make_pair(w, prec)[1]
    assert np.array_equal(to_np(s.llg_rhs(dm)), to_np(s2.llg_rhs(dm)))


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("integ", [wl.RK4, wl.DOPRI5, wl.CAYLEY_RK4])
def test_fixed_dt_steps_with_everything_on(integ, prec):
    """Five fixed-dt steps with the thermal field (fresh per step: the device attempt counter must advance like the
    oracle's), Zhang-Li and Slonczewski terms, all field terms and a mask — every integrator, m cell by cell."""
    w = problem(32, 32, 4)
    w.integrator = integ
    o, s = make_pair(w, prec)
    both(o, s, "set_zhang_li", 80.0, 0.0, -30.0, 0.2)
    both(o, s, "set_slonczewski", 2e9, 5e8, 0.0, 1.0, 1.0)
    both(o, s, "set_temperature", 300.0, 77)
    m = masked_m(w)
    dm = s.to_device(m)
    for i in range(5):
        ro = o.step(m, w.dt)
        rs = s.step(dm, w.dt, sync=(i != 2))        # one step without a host read-back in between
        if i != 2:
            assert ro[0] and rs[0]
            assert np.isclose(rs[3], ro[3], rtol=1e-9 if prec == F64 else 1e-3)
    g = to_np(dm)
    Ms = w.Ms_array()
    assert np.abs(g - m).max() <= (1e-9 if prec == F64 else 2e-3), np.abs(g - m).max()
    assert np.abs(avg_m(g, Ms) - avg_m(m, Ms)).max() <= (1e-8 if prec == F64 else 1e-3)
    assert np.all(g[:, Ms == 0] == 0)
    nrm = np.sqrt((g * g).sum(axis=0))[Ms > 0]
    assert np.abs(nrm - 1).max() < (1e-13 if prec == F64 else 5e-6)
    assert np.isclose(s.time(), 5 * w.dt, rtol=1e-12)


def test_cayley_fp32_modulus_drift_over_a_long_run():
    """MM_CAYLEY_RK4 applies no projection (Q(omega) is a rotation); in fp32 the rounding of Q m lets |m|
    random-walk.  20 000 steps of a small film: the drift stays at the 1e-7 sqrt(steps) scale, far inside
    the fp32 trajectory tolerance; include/mm.h tells long-run callers to renormalise themselves."""
    w = problem(16, 16, 1, demag=False)
    w.integrator = wl.CAYLEY_RK4
    s = make_pair(w, F32)[1]
    Ms = w.Ms_array()
    dm = s.to_device(masked_m(w))
    for _ in range(20000):
        s.step(dm, 2e-14, sync=False)
    g = to_np(dm)
    drift = np.abs(np.sqrt((g * g).sum(axis=0))[Ms > 0] - 1).max()
    print(f"Cayley fp32 |m| drift after 20000 steps: {drift:.3e}")
    assert drift < 1e-4, drift


def test_adaptive_control_is_refused_with_the_thermal_field():
    """T > 0 and error control together are refused (include/mm.h, mm_set_temperature): a rejected attempt would redraw
    the noise.  Fixed steps still run, and T = 0 brings the adaptive calls back."""
    from paper_2406_16064_b200 import MMError
    w = problem(16, 16, 2)
    w.integrator = wl.DOPRI5
    s = make_pair(w, F64)[1]
    dm = s.to_device(masked_m(w))
    s.set_temperature(300.0, 9)
    for call in (lambda: s.step(dm, w.dt, tol=1e-6), lambda: s.relax(dm, 1e-6, 1e3, 4, dt0=w.dt),
                 lambda: s.run_until(dm, 10 * w.dt, 1e-6, dt0=w.dt),
                 lambda: s.run_host(dm.cpu(), 2, w.dt, tol=1e-6)):
        with pytest.raises(MMError, match="MM_ERR_UNSUPPORTED"):
            call()
    assert s.step(dm, w.dt)[0]                       # fixed step: fine
    s.set_temperature(0.0, 9)
    assert s.step(dm, w.dt, tol=1e-3)[1] >= 0.0      # T = 0: adaptive again


@pytest.mark.parametrize("prec", [F64, F32])
def test_cayley_macrospin_follows_eq_53(prec):
    """1x1x1 mesh (one-cell-per-thread kernel), Fig. 3 parameters: the GPU Cayley-RK4 trajectory equals the oracle's and
    sits at the closed form within the integrator's error; |m| = 1 without projection."""
    w = wl.Workload("macrospin", 1, 1, 1, 1e-9, 1e-9, 1e-9, Ms=8e5, alpha=0.5, gamma=GAMMA, H_ext=(0.0, 0.0, 1e5), integrator=wl.CAYLEY_RK4,
                    demag=False)
    w.m0 = np.array([1.0, 0.0, 0.0]).reshape(3, 1, 1, 1)
    o, s = make_pair(w, prec)
    m = np.ascontiguousarray(w.m0)
    dm = s.to_device(m)
    dt, n = 2e-12, 200
    for _ in range(n):
        o.step(m, dt)
        s.step(dm, dt, sync=False)
    g = to_np(dm).reshape(3)
    t = n * dt
    gp = GAMMA / 1.25
    ref = np.array([np.cos(gp * 1e5 * t) / np.cosh(0.5 * gp * 1e5 * t), np.sin(gp * 1e5 * t) / np.cosh(0.5 * gp * 1e5 * t), np.tanh(0.5 * gp * 1e5 * t)])
    assert np.abs(g - m.reshape(3)).max() <= (1e-12 if prec == F64 else 2e-5)
    assert np.abs(g - ref).max() <= (1e-7 if prec == F64 else 2e-5)
    assert abs(np.linalg.norm(g) - 1) <= (1e-14 if prec == F64 else 2e-5)


def test_domain_wall_motion_on_the_gpu_is_eq_54():
    """the head-to-head wall of Eq. 54 stepped on the GPU (fp64, RK4): wall velocity and tilt rate."""
    nx, dx, alpha, beta, A, K, u = 512, 1e-9, 0.1, 0.3, 1.3e-11, 1e5, 100.0
    Delta = np.sqrt(A / K)
    w = wl.Workload("wall", nx, 1, 1, dx, dx, dx, Ms=8e5, A=A, Ku=K, axis=(1.0, 0.0, 0.0), alpha=alpha, gamma=GAMMA, integrator=wl.RK4, demag=False)
    x = (np.arange(nx) + 0.5) * dx
    m = np.zeros((3, 1, 1, nx))
    m[0, 0, 0] = -np.tanh((x - 300e-9) / Delta)
    m[1, 0, 0] = 1 / np.cosh((x - 300e-9) / Delta)
    w.m0 = m
    s = make_pair(w, F64)[1]
    dm = s.to_device(m)

    def wall(t):
        a = to_np(t)
        return 0.5 * nx * dx * (1 + a[0].mean()), np.arctan2(a[2].sum(), a[1].sum())

    dt = 1e-13
    for _ in range(200):
        s.step(dm, dt, sync=False)
    s.set_zhang_li(u, 0, 0, beta)
    p0, f0 = wall(dm)
    for _ in range(4000):
        s.step(dm, dt, sync=False)
    p1, f1 = wall(dm)
    T = 4000 * dt
    v_ref = -(1 + alpha * beta) * u / (1 + alpha**2)
    w_ref = (alpha - beta) * u / ((1 + alpha**2) * Delta)
    assert abs((p1 - p0) / T - v_ref) <= 0.01 * abs(v_ref)
    assert abs((f1 - f0) / T - w_ref) <= 0.02 * abs(w_ref)


@pytest.mark.parametrize("prec", [F64, F32])
def test_equilibrium_distribution_on_the_gpu(prec):
    """PAPER.md:458-470 (Eq. 55-56, Fig. 6) on the GPU: 128 x 128 non-interacting nanoparticles at 300 K, RK4 with the
    thermal field of Eq. 42: <m_z^2> against the exact integral of P_eq ~ exp(-chi (1 - m_z^2))."""
    from conftest import load_golden
    g = load_golden("nanoparticle_eq56.txt")
    K, V, T, Ms = g["K"][0], g["V"][0], g["T"][0], g["Ms"][0]
    chi = K * V / (1.380649e-23 * T)
    n, edge = 128, V ** (1.0 / 3.0)
    w = wl.Workload("particles", n, n, 1, edge, edge, edge, Ms=Ms, Ku=K, axis=(0.0, 0.0, 1.0), alpha=0.1, gamma=GAMMA, integrator=wl.RK4, demag=False)
    w.m0 = wl.random_unit(8, n, n, 1)
    s = make_pair(w, prec)[1]
    s.set_temperature(T, 2025)
    dm = s.to_device(w.m0)
    mz2 = []
    for i in range(6000):
        s.step(dm, 1e-13, sync=False)
        if i >= 3000 and i % 600 == 599:
            a = to_np(dm)
            mz2.append(np.mean(a[2] ** 2))
    x, wq = np.polynomial.legendre.leggauss(400)
    p = np.exp(-chi * (1 - x * x))
    ref2 = np.sum(wq * p * x * x) / np.sum(wq * p)
    assert abs(np.mean(mz2) - ref2) < 4 * 0.3 / np.sqrt(n * n * len(mz2)) + 0.01
    assert np.abs(np.sqrt((a * a).sum(axis=0)) - 1).max() < (1e-12 if prec == F64 else 1e-5)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("integ", [wl.RK4, wl.DOPRI5, wl.CAYLEY_RK4])
def test_time_dependent_current_matches_oracle(integ, prec):
    """u(t) = u exp(-b t) cos(w t) evaluated at every stage's own time on the device: ten fixed-dt steps
    from a non-zero start time against the oracle, every integrator; and the right-hand side alone at that time."""
    w = problem(32, 16, 2)
    w.integrator = integ
    o, s = make_pair(w, prec)
    both(o, s, "set_zhang_li", 200.0, -50.0, 30.0, 0.25)
    both(o, s, "set_zhang_li_pulse", 5e8, 2e9)
    both(o, s, "set_time", 3.7e-10)
    m = masked_m(w)
    dm = s.to_device(m)
    kref = o.llg_rhs(m)
    k = to_np(s.llg_rhs(dm))
    assert np.abs(k - kref).max() <= (1e-9 if prec == F64 else 2e-4) * np.abs(kref).max()
    dt = 4e-13 if integ != wl.DOPRI5 else 1e-13       # large steps: a current frozen at the step start would show
    for _ in range(10):
        o.step(m, dt)
        s.step(dm, dt, sync=False)
    assert np.abs(to_np(dm) - m).max() <= (1e-9 if prec == F64 else 5e-3)
    assert np.isclose(s.time(), o.time(), rtol=1e-12)


def test_domain_wall_under_the_papers_pulse_on_the_gpu():
    """PAPER.md:433-446, Fig. 5 on the GPU (fp64, DOPRI5): wall position and tilt under u0 exp(-b t) cos(w t) against
    Eq. 54 integrated in closed form."""
    nx, dx, alpha, beta, A, K, u0, b, om = 512, 1e-9, 0.1, 0.3, 1.3e-11, 1e5, 300.0, 5e8, 2e9
    Delta = np.sqrt(A / K)
    w = wl.Workload("wall", nx, 1, 1, dx, dx, dx, Ms=8e5, A=A, Ku=K, axis=(1.0, 0.0, 0.0), alpha=alpha, gamma=GAMMA, integrator=wl.DOPRI5, demag=False)
    x = (np.arange(nx) + 0.5) * dx
    m = np.zeros((3, 1, 1, nx))
    m[0, 0, 0] = -np.tanh((x - 256e-9) / Delta)
    m[1, 0, 0] = 1 / np.cosh((x - 256e-9) / Delta)
    w.m0 = m
    s = make_pair(w, F64)[1]
    dm = s.to_device(m)

    def wall():
        a = to_np(dm)
        return 0.5 * nx * dx * (1 + a[0].mean()), np.arctan2(a[2].sum(), a[1].sum())

    dt = 1e-13
    for _ in range(200):
        s.step(dm, dt, sync=False)
    s.set_time(0.0)
    s.set_zhang_li(u0, 0, 0, beta)
    s.set_zhang_li_pulse(b, om)
    p0, f0 = wall()
    U = lambda t: u0 * (np.exp(-b * t) * (om * np.sin(om * t) - b * np.cos(om * t)) + b) / (b * b + om * om)
    Umax = abs(U(7.85e-10))
    for i in range(1, 12001):
        s.step(dm, dt, sync=False)
        if i % 3000 == 0:
            t = i * dt
            p, f = wall()
            assert abs((p - p0) + (1 + alpha * beta) * U(t) / (1 + alpha**2)) <= 0.01 * Umax + 2e-11
            assert abs((f - f0) - (alpha - beta) * U(t) / ((1 + alpha**2) * Delta)) <= 0.02 * abs(alpha - beta) * Umax / Delta
