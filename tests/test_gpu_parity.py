"""GPU parity: libmm.so (through the C ABI) against the oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json's: max|dH|/Ms <= 1e-10 (fp64), 2e-4 (fp32);
<m> after fixed-dt steps <= 1e-8 (fp64), 1e-3 (fp32)."""
import numpy as np
import pytest

import oracle
from gpu_common import avg_m, make_pair, masked_m, to_np
from paper_2406_16064_b200 import workloads as wl

pytestmark = pytest.mark.gpu
F32, F64 = 0, 1
HTOL = {F64: 1e-10, F32: 2e-4}
MTOL = {F64: 1e-8, F32: 1e-3}


def small3d(nx=32, ny=16, nz=8, mask=True, kind=wl.DMI_BULK):
    w = wl.cfg4(nx, ny, nz)
    w.dmi_kind = kind
    if mask:
        w.Ms = 8.6e5 * wl.random_mask(77, nx, ny, nz, 0.85)
    return w


def film(n, mask=False):
    w = wl.cfg5(n)
    if mask:
        w.Ms = 8e5 * wl.random_mask(78, n, n, 1, 0.9)
    return w


# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,cell", [((32, 16, 4), (2e-9, 1.5e-9, 3e-9)), ((64, 64, 1), (3.90625e-9, 3.90625e-9, 3e-9)),
                                        ((16, 32, 16), (2.5e-9, 2.5e-9, 2.5e-9)), ((128, 8, 2), (2e-9, 2e-9, 1e-9))])
def test_demag_tensor_matches_oracle(shape, cell):
    """S0: near-field quad closed forms + far-field quadrature vs the oracle's quad tensor everywhere."""
    nx, ny, nz = shape
    w = wl.Workload("t", nx, ny, nz, *cell, Ms=8e5)
    w.m0 = wl.random_unit(1, nx, ny, nz)
    o, s = make_pair(w, F64)
    for c in range(6):
        ref = o.demag_kernel(c)
        got = to_np(s.demag_kernel(c))
        assert np.abs(got - ref).max() < 2e-15, (c, np.abs(got - ref).max())


@pytest.mark.parametrize("prec", [F64, F32])
def test_cfg1_field_vs_direct_sum(prec):
    w = wl.cfg1()
    o, s = make_pair(w, prec, oracle_demag=oracle.DEMAG_DIRECT)
    m = masked_m(w)
    Href = o.effective_field(m)
    H = to_np(s.effective_field(s.to_device(m)))
    assert np.abs(H - Href).max() / w.Ms_max <= HTOL[prec]


CASES = {
    "cfg2": lambda: wl.cfg2(),
    "cfg3_64": lambda: wl.cfg3(64),
    "cfg3_256": lambda: wl.cfg3(256),
    "slab_32x16x8_bulk": lambda: small3d(),
    "slab_64x64x16": lambda: small3d(64, 64, 16),
    "slab_16x64x2_interfacial": lambda: small3d(16, 64, 2, kind=wl.DMI_INTERFACIAL),
    "slab_128x32x4": lambda: small3d(128, 32, 4),
    "film_128_masked": lambda: film(128, mask=True),
    "film_512": lambda: film(512),
    "slab_32x1024x2_b7_ny1024": lambda: small3d(32, 1024, 2),
    "film_64x1024_b7_ny1024": lambda: small3d(64, 1024, 1, kind=wl.DMI_INTERFACIAL),
    "film_4x2": lambda: wl.cfg5(4).__class__("tiny", 4, 2, 1, 4e-9, 4e-9, 4e-9, Ms=8e5, A=1.3e-11, m0=wl.random_unit(3, 4, 2, 1)),
}


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("case", sorted(CASES))
def test_effective_field_and_rhs(case, prec):
    w = CASES[case]()
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    Href = o.effective_field(m)
    H = to_np(s.effective_field(dm))
    assert np.abs(H - Href).max() / w.Ms_max <= HTOL[prec], np.abs(H - Href).max() / w.Ms_max
    kref = o.llg_rhs(m)
    k = to_np(s.llg_rhs(dm))
    scale = np.abs(kref).max()
    assert np.abs(k - kref).max() <= (1e-9 if prec == F64 else 2e-4) * scale
    live = w.Ms_array() > 0
    assert np.all(H[:, ~live] == 0) and np.all(k[:, ~live] == 0)


@pytest.mark.parametrize("prec", [F64, F32])
def test_demag_only_and_local_only(prec):
    w = small3d(32, 32, 4)
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    # local terms only
    s.set_demag(0); o.set_demag(0)
    H = to_np(s.effective_field(dm))
    Href = o.effective_field(m)
    assert np.abs(H - Href).max() / w.Ms_max <= (1e-12 if prec == F64 else 2e-5)
    # demag only
    s.set_demag(1); o.set_demag(1)
    for x in (s, o):
        x.set_A(0.0); x.set_D(0.0, 0); x.set_Ku(0.0); x.set_H_ext(0, 0, 0)
    H = to_np(s.effective_field(dm))
    Href = o.effective_field(m)
    assert np.abs(H - Href).max() / w.Ms_max <= (1e-12 if prec == F64 else 2e-5)


# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [F64, F32])
def test_cfg1_200_rk4_steps(prec):
    w = wl.cfg1()
    o, s = make_pair(w, prec, oracle_demag=oracle.DEMAG_DIRECT)
    m = masked_m(w)
    dm = s.to_device(m)
    E = [s.energy(dm)[0]]
    for i in range(200):
        o.step(m, w.dt)
        s.step(dm, w.dt, sync=(i % 50 == 49))
        if i % 20 == 19:
            E.append(s.energy(dm)[0])
    g = to_np(dm)
    Ms = w.Ms_array()
    assert np.abs(avg_m(g, Ms) - avg_m(m, Ms)).max() <= MTOL[prec]
    assert np.abs(g - m).max() <= (1e-8 if prec == F64 else 5e-3)
    assert np.abs(np.sqrt((g * g).sum(axis=0)) - 1).max() < (1e-14 if prec == F64 else 1e-6)
    assert all(E[i + 1] < E[i] for i in range(len(E) - 1))
    assert np.isclose(s.time(), 200 * w.dt, rtol=1e-12)
    Eo = o.energy(m)[0]
    assert np.isclose(E[-1], Eo, rtol=1e-9 if prec == F64 else 1e-4)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("case,nsteps", [("cfg2", 20), ("cfg3_64", 20), ("cfg3_256", 20), ("slab_32x16x8_bulk", 5), ("slab_64x64x16", 5)])
def test_fixed_dt_dopri5_steps(case, nsteps, prec):
    w = CASES[case]()
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    for i in range(nsteps):
        ok_o, err_o, _, md_o = o.step(m, w.dt)
        ok, err, dn, md = s.step(dm, w.dt)
        assert ok and ok_o and dn == w.dt
        assert np.isclose(md, md_o, rtol=1e-9 if prec == F64 else 1e-3)
        if prec == F64:
            assert np.isclose(err, err_o, rtol=1e-5)
        else:
            # E = dt sum_j e_j k_j with sum_j e_j = 0: the estimate is a small residual of terms of size dt |k|, each
            # carrying fp32 rounding 2^-24 |k|-relative; seven of them add in quadrature-ish: |d err| <~ 2^-23 sqrt(7) dt max|k|
            # (measured 1e-9 .. 8e-8 dt max|k|).  A wrong e_j would move err by ~1e-3 dt max|k|.
            assert abs(err - err_o) <= 2.0**-23 * np.sqrt(7.0) * w.dt * md_o, (err, err_o)
    g = to_np(dm)
    Ms = w.Ms_array()
    assert np.abs(avg_m(g, Ms) - avg_m(m, Ms)).max() <= MTOL[prec]
    assert np.abs(g - m).max() <= (1e-8 if prec == F64 else 5e-3)
    assert np.allclose(s.average_m(dm), avg_m(g, Ms), atol=1e-12 if prec == F64 else 1e-6)


def test_adaptive_step_accept_reject_matches_oracle():
    w = wl.cfg2()
    w.alpha = 0.5
    o, s = make_pair(w, F64)
    m = masked_m(w)
    dm = s.to_device(m)
    m_before = m.copy()
    ok_o, err_o, dn_o, _ = o.step(m, 5e-12, 1e-6)            # too large: rejected on both sides
    ok, err, dn, _ = s.step(dm, 5e-12, 1e-6)
    assert (not ok) and (not ok_o)
    assert np.isclose(err, err_o, rtol=1e-6) and np.isclose(dn, dn_o, rtol=1e-6)
    assert np.array_equal(to_np(dm), m_before) and s.time() == 0.0
    ok_o, err_o, dn_o, _ = o.step(m, 2e-13, 1e-6)
    ok, err, dn, _ = s.step(dm, 2e-13, 1e-6)
    assert ok and ok_o and np.isclose(err, err_o, rtol=1e-5) and np.isclose(dn, dn_o, rtol=1e-5)
    assert np.abs(to_np(dm) - m).max() < 1e-10
    assert s.stats() == (1, 1, 14)                           # mm_get_stats: one rejected + one accepted DOPRI5 attempt
    s.set_integrator(wl.RK4)
    s.step(dm, 1e-13, sync=False)
    assert s.stats() == (2, 1, 18)                           # totals run on across calls; an RK4 attempt is 4 evaluations


@pytest.mark.parametrize("prec", [F64, F32])
def test_cfg2_relax_then_run(prec):
    """configs[1] shape: relax with alpha=0.5, apply the field, run adaptive DOPRI5; observables vs the
    oracle at a fixed time (a short 20 ps window keeps the oracle affordable). DESIGN.md R8, R10."""
    w = wl.cfg2()
    w.alpha = 0.5
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    tol = 1e-6
    n_o, md_o = o.relax(m, tol, 2e9, 400, 1e-13)
    n_s, md_s = s.relax(dm, tol, 2e9, 400, 1e-13)
    acc, rej, nrhs = s.stats()                               # attempts enqueued after the stop do not count
    assert acc + rej == n_s and nrhs == 7 * n_s and acc >= 1
    Ms = w.Ms_array()
    loose = 1e-4 if prec == F64 else 1e-2
    assert md_s < 2e9 and md_o < 2e9
    assert np.abs(avg_m(to_np(dm), Ms) - avg_m(m, Ms)).max() < loose
    for x in (o, s):
        x.set_alpha(0.02)
        x.set_H_ext(*wl.CFG2_FIELD)
        x.set_time(0.0)
    t_end = 20e-12
    s.run_until(dm, t_end, tol, 1e-13)
    dt = 1e-13
    while o.time() < t_end * (1 - 1e-12):
        dt = min(dt, t_end - o.time())
        ok, err, dn, _ = o.step(m, dt, tol)
        dt = dn
    assert np.isclose(s.time(), t_end, rtol=1e-9)
    assert np.abs(avg_m(to_np(dm), Ms) - avg_m(m, Ms)).max() < loose
    Es, Eo = s.energy(dm)[0], o.energy(m)[0]
    assert np.isclose(Es, Eo, rtol=loose)


def test_macrospin_eq53_on_gpu():
    """PAPER.md:409-417 on a 1x1x1 mesh (demag off: the library needs nx >= 4 for demag)."""
    from paper_2406_16064_b200 import Sim
    s = Sim(1, 1, 1, 1e-9, 1e-9, 1e-9, prec=F64)
    s.set_Ms(8e5); s.set_alpha(0.5); s.set_gamma(2.21e5); s.set_H_ext(0, 0, 1e5); s.set_demag(0)
    dm = s.to_device(np.array([1.0, 0, 0]).reshape(3, 1, 1, 1))
    T, n = 0.2e-9, 400
    for _ in range(n):
        s.step(dm, T / n, sync=False)
    g = 2.21e5 / 1.25
    ref = [np.cos(g * 1e5 * T) / np.cosh(0.5 * g * 1e5 * T), np.sin(g * 1e5 * T) / np.cosh(0.5 * g * 1e5 * T), np.tanh(0.5 * g * 1e5 * T)]
    assert np.allclose(to_np(dm).reshape(3), ref, atol=1e-9)


def test_host_buffer_entry_points():
    import torch
    w = small3d(32, 16, 8)
    o, s = make_pair(w, F64)
    m = masked_m(w)
    hm = torch.from_numpy(m.copy()).pin_memory()
    hk = torch.empty_like(hm).pin_memory()
    s.llg_rhs_host(hm, hk)
    kref = o.llg_rhs(m)
    assert np.abs(hk.numpy() - kref).max() <= 1e-9 * np.abs(kref).max()
    s.run_host(hm, 3, w.dt)
    for _ in range(3):
        o.step(m, w.dt)
    assert np.abs(hm.numpy() - m).max() < 1e-9


def test_edge_cases_and_errors():
    from paper_2406_16064_b200 import Sim, MMError
    import torch
    s = Sim(16, 16, 1, 2e-9, 2e-9, 2e-9, prec=F32)
    m = s.to_device(wl.random_unit(5, 16, 16, 1))
    with pytest.raises(MMError):                      # Ms not set
        s.effective_field(m)
    s.set_Ms(8e5)
    with pytest.raises(MMError):                      # demag enabled, not initialised
        s.effective_field(m)
    s.set_Ms(np.zeros((1, 16, 16)))                   # all vacuum: everything is zero
    s.init_demag()
    assert float(s.effective_field(m).abs().max()) == 0.0
    assert float(s.llg_rhs(m).abs().max()) == 0.0
    with pytest.raises(MMError):
        Sim(2, 16, 1, 1e-9, 1e-9, 1e-9).init_demag()   # nx < 4
    Sim(24, 16, 1, 1e-9, 1e-9, 1e-9).init_demag()     # not a power of two: embedded (tests/test_gpu_anysize.py)
    with pytest.raises(MMError):
        Sim(0, 16, 1, 1e-9, 1e-9, 1e-9)               # empty mesh
    # NaN in m is reported, not silently propagated
    s2 = Sim(16, 16, 1, 2e-9, 2e-9, 2e-9, prec=F32)
    s2.set_Ms(8e5); s2.set_A(1.3e-11); s2.init_demag()
    bad = s2.to_device(wl.random_unit(5, 16, 16, 1))
    bad[0, 0, 3, 3] = float("nan")
    with pytest.raises(MMError):
        s2.step(bad, 1e-14, 1e-6)


# ---------------------------------------------------------------------------------------------
# Full BASELINE.json sizes, in the launch configuration bench.py times (default Sim of the workload)
# ---------------------------------------------------------------------------------------------
def test_cfg4_full_size_sampled_direct_sum():
    """configs[3] (512x512x16): the demag field of Eq. 8 at sampled cells, each computed by the oracle as
    the plain O(N) sum over all source cells with its quad-precision tensor; fp64 and fp32."""
    from paper_2406_16064_b200 import Sim
    w = wl.cfg4()
    o = oracle.Oracle(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz)
    o.set_Ms(w.Ms_array())
    o.init_demag()
    m = np.ascontiguousarray(w.m0)
    rng = np.random.default_rng(4004)
    cells = [0, w.nx - 1, w.N - 1, (w.nx * w.ny) * 7 + w.nx * 255 + 256] + [int(c) for c in rng.integers(0, w.N, 20)]
    ref = np.array([o.demag_direct_at(m, c) for c in cells])
    for prec in (F64, F32):
        s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=prec)
        wl.apply(s, w)
        s.set_A(0.0); s.set_D(0.0, 0); s.set_Ku(0.0); s.set_H_ext(0, 0, 0)      # demag term alone
        H = to_np(s.effective_field(s.to_device(m))).reshape(3, -1)
        got = np.array([H[:, c] for c in cells])
        assert np.abs(got - ref).max() / w.Ms_max <= HTOL[prec], (prec, np.abs(got - ref).max() / w.Ms_max)
        del s


@pytest.mark.parametrize("case", ["cfg4", "film4096_f32", "film4096_f64", "film2048_f64", "film1024_f64", "film2048_f32", "film1024_f32"])
def test_full_size_block_aggregation_identity(case):
    """Uniformly magnetised full mesh: the MEAN demag field is -Ms N_self(block) m exactly, with N_self the
    Newell self term of the whole block as one cell (SURVEY.md §8c pins; holds at any size)."""
    from paper_2406_16064_b200 import Sim
    if case == "cfg4":
        w, precs = wl.cfg4(with_m=False), (F64, F32)
    else:
        n = int(case.split("_")[0][4:])
        w, precs = wl.cfg5(n, with_m=False), ((F32,) if case.endswith("f32") else (F64,))
    nself = oracle.newell_point(0, 0, 0, w.nx * w.dx, w.ny * w.dy, w.nz * w.dz)[:3]
    u = np.array([0.36, -0.48, 0.8])
    m = np.ascontiguousarray(np.broadcast_to(u.reshape(3, 1, 1, 1), (3, w.nz, w.ny, w.nx)))
    for prec in precs:
        s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=prec)
        wl.apply(s, w)
        s.set_A(0.0); s.set_D(0.0, 0); s.set_Ku(0.0); s.set_H_ext(0, 0, 0)
        H = s.effective_field(s.to_device(m)).double().reshape(3, -1).mean(dim=1).cpu().numpy()
        ref = -w.Ms_max * np.array(nself) * u
        assert np.abs(H - ref).max() / w.Ms_max <= (1e-10 if prec == F64 else 2e-5), (case, prec, H, ref)
        del s


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("n", [4096, 2048, 1024])
def test_film_point_source_is_the_newell_tensor(n, prec):
    """configs[4] at N = 4096 (fp64 runs the cluster pass B: a full 8192-row tile does not fit one CTA), 2048 (fp32: the
    generic TMA pass B at 2-column tiles and the padded x tile at 4 lines per CTA) and 1024: the field of ONE
    magnetised cell is -Ms N(r - r0) m at every cell; sampled cells against the oracle's quad-precision tensor,
    including the far corners of the film and the source's neighbours."""
    from paper_2406_16064_b200 import Sim
    import torch
    w = wl.cfg5(n, with_m=False)
    s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=prec)
    wl.apply(s, w)
    s.set_A(0.0); s.set_H_ext(0, 0, 0)
    i0, j0 = (1234 * n) // 4096, (3071 * n) // 4096
    mvec = np.array([0.6, -0.64, 0.48])
    dm = torch.zeros((3, 1, n, n), dtype=s.dtype, device=s.device)
    dm[:, 0, j0, i0] = torch.tensor(mvec, dtype=s.dtype)
    H = s.effective_field(dm)
    rng = np.random.default_rng(7)
    cells = [(i0, j0), (i0 + 1, j0), (i0, j0 - 1), (i0 - 1, j0 + 1), (0, 0), (n - 1, n - 1), (0, n - 1), (n - 1, 0), (i0, 0), (n // 2, n // 2)]
    cells += [(int(a), int(b)) for a, b in rng.integers(0, n, (30, 2))]
    cells += [(i0 + int(a), j0 + int(b)) for a, b in rng.integers(-12, 13, (30, 2))]
    worst = 0.0
    for (i, j) in cells:
        n = oracle.newell_point((i - i0) * w.dx, (j - j0) * w.dy, 0.0, w.dx, w.dy, w.dz)      # xx yy zz xy xz yz
        N = np.array([[n[0], n[3], n[4]], [n[3], n[1], n[5]], [n[4], n[5], n[2]]])
        ref = -w.Ms_max * N @ mvec
        got = H[:, 0, j, i].double().cpu().numpy()
        worst = max(worst, np.abs(got - ref).max() / w.Ms_max)
    assert worst <= (1e-12 if prec == F64 else 2e-7), worst
    del s


@pytest.mark.parametrize("prec", [F64, F32])
def test_pass_b_half_tile_form(monkeypatch, prec):
    """The half-tile form of pass B (mm_passB3.cuh, the long-line path) forced on small meshes (MM_B3): 3-D and film,
    both precisions, against the oracle."""
    monkeypatch.setenv("MM_B3", "1")
    w = small3d(64, 64, 16)
    o, s = make_pair(w, prec)
    m = masked_m(w)
    assert np.abs(to_np(s.effective_field(s.to_device(m))) - o.effective_field(m)).max() / w.Ms_max <= HTOL[prec]
    wf = film(512)
    o, s = make_pair(wf, prec)
    H = to_np(s.effective_field(s.to_device(wf.m0)))
    assert np.abs(H - o.effective_field(np.ascontiguousarray(wf.m0))).max() / wf.Ms_max <= HTOL[prec]
    wn = small3d(32, 16, 2)
    o, s = make_pair(wn, prec)
    m = masked_m(wn)
    dm = s.to_device(m)
    for _ in range(3):
        o.step(m, wn.dt); s.step(dm, wn.dt, sync=False)
    assert np.abs(to_np(dm) - m).max() <= (1e-9 if prec == F64 else 2e-3)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("Q", ["2", "4"])
def test_pass_b_cluster_form(monkeypatch, prec, Q):
    """The cluster form of pass B (mm_passB4.cuh: Q CTAs share one long y line through distributed shared memory) forced
    on small meshes (MM_B4, MM_Q): 3-D and film, both precisions, against the oracle; then a few steps."""
    monkeypatch.setenv("MM_B4", "1")
    monkeypatch.setenv("MM_Q", Q)
    w = small3d(64, 64, 16)
    o, s = make_pair(w, prec)
    m = masked_m(w)
    assert np.abs(to_np(s.effective_field(s.to_device(m))) - o.effective_field(m)).max() / w.Ms_max <= HTOL[prec]
    wf = film(512)
    o, s = make_pair(wf, prec)
    H = to_np(s.effective_field(s.to_device(wf.m0)))
    assert np.abs(H - o.effective_field(np.ascontiguousarray(wf.m0))).max() / wf.Ms_max <= HTOL[prec]
    wn = small3d(32, 32, 2)
    o, s = make_pair(wn, prec)
    m = masked_m(wn)
    dm = s.to_device(m)
    for _ in range(3):
        o.step(m, wn.dt); s.step(dm, wn.dt, sync=False)
    assert np.abs(to_np(dm) - m).max() <= (1e-9 if prec == F64 else 2e-3)


@pytest.mark.parametrize("prec", [F64, F32])
def test_step_graph_replay_is_bitwise_the_eager_path(monkeypatch, prec):
    """Whole-step CUDA graphs (captured on the second step, replayed afterwards) must give exactly what kernel-by-kernel
    launches give: fixed-dt steps, a parameter change in between (new key -> new capture), adaptive steps."""
    w = small3d(32, 32, 4)
    m0 = masked_m(w)
    res = []
    for no_graph in ("", "1"):
        if no_graph:
            monkeypatch.setenv("MM_NO_GRAPH", "1")
        s = make_pair(w, prec)[1]
        dm = s.to_device(m0)
        for _ in range(5):
            s.step(dm, w.dt, sync=False)
        s.set_alpha(0.3)
        for _ in range(4):
            s.step(dm, w.dt, sync=False)
        n, _ = s.relax(dm, 1e-5, 0.0, 12, 1e-14)
        assert n == 12
        res.append((to_np(dm), s.time(), s.launch_count()))
    assert np.array_equal(res[0][0], res[1][0])
    assert res[0][1] == res[1][1] and res[0][2] == res[1][2]


def test_cfg4_full_size_step_invariants():
    """configs[3] in bench.py's configuration (fp32, fixed-dt DOPRI5): |m| = 1 after every step, finite,
    and the energy does not increase (alpha > 0, constant field)."""
    from paper_2406_16064_b200 import Sim
    import torch
    w = wl.cfg4()
    s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=F32)
    wl.apply(s, w)
    dm = s.to_device(w.m0)
    E0 = s.energy(dm)[0]
    for _ in range(5):
        s.step(dm, w.dt, sync=False)
    nrm = torch.sqrt((dm.double() ** 2).sum(dim=0))
    assert bool(torch.isfinite(dm).all()) and float((nrm - 1).abs().max()) < 1e-5
    assert s.energy(dm)[0] < E0


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("tma", ["0", "1"])
def test_pass_b_tma_and_register_forms(monkeypatch, prec, tma):
    """Pass B has two forms (TMA box copies into a component-major tile / thread-issued loads into a row-major
    tile); the library picks one per precision.  Both are checked against the oracle here (MM_TMA forces one)."""
    monkeypatch.setenv("MM_TMA", tma)
    w = small3d(64, 64, 16)
    o, s = make_pair(w, prec)
    m = masked_m(w)
    H = to_np(s.effective_field(s.to_device(m)))
    Href = o.effective_field(m)
    assert np.abs(H - Href).max() / w.Ms_max <= HTOL[prec]
    wf = film(512)
    o, s = make_pair(wf, prec)
    H = to_np(s.effective_field(s.to_device(wf.m0)))
    Href = o.effective_field(np.ascontiguousarray(wf.m0))
    assert np.abs(H - Href).max() / wf.Ms_max <= HTOL[prec]
