"""GPU parity on meshes whose sizes are NOT powers of two: the library embeds them in the next
power of two with vacuum cells; every ABI call that takes cell arrays must behave as if it ran on the caller's own
nx x ny x nz mesh.  The oracle runs the caller's mesh directly (its demag is the defining direct sum there)."""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import avg_m, make_pair, masked_m, to_np
from paper_2406_16064_b200 import workloads as wl

pytestmark = pytest.mark.gpu
F32, F64 = 0, 1
HTOL = {F64: 1e-10, F32: 2e-4}
SHAPES = [(12, 10, 3), (100, 60, 1), (5, 7, 2), (24, 24, 5), (17, 4, 4)]


def problem(nx, ny, nz, kind=wl.DMI_BULK, mask=True, demag=True):
    w = wl.cfg4(nx, ny, nz)
    w.dmi_kind = kind
    if mask:
        w.Ms = 8.6e5 * wl.random_mask(95, nx, ny, nz, 0.85)
    w.demag = demag
    return w


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("shape", SHAPES)
def test_field_rhs_tensor(shape, prec):
    w = problem(*shape, kind=wl.DMI_INTERFACIAL if shape[2] == 1 else wl.DMI_BULK)
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    Href = o.effective_field(m)
    H = to_np(s.effective_field(dm))
    assert H.shape == Href.shape
    assert np.abs(H - Href).max() / w.Ms_max <= HTOL[prec], np.abs(H - Href).max() / w.Ms_max
    kref = o.llg_rhs(m)
    k = to_np(s.llg_rhs(dm))
    assert np.abs(k - kref).max() <= (1e-9 if prec == F64 else 2e-4) * np.abs(kref).max()
    live = w.Ms_array() > 0
    assert np.all(H[:, ~live] == 0) and np.all(k[:, ~live] == 0)
    if prec == F64:
        for c in (0, 3, 5):
            assert np.abs(to_np(s.demag_kernel(c)) - o.demag_kernel(c)).max() < 2e-15
    assert np.allclose(s.average_m(dm), o.average_m(m), atol=1e-12 if prec == F64 else 1e-6)
    Es, Eo = s.energy(dm), o.energy(m)
    assert np.isclose(Es[0], Eo[0], rtol=1e-9 if prec == F64 else 1e-4)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("integ", [wl.DOPRI5, wl.RK4, wl.CAYLEY_RK4])
def test_steps_host_path_and_thermal_indexing(integ, prec):
    """Fixed-dt steps in place on the caller's array, the host-buffer path, and the thermal field keyed by the
    caller's cell index (not the padded one)."""
    w = problem(20, 12, 3)
    w.integrator = integ
    o, s = make_pair(w, prec)
    for x in (o, s):
        x.set_temperature(300.0, 5)
        x.set_zhang_li(60.0, 20.0, 0.0, 0.1)
    xi = to_np(s.thermal_field(w.dt, 3))
    assert np.abs(xi - o.thermal_field(w.dt, 3)).max() <= (1e-12 if prec == F64 else 2e-7) * np.abs(xi).max()
    m = masked_m(w)
    dm = s.to_device(m)
    for i in range(4):
        ro = o.step(m, w.dt)
        rs = s.step(dm, w.dt, sync=(i % 2 == 0))
        if i % 2 == 0:
            assert np.isclose(rs[3], ro[3], rtol=1e-9 if prec == F64 else 1e-3)
    g = to_np(dm)
    assert np.abs(g - m).max() <= (1e-9 if prec == F64 else 2e-3)
    # host-buffer path: two more steps
    hm = torch.from_numpy(g.copy()).to(s.dtype).contiguous()
    s.run_host(hm, 2, w.dt)
    for _ in range(2):
        o.step(m, w.dt)
    assert np.abs(hm.numpy().astype(np.float64) - m).max() <= (1e-9 if prec == F64 else 2e-3)
    assert np.isclose(s.time(), 6 * w.dt, rtol=1e-12)


@pytest.mark.parametrize("prec", [F64, F32])
def test_adaptive_relax_minimize_and_cell_params(prec):
    w = problem(14, 9, 2, kind=wl.DMI_D2D)
    wl.cell_params(w, 4100, kind=wl.DMI_D2D, Kc=-3e4)
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    assert np.abs(to_np(s.effective_field(dm)) - o.effective_field(m)).max() / w.Ms_max <= HTOL[prec]
    no, go, to = o.minimize(m, 1e-8, 1e-12, 1e-4, 0.0, 8)
    ns, gs, ts = s.minimize(dm, 1e-8, 1e-12, 1e-4, 0.0, 8)
    assert no == ns == 8 and np.isclose(gs, go, rtol=1e-7 if prec == F64 else 2e-2)
    assert np.abs(to_np(dm) - m).max() <= (1e-8 if prec == F64 else 2e-2)
    # adaptive relaxation for a fixed number of attempts, then run_until: observables
    m2 = masked_m(w)
    dm2 = s.to_device(m2)
    n_o, _ = o.relax(m2, 1e-6 if prec == F64 else 1e-5, 0.0, 30, 1e-14)
    n_s, _ = s.relax(dm2, 1e-6 if prec == F64 else 1e-5, 0.0, 30, 1e-14)
    assert n_o == n_s == 30
    Ms = w.Ms_array()
    assert np.abs(avg_m(to_np(dm2), Ms) - avg_m(m2, Ms)).max() <= (1e-6 if prec == F64 else 1e-3)
    t_end = s.time() + 2e-13
    s.run_until(dm2, t_end, 1e-6)
    assert np.isclose(s.time(), t_end, rtol=1e-12)


def test_power_of_two_meshes_keep_the_direct_path():
    """No embedding (and no extra launches) when every size is a power of two."""
    w = problem(16, 8, 2)
    s = make_pair(w, F32)[1]
    dm = s.to_device(masked_m(w))
    l0 = s.launch_count()
    s.llg_rhs(dm)
    assert s.launch_count() - l0 == 5          # set_state + passes A, B, C + stage kernel
    w2 = problem(15, 8, 2)
    s2 = make_pair(w2, F32)[1]
    dm2 = s2.to_device(masked_m(w2))
    l0 = s2.launch_count()
    s2.llg_rhs(dm2)
    assert s2.launch_count() - l0 == 7         # + pack, + unpack
