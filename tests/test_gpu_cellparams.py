"""GPU parity for SURVEY.md 8(f)2: cell-based A and D with harmonic-mean bond values, the D2d
DMI table (Eq. 14), cubic anisotropy (Eq. 33-34, continuum reading
R6) and a per-cell external field (Eq. 35) — libmm.so through the C ABI against the oracle, element by element."""
import numpy as np
import pytest

from gpu_common import avg_m, make_pair, masked_m, to_np
from paper_2406_16064_b200 import workloads as wl

pytestmark = pytest.mark.gpu
F32, F64 = 0, 1
HTOL = {F64: 1e-10, F32: 2e-4}


def general(nx, ny, nz, kind, use="all", mask=True, demag=True):
    w = wl.cfg4(nx, ny, nz)
    if mask:
        w.Ms = 8.6e5 * wl.random_mask(79, nx, ny, nz, 0.85)
    wl.cell_params(w, 4000 + nx + ny + nz, kind=kind, Kc=-3e4)
    if "A" not in use and use != "all":
        w.A_cell = None
    if "D" not in use and use != "all":
        w.D_cell = None
    if "H" not in use and use != "all":
        w.H_ext_cell = None
    if "K" not in use and use != "all":
        w.Kc = 0.0
    w.demag = demag
    return w


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("kind", [wl.DMI_BULK, wl.DMI_INTERFACIAL, wl.DMI_D2D])
@pytest.mark.parametrize("use", ["A", "D", "H", "K", "all"])
def test_local_terms_only(kind, use, prec):
    """Local terms alone (no demag) on a masked 3-D mesh spanning several thread blocks with ragged rows: the field and
    the torque at every cell; vacuum cells stay exactly 0."""
    w = general(32, 16, 4, kind, use, demag=False)
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    Href = o.effective_field(m)
    H = to_np(s.effective_field(dm))
    assert np.abs(H - Href).max() / w.Ms_max <= (1e-12 if prec == F64 else 2e-5), np.abs(H - Href).max() / w.Ms_max
    kref = o.llg_rhs(m)
    k = to_np(s.llg_rhs(dm))
    assert np.abs(k - kref).max() <= (1e-11 if prec == F64 else 2e-5) * np.abs(kref).max()
    live = w.Ms_array() > 0
    assert np.all(H[:, ~live] == 0) and np.all(k[:, ~live] == 0)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("shape,kind", [((64, 32, 8), wl.DMI_BULK), ((128, 64, 1), wl.DMI_D2D), ((32, 64, 2), wl.DMI_INTERFACIAL),
                                        ((2, 16, 4), wl.DMI_D2D)])
def test_full_field_with_demag(shape, kind, prec):
    """All terms together, demag included, films and 3-D, the narrowest mesh the vectorised stage kernel takes."""
    w = general(*shape, kind)
    if shape[0] < 4:
        w.demag = False
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    Href = o.effective_field(m)
    H = to_np(s.effective_field(dm))
    assert np.abs(H - Href).max() / w.Ms_max <= HTOL[prec], np.abs(H - Href).max() / w.Ms_max


@pytest.mark.parametrize("prec", [F64, F32])
def test_uniform_arrays_reduce_to_uniform_constants(prec):
    """Constant A_i = A, D_i = D, H_i = H_ext must give the field of the uniform setters (harmonic mean of equal
    values is the value) to rounding; switching back with NULL restores the uniform path bit for bit."""
    w = wl.cfg4(32, 16, 4)
    w.Ms = 8.6e5 * wl.random_mask(80, 32, 16, 4, 0.9)
    o, s = make_pair(w, prec, demag=False)
    m = masked_m(w)
    dm = s.to_device(m)
    H0 = to_np(s.effective_field(dm))
    s.set_A_cell(np.full((4, 16, 32), w.A))
    s.set_D_cell(np.full((4, 16, 32), w.D), w.dmi_kind)
    s.set_H_ext_cell(np.broadcast_to(np.array(w.H_ext)[:, None, None, None], (3, 4, 16, 32)).copy())
    H1 = to_np(s.effective_field(dm))
    assert np.abs(H1 - H0).max() <= (1e-13 if prec == F64 else 2e-6) * np.abs(H0).max()
    s.set_A_cell(None); s.set_D_cell(None, w.dmi_kind); s.set_H_ext_cell(None)
    s.set_A(w.A); s.set_D(w.D, w.dmi_kind)
    assert np.array_equal(to_np(s.effective_field(dm)), H0)


def test_set_D_cell_null_keeps_the_uniform_kind():
    """mm_set_D_cell(NULL, kind) only switches back to the uniform D: the kind given with NULL is ignored, the one of the
    last mm_set_D stays (include/mm.h).  A cell array set with another kind does change the field."""
    w = wl.cfg4(32, 16, 4)
    o, s = make_pair(w, F64, demag=False)          # cfg4: bulk DMI
    dm = s.to_device(masked_m(w))
    H0 = to_np(s.effective_field(dm))
    s.set_D_cell(np.full((4, 16, 32), w.D), wl.DMI_D2D)
    assert np.abs(to_np(s.effective_field(dm)) - H0).max() > 1e-3 * np.abs(H0).max()
    s.set_D_cell(None, wl.DMI_INTERFACIAL)
    s.set_D(w.D, wl.DMI_BULK)
    assert np.array_equal(to_np(s.effective_field(dm)), H0)
    s.set_D_cell(None, wl.DMI_INTERFACIAL)         # uniform D already active: the kind must not move
    assert np.array_equal(to_np(s.effective_field(dm)), H0)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("kind", [wl.DMI_BULK, wl.DMI_D2D])
def test_fixed_dt_steps_and_energy(kind, prec):
    """Five fixed-dt DOPRI5 steps with every (f)2 term on, against the oracle; the energy (cubic term inside the
    anisotropy slot, weight 1/4) agrees and decreases."""
    w = general(32, 32, 4, kind)
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    E0, T0 = s.energy(dm)
    Eo, To = o.energy(m)
    assert np.isclose(E0, Eo, rtol=1e-10 if prec == F64 else 1e-4)
    assert np.allclose(T0, To, rtol=1e-9 if prec == F64 else 1e-3, atol=abs(Eo) * (1e-12 if prec == F64 else 1e-5))
    for _ in range(5):
        ro = o.step(m, w.dt)
        rs = s.step(dm, w.dt)
        assert ro[0] and rs[0]
        assert np.isclose(rs[3], ro[3], rtol=1e-9 if prec == F64 else 1e-3)
    g = to_np(dm)
    Ms = w.Ms_array()
    assert np.abs(g - m).max() <= (1e-9 if prec == F64 else 2e-3)
    assert np.abs(avg_m(g, Ms) - avg_m(m, Ms)).max() <= (1e-8 if prec == F64 else 1e-3)
    assert s.energy(dm)[0] < E0


@pytest.mark.parametrize("prec", [F64, F32])
def test_minimize_with_cell_params(prec):
    """mm_minimize (Eq. 50-52) uses the same general local field: a fixed number of updates against the oracle."""
    w = general(16, 16, 2, wl.DMI_INTERFACIAL, use="AD")
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    no, go, to = o.minimize(m, 1e-8, 1e-12, 1e-4, 0.0, 10)
    ns, gs, ts = s.minimize(dm, 1e-8, 1e-12, 1e-4, 0.0, 10)
    assert no == ns == 10
    assert np.isclose(ts, to, rtol=1e-7 if prec == F64 else 2e-2)
    assert np.isclose(gs, go, rtol=1e-7 if prec == F64 else 2e-2)
    assert np.abs(to_np(dm) - m).max() <= (1e-8 if prec == F64 else 2e-2)
