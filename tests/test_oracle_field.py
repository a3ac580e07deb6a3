"""Pins for the oracle's field terms (oracle/mo.c: demag_direct, demag_fft, local_field_add)."""
import numpy as np
import pytest

import oracle
from conftest import load_golden
from paper_2406_16064_b200 import workloads as wl

G = load_golden("newell_values.txt")
MU0 = 4e-7 * np.pi


def make(nx, ny, nz, cell, Ms=8e5, demag=oracle.DEMAG_FFT):
    o = oracle.Oracle(nx, ny, nz, *cell)
    o.set_Ms(Ms)
    o.set_demag(demag)
    if demag:
        o.init_demag()
    return o


def test_two_cell_worked_example():
    o = make(2, 1, 1, (1.0, 1.0, 1.0), Ms=1.0, demag=oracle.DEMAG_DIRECT)
    m = np.zeros((3, 1, 1, 2))
    m[0, 0, 0, 0] = 1.0
    m[1, 0, 0, 1] = 1.0
    H = o.field_terms(m, oracle.TERM_DEMAG)
    assert np.allclose(H[:, 0, 0, 0], G["twocell_H1"], atol=2e-15)
    assert np.allclose(H[:, 0, 0, 1], G["twocell_H2"], atol=2e-15)
    o.set_demag(oracle.DEMAG_FFT)
    H2 = o.field_terms(m, oracle.TERM_DEMAG)
    assert np.allclose(H2, H, atol=1e-15)


@pytest.mark.parametrize("shape,cell", [((8, 4, 2), (1e-9, 2e-9, 0.5e-9)), ((16, 16, 4), (2e-9, 1.5e-9, 3e-9)),
                                        ((16, 8, 1), (3.90625e-9, 3.90625e-9, 3e-9)), ((1, 4, 8), (1e-9, 1e-9, 2e-9))])
def test_fft_path_equals_direct_sum(shape, cell):
    nx, ny, nz = shape
    Ms = 8e5 * wl.random_mask(11, nx, ny, nz, 0.8)
    m = wl.random_unit(12, nx, ny, nz) * (Ms > 0)
    o = make(nx, ny, nz, cell, Ms=Ms)
    Hf = o.field_terms(m, oracle.TERM_DEMAG)
    o.set_demag(oracle.DEMAG_DIRECT)
    Hd = o.field_terms(m, oracle.TERM_DEMAG)
    assert np.abs(Hf - Hd).max() <= 1e-13 * 8e5
    assert np.abs(Hd).max() > 1e4
    assert o.khat_imag_ratio() < 1e-15
    # single sampled output of Eq. 8
    cell_id = int(np.flatnonzero(Ms.reshape(-1) > 0)[3])
    h = o.demag_direct_at(m, cell_id)
    assert np.allclose(h, Hd.reshape(3, -1)[:, cell_id], atol=1e-15 * 8e5)


def test_block_aggregation_cfg1_printed_value():
    """Uniform m on the full cfg1 mesh (16x16x1 of 2 nm): mean H_d = -Ms N_self(32,32,2 nm) m."""
    for axis, c in [((1.0, 0, 0), 0), ((0, 0, 1.0), 2)]:
        o = make(16, 16, 1, (2e-9, 2e-9, 2e-9), Ms=8e5)
        m = np.zeros((3, 1, 16, 16))
        m[c] = 1.0
        H = o.field_terms(m, oracle.TERM_DEMAG)
        assert abs(H[c].mean() / 8e5 + G["block_32_32_2"][c]) < 1e-14


def test_thin_film_limit():
    """Uniform out-of-plane film: H_d ~ -Ms m_z z^ (mean demag factor -> 1 as the film widens)."""
    o = make(64, 64, 1, (4e-9, 4e-9, 4e-9), Ms=8e5)
    m = np.zeros((3, 1, 64, 64))
    m[2] = 1.0
    H = o.field_terms(m, oracle.TERM_DEMAG)
    assert abs(H[2].mean() / 8e5 + G["block_256_256_4_zz"][0]) < 1e-13
    assert -1.0 < H[2, 0, 32, 32] / 8e5 < -0.97           # centre of the film close to -Ms
    # in-plane components: odd under the film's mirror symmetries, so they cancel in the mean (not cell by cell: they are
    # of order 1e-2 Ms at the edges)
    assert np.abs(H[:2].mean(axis=(1, 2, 3))).max() / 8e5 < 1e-13


def test_demag_energy_nonnegative_and_masked_cells_zero():
    Ms = 8e5 * wl.random_mask(3, 8, 8, 2, 0.7)
    m = wl.random_unit(4, 8, 8, 2) * (Ms > 0)
    o = make(8, 8, 2, (2e-9, 2e-9, 1e-9), Ms=Ms)
    H = o.field_terms(m, oracle.TERM_DEMAG)
    assert np.all(H[:, Ms == 0] == 0)
    E, terms = o.energy(m)
    assert terms[0] > 0


# ---------------------------------------------------------------- local terms ----------
def local(nx, ny, nz, cell, **kw):
    o = make(nx, ny, nz, cell, Ms=kw.pop("Ms", 8e5), demag=oracle.DEMAG_OFF)
    for k, v in kw.items():
        getattr(o, "set_" + k)(*v) if isinstance(v, tuple) else getattr(o, "set_" + k)(v)
    return o


def test_exchange_uniform_zero_and_spiral():
    A, Ms, d = 1.3e-11, 8e5, 2e-9
    o = local(32, 4, 3, (d, d, d), A=A)
    m = np.zeros((3, 3, 4, 32))
    m[0], m[1], m[2] = 0.6, 0.0, 0.8
    assert np.abs(o.field_terms(m, oracle.TERM_EXCHANGE)).max() == 0.0
    q = 2 * np.pi / (12.3 * d)
    x = np.arange(32) * d
    m[0], m[1], m[2] = np.cos(q * x), np.sin(q * x), 0.0
    H = o.field_terms(m, oracle.TERM_EXCHANGE)
    ref = (2 * A / (MU0 * Ms)) * (2 * (np.cos(q * d) - 1) / d**2) * m
    assert np.allclose(H[..., 1:-1], ref[..., 1:-1], rtol=1e-12, atol=1e-6)
    assert not np.allclose(H[..., 0], ref[..., 0], rtol=1e-3)          # free boundary: one neighbour missing


def test_exchange_anisotropic_cells_and_mask():
    """Each axis uses its own spacing; a Ms=0 neighbour is absent."""
    A, Ms = 1.0e-11, 5e5
    cell = (1e-9, 2e-9, 4e-9)
    o = local(3, 3, 3, cell, A=A, Ms=Ms)
    m = np.zeros((3, 3, 3, 3))
    m[2] = 1.0
    m[:, 1, 1, 1] = (1.0, 0.0, 0.0)                      # centre cell differs
    H = o.field_terms(m, oracle.TERM_EXCHANGE)
    f = 2 * A / (MU0 * Ms)
    # centre: six neighbours each contribute (z^ - x^)/d^2
    s = 2 / cell[0]**2 + 2 / cell[1]**2 + 2 / cell[2]**2
    assert np.allclose(H[:, 1, 1, 1], f * s * np.array([-1.0, 0, 1.0]), rtol=1e-13)
    # +x neighbour of the centre sees (x^ - z^)/dx^2 only
    assert np.allclose(H[:, 1, 1, 2], f / cell[0]**2 * np.array([1.0, 0, -1.0]), rtol=1e-13)
    assert np.allclose(H[:, 2, 1, 1], f / cell[2]**2 * np.array([1.0, 0, -1.0]), rtol=1e-13)
    Msa = np.full((3, 3, 3), Ms)
    Msa[1, 1, 2] = 0.0                                   # remove the +x neighbour
    o.set_Ms(Msa)
    mm = m.copy()
    mm[:, 1, 1, 2] = 0
    H2 = o.field_terms(mm, oracle.TERM_EXCHANGE)
    s2 = 1 / cell[0]**2 + 2 / cell[1]**2 + 2 / cell[2]**2
    assert np.allclose(H2[:, 1, 1, 1], f * s2 * np.array([-1.0, 0, 1.0]), rtol=1e-13)
    assert np.all(H2[:, 1, 1, 2] == 0)


def test_dmi_bulk_helix_and_interfacial_cycloid():
    D, Ms, d = 1.5e-3, 8.6e5, 2.5e-9
    q = 2 * np.pi / (9.7 * d)
    x = np.arange(40) * d
    amp = 2 * D * np.sin(q * d) / (MU0 * Ms * d)
    m = np.zeros((3, 1, 1, 40))
    o = local(40, 1, 1, (d, d, d), Ms=Ms, D=(D, oracle.DMI_BULK))
    m[0], m[1], m[2] = 0.0, np.cos(q * x), np.sin(q * x)              # helix along x
    H = o.field_terms(m, oracle.TERM_DMI)
    assert np.allclose(H[..., 1:-1], amp * m[..., 1:-1], rtol=1e-12, atol=1e-6)
    o = local(40, 1, 1, (d, d, d), Ms=Ms, D=(D, oracle.DMI_INTERFACIAL))
    m[0], m[1], m[2] = np.sin(q * x), 0.0, np.cos(q * x)              # cycloid along x
    H = o.field_terms(m, oracle.TERM_DMI)
    assert np.allclose(H[..., 1:-1], amp * m[..., 1:-1], rtol=1e-12, atol=1e-6)


def test_dmi_y_and_z_directions_match_continuum_curl():
    """Bulk DMI (Eq. 11): H = -(2D/mu0 Ms) curl m with central differences, helices along y and z."""
    D, Ms, d = 1.5e-3, 8.6e5, 2.5e-9
    q = 2 * np.pi / (11.0 * d)
    amp = 2 * D * np.sin(q * d) / (MU0 * Ms * d)
    o = local(1, 40, 1, (d, d, d), Ms=Ms, D=(D, oracle.DMI_BULK))
    y = np.arange(40) * d
    m = np.zeros((3, 1, 40, 1))
    m[0, 0, :, 0], m[2, 0, :, 0] = np.sin(q * y), np.cos(q * y)        # helix along y: (sin, 0, cos)
    H = o.field_terms(m, oracle.TERM_DMI)
    assert np.allclose(H[:, :, 1:-1], amp * m[:, :, 1:-1], rtol=1e-12, atol=1e-6)
    o = local(1, 1, 40, (d, d, d), Ms=Ms, D=(D, oracle.DMI_BULK))
    m = np.zeros((3, 40, 1, 1))
    m[0, :, 0, 0], m[1, :, 0, 0] = np.cos(q * y), np.sin(q * y)        # helix along z: (cos, sin, 0)
    H = o.field_terms(m, oracle.TERM_DMI)
    assert np.allclose(H[:, 1:-1], amp * m[:, 1:-1], rtol=1e-12, atol=1e-6)
    # interfacial (Eq. 13), cycloid along y: (0, sin, cos)
    o = local(1, 40, 1, (d, d, d), Ms=Ms, D=(D, oracle.DMI_INTERFACIAL))
    m = np.zeros((3, 1, 40, 1))
    m[1, 0, :, 0], m[2, 0, :, 0] = np.sin(q * y), np.cos(q * y)
    H = o.field_terms(m, oracle.TERM_DMI)
    assert np.allclose(H[:, :, 1:-1], amp * m[:, :, 1:-1], rtol=1e-12, atol=1e-6)


def test_dmi_uniform_interior_zero_edge_value():
    D, Ms, d = 3.0e-3, 5.8e5, 2e-9
    o = local(8, 8, 1, (d, d, 1e-9), Ms=Ms, D=(D, oracle.DMI_INTERFACIAL))
    m = np.zeros((3, 1, 8, 8))
    m[2] = 1.0
    H = o.field_terms(m, oracle.TERM_DMI)
    assert np.abs(H[:, :, 1:-1, 1:-1]).max() == 0.0
    edge = np.linalg.norm(H[:, 0, 4, 0])
    assert np.isclose(edge, D / (MU0 * Ms * d), rtol=1e-13)            # DESIGN.md reading R4
    # interfacial DMI has no z neighbours: stacking layers changes nothing
    o3 = local(8, 8, 3, (d, d, 1e-9), Ms=Ms, D=(D, oracle.DMI_INTERFACIAL))
    m3 = np.zeros((3, 3, 8, 8))
    m3[2] = 1.0
    H3 = o3.field_terms(m3, oracle.TERM_DMI)
    assert np.allclose(H3[:, 1], H[:, 0])


def test_anisotropy_and_zeeman():
    Ku, Ms = 5e4, 8e5
    o = local(4, 4, 4, (1e-9, 1e-9, 1e-9), Ms=Ms, Ku=Ku, axis=(1.0, 1.0, 0.0), H_ext=(1.0, -2.0, 3.0))
    u = np.array([1.0, 1.0, 0.0]) / np.sqrt(2)
    m = np.zeros((3, 4, 4, 4))
    m[0], m[1] = u[0], u[1]
    H = o.field_terms(m, oracle.TERM_ANIS)
    assert np.allclose(H[:, 0, 0, 0], 2 * Ku / (MU0 * Ms) * u, rtol=1e-14)
    m[:] = 0
    m[2] = 1.0                                                        # m perpendicular to u
    assert np.abs(o.field_terms(m, oracle.TERM_ANIS)).max() < 1e-9
    m[0], m[2] = 0.6, 0.8
    H = o.field_terms(m, oracle.TERM_ANIS)
    assert np.allclose(H[:, 1, 2, 3], 2 * Ku / (MU0 * Ms) * (0.6 * u[0]) * u, rtol=1e-14)
    Hz = o.field_terms(m, oracle.TERM_ZEEMAN)
    assert np.all(Hz[0] == 1.0) and np.all(Hz[1] == -2.0) and np.all(Hz[2] == 3.0)
    # terms add up
    Hall = o.effective_field(m)
    assert np.allclose(Hall, H + Hz + o.field_terms(m, oracle.TERM_EXCHANGE) + o.field_terms(m, oracle.TERM_DMI))
