"""Pins for the oracle's demag tensor (oracle/mo.c: newell_f, newell_g, stencil, permutations)."""
import numpy as np
import pytest

import oracle
from conftest import load_golden

G = load_golden("newell_values.txt")
IDX = {"xx": 0, "yy": 1, "zz": 2, "xy": 3, "xz": 4, "yz": 5}


def test_cube_self_term_is_one_third():
    n = oracle.newell_point(0, 0, 0, 1.0, 1.0, 1.0)
    assert np.allclose(n[:3], 1.0 / 3.0, atol=1e-15)
    assert np.allclose(n[3:], 0.0, atol=1e-15)
    n = oracle.newell_point(0, 0, 0, 2.5e-9, 2.5e-9, 2.5e-9)        # scale invariance
    assert np.allclose(n[:3], 1.0 / 3.0, atol=1e-15)


@pytest.mark.parametrize("key", ["xx_100", "yy_100", "zz_100", "xx_110", "zz_110", "xy_110", "xy_111", "xx_200"])
def test_printed_values_unit_cubes(key):
    comp, off = key.split("_")
    X, Y, Z = (float(c) for c in off)
    n = oracle.newell_point(X, Y, Z, 1.0, 1.0, 1.0)
    assert abs(n[IDX[comp]] - G[key][0]) < 2e-15


def test_printed_self_terms_noncubic():
    assert np.allclose(oracle.newell_point(0, 0, 0, 1, 1, 0.5)[:3], G["self_1_1_0.5"], atol=2e-15)
    assert np.allclose(oracle.newell_point(0, 0, 0, 2, 3, 5)[:3], G["self_2_3_5"], atol=2e-15)


def test_trace_is_one_at_origin_zero_elsewhere():
    rng = np.random.default_rng(5)
    for cell in [(1, 1, 1), (1, 2, 0.5), (3.90625, 3.90625, 3.0)]:
        assert abs(oracle.newell_point(0, 0, 0, *cell)[:3].sum() - 1.0) < 1e-15
        for _ in range(20):
            o = rng.integers(-6, 7, size=3)
            if not o.any():
                continue
            n = oracle.newell_point(o[0] * cell[0], o[1] * cell[1], o[2] * cell[2], *cell)
            assert abs(n[:3].sum()) < 1e-16


def test_parity_symmetries():
    cell = (1.0, 1.5, 0.75)
    p = oracle.newell_point(2 * cell[0], 1 * cell[1], 3 * cell[2], *cell)
    for sx, sy, sz in [(-1, 1, 1), (1, -1, 1), (1, 1, -1), (-1, -1, -1)]:
        q = oracle.newell_point(sx * 2 * cell[0], sy * 1 * cell[1], sz * 3 * cell[2], *cell)
        assert np.allclose(q[:3], p[:3], atol=1e-17)
        assert np.allclose(q[3:], p[3:] * np.array([sx * sy, sx * sz, sy * sz]), atol=1e-17)
    m = oracle.newell_point(-2 * cell[0], -1 * cell[1], -3 * cell[2], *cell)     # N(-r) = N(r)
    assert np.allclose(m, p, atol=1e-17)


def test_dipole_limit():
    """N_ab -> -(V / 4 pi r^3)(3 r^_a r^_b - delta_ab) far away (point-dipole field)."""
    cell = (1.0, 1.0, 1.0)
    r = np.array([40.0, 25.0, 30.0])
    n = oracle.newell_point(*r, *cell)
    R = np.linalg.norm(r)
    rh = r / R
    D = -(1.0 / (4 * np.pi * R**3)) * (3 * np.outer(rh, rh) - np.eye(3))
    ref = np.array([D[0, 0], D[1, 1], D[2, 2], D[0, 1], D[0, 2], D[1, 2]])
    assert np.allclose(n, ref, rtol=0, atol=2e-3 * np.abs(ref).max())      # O((cell/R)^2) correction
    assert np.abs(n - ref).max() > 0                                       # not literally the dipole formula


def _tensor_by_quadrature(off, cell, npts=24):
    """Independent of the closed forms: N_ab(r) = -(1/(4 pi V)) int int d_a d_b (1/|r+u-u'|) du du'
    over two cells, reduced to the 3-D integral over s = u-u' with triangular weights
    prod_i (cell_i - |s_i|), Gauss-Legendre on each half interval."""
    x, w = np.polynomial.legendre.leggauss(npts)
    axes = []
    for d in cell:
        s = np.concatenate([(x - 1) * d / 2, (x + 1) * d / 2])          # [-d,0] and [0,d]
        ww = np.concatenate([w, w]) * d / 2 * (d - np.abs(s))
        axes.append((s, ww))
    S = np.meshgrid(axes[0][0], axes[1][0], axes[2][0], indexing="ij")
    W = axes[0][1][:, None, None] * axes[1][1][None, :, None] * axes[2][1][None, None, :]
    r = [off[i] * cell[i] + S[i] for i in range(3)]
    R2 = r[0] ** 2 + r[1] ** 2 + r[2] ** 2
    R5 = R2 ** 2.5
    V = cell[0] * cell[1] * cell[2]
    out = []
    for a, b in [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]:
        dd = (3 * r[a] * r[b] - (R2 if a == b else 0.0)) / R5           # d_a d_b (1/r)
        out.append(-(W * dd).sum() / (4 * np.pi * V))
    return np.array(out)


@pytest.mark.parametrize("off,cell", [((2, 0, 0), (1.0, 1.0, 1.0)), ((3, 1, 2), (1.0, 1.0, 1.0)),
                                      ((2, 3, 1), (1.0, 0.5, 2.0)), ((0, 2, 5), (3.90625, 3.90625, 3.0))])
def test_against_defining_dipole_integral(off, cell):
    q = _tensor_by_quadrature(off, cell)
    n = oracle.newell_point(off[0] * cell[0], off[1] * cell[1], off[2] * cell[2], *cell)
    assert np.allclose(n, q, rtol=0, atol=1e-12)


def test_block_aggregation_identity_small():
    """Mean demag factor of a uniformly magnetised block of cells = self term of the block as one cell."""
    nx, ny, nz = 6, 4, 3
    cell = (1.0, 1.5, 0.5)
    T = np.zeros((6, nz, ny, nx))
    oracle.lib().mo_newell_tensor(nx, ny, nz, *cell, T.ctypes.data_as(oracle._dp))
    acc = np.zeros(3)
    for c in range(3):
        for k in range(-nz + 1, nz):
            for j in range(-ny + 1, ny):
                for i in range(-nx + 1, nx):
                    acc[c] += (nx - abs(i)) * (ny - abs(j)) * (nz - abs(k)) * T[c, abs(k), abs(j), abs(i)]
    acc /= nx * ny * nz
    blk = oracle.newell_point(0, 0, 0, nx * cell[0], ny * cell[1], nz * cell[2])[:3]
    assert np.allclose(acc, blk, atol=1e-14)


@pytest.mark.parametrize("shape,cell", [((5, 4, 3), (1.0, 0.8, 1.3)), ((12, 7, 1), (3.90625, 3.90625, 3.0)), ((6, 9, 4), (2.0, 1.0, 0.5)),
                                        # larger than the library's near box (8 cell edges per direction): offsets where the
                                        # table's index arithmetic is furthest from the origin, with and without a z extent
                                        ((40, 24, 3), (2.5, 2.5, 2.5)), ((40, 24, 1), (4.0, 4.0, 4.0))])
def test_tabulated_tensor_equals_pointwise(shape, cell):
    """mo_newell_tensor (lattice tabulation of f / g + 27-point stencil + odd-axis signs) against the independent
    point evaluation mo_newell_point at EVERY offset of the mesh, all six components (one mesh has nz = 1)."""
    nx, ny, nz = shape
    T = np.zeros((6, nz, ny, nx))
    oracle.lib().mo_newell_tensor(nx, ny, nz, *cell, T.ctypes.data_as(oracle._dp))
    worst = 0.0
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                p = oracle.newell_point(i * cell[0], j * cell[1], k * cell[2], *cell)
                worst = max(worst, np.abs(T[:, k, j, i] - p).max())
    assert worst < 1e-16, worst


def test_printed_block_values():
    for key, dims in [("block_32_32_2", (32, 32, 2)), ("block_500_125_3", (500, 125, 3)),
                      ("block_1280_1280_40", (1280, 1280, 40))]:
        assert np.allclose(oracle.newell_point(0, 0, 0, *dims)[:3], G[key], atol=2e-15)
    assert abs(oracle.newell_point(0, 0, 0, 256, 256, 4)[2] - G["block_256_256_4_zz"][0]) < 2e-15
    assert abs(oracle.newell_point(0, 0, 0, 16384, 16384, 4)[2] - G["block_16384_16384_4_zz"][0]) < 2e-15
