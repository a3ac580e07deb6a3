"""ctypes binding of the CPU oracle (oracle/mo.c).  TEST INFRASTRUCTURE — see mo.c header.

All arrays are numpy float64, C-contiguous, SoA: m[3, nz, ny, nx] (x fastest), Ms[nz, ny, nx].
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

_lib = None

DMI_NONE, DMI_BULK, DMI_INTERFACIAL, DMI_D2D = 0, 1, 2, 3
RK4, DOPRI5, CAYLEY_RK4 = 0, 1, 2
DEMAG_OFF, DEMAG_FFT, DEMAG_DIRECT = 0, 1, 2
TERM_EXCHANGE, TERM_DMI, TERM_ANIS, TERM_ZEEMAN, TERM_DEMAG, TERM_CUBIC = 1, 2, 4, 8, 16, 32

_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.mo_time.restype = C.c_double
        L.mo_khat_imag_ratio.restype = C.c_double
        L.mo_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]
        for name in ("mo_set_Ms_uniform", "mo_set_A", "mo_set_Ku", "mo_set_Kc", "mo_set_alpha", "mo_set_gamma", "mo_set_time"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_double]
        L.mo_set_D.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.mo_set_axis.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.mo_set_H_ext.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.mo_set_integrator.argtypes = [C.c_void_p, C.c_int]
        L.mo_set_demag.argtypes = [C.c_void_p, C.c_int]
        L.mo_set_Ms.argtypes = [C.c_void_p, _dp]
        L.mo_set_A_cell.argtypes = [C.c_void_p, _dp]
        L.mo_set_D_cell.argtypes = [C.c_void_p, _dp, C.c_int]
        L.mo_set_H_ext_cell.argtypes = [C.c_void_p, _dp]
        L.mo_init_demag.argtypes = [C.c_void_p]
        L.mo_destroy.argtypes = [C.c_void_p]
        L.mo_time.argtypes = [C.c_void_p]
        L.mo_khat_imag_ratio.argtypes = [C.c_void_p]
        L.mo_effective_field.argtypes = [C.c_void_p, _dp, _dp]
        L.mo_llg_rhs.argtypes = [C.c_void_p, _dp, _dp]
        L.mo_field_terms.argtypes = [C.c_void_p, _dp, _dp, C.c_int]
        L.mo_step.argtypes = [C.c_void_p, _dp, C.c_double, C.c_double, C.POINTER(C.c_int), _dp, _dp, _dp]
        L.mo_relax.argtypes = [C.c_void_p, _dp, C.c_double, C.c_double, C.c_long, C.c_double,
                               C.POINTER(C.c_long), _dp]
        L.mo_minimize.argtypes = [C.c_void_p, _dp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_long,
                                  C.POINTER(C.c_long), _dp, _dp]
        L.mo_sd_update.argtypes = [C.c_void_p, _dp, _dp, C.c_double]
        L.mo_sd_update.restype = None
        L.mo_energy.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.mo_average_m.argtypes = [C.c_void_p, _dp, _dp]
        L.mo_get_demag_kernel.argtypes = [C.c_void_p, C.c_int, _dp]
        L.mo_demag_direct_at.argtypes = [C.c_void_p, _dp, C.c_long, _dp]
        L.mo_newell_point.argtypes = [C.c_double] * 6 + [_dp]
        L.mo_newell_tensor.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [_dp]
        L.mo_dopri5_tableau.argtypes = [_dp, _dp]
        _up = C.POINTER(C.c_uint)
        L.mo_philox4x32_10.argtypes = [_up, _up, _up]
        L.mo_philox4x32_10.restype = None
        L.mo_normals3.argtypes = [C.c_ulonglong, C.c_ulonglong, C.c_ulonglong, _dp]
        L.mo_normals3.restype = None
        L.mo_thermal_field.argtypes = [C.c_void_p, C.c_double, C.c_ulonglong, _dp]
        L.mo_stt_tau.argtypes = [C.c_void_p, _dp, _dp]
        L.mo_cayley_apply.argtypes = [_dp, _dp, _dp]
        L.mo_cayley_apply.restype = None
        L.mo_set_zhang_li.argtypes = [C.c_void_p] + [C.c_double] * 4
        L.mo_set_zhang_li_pulse.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.mo_set_slonczewski.argtypes = [C.c_void_p] + [C.c_double] * 5
        L.mo_set_temperature.argtypes = [C.c_void_p, C.c_double, C.c_ulonglong]
        _lib = L
    return _lib


def _p(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with status {rc}")


def newell_point(X, Y, Z, dx, dy, dz):
    out = np.zeros(6)
    lib().mo_newell_point(X, Y, Z, dx, dy, dz, _p(out))
    return out


def philox4x32_10(ctr, key):
    c = (C.c_uint * 4)(*ctr)
    k = (C.c_uint * 2)(*key)
    o = (C.c_uint * 4)()
    lib().mo_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def normals3(seed, step, cell):
    out = np.zeros(3)
    lib().mo_normals3(seed, step, cell, _p(out))
    return out


def cayley_apply(w, m0):
    out = np.zeros(3)
    lib().mo_cayley_apply(_p(np.ascontiguousarray(w, dtype=np.float64)), _p(np.ascontiguousarray(m0, dtype=np.float64)), _p(out))
    return out


def dopri5_tableau():
    a = np.zeros(42)
    e = np.zeros(7)
    lib().mo_dopri5_tableau(_p(a), _p(e))
    return a.reshape(7, 6), e


class Oracle:
    """Mirror of the mm_* C ABI on host arrays (fp64)."""

    def __init__(self, nx, ny, nz, dx, dy, dz):
        self.L = lib()
        self.h = C.c_void_p()
        _chk(self.L.mo_create(C.byref(self.h), nx, ny, nz, dx, dy, dz), "create")
        self.nx, self.ny, self.nz = nx, ny, nz
        self.N = nx * ny * nz

    def __del__(self):
        if getattr(self, "h", None):
            self.L.mo_destroy(self.h)
            self.h = None

    # setters -------------------------------------------------------------------------
    def set_Ms(self, Ms):
        if np.isscalar(Ms):
            _chk(self.L.mo_set_Ms_uniform(self.h, float(Ms)), "set_Ms_uniform")
        else:
            a = np.ascontiguousarray(Ms, dtype=np.float64).reshape(-1)
            assert a.size == self.N
            _chk(self.L.mo_set_Ms(self.h, _p(a)), "set_Ms")

    def set_A(self, A): _chk(self.L.mo_set_A(self.h, A), "set_A")
    def set_D(self, D, kind): _chk(self.L.mo_set_D(self.h, D, kind), "set_D")
    def set_Ku(self, Ku): _chk(self.L.mo_set_Ku(self.h, Ku), "set_Ku")
    def set_Kc(self, Kc): _chk(self.L.mo_set_Kc(self.h, Kc), "set_Kc")

    def _cell(self, a, n):
        if a is None:
            return None
        a = np.ascontiguousarray(a, dtype=np.float64).reshape(-1)
        assert a.size == n
        return _p(a)

    def set_A_cell(self, A): _chk(self.L.mo_set_A_cell(self.h, self._cell(A, self.N)), "set_A_cell")
    def set_D_cell(self, D, kind): _chk(self.L.mo_set_D_cell(self.h, self._cell(D, self.N), kind), "set_D_cell")
    def set_H_ext_cell(self, H): _chk(self.L.mo_set_H_ext_cell(self.h, self._cell(H, 3 * self.N)), "set_H_ext_cell")
    def set_zhang_li(self, ux, uy, uz, beta): _chk(self.L.mo_set_zhang_li(self.h, ux, uy, uz, beta), "set_zhang_li")
    def set_zhang_li_pulse(self, b, w): _chk(self.L.mo_set_zhang_li_pulse(self.h, b, w), "set_zhang_li_pulse")
    def set_slonczewski(self, aJ, bJ, px, py, pz): _chk(self.L.mo_set_slonczewski(self.h, aJ, bJ, px, py, pz), "set_slonczewski")
    def set_temperature(self, T, seed): _chk(self.L.mo_set_temperature(self.h, T, seed), "set_temperature")
    def set_axis(self, ux, uy, uz): _chk(self.L.mo_set_axis(self.h, ux, uy, uz), "set_axis")
    def set_H_ext(self, hx, hy, hz): _chk(self.L.mo_set_H_ext(self.h, hx, hy, hz), "set_H_ext")
    def set_alpha(self, a): _chk(self.L.mo_set_alpha(self.h, a), "set_alpha")
    def set_gamma(self, g): _chk(self.L.mo_set_gamma(self.h, g), "set_gamma")
    def set_integrator(self, i): _chk(self.L.mo_set_integrator(self.h, i), "set_integrator")
    def set_demag(self, mode): _chk(self.L.mo_set_demag(self.h, mode), "set_demag")
    def init_demag(self): _chk(self.L.mo_init_demag(self.h), "init_demag")
    def time(self): return self.L.mo_time(self.h)
    def set_time(self, t): _chk(self.L.mo_set_time(self.h, t), "set_time")

    # compute -------------------------------------------------------------------------
    def _m(self, m):
        a = np.ascontiguousarray(m, dtype=np.float64).reshape(-1)
        assert a.size == 3 * self.N
        return a

    def effective_field(self, m):
        a = self._m(m)
        H = np.zeros_like(a)
        _chk(self.L.mo_effective_field(self.h, _p(a), _p(H)), "effective_field")
        return H.reshape(3, self.nz, self.ny, self.nx)

    def field_terms(self, m, which):
        a = self._m(m)
        H = np.zeros_like(a)
        _chk(self.L.mo_field_terms(self.h, _p(a), _p(H), which), "field_terms")
        return H.reshape(3, self.nz, self.ny, self.nx)

    def thermal_field(self, dt, step):
        xi = np.zeros(3 * self.N)
        _chk(self.L.mo_thermal_field(self.h, dt, step, _p(xi)), "thermal_field")
        return xi.reshape(3, self.nz, self.ny, self.nx)

    def stt_tau(self, m):
        a = self._m(m)
        t = np.zeros_like(a)
        _chk(self.L.mo_stt_tau(self.h, _p(a), _p(t)), "stt_tau")
        return t.reshape(3, self.nz, self.ny, self.nx)

    def llg_rhs(self, m):
        a = self._m(m)
        k = np.zeros_like(a)
        _chk(self.L.mo_llg_rhs(self.h, _p(a), _p(k)), "llg_rhs")
        return k.reshape(3, self.nz, self.ny, self.nx)

    def step(self, m, dt, tol=0.0):
        """In-place on m (must be a contiguous float64 array). Returns (accepted, err, dt_next, max_dmdt)."""
        assert m.dtype == np.float64 and m.flags["C_CONTIGUOUS"] and m.size == 3 * self.N
        acc = C.c_int()
        err, dn, md = np.zeros(1), np.zeros(1), np.zeros(1)
        _chk(self.L.mo_step(self.h, _p(m.reshape(-1)), dt, tol, C.byref(acc), _p(err), _p(dn), _p(md)), "step")
        return bool(acc.value), float(err[0]), float(dn[0]), float(md[0])

    def relax(self, m, tol, stop_dmdt, max_steps, dt0=1e-13):
        assert m.dtype == np.float64 and m.flags["C_CONTIGUOUS"] and m.size == 3 * self.N
        n = C.c_long()
        md = np.zeros(1)
        _chk(self.L.mo_relax(self.h, _p(m.reshape(-1)), tol, stop_dmdt, max_steps, dt0, C.byref(n), _p(md)), "relax")
        return n.value, float(md[0])

    def minimize(self, m, tau0, tau_min, tau_max, stop_torque, max_steps):
        """Steepest descent with Barzilai-Borwein steps, in place.
        Returns (updates done, max|m x (m x H)| at the last evaluation, last tau)."""
        assert m.dtype == np.float64 and m.flags["C_CONTIGUOUS"] and m.size == 3 * self.N
        n = C.c_long()
        mg, tl = np.zeros(1), np.zeros(1)
        _chk(self.L.mo_minimize(self.h, _p(m.reshape(-1)), tau0, tau_min, tau_max, stop_torque, max_steps, C.byref(n), _p(mg), _p(tl)),
             "minimize")
        return n.value, float(mg[0]), float(tl[0])

    def sd_update(self, m, H, tau):
        """One update of Eq. 51 with the given tau, in place on m."""
        assert m.dtype == np.float64 and m.flags["C_CONTIGUOUS"] and m.size == 3 * self.N
        self.L.mo_sd_update(self.h, _p(m.reshape(-1)), _p(np.ascontiguousarray(H, dtype=np.float64).reshape(-1)), tau)

    def energy(self, m):
        a = self._m(m)
        tot, terms = np.zeros(1), np.zeros(5)
        _chk(self.L.mo_energy(self.h, _p(a), _p(tot), _p(terms)), "energy")
        return float(tot[0]), terms

    def average_m(self, m):
        a = self._m(m)
        out = np.zeros(3)
        _chk(self.L.mo_average_m(self.h, _p(a), _p(out)), "average_m")
        return out

    def demag_kernel(self, comp):
        out = np.zeros(self.N)
        _chk(self.L.mo_get_demag_kernel(self.h, comp, _p(out)), "get_demag_kernel")
        return out.reshape(self.nz, self.ny, self.nx)

    def demag_direct_at(self, m, cell):
        a = self._m(m)
        out = np.zeros(3)
        self.L.mo_demag_direct_at(self.h, _p(a), int(cell), _p(out))
        return out

    def khat_imag_ratio(self):
        return self.L.mo_khat_imag_ratio(self.h)
