"""ctypes binding of include/mm.h — argument marshalling only; every step runs in libmm.so's kernels.

PyTorch is used for device memory (m, H, workspace tensors) and the CUDA stream, nothing else.
"""
import ctypes as C
import os

F32, F64 = 0, 1
RK4, DOPRI5, CAYLEY_RK4 = 0, 1, 2
DMI_NONE, DMI_BULK, DMI_INTERFACIAL, DMI_D2D = 0, 1, 2, 3
_STATUS = {0: "MM_OK", -1: "MM_ERR_ARG", -2: "MM_ERR_UNSUPPORTED", -3: "MM_ERR_STATE", -4: "MM_ERR_CUDA",
           -5: "MM_ERR_NOMEM", -6: "MM_ERR_NAN", -7: "MM_ERR_INTERNAL"}
HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmm.so")
_lib = None

# name -> (restype, argtypes): every symbol include/mm.h declares
_vp, _d, _i, _l = C.c_void_p, C.c_double, C.c_int, C.c_long
_dp, _ip, _lp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_long)
SIGNATURES = {
    "mm_create": (_i, [C.POINTER(_vp), _i, _i, _i, _d, _d, _d, _i, _i, _vp]),
    "mm_destroy": (_i, [_vp]),
    "mm_workspace_bytes": (C.c_size_t, [_vp]),
    "mm_set_workspace": (_i, [_vp, _vp, C.c_size_t]),
    "mm_set_Ms_uniform": (_i, [_vp, _d]),
    "mm_set_Ms": (_i, [_vp, _vp]),
    "mm_set_A": (_i, [_vp, _d]),
    "mm_set_D": (_i, [_vp, _d, _i]),
    "mm_set_Ku": (_i, [_vp, _d]),
    "mm_set_Kc": (_i, [_vp, _d]),
    "mm_set_zhang_li": (_i, [_vp, _d, _d, _d, _d]),
    "mm_set_zhang_li_pulse": (_i, [_vp, _d, _d]),
    "mm_set_slonczewski": (_i, [_vp, _d, _d, _d, _d, _d]),
    "mm_set_temperature": (_i, [_vp, _d, C.c_ulonglong]),
    "mm_thermal_field": (_i, [_vp, _d, C.c_ulonglong, _vp]),
    "mm_set_A_cell": (_i, [_vp, _vp]),
    "mm_set_D_cell": (_i, [_vp, _vp, _i]),
    "mm_set_H_ext_cell": (_i, [_vp, _vp]),
    "mm_set_axis": (_i, [_vp, _d, _d, _d]),
    "mm_set_H_ext": (_i, [_vp, _d, _d, _d]),
    "mm_set_alpha": (_i, [_vp, _d]),
    "mm_set_gamma": (_i, [_vp, _d]),
    "mm_set_integrator": (_i, [_vp, _i]),
    "mm_set_demag": (_i, [_vp, _i]),
    "mm_init_demag": (_i, [_vp]),
    "mm_effective_field": (_i, [_vp, _vp, _vp]),
    "mm_llg_rhs": (_i, [_vp, _vp, _vp]),
    "mm_step": (_i, [_vp, _vp, _d, _d, _ip, _dp, _dp, _dp]),
    "mm_relax": (_i, [_vp, _vp, _d, _d, _l, _d, _lp, _dp]),
    "mm_run_until": (_i, [_vp, _vp, _d, _d, _d, _l, _lp]),
    "mm_minimize": (_i, [_vp, _vp, _d, _d, _d, _d, _l, _lp, _dp, _dp]),
    "mm_run_host": (_i, [_vp, _vp, _i, _d, _d]),
    "mm_llg_rhs_host": (_i, [_vp, _vp, _vp]),
    "mm_time": (_d, [_vp]),
    "mm_set_time": (_i, [_vp, _d]),
    "mm_average_m": (_i, [_vp, _vp, _dp]),
    "mm_average_m_static": (_i, [_i, _vp, _i, _l, _vp, _vp, _vp]),
    "mm_static_last_error": (C.c_char_p, []),
    "mm_energy": (_i, [_vp, _vp, _dp, _dp]),
    "mm_get_demag_kernel": (_i, [_vp, _i, _vp]),
    "mm_set_profiling": (_i, [_vp, _i]),
    "mm_get_profile": (_i, [_vp, _dp, _lp]),
    "mm_get_stats": (_i, [_vp, _lp, _lp, _lp]),
    "mm_launch_count": (_l, [_vp]),
    "mm_last_error": (C.c_char_p, [_vp]),
    "mm_version": (C.c_char_p, []),
}


class MMError(RuntimeError):
    pass


def load_library(path=LIB_PATH):
    """Load libmm.so; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(path):
            raise MMError(f"{path} not found: build it with `python -m paper_2406_16064_b200.build` "
                          "(there is no CPU fallback)")
        L = C.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


STATIC_MAX_CELLS = 1 << 26   # MM_STATIC_MAX_CELLS of include/mm.h


def average_m_static(m, Ms, out=None):
    """mm_average_m_static: <m> over the cells with Ms != 0, for callers that can hand the library no workspace.

    The partial sums go to an array built into libmm.so, so the C call allocates nothing; no Sim (and therefore no
    workspace tensor) is needed.  m: CUDA tensor of 3N reals (float32 or float64), Ms: N reals of the same dtype and
    device.  Returns `out`, 3 float64 values on the same device (pass your own tensor if this wrapper must not
    allocate either), filled asynchronously on torch's current stream.  At most STATIC_MAX_CELLS cells; calls that
    may overlap on the GPU (different streams) share the built-in array and must be ordered by the caller.  Make the
    first call on each device during start-up (include/mm.h)."""
    import torch
    if not (torch.is_tensor(m) and m.is_cuda):
        raise MMError("no CUDA tensor: the mm library has no CPU path")
    L = load_library()
    assert m.dtype in (torch.float32, torch.float64) and Ms.dtype == m.dtype and Ms.device == m.device
    assert m.is_contiguous() and Ms.is_contiguous() and m.numel() == 3 * Ms.numel()
    if out is None:
        out = torch.empty(3, dtype=torch.float64, device=m.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() == 3 and out.is_contiguous()
    dev = m.device.index if m.device.index is not None else torch.cuda.current_device()
    stream = torch.cuda.current_stream(m.device)
    rc = L.mm_average_m_static(dev, _vp(stream.cuda_stream), F64 if m.dtype == torch.float64 else F32, Ms.numel(),
                               _vp(m.data_ptr()), _vp(Ms.data_ptr()), _vp(out.data_ptr()))
    if rc != 0:
        raise MMError(f"mm_average_m_static: {_STATUS.get(rc, rc)} ({L.mm_static_last_error().decode()})")
    return out


class Sim:
    """One mm_sim handle.  Device arrays are torch CUDA tensors shaped [3, nz, ny, nx] / [nz, ny, nx]."""

    def __init__(self, nx, ny, nz, dx, dy, dz, prec=F32, device=0):
        import torch
        if not torch.cuda.is_available():
            raise MMError("no CUDA device: the mm library has no CPU path")
        self.torch = torch
        self.L = load_library()
        self.nx, self.ny, self.nz, self.N = nx, ny, nz, nx * ny * nz
        self.prec = prec
        self.dtype = torch.float64 if prec == F64 else torch.float32
        self.device = torch.device("cuda", device)
        self.stream = torch.cuda.current_stream(self.device)
        self.h = _vp()
        rc = self.L.mm_create(C.byref(self.h), nx, ny, nz, dx, dy, dz, prec, device, _vp(self.stream.cuda_stream))
        if rc != 0:
            raise MMError(f"mm_create: {_STATUS.get(rc, rc)}")
        nbytes = self.L.mm_workspace_bytes(self.h)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self.workspace.data_ptr() + 255) & ~255
        self._chk(self.L.mm_set_workspace(self.h, _vp(ptr), nbytes), "mm_set_workspace")

    def __del__(self):
        if getattr(self, "h", None) and self.h.value:
            self.L.mm_destroy(self.h)
            self.h = _vp()

    def _chk(self, rc, what):
        if rc != 0:
            msg = self.L.mm_last_error(self.h)
            raise MMError(f"{what}: {_STATUS.get(rc, rc)} ({msg.decode() if msg else ''})")

    # tensors ---------------------------------------------------------------------------
    def to_device(self, a):
        return self.torch.as_tensor(a, dtype=self.dtype).contiguous().to(self.device)

    def _dev(self, t, n):
        assert t.is_cuda and t.dtype == self.dtype and t.is_contiguous() and t.numel() == n, "bad device tensor"
        assert t.data_ptr() % 16 == 0, "device pointers must be 16-byte aligned (include/mm.h)"
        return _vp(t.data_ptr())

    def empty_field(self):
        return self.torch.empty((3, self.nz, self.ny, self.nx), dtype=self.dtype, device=self.device)

    # setters ---------------------------------------------------------------------------
    def set_Ms(self, Ms):
        import numpy as np
        if np.isscalar(Ms):
            self._chk(self.L.mm_set_Ms_uniform(self.h, float(Ms)), "mm_set_Ms_uniform")
        else:
            t = Ms if self.torch.is_tensor(Ms) else self.to_device(Ms)
            self._chk(self.L.mm_set_Ms(self.h, self._dev(t, self.N)), "mm_set_Ms")
            self.torch.cuda.current_stream(self.device).synchronize()

    def set_A(self, A): self._chk(self.L.mm_set_A(self.h, A), "mm_set_A")
    def set_D(self, D, kind): self._chk(self.L.mm_set_D(self.h, D, kind), "mm_set_D")
    def set_Ku(self, Ku): self._chk(self.L.mm_set_Ku(self.h, Ku), "mm_set_Ku")
    def set_Kc(self, Kc): self._chk(self.L.mm_set_Kc(self.h, Kc), "mm_set_Kc")
    def set_zhang_li(self, ux, uy, uz, beta): self._chk(self.L.mm_set_zhang_li(self.h, ux, uy, uz, beta), "mm_set_zhang_li")
    def set_zhang_li_pulse(self, b, w): self._chk(self.L.mm_set_zhang_li_pulse(self.h, b, w), "mm_set_zhang_li_pulse")
    def set_slonczewski(self, aJ, bJ, px, py, pz): self._chk(self.L.mm_set_slonczewski(self.h, aJ, bJ, px, py, pz), "mm_set_slonczewski")
    def set_temperature(self, T, seed): self._chk(self.L.mm_set_temperature(self.h, T, seed), "mm_set_temperature")

    def thermal_field(self, dt, step):
        out = self.empty_field()
        self._chk(self.L.mm_thermal_field(self.h, dt, step, self._dev(out, 3 * self.N)), "mm_thermal_field")
        return out

    def _cell(self, a, n):
        """Device pointer of a per-cell array (numpy or tensor, copied by the library), or NULL for None."""
        if a is None:
            return None, None
        t = a if self.torch.is_tensor(a) else self.to_device(a)
        return t, self._dev(t, n)

    def set_A_cell(self, A):
        t, p = self._cell(A, self.N)
        self._chk(self.L.mm_set_A_cell(self.h, p), "mm_set_A_cell")
        self.torch.cuda.current_stream(self.device).synchronize()

    def set_D_cell(self, D, kind):
        t, p = self._cell(D, self.N)
        self._chk(self.L.mm_set_D_cell(self.h, p, kind), "mm_set_D_cell")
        self.torch.cuda.current_stream(self.device).synchronize()

    def set_H_ext_cell(self, H):
        t, p = self._cell(H, 3 * self.N)
        self._chk(self.L.mm_set_H_ext_cell(self.h, p), "mm_set_H_ext_cell")
        self.torch.cuda.current_stream(self.device).synchronize()
    def set_axis(self, ux, uy, uz): self._chk(self.L.mm_set_axis(self.h, ux, uy, uz), "mm_set_axis")
    def set_H_ext(self, hx, hy, hz): self._chk(self.L.mm_set_H_ext(self.h, hx, hy, hz), "mm_set_H_ext")
    def set_alpha(self, a): self._chk(self.L.mm_set_alpha(self.h, a), "mm_set_alpha")
    def set_gamma(self, g): self._chk(self.L.mm_set_gamma(self.h, g), "mm_set_gamma")
    def set_integrator(self, i): self._chk(self.L.mm_set_integrator(self.h, i), "mm_set_integrator")
    def set_demag(self, on): self._chk(self.L.mm_set_demag(self.h, int(on)), "mm_set_demag")
    def init_demag(self): self._chk(self.L.mm_init_demag(self.h), "mm_init_demag")
    def time(self): return self.L.mm_time(self.h)
    def set_time(self, t): self._chk(self.L.mm_set_time(self.h, t), "mm_set_time")
    def launch_count(self): return self.L.mm_launch_count(self.h)

    # compute ---------------------------------------------------------------------------
    def effective_field(self, m, H=None):
        H = self.empty_field() if H is None else H
        self._chk(self.L.mm_effective_field(self.h, self._dev(m, 3 * self.N), self._dev(H, 3 * self.N)), "mm_effective_field")
        return H

    def llg_rhs(self, m, out=None):
        out = self.empty_field() if out is None else out
        self._chk(self.L.mm_llg_rhs(self.h, self._dev(m, 3 * self.N), self._dev(out, 3 * self.N)), "mm_llg_rhs")
        return out

    def step(self, m, dt, tol=0.0, sync=True):
        if not sync:
            self._chk(self.L.mm_step(self.h, self._dev(m, 3 * self.N), dt, tol, None, None, None, None), "mm_step")
            return None
        acc, err, dn, md = C.c_int(), C.c_double(), C.c_double(), C.c_double()
        self._chk(self.L.mm_step(self.h, self._dev(m, 3 * self.N), dt, tol, C.byref(acc), C.byref(err), C.byref(dn),
                                 C.byref(md)), "mm_step")
        return bool(acc.value), err.value, dn.value, md.value

    def relax(self, m, tol, stop_dmdt, max_steps, dt0=1e-13):
        n, md = C.c_long(), C.c_double()
        self._chk(self.L.mm_relax(self.h, self._dev(m, 3 * self.N), tol, stop_dmdt, max_steps, dt0, C.byref(n),
                                  C.byref(md)), "mm_relax")
        return n.value, md.value

    def run_until(self, m, t_end, tol, dt0=1e-13, max_steps=1000000):
        n = C.c_long()
        self._chk(self.L.mm_run_until(self.h, self._dev(m, 3 * self.N), t_end, tol, dt0, max_steps, C.byref(n)), "mm_run_until")
        return n.value

    def minimize(self, m, tau0, tau_min, tau_max, stop_torque, max_steps):
        """Steepest descent with Barzilai-Borwein steps (mm_minimize), in place on m.
        Returns (updates done, max|m x (m x H)| at the last evaluation, last tau)."""
        n = C.c_long()
        mg, tl = C.c_double(), C.c_double()
        self._chk(self.L.mm_minimize(self.h, self._dev(m, 3 * self.N), tau0, tau_min, tau_max, stop_torque, max_steps,
                                     C.byref(n), C.byref(mg), C.byref(tl)), "mm_minimize")
        return n.value, mg.value, tl.value

    def run_host(self, host_m, nsteps, dt, tol=0.0):
        """host_m: pinned (or pageable) CPU tensor [3,nz,ny,nx] of the sim dtype, updated in place."""
        assert (not host_m.is_cuda) and host_m.dtype == self.dtype and host_m.is_contiguous()
        self._chk(self.L.mm_run_host(self.h, _vp(host_m.data_ptr()), nsteps, dt, tol), "mm_run_host")

    def llg_rhs_host(self, host_m, host_out):
        assert (not host_m.is_cuda) and (not host_out.is_cuda) and host_m.dtype == self.dtype
        self._chk(self.L.mm_llg_rhs_host(self.h, _vp(host_m.data_ptr()), _vp(host_out.data_ptr())), "mm_llg_rhs_host")

    def average_m(self, m):
        out = (C.c_double * 3)()
        self._chk(self.L.mm_average_m(self.h, self._dev(m, 3 * self.N), out), "mm_average_m")
        return [out[0], out[1], out[2]]

    def energy(self, m):
        tot, terms = C.c_double(), (C.c_double * 5)()
        self._chk(self.L.mm_energy(self.h, self._dev(m, 3 * self.N), C.byref(tot), terms), "mm_energy")
        return tot.value, list(terms)

    def stats(self):
        """(accepted attempts, rejected attempts, RHS evaluations of the steppers) since the workspace was set."""
        a, r, n = C.c_long(), C.c_long(), C.c_long()
        self._chk(self.L.mm_get_stats(self.h, C.byref(a), C.byref(r), C.byref(n)), "mm_get_stats")
        return a.value, r.value, n.value

    def set_profiling(self, on): self._chk(self.L.mm_set_profiling(self.h, int(on)), "mm_set_profiling")

    def get_profile(self):
        ms, cnt = (C.c_double * 4)(), (C.c_long * 4)()
        self._chk(self.L.mm_get_profile(self.h, ms, cnt), "mm_get_profile")
        return list(ms), list(cnt)

    def demag_kernel(self, comp):
        out = self.torch.empty((self.nz, self.ny, self.nx), dtype=self.torch.float64, device=self.device)
        self._chk(self.L.mm_get_demag_kernel(self.h, comp, _vp(out.data_ptr())), "mm_get_demag_kernel")
        self.torch.cuda.current_stream(self.device).synchronize()
        return out
