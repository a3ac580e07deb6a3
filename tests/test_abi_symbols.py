"""The C-ABI library builds, loads and exports every symbol include/mm.h declares (no compute)."""
import ctypes as C
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "mm.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(mm_[a-zA-Z_0-9]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    from paper_2406_16064_b200.build import build
    from paper_2406_16064_b200 import binding
    lib = C.CDLL(build())
    names = declared_symbols()
    assert len(names) >= 30
    for n in names:
        assert hasattr(lib, n), f"{n} declared in mm.h but not exported"
    assert set(names) == set(binding.SIGNATURES), "binding.SIGNATURES out of sync with mm.h"
    lib.mm_version.restype = C.c_char_p
    assert b"sm_100a" in lib.mm_version()


def test_argument_errors_without_gpu():
    """Argument validation that needs no device."""
    from paper_2406_16064_b200.build import build
    lib = C.CDLL(build())
    h = C.c_void_p()
    f = lib.mm_create
    f.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, C.c_void_p]
    assert f(C.byref(h), 0, 4, 4, 1e-9, 1e-9, 1e-9, 0, 0, None) == -1          # MM_ERR_ARG
    assert f(C.byref(h), 4, 4, 4, -1e-9, 1e-9, 1e-9, 0, 0, None) == -1
    assert f(C.byref(h), 1 << 21, 4, 4, 1e-9, 1e-9, 1e-9, 0, 0, None) == -2    # MM_ERR_UNSUPPORTED (too large)
    assert f(C.byref(h), 12, 5, 3, 1e-9, 1e-9, 1e-9, 0, 0, None) == 0           # not 2^k: embedded in 16 x 8 x 4
    lib.mm_workspace_bytes.restype = C.c_size_t
    lib.mm_workspace_bytes.argtypes = [C.c_void_p]
    lib.mm_destroy.argtypes = [C.c_void_p]
    emb = lib.mm_workspace_bytes(h)
    assert lib.mm_destroy(h) == 0
    assert f(C.byref(h), 16, 8, 4, 1e-9, 1e-9, 1e-9, 0, 0, None) == 0
    assert emb > lib.mm_workspace_bytes(h)                                       # two extra inner-layout slots
    assert lib.mm_destroy(h) == 0
    assert f(C.byref(h), 16, 16, 1, 1e-9, 1e-9, 1e-9, 1, 0, None) == 0
    lib.mm_workspace_bytes.restype = C.c_size_t
    lib.mm_workspace_bytes.argtypes = [C.c_void_p]
    assert lib.mm_workspace_bytes(h) > 16 * 16 * 8 * 30
    lib.mm_set_axis.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
    assert lib.mm_set_axis(h, 0.0, 0.0, 0.0) == -1
    lib.mm_init_demag.argtypes = [C.c_void_p]
    assert lib.mm_init_demag(h) == -3                                            # MM_ERR_STATE: no workspace
    lib.mm_destroy.argtypes = [C.c_void_p]
    assert lib.mm_destroy(h) == 0


def test_binding_fails_loudly_without_gpu():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2406_16064_b200 import Sim, MMError
    with pytest.raises(MMError):
        Sim(16, 16, 1, 1e-9, 1e-9, 1e-9)
