"""mm_average_m_static — <m> without a workspace (include/mm.h, csrc/mm_noalloc.cu).

Why the entry point exists: every other compute call of the library needs a workspace the caller allocates.  A caller
that cannot allocate device memory — a logging hook inside an application whose memory pool has taken all of HBM, code
in a latency-critical loop that must not trigger cudaMalloc's device-wide wait, a plug-in that gets two arrays and a
stream and nothing else — uses this call instead; its partial sums live in an array built into libmm.so.

What is checked here: the new call returns the same <m> as the existing path (Sim.average_m = mm_average_m, which
keeps its partial sums in the workspace), on two calls in a row with different inputs.  The second call finds the
first call's partial sums and a used block counter in the built-in array, so a missing reset, or a slot that is read
without having been rewritten, shows up as a wrong second result.  Both paths add the same values in fp64 and differ
only in the order of the additions, so the tolerance is 1e-12 in both precisions (the other average_m tests use 1e-12
for fp64 and 1e-6 for fp32).

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide the parity
tests), and it depends on no state the earlier tests leave: it passes alone in a fresh process and at the end of
the whole run.
"""
import ctypes as C

import numpy as np
import pytest


def test_sizes_beyond_the_built_in_array_are_refused_without_a_gpu():
    """The size check comes before any CUDA call: it can be exercised on a box with no GPU."""
    from paper_2406_16064_b200 import binding
    L = binding.load_library()
    buf = (C.c_double * 4)()
    p = C.cast(buf, C.c_void_p)
    rc = L.mm_average_m_static(0, None, binding.F64, binding.STATIC_MAX_CELLS + 1, p, p, p)
    assert rc == -2                                                                 # MM_ERR_UNSUPPORTED
    msg = L.mm_static_last_error().decode()
    assert str(binding.STATIC_MAX_CELLS) in msg and str(binding.STATIC_MAX_CELLS + 1) in msg
    assert L.mm_average_m_static(0, None, binding.F64, 0, p, p, p) == -1            # MM_ERR_ARG
    assert L.mm_average_m_static(0, None, binding.F64, 8, None, p, p) == -1
    assert L.mm_average_m_static(0, None, 7, 8, p, p, p) == -1
    assert L.mm_average_m_static(-1, None, binding.F64, 8, p, p, p) == -1


@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_static_average_matches_the_workspace_path_twice_in_a_row(prec):
    import torch
    from paper_2406_16064_b200 import Sim, F32, F64, workloads as wl
    from paper_2406_16064_b200.binding import average_m_static

    # 100 x 50 x 3 = 15 000 cells: three full 4096-cell blocks and a ragged fourth; a quarter of the cells vacuum
    nx, ny, nz = 100, 50, 3
    w = wl.cfg4(nx, ny, nz)
    w.Ms = 8.6e5 * wl.random_mask(21, nx, ny, nz, 0.75)
    s = Sim(nx, ny, nz, w.dx, w.dy, w.dz, prec=F64 if prec == "f64" else F32)
    wl.apply(s, w, with_demag=False)
    Ms = s.to_device(w.Ms_array())
    live = w.Ms_array() > 0
    out = torch.full((3,), float("nan"), dtype=torch.float64, device=Ms.device)

    rng = np.random.default_rng(5)
    for call in range(2):
        m = rng.normal(size=(3, nz, ny, nx)) + (0.3, -0.2, 0.1)[call] * (call + 1)
        m /= np.linalg.norm(m, axis=0)
        dm = s.to_device(m)                      # NOT masked: cells with Ms = 0 must be skipped by the kernel itself
        got = average_m_static(dm, Ms, out=out).cpu().numpy()
        ref = np.array(s.average_m(dm))
        assert np.all(np.isfinite(got))
        assert np.abs(got - ref).max() <= 1e-12, (call, got, ref)
        # and both agree with the definition, evaluated on the values the device holds
        mh = dm.cpu().numpy().astype(np.float64)
        mean = np.array([mh[c][live].mean() for c in range(3)])
        assert np.abs(got - mean).max() <= 1e-12, (call, got, mean)


@pytest.mark.gpu
def test_static_average_of_an_all_vacuum_mesh_is_zero_and_large_inputs_run():
    import torch
    from paper_2406_16064_b200.binding import average_m_static

    m = torch.ones(3 * 5000, dtype=torch.float32, device="cuda")
    assert average_m_static(m, torch.zeros(5000, dtype=torch.float32, device="cuda")).cpu().tolist() == [0.0, 0.0, 0.0]
    # 2048 x 2048 x 1 cells = 1024 blocks: the last block's fixed-order sum spans several rounds per thread
    N = 2048 * 2048
    g = torch.Generator(device="cuda").manual_seed(3)
    m = torch.rand(3 * N, dtype=torch.float32, device="cuda", generator=g) - 0.25
    Ms = (torch.rand(N, dtype=torch.float32, device="cuda", generator=g) > 0.1).float() * 8e5
    got = average_m_static(m, Ms).cpu().numpy()
    md = m.double().view(3, N)[:, Ms > 0]
    assert np.abs(got - md.mean(dim=1).cpu().numpy()).max() <= 1e-12
