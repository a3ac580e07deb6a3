"""GPU parity at BASELINE.json's full sizes and run lengths (VERDICT r1 "parity" items): the whole field and
fixed-dt steps of configs[3] against the oracle at every cell, the full 5000-step relaxation of configs[2]
and the full 1 ns run of configs[1] with the invariants that hold at any length, and the host-mirror fix
of mm_run_until.  The oracle is compared where it is affordable (start windows, small twins)."""
import numpy as np
import pytest

import oracle
from gpu_common import avg_m, make_pair, masked_m, to_np
from paper_2406_16064_b200 import workloads as wl

pytestmark = pytest.mark.gpu
F32, F64 = 0, 1
HTOL = {F64: 1e-10, F32: 2e-4}
MTOL = {F64: 1e-8, F32: 1e-3}


@pytest.mark.slow
def test_cfg4_full_size_every_cell():
    """configs[3], 512x512x16, in bench.py's launch configuration: the WHOLE effective field (demag + exchange +
    bulk DMI + anisotropy + Zeeman) and two fixed-dt DOPRI5 steps against the oracle's FFT path at every cell,
    fp64 <= 1e-10 Ms and fp32 <= 2e-4 Ms."""
    from paper_2406_16064_b200 import Sim
    w = wl.cfg4()
    o = oracle.Oracle(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz)
    wl.apply(o, w)
    m0 = np.ascontiguousarray(w.m0)
    Href = o.effective_field(m0)
    mo = m0.copy()
    step_ref = []
    for _ in range(2):
        step_ref.append(o.step(mo, w.dt))
    for prec in (F64, F32):
        s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=prec)
        wl.apply(s, w)
        dm = s.to_device(m0)
        H = to_np(s.effective_field(dm))
        eh = np.abs(H - Href).max() / w.Ms_max
        assert eh <= HTOL[prec], (prec, eh)
        for i in range(2):
            ok, err, dn, md = s.step(dm, w.dt)
            ok_o, err_o, _, md_o = step_ref[i]
            assert ok and ok_o
            assert np.isclose(md, md_o, rtol=1e-9 if prec == F64 else 1e-3)
            if prec == F64:
                assert np.isclose(err, err_o, rtol=1e-5)
            else:
                assert abs(err - err_o) <= 2.0**-23 * np.sqrt(7.0) * w.dt * md_o
        g = to_np(dm)
        assert np.abs(g - mo).max() <= (1e-8 if prec == F64 else 5e-3), (prec, np.abs(g - mo).max())
        assert np.abs(g.reshape(3, -1).mean(axis=1) - mo.reshape(3, -1).mean(axis=1)).max() <= MTOL[prec]
        del s, dm


def test_cfg3_full_5000_adaptive_steps():
    """configs[2]: the full 5000-step adaptive DOPRI5 relaxation of the 256x256 skyrmion disk in fp32 on the GPU
    (the oracle cannot afford it; it is compared on a 64x64 twin below and on the first steps in
    test_gpu_parity.py).  Invariants: |m| = 1 on the disk, m = 0 outside, E non-increasing chunk to chunk up to
    fp32 rounding of the sum, the reversed core survives, the mean stays that of a single skyrmion."""
    from paper_2406_16064_b200 import Sim
    w = wl.cfg3(256)
    s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=F32)
    wl.apply(s, w)
    m = masked_m(w)
    dm = s.to_device(m)
    Ms = w.Ms_array()
    E = [s.energy(dm)[0]]
    steps = 0
    for _ in range(10):
        n, md = s.relax(dm, 1e-5, 0.0, 500, 1e-14)
        steps += n
        E.append(s.energy(dm)[0])
    assert steps == 5000
    g = to_np(dm)
    nrm = np.sqrt((g * g).sum(axis=0))
    assert np.abs(nrm[Ms > 0] - 1).max() < 5e-7 and np.all(g[:, Ms == 0] == 0)
    assert E[-1] < E[0]
    assert all(E[i + 1] <= E[i] + 1e-7 * abs(E[i]) for i in range(len(E) - 1)), E
    assert g[2, 0, 128, 128] < -0.9                      # core still reversed
    assert 0.98 < avg_m(g, Ms)[2] < 1.0
    assert s.time() > 5e-10


@pytest.mark.parametrize("prec", [F64, F32])
def test_cfg3_twin_end_state_vs_oracle(prec):
    """The same relaxation on a 64x64 twin (disk radius and core scaled with n), 400 adaptive steps on both sides:
    end-state <m_z> and E within 1e-2 relative (R8/R10: accept/reject sequences
    may differ by rounding, observables are compared)."""
    w = wl.cfg3(64)
    o, s = make_pair(w, prec)
    m = masked_m(w)
    dm = s.to_device(m)
    n_o, _ = o.relax(m, 1e-5, 0.0, 400, 1e-14)
    n_s, _ = s.relax(dm, 1e-5, 0.0, 400, 1e-14)
    assert n_o == 400 and n_s == 400
    Ms = w.Ms_array()
    g = to_np(dm)
    assert abs(avg_m(g, Ms)[2] - avg_m(m, Ms)[2]) <= 1e-2 * abs(avg_m(m, Ms)[2])
    Es, Eo = s.energy(dm)[0], o.energy(m)[0]
    assert abs(Es - Eo) <= 1e-2 * abs(Eo)
    assert np.isclose(s.time(), o.time(), rtol=2e-2)


@pytest.mark.parametrize("prec", [F64, F32])
def test_cfg2_full_relax_and_1ns_run(prec):
    """configs[1] in full on the GPU: relax at alpha = 0.5 until max|dm/dt| < 1e7 rad/s, switch the field on, run
    adaptive DOPRI5 (tol 1e-6) to exactly 1 ns.  At the 0.1 ns marks: |m| = 1, t lands on the mark, E (constant field,
    alpha > 0) never increases, and <m> agrees with the ORACLE's run of the same procedure within 1e-4 (fp64) / 1e-2
    (fp32).  The oracle's values are stored in tests/golden/cfg2_trajectory.txt, written by
    tests/golden/make_cfg2_trajectory.py, which calls only oracle/ (ten minutes of CPU, so not re-run here)."""
    from conftest import load_golden
    from paper_2406_16064_b200 import Sim
    gold = load_golden("cfg2_trajectory.txt")
    mtol = 1e-4 if prec == F64 else 1e-2
    w = wl.cfg2()
    w.alpha = 0.5
    s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=prec)
    wl.apply(s, w)
    dm = s.to_device(masked_m(w))
    n, md = s.relax(dm, 1e-6, 1e7, 200000, 1e-13)
    assert md < 1e7 and 100 < n < 200000
    s.set_alpha(0.02)
    s.set_H_ext(*wl.CFG2_FIELD)
    s.set_time(0.0)
    Ms = w.Ms_array()
    # the relaxation ends where max|dm/dt| crosses the threshold on a very flat tail: a few attempts either way
    assert abs(n - gold["relax_steps"][0]) <= 0.05 * gold["relax_steps"][0]
    assert np.abs(avg_m(to_np(dm), Ms) - np.array(gold["m_0"])).max() < mtol
    E = [s.energy(dm)[0]]
    tot = 0
    worst = 0.0
    for k in range(1, 11):
        tot += s.run_until(dm, k * 1e-10, 1e-6, 1e-13)
        assert np.isclose(s.time(), k * 1e-10, rtol=1e-12)
        g = to_np(dm)
        assert np.abs(np.sqrt((g * g).sum(axis=0)) - 1).max() < (1e-14 if prec == F64 else 5e-7)
        E.append(s.energy(dm)[0])
        worst = max(worst, np.abs(avg_m(g, Ms) - np.array(gold[f"m_{k}"])).max())
    print(f"cfg2 1 ns prec={prec}: max |<m> - oracle| over the ten marks = {worst:.3e}, attempts {tot} (oracle {gold['run_attempts'][0]:.0f})")
    assert worst < mtol, worst
    assert all(E[i + 1] < E[i] for i in range(10)), E
    assert abs(tot - gold["run_attempts"][0]) <= 0.05 * gold["run_attempts"][0]


def test_run_until_after_unsynchronised_steps():
    """mm_run_until must clip against the DEVICE clock: steps enqueued with sync=False advance it without
    refreshing the host mirror.  The run must end exactly at t_end and reject a t_end in the past."""
    from paper_2406_16064_b200 import Sim, MMError
    w = wl.cfg2()
    s = Sim(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec=F64)
    wl.apply(s, w)
    dm = s.to_device(masked_m(w))
    for _ in range(5):
        s.step(dm, 2e-13, sync=False)                  # device t = 1e-12, host mirror still 0
    t_end = 1.05e-12
    s.run_until(dm, t_end, 1e-6, 2e-13)                # dt0 larger than what is left
    assert np.isclose(s.time(), t_end, rtol=1e-12)
    for _ in range(3):
        s.step(dm, 2e-13, sync=False)
    with pytest.raises(MMError):
        s.run_until(dm, 1.2e-12, 1e-6, 1e-13)          # already past it
