"""swe_cfl_dt_static (include/swe.h): the CFL time step with no handle, no workspace and no allocation,
its scratch in a fixed device array inside the library, against the existing handle-based path
(swe_compute_dt) on the same states.  dt tolerance as everywhere in tests/: 1e-12 relative.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after
the other GPU tests: it depends on nothing they leave behind, and the shared scratch array keeps
whatever the previous call wrote (the second call below is smaller than the first, so stale partial
maxima of the first sit right behind the ones it uses).
"""
import numpy as np
import pytest

from paper_2010_14416_b200 import binding as B
from paper_2010_14416_b200 import workloads as W

STATIC_MAX_CELLS = 1 << 26      # SWE_STATIC_MAX_CELLS


def _existing_path(w, nsteps):
    """State after nsteps of the shipped solver and the time step swe_compute_dt gives for it."""
    m = B.SweMesh.from_workload(w).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    m.run(nsteps)
    h, hu, hv = m.get_state()[:3]
    dt = m.compute_dt()
    rin = m.get_tables()["inradius"]
    m.destroy()
    return h, hu, hv, rin, dt


@pytest.mark.gpu
def test_static_scratch_dt_matches_compute_dt_twice_in_a_row():
    import torch
    big = W.canal_dam_break(300, 30, h_left=1.0, h_right=0.0, manning=0.03, seed=77, cfl=0.9)    # 18000 cells: 18 blocks, ragged tail
    small = W.config1()                                                                            # 2000 cells: 2 blocks
    cases = [(big, _existing_path(big, 60)), (small, _existing_path(small, 40))]
    assert cases[0][1][4] != pytest.approx(cases[1][1][4], rel=1e-3)     # two different answers
    dev = torch.device("cuda", 0)
    stream = torch.cuda.Stream(dev)
    outs, keep = [], []
    with torch.cuda.stream(stream):
        for w, (h, hu, hv, rin, _) in cases:
            t = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (h, hu, hv, rin)]
            out = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
            keep.append(t)
            outs.append(out)
        # two calls in a row on one stream, nothing in between
        for (w, _), t, out in zip(cases, keep, outs):
            B.cfl_dt_static(t[0].data_ptr(), t[1].data_ptr(), t[2].data_ptr(), t[3].data_ptr(), w.ncells,
                            w.g, w.cfl, w.h_dry, out.data_ptr(), stream.cuda_stream)
    stream.synchronize()
    for (w, (_, _, _, _, dt_ref)), out in zip(cases, outs):
        assert dt_ref > 0.0
        assert float(out.item()) == pytest.approx(dt_ref, rel=1e-12)
    # the same two calls again, in the other order: the array now holds the small case's partials in front
    with torch.cuda.stream(stream):
        for k in (1, 0):
            w, t, out = cases[k][0], keep[k], outs[k]
            out.fill_(-1.0)
            B.cfl_dt_static(t[0].data_ptr(), t[1].data_ptr(), t[2].data_ptr(), t[3].data_ptr(), w.ncells,
                            w.g, w.cfl, w.h_dry, out.data_ptr(), stream.cuda_stream)
    stream.synchronize()
    for (w, (_, _, _, _, dt_ref)), out in zip(cases, outs):
        assert float(out.item()) == pytest.approx(dt_ref, rel=1e-12)


@pytest.mark.gpu
def test_static_scratch_dt_against_the_oracle():
    """The oracle's own eq.(15) on its own geometry (inradius included), for a state with velocities."""
    import torch
    from oracle.swe_oracle import OracleSolver
    w = W.canal_dam_break(120, 12, h_left=1.0, h_right=0.3, seed=9)          # 2880 cells
    o = OracleSolver.from_workload(w)
    o.run(25)                                   # get some velocities
    h, hu, hv = o.get_state()[:3]
    o2 = OracleSolver.from_workload(w)
    o2.set_state(h, hu, hv)
    dt_ref = o2.compute_dt()
    rin = o.geometry()["rin"]
    dev = torch.device("cuda", 0)
    t = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (h, hu, hv, rin)]
    out = torch.zeros(1, dtype=torch.float64, device=dev)
    B.cfl_dt_static(t[0].data_ptr(), t[1].data_ptr(), t[2].data_ptr(), t[3].data_ptr(), w.ncells, w.g, w.cfl, w.h_dry,
                    out.data_ptr(), None)
    torch.cuda.synchronize()
    assert dt_ref > 0.0 and float(out.item()) == pytest.approx(dt_ref, rel=1e-12)


@pytest.mark.gpu
def test_static_scratch_all_dry_gives_zero():
    import torch
    dev = torch.device("cuda", 0)
    n = 3000
    z = torch.zeros(n, dtype=torch.float64, device=dev)
    rin = torch.ones(n, dtype=torch.float64, device=dev)
    out = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    B.cfl_dt_static(z.data_ptr(), z.data_ptr(), z.data_ptr(), rin.data_ptr(), n, 9.81, 0.9, 1e-6, out.data_ptr(), None)
    torch.cuda.synchronize()
    assert float(out.item()) == 0.0


def test_static_scratch_rejects_sizes_beyond_the_maximum():
    """Checked before any CUDA call: runs without a GPU (the addresses are never dereferenced)."""
    with pytest.raises(B.SweError) as ei:
        B.cfl_dt_static(256, 256, 256, 256, STATIC_MAX_CELLS + 1, 9.81, 0.9, 1e-6, 256, None)
    assert ei.value.code == -1 and "SWE_STATIC_MAX_CELLS" in str(ei.value)
    with pytest.raises(B.SweError):
        B.cfl_dt_static(256, 256, 256, 256, 0, 9.81, 0.9, 1e-6, 256, None)
    with pytest.raises(B.SweError):
        B.cfl_dt_static(None, 256, 256, 256, 10, 9.81, 0.9, 1e-6, 256, None)
