"""GPU-vs-oracle parity through the C ABI (north_star tolerances, written here):

  |x_gpu - x_oracle| <= 1e-10 + 1e-10 |x_oracle|   for h, hu, hv after the stated steps
  dt matched to 1e-12 relative, simulated time likewise
  dry-cell mask (h <= h_dry) identical

Both sides get the same seeded arrays from paper_2010_14416_b200.workloads.
"""
import numpy as np
import pytest

from oracle.swe_oracle import OracleSolver
from paper_2010_14416_b200 import binding as B
from paper_2010_14416_b200 import workloads as W
from tests.analytic import stoker_profile

pytestmark = pytest.mark.gpu

RTOL = ATOL = 1e-10


def run_both(w, nsteps, **kw):
    m = B.SweMesh.from_workload(w, **kw).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    o = OracleSolver.from_workload(w)
    dt0_g, dt0_o = m.compute_dt(), o.compute_dt()
    assert dt0_g == pytest.approx(dt0_o, rel=1e-12)
    m.run(nsteps)
    done = o.run(nsteps)
    assert done == nsteps
    return m, o


def assert_parity(m, o, w):
    hg, hug, hvg, tg, dtg = m.get_state()
    ho, huo, hvo, to, dto = o.get_state()
    np.testing.assert_array_equal(hg <= w.h_dry, ho <= w.h_dry)
    np.testing.assert_allclose(hg, ho, rtol=RTOL, atol=ATOL)
    np.testing.assert_allclose(hug, huo, rtol=RTOL, atol=ATOL)
    np.testing.assert_allclose(hvg, hvo, rtol=RTOL, atol=ATOL)
    assert tg == pytest.approx(to, rel=1e-12)
    assert dtg == pytest.approx(dto, rel=1e-12)
    sg, so = m.get_stats(), o.stats()
    assert sg["n_clamped"] == 0 and so["nclamp"] == 0 and sg["n_nonfinite"] == 0
    assert sg["n_dry"] == so["ndry"]
    assert sg["volume"] == pytest.approx(so["volume"], rel=1e-12)
    assert sg["steps"] == so["steps"]
    return hg, hug, hvg, tg


LOOPS = [B.LOOP_GRAPH, B.LOOP_PERSISTENT, B.LOOP_LAUNCH, B.LOOP_CLUSTER]


@pytest.mark.parametrize("loop_mode", LOOPS)
def test_config1_wetwet_dambreak(loop_mode):
    """BASELINE configs[0] in full: 2000 cells, 500 steps, every loop mode."""
    w = W.config1()
    m, o = run_both(w, w.nsteps, loop_mode=loop_mode)
    h, hu, hv, t = assert_parity(m, o, w)
    assert m.get_launch_info()["loop_mode"] == B.LOOP_NAMES[loop_mode]
    v0 = float(np.sum(w.h * OracleSolver.from_workload(w).geometry()["area"]))
    assert m.get_stats()["volume"] == pytest.approx(v0, rel=1e-12)


def test_config1_stoker_profile():
    """The GPU result itself against the closed-form Stoker solution before wall reflection."""
    w = W.config1()
    m = B.SweMesh.from_workload(w).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    while True:
        m.run(20)
        h, hu, hv, t, _ = m.get_state()
        if t >= 8.0:
            break
    cx = W.centroids(w.nodes_xy, w.tris)[:, 0]
    hex_, _ = stoker_profile((cx - 50.0) / t, 1.0, 0.5)
    area = m.get_tables()["area"]
    assert float(np.sum(np.abs(h - hex_) * area) / area.sum()) < 0.012


@pytest.mark.parametrize("ordering", [B.ORDER_IDENTITY, B.ORDER_HILBERT, B.ORDER_RCM])
def test_config2_wetdry_dambreak_full(ordering):
    """BASELINE configs[1] in full: 200k cells, Manning 0.03, wet/dry front, 2000 steps."""
    w = W.config2()
    m, o = run_both(w, w.nsteps, ordering=ordering)
    assert_parity(m, o, w)


def test_config3_lake_at_rest_reduced_full_steps():
    """configs[2] shape (bumps, islands, Manning 0.025) at 400x200 squares, all 1000 steps."""
    w = W.config3(nx=400, ny=200)
    m, o = run_both(w, 1000)
    h, hu, hv, _ = assert_parity(m, o, w)
    z = m.get_tables()["cell_z"]
    wet = h > w.h_dry
    np.testing.assert_array_equal(~wet, w.h <= w.h_dry)
    assert np.abs(h[wet] + z[wet] - 2.0).max() < 1e-12
    assert np.abs(hu[wet] / h[wet]).max() < 1e-10 and np.abs(hv[wet] / h[wet]).max() < 1e-10


def test_config4_river_reduced_full_steps():
    """configs[3] shape (channel, noise terrain, varying Manning, inflow/outflow) at 640x160."""
    w = W.config4(nx=640, ny=160)
    m, o = run_both(w, 2000)
    assert_parity(m, o, w)
    st, so = m.get_stats(), o.stats()
    v0 = float(np.sum(w.h * m.get_tables()["area"]))
    # mass balance against the oracle's boundary-flux integral (R-20)
    assert st["volume"] - v0 == pytest.approx(-so["boundary_volume_out"], rel=1e-8)


def test_ordering_invariance_bitwise():
    """R-17: renumbering permutes cells only, so results agree bit for bit in caller numbering."""
    w = W.config4(nx=200, ny=50)
    out = []
    for ordering in (B.ORDER_IDENTITY, B.ORDER_HILBERT, B.ORDER_RCM):
        m = B.SweMesh.from_workload(w, ordering=ordering, loop_mode=B.LOOP_GRAPH).bind_device()
        m.set_state(w.h, w.hu, w.hv)
        m.run(300)
        out.append(m.get_state())
    for other in out[1:]:
        for a, b in zip(out[0][:3], other[:3]):
            np.testing.assert_array_equal(a, b)
        assert out[0][3] == other[3] and out[0][4] == other[4]


def test_determinism_and_loop_modes_bitwise():
    """Two runs, and the three loop modes, give identical bits (no atomics in the data path)."""
    w = W.config2(nx=300, ny=30)
    ref = None
    for loop_mode in (B.LOOP_GRAPH, B.LOOP_GRAPH, B.LOOP_PERSISTENT, B.LOOP_LAUNCH):
        m = B.SweMesh.from_workload(w, loop_mode=loop_mode).bind_device()
        m.set_state(w.h, w.hu, w.hv)
        m.run(137)
        m.run(64)
        m.step()
        got = m.get_state()
        if ref is None:
            ref = got
        else:
            for a, b in zip(ref[:3], got[:3]):
                np.testing.assert_array_equal(a, b)
            assert ref[3] == got[3] and ref[4] == got[4]


def test_cluster_loop_bitwise_equal_to_the_other_loop_modes():
    """Small meshes (<= 16 tiles): one thread-block cluster runs the whole swe_run with the state in
    shared memory, halo records through distributed shared memory and the cluster barrier per step.
    Same bits as the graph / persistent loops (different tile size included), AUTO picks it, and a
    run split into several calls (state written back and reloaded) changes nothing."""
    for w in (W.config1(), W.config4(nx=40, ny=10), W.canal_dam_break(37, 7, seed=9, length=37.0, manning=0.02, h_right=0.0)):
        ref = None
        for loop_mode, block in ((B.LOOP_GRAPH, 192), (B.LOOP_PERSISTENT, 128), (B.LOOP_CLUSTER, 0), (B.LOOP_AUTO, 0),
                                 (B.LOOP_CLUSTER, 192), (B.LOOP_CLUSTER, 256)):
            m = B.SweMesh.from_workload(w, loop_mode=loop_mode, block_size=block).bind_device()
            m.set_state(w.h, w.hu, w.hv)
            m.run(137); m.run(64); m.step()
            got = m.get_state()
            info = m.get_launch_info()
            if loop_mode in (B.LOOP_CLUSTER, B.LOOP_AUTO):
                assert info["loop_mode"] == "cluster" and info["block"] == (block or 128)
            if ref is None:
                ref = got
                vol = m.get_boundary_volumes()
            else:
                for a, b in zip(ref[:3], got[:3]):
                    np.testing.assert_array_equal(a, b)
                assert ref[3] == got[3] and ref[4] == got[4]
                np.testing.assert_array_equal(vol, m.get_boundary_volumes())
                assert m.get_stats()["steps"] == 202
    # run_until in cluster mode ends on t_end exactly, in as many steps as the oracle
    w = W.config1()
    m = B.SweMesh.from_workload(w, loop_mode=B.LOOP_CLUSTER).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    o = OracleSolver.from_workload(w)
    assert m.run_until(2.0) == o.run_until(2.0)
    assert m.get_state()[3] == 2.0
    # a mesh with more than 16 tiles falls back to the graph loop
    w = W.config2(nx=100, ny=20)
    m = B.SweMesh.from_workload(w, loop_mode=B.LOOP_CLUSTER).bind_device()
    assert m.get_launch_info()["loop_mode"] == "graph"


def test_edge_cases():
    # all dry: no time step, state unchanged, error code from compute_dt
    w = W.canal_dam_break(10, 3, h_left=0.0, h_right=0.0, length=10.0)
    m = B.SweMesh.from_workload(w).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    with pytest.raises(B.SweError) as e:
        m.compute_dt()
    assert e.value.code == B.ERR_ALL_DRY
    m.run(3)
    h, hu, hv, t, dt = m.get_state()
    assert (h == 0).all() and t == 0.0 and dt == 0.0
    # two cells (the smallest mesh), ragged tail of one partial warp
    w = W.two_triangles()
    m, o = run_both(w, 25)
    assert_parity(m, o, w)
    # a mesh size that is not a multiple of the block size, several blocks, tiny block size
    w = W.canal_dam_break(37, 7, seed=9, length=37.0, manning=0.02, h_right=0.0)
    m, o = run_both(w, 200, block_size=64)
    assert_parity(m, o, w)
    # state with momentum in dry cells is sanitised identically on both sides (R-15)
    w = W.canal_dam_break(20, 4, seed=4, length=20.0, h_right=5e-7)
    w.hu[:] = 0.01
    m, o = run_both(w, 30)
    assert_parity(m, o, w)
    # invalid state is rejected
    bad = w.h.copy(); bad[3] = -1.0
    with pytest.raises(B.SweError) as e:
        m.set_state(bad, w.hu, w.hv)
    assert e.value.code == -5


def test_device_state_roundtrip():
    import torch
    w = W.config1()
    m = B.SweMesh.from_workload(w).bind_device()
    with torch.cuda.stream(m.stream):
        d = [torch.from_numpy(x.copy()).cuda() for x in (w.h, w.hu, w.hv)]
        m.set_state_device(*d)
        m.run(10)
        out = [torch.empty(w.ncells, dtype=torch.float64, device="cuda") for _ in range(3)]
        m.get_state_device(*out)
    m.sync()
    h, hu, hv, _, _ = m.get_state()
    np.testing.assert_array_equal(out[0].cpu().numpy(), h)
    np.testing.assert_array_equal(out[1].cpu().numpy(), hu)
    np.testing.assert_array_equal(out[2].cpu().numpy(), hv)


def test_clockwise_input_and_permuted_tags_on_the_device():
    """Every other triangle given clockwise with its edge tags permuted accordingly (river case:
    inflow, outflow, walls, bed, friction): the device run matches the oracle on the same flipped
    input, and is bit-identical to the run on the counter-clockwise input."""
    w = W.config4(nx=240, ny=60)
    f = W.config4(nx=240, ny=60)
    flip = np.arange(w.ncells) % 2 == 0
    f.tris[flip] = f.tris[flip][:, [0, 2, 1]]
    f.bc_tags[flip] = f.bc_tags[flip][:, [2, 1, 0]]
    m, o = run_both(f, 400)
    got = assert_parity(m, o, f)
    r = B.SweMesh.from_workload(w).bind_device()
    r.set_state(w.h, w.hu, w.hv)
    r.run(400)
    for a, b in zip(got[:3], r.get_state()[:3]):
        np.testing.assert_array_equal(a, b)
    np.testing.assert_array_equal(m.get_boundary_volumes(), r.get_boundary_volumes())


def test_eq22_clamp_branch_strongly_diverging_flow():
    """R-6: two halves of a canal moving apart at |u| = 15 m/s with h = 1 m (u_R - u_L > 8 a, so
    the bracket of eq.(22) is negative and its unclamped square would exceed h_k): the edges along
    the parting line take the clamped branch on both sides; a dry bed opens between them."""
    w = W.canal_dam_break(120, 12, h_left=1.0, h_right=1.0, manning=0.02, length=120.0, seed=77)
    w.bc_tags[w.bc_tags > 0] = W.BC_TRANSMISSIVE
    cx = W.centroids(w.nodes_xy, w.tris)[:, 0]
    w.hu[:] = np.where(cx < 60.0, -15.0, 15.0) * w.h
    assert 30.0 > 8.0 * np.sqrt(9.81 * 1.0)
    from oracle.swe_oracle import hllc
    assert hllc(1.0, -15.0, 0.0, 1.0, 15.0, 0.0)[1]["hs"] == 0.0        # the branch in question
    m, o = run_both(w, 60)
    h, hu, hv, t = assert_parity(m, o, w)
    assert h.min() < 0.2 and (np.abs(hu) > 1.0).any()                   # the bed is emptying at the parting line


def test_dry_inflow_cells():
    """R-20, dry branch: the whole left edge is an inflow boundary, including the dry floodplain
    cells, which receive the mass flux q_n and no momentum flux while they are dry."""
    w = W.config4(nx=480, ny=120)
    cx = W.centroids(w.nodes_xy, w.tris)[:, 0]
    for k in range(3):
        xa = w.nodes_xy[w.tris[:, k], 0]
        xb = w.nodes_xy[w.tris[:, (k + 1) % 3], 0]
        w.bc_tags[(xa == 0.0) & (xb == 0.0), k] = W.BC_INFLOW0
    left = (w.bc_tags == W.BC_INFLOW0).any(axis=1)
    assert (w.h[left] <= w.h_dry).any() and (w.h[left] > w.h_dry).any()
    m, o = run_both(w, 500)
    h, hu, hv, t = assert_parity(m, o, w)
    assert (h[left] > w.h_dry).all()                                     # the dry inflow cells have filled
    vg, vo = m.get_boundary_volumes(), o.boundary_volumes()
    np.testing.assert_allclose(vg, vo, rtol=1e-10, atol=1e-10)
    assert vg[W.BC_INFLOW0] == pytest.approx(-500.0 * t, rel=1e-12)


@pytest.mark.parametrize("ordering", [B.ORDER_IDENTITY, B.ORDER_HILBERT])
def test_config5_sweep_2M_both_orderings(ordering):
    """BASELINE configs[4], the 2M-cell sweep mesh (1,997,120 cells), all 200 steps, with the
    caller's random numbering kept and with the Hilbert renumbering: every cell against the oracle."""
    w = W.config5("2M")
    m, o = run_both(w, w.nsteps, ordering=ordering)
    assert_parity(m, o, w)


# ---- NEXT-2: the edge-centric two-pass kernels (PAPER.md:393, :617 leave the kernel split open) ----
@pytest.mark.parametrize("loop_mode", [B.LOOP_GRAPH, B.LOOP_LAUNCH])
def test_edge_two_pass_kernel_matches_oracle_and_tiled_kernel(loop_mode):
    """Pass 1 (one thread per edge of the mesh) + pass 2 (one thread per cell): the same scheme as
    the fused tile kernel, against the oracle at the same bar, river case with inflow / outflow /
    wet-dry fronts / friction; and against the tile kernel itself (same edge and cell arithmetic,
    same order k = 0,1,2, every fused multiply-add written out and --fmad=false: identical bits)."""
    w = W.config4(nx=320, ny=80)
    m, o = run_both(w, 600, kernel=B.KERNEL_EDGE_TWO_PASS, loop_mode=loop_mode)
    got = assert_parity(m, o, w)
    np.testing.assert_allclose(m.get_boundary_volumes(), o.boundary_volumes(), rtol=1e-10, atol=1e-10)
    r = B.SweMesh.from_workload(w).bind_device()
    r.set_state(w.h, w.hu, w.hv)
    r.run(600)
    ref = r.get_state()
    for a, b in zip(got[:3], ref[:3]):
        np.testing.assert_array_equal(a, b)
    assert got[3] == ref[3]


def test_quiet_tiles_bitwise_against_the_kernels_without_shortcuts():
    """A mesh large enough for the quiet-tile path (blocks with >= 8 tiles, most of them on the dry
    floodplain): the tile kernel copies all-dry tiles and leaves quiet tiles untouched (both state
    buffers hold their records already), the edge-centric kernels compute every edge and every
    cell of every step.  Identical bits, while the wet front keeps moving into quiet territory; and parity with
    the oracle at the usual bar."""
    w = W.config4(nx=1600, ny=400)
    m, o = run_both(w, 300, block_size=64)
    got = assert_parity(m, o, w)
    st, ti = m.get_stats(), m.get_tile_info()
    assert st["quiet_tile_steps"] > 0.5 * 300 * ti["ntiles"]                  # most tile-steps took the quiet path
    assert 0 < st["active_tile_steps"] < 0.3 * 300 * ti["ntiles"]
    assert st["quiet_tile_steps"] + st["active_tile_steps"] < 300 * ti["ntiles"]   # the rest were voted all dry
    e = B.SweMesh.from_workload(w, kernel=B.KERNEL_EDGE_TWO_PASS).bind_device()
    e.set_state(w.h, w.hu, w.hv)
    e.run(300)
    ref = e.get_state()
    for a, b in zip(got[:3], ref[:3]):
        np.testing.assert_array_equal(a, b)
    assert got[3] == ref[3]
    np.testing.assert_array_equal(m.get_boundary_volumes(), e.get_boundary_volumes())
    # the persistent loop takes the same path and gives the same bits
    p = B.SweMesh.from_workload(w, block_size=64, loop_mode=B.LOOP_PERSISTENT).bind_device()
    p.set_state(w.h, w.hu, w.hv)
    p.run(300)
    for a, b in zip(got[:3], p.get_state()[:3]):
        np.testing.assert_array_equal(a, b)
    assert p.get_stats()["quiet_tile_steps"] == st["quiet_tile_steps"]


def test_untouched_quiet_tiles_and_work_stealing_across_run_calls_and_a_new_state():
    """Quiet tiles are not written, which is right only while both state buffers hold their records;
    blocks take tiles from each other's lists, which must not change a bit.  Uneven swe_run calls
    (the buffer parity flips between calls), read-backs in between, then a NEW state whose wet region
    lies where the old one was quiet (swe_set_state must forget what the tiles were), against the
    edge-centric kernels, which have neither shortcut, with the same sequence of calls."""
    w = W.config4(nx=1600, ny=400)
    t = B.SweMesh.from_workload(w, block_size=64).bind_device()
    e = B.SweMesh.from_workload(w, kernel=B.KERNEL_EDGE_TWO_PASS).bind_device()

    def both(fn):
        return fn(t), fn(e)

    def same_state():
        a, b = both(lambda m: m.get_state())
        for x, y in zip(a[:3], b[:3]):
            np.testing.assert_array_equal(x, y)
        assert a[3] == b[3] and a[4] == b[4]
        return a

    both(lambda m: m.set_state(w.h, w.hu, w.hv))
    for chunk in (1, 2, 3, 7, 30, 1, 101):
        both(lambda m: m.run(chunk))
        same_state()
    st, ti = t.get_stats(), t.get_tile_info()
    assert st["steps"] == 145
    assert st["quiet_tile_steps"] > 0.5 * 145 * ti["ntiles"]
    assert st["stolen_tile_steps"] > 0                      # the wet channel is a small part of the mesh: idle blocks took tiles
    assert e.get_stats()["stolen_tile_steps"] == 0
    # a new state: the old one mirrored in y (the channel meanders, so water now stands on cells that were quiet)
    h, hu, hv = same_state()[:3]
    cy = W.centroids(w.nodes_xy, w.tris)[:, 1]
    order = np.argsort(cy, kind="stable")
    h2, hu2, hv2 = h.copy(), np.zeros_like(hu), np.zeros_like(hv)
    h2[order] = h[order[::-1]]
    assert np.count_nonzero((h2 > w.h_dry) & (h <= w.h_dry)) > 1000
    both(lambda m: m.set_state(h2, hu2, hv2))
    for chunk in (5, 64):
        both(lambda m: m.run(chunk))
        same_state()
    assert t.get_stats()["n_clamped"] == e.get_stats()["n_clamped"]
    np.testing.assert_array_equal(t.get_boundary_volumes(), e.get_boundary_volumes())


def test_full_size_river_graph_and_persistent_loops_bitwise_whatever_is_stolen():
    """BASELINE configs[3] at full size (13 M cells, bench.py's launch configuration): the CUDA-graph loop and the
    cooperative persistent loop give the same bits and skip the same quiet tiles, although which block computes
    which tile depends on timing (the stolen-tile counts of two runs differ)."""
    w = W.config4()
    res = []
    for loop_mode in (B.LOOP_GRAPH, B.LOOP_PERSISTENT):
        m = B.SweMesh.from_workload(w, loop_mode=loop_mode).bind_device()
        m.set_state(w.h, w.hu, w.hv)
        for chunk in (1, 7, 192):
            m.run(chunk)
        res.append((m.get_state(), m.get_stats()))
        m.destroy()
    (a, sa), (b, sb) = res
    for x, y in zip(a[:3], b[:3]):
        np.testing.assert_array_equal(x, y)
    assert a[3] == b[3] and a[4] == b[4]
    assert sa["steps"] == sb["steps"] == 200
    assert sa["quiet_tile_steps"] == sb["quiet_tile_steps"] > 0
    assert sa["active_tile_steps"] == sb["active_tile_steps"] > 0
    assert sa["stolen_tile_steps"] > 0 and sb["stolen_tile_steps"] > 0


def test_edge_two_pass_kernel_ordering_invariance_and_run_until():
    w = W.config2(nx=300, ny=30)
    out = []
    for ordering in (B.ORDER_IDENTITY, B.ORDER_HILBERT):
        m = B.SweMesh.from_workload(w, ordering=ordering, kernel=B.KERNEL_EDGE_TWO_PASS).bind_device()
        m.set_state(w.h, w.hu, w.hv)
        n = m.run_until(1.5)
        out.append(m.get_state() + (n,))
    for a, b in zip(out[0][:3], out[1][:3]):
        np.testing.assert_array_equal(a, b)
    assert out[0][3] == out[1][3] == 1.5 and out[0][5] == out[1][5]
    o = OracleSolver.from_workload(w)
    assert o.run_until(1.5) == out[0][5]
    for a, b in zip(out[0][:3], o.get_state()[:3]):
        np.testing.assert_allclose(a, b, rtol=RTOL, atol=ATOL)


def test_mixed32_state_storage_against_the_oracle():
    """SWE_FP_MIXED32 (the paper's floating-point kind is configurable): FP32 state
    records in HBM, FP64 arithmetic, on the edge-centric two-pass kernels.  Bar:
    both sides round the same quantities to float after every step, so they differ only where a
    rounding falls the other way (2^-24 of the value each time, and through the fluxes 2^-24 of
    the neighbours' values): 2e-5 of the field's scale, absolute + relative, after 600 steps;
    against the all-double oracle the same bar holds with the accumulated float round-off."""
    w = W.config4(nx=320, ny=80)
    m = B.SweMesh.from_workload(w, kernel=B.KERNEL_EDGE_TWO_PASS, fp_kind=B.FP_MIXED32).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    o = OracleSolver.from_workload(w, storage32=True)
    o64 = OracleSolver.from_workload(w)
    m.run(600)
    assert o.run(600) == 600 and o64.run(600) == 600
    hg, hug, hvg, tg, dtg = m.get_state()
    for ref, tol in ((o, 2e-5), (o64, 2e-5)):
        ho, huo, hvo, to, dto = ref.get_state()
        for a, b in ((hg, ho), (hug, huo), (hvg, hvo)):
            np.testing.assert_allclose(a, b, rtol=tol, atol=tol * max(1.0, float(np.abs(b).max())))
        assert tg == pytest.approx(to, rel=1e-6) and dtg == pytest.approx(dto, rel=1e-5)
        differ = (hg <= w.h_dry) != (ho <= w.h_dry)
        assert (np.abs(ho[differ] - w.h_dry) < tol).all()       # the mask may differ only at the threshold
    np.testing.assert_array_equal(hg, hg.astype(np.float32).astype(np.float64))     # the state IS single precision
    st = m.get_stats()
    assert st["n_clamped"] == 0 and st["n_nonfinite"] == 0 and st["steps"] == 600
    # the tile kernel has no such variant: the combination is refused at create time
    with pytest.raises(B.SweError) as e:
        B.SweMesh.from_workload(w, fp_kind=B.FP_MIXED32)
    assert e.value.code == -1


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times (defaults) ----------
def test_config3_full_size_every_cell_then_invariants():
    """configs[2] at 2000x1000 squares (4,000,000 cells): every cell against the oracle after 40
    steps, then the remaining steps of the 1000 on the GPU alone, checked by what holds at any
    size: state at rest to round-off, dry mask unchanged, mass to round-off, dt constant."""
    w = W.config3()
    m, o = run_both(w, 40)
    assert_parity(m, o, w)
    info = m.get_launch_info()
    assert info["loop_mode"] == "graph" and info["block"] == 192
    dt40 = m.get_state()[4]
    m.run(w.nsteps - 40)
    h, hu, hv, t, dt = m.get_state()
    st = m.get_stats()
    assert st["steps"] == w.nsteps and st["n_clamped"] == 0 and st["n_nonfinite"] == 0
    tab = m.get_tables()
    wet = h > w.h_dry
    np.testing.assert_array_equal(~wet, w.h <= w.h_dry)
    assert np.abs(h[wet] + tab["cell_z"][wet] - 2.0).max() < 1e-12
    assert np.abs(hu[wet] / h[wet]).max() < 1e-10 and np.abs(hv[wet] / h[wet]).max() < 1e-10
    assert st["volume"] == pytest.approx(float(np.sum(w.h * tab["area"])), rel=1e-12)
    assert dt == pytest.approx(dt40, rel=1e-12)


def test_config4_full_size_every_cell_then_mass_balance():
    """configs[3] at 5100x1275 squares (13,005,000 cells): every cell against the oracle after 25
    steps; then 2000 steps in all on the GPU: no clamp, nothing non-finite, and the volume gained
    is the prescribed inflow (exactly, while the outlet is dry) minus what left through the outlet."""
    w = W.config4()
    m, o = run_both(w, 25)
    assert_parity(m, o, w)
    assert m.get_launch_info()["loop_mode"] == "graph"
    v0 = float(np.sum(w.h * m.get_tables()["area"]))
    m.run(w.nsteps - 25)
    st = m.get_stats()
    assert st["steps"] == w.nsteps and st["n_clamped"] == 0 and st["n_nonfinite"] == 0
    h, hu, hv, t, dt = m.get_state()
    assert h.min() >= 0.0 and dt > 0.0
    cx = W.centroids(w.nodes_xy, w.tris)[:, 0]
    outlet_wet = (cx > 0.999 * w.nodes_xy[:, 0].max()) & (h > w.h_dry) & (hu > 0)
    gained = st["volume"] - v0
    if not outlet_wet.any():
        assert gained == pytest.approx(500.0 * t, rel=1e-9)     # R-20: all of Q enters, nothing leaves
    else:                       # the outlet only removes water: the gain cannot exceed the inflow
        assert gained <= 500.0 * t * (1 + 1e-9)


def test_random_caller_numbering_without_locality_pass():
    """config 5's 'random permutation' arm: ORDER_IDENTITY keeps the caller's random numbering,
    so every neighbour lives in another tile (3 edge evaluations per cell, halo = 3 x tile)."""
    w = W.config5("0.1M", nsteps=200)
    m, o = run_both(w, 200, ordering=B.ORDER_IDENTITY)
    assert_parity(m, o, w)
    ti = m.get_tile_info()
    assert ti["edges_per_cell"] > 2.9
    m2 = B.SweMesh.from_workload(w, ordering=B.ORDER_HILBERT).bind_device()
    m2.set_state(w.h, w.hu, w.hv)
    m2.run(200)
    for a, b in zip(m.get_state()[:3], m2.get_state()[:3]):
        np.testing.assert_array_equal(a, b)                        # R-17, bitwise


# ---- boundary discharge diagnostics and run-until-time -------------
@pytest.mark.parametrize("loop_mode", [B.LOOP_GRAPH, B.LOOP_PERSISTENT])
def test_boundary_volumes_and_run_until_match_oracle(loop_mode):
    w = W.config4(nx=320, ny=80)
    m = B.SweMesh.from_workload(w, loop_mode=loop_mode).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    o = OracleSolver.from_workload(w)
    t_end = 12.5
    n_gpu, n_cpu = m.run_until(t_end), o.run_until(t_end)
    assert n_gpu == n_cpu
    hg, hug, hvg, tg = assert_parity(m, o, w)
    assert tg == t_end
    vg, vo = m.get_boundary_volumes(), o.boundary_volumes()
    np.testing.assert_allclose(vg, vo, rtol=1e-10, atol=1e-10)
    assert vg[W.BC_INFLOW0] == pytest.approx(-500.0 * t_end, rel=1e-12) and vg[W.BC_WALL] == 0.0
    v0 = float(np.sum(w.h * m.get_tables()["area"]))
    assert m.get_stats()["volume"] - v0 == pytest.approx(-vg.sum(), rel=1e-9)
    # continuing with plain steps after run_until works (t_end is disarmed) and max_steps binds
    assert m.run_until(1e30, max_steps=7) == 7 and o.run_until(1e30, max_steps=7) == 7
    assert_parity(m, o, w)


def test_config4_full_size_exact_mass_balance():
    """13,005,000 cells, bench.py's launch configuration: after 300 steps the volume in the domain
    has changed by exactly what crossed the boundary (inflow tag: -Q t)."""
    w = W.config4()
    m = B.SweMesh.from_workload(w).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    v0 = float(np.sum(w.h * m.get_tables()["area"]))
    m.run(300)
    st, vol = m.get_stats(), m.get_boundary_volumes()
    assert vol[W.BC_INFLOW0] == pytest.approx(-500.0 * st["t"], rel=1e-12)
    assert st["volume"] - v0 == pytest.approx(-vol.sum(), rel=1e-9)


@pytest.mark.parametrize("block_size", [64, 128, 256])
def test_other_tile_sizes(block_size):
    """Every supported tile size (threads per block) gives the default's bits: the tile decomposition
    only changes who evaluates an edge, never how (R-17, R-23)."""
    w = W.config4(nx=200, ny=50)
    ref = B.SweMesh.from_workload(w).bind_device()
    ref.set_state(w.h, w.hu, w.hv)
    ref.run(150)
    m = B.SweMesh.from_workload(w, block_size=block_size).bind_device()
    assert m.get_launch_info()["block"] == block_size
    m.set_state(w.h, w.hu, w.hv)
    m.run(150)
    for a, b in zip(ref.get_state()[:3], m.get_state()[:3]):
        np.testing.assert_array_equal(a, b)


def test_zero_threshold_and_zero_steps():
    """h_dry = 0 (the library floors it at 1e-250 so that every rsqrt argument stays normal) and
    swe_run(0) / a reached t_end leave the state bitwise unchanged."""
    w = W.canal_dam_break(60, 6, h_right=0.0, manning=0.03, length=60.0, seed=21)
    w.h_dry = 0.0
    m, o = run_both(w, 120)
    hg, hug, hvg, tg, _ = m.get_state()
    ho, huo, hvo, to, _ = o.get_state()
    np.testing.assert_allclose(hg, ho, rtol=RTOL, atol=ATOL)
    np.testing.assert_allclose(hug, huo, rtol=RTOL, atol=ATOL)
    np.testing.assert_allclose(hvg, hvo, rtol=RTOL, atol=ATOL)
    assert tg == pytest.approx(to, rel=1e-12) and np.isfinite(hg).all()
    before = m.get_state()
    m.run(0)
    assert m.run_until(before[3]) == 0          # t_end already reached: no step
    after = m.get_state()
    for a, b in zip(before[:3], after[:3]):
        np.testing.assert_array_equal(a, b)
    assert before[3] == after[3]


def test_asynchronous_snapshot_on_a_side_stream():
    """swe_snapshot_begin: the snapshot holds the state at the moment of the call although more
    steps are queued right behind it, and it does not disturb them."""
    import torch
    w = W.config2(nx=600, ny=60)
    ref = B.SweMesh.from_workload(w).bind_device()
    ref.set_state(w.h, w.hu, w.hv)
    ref.run(150)
    mid = ref.get_state()
    ref.run(250)
    end = ref.get_state()
    m = B.SweMesh.from_workload(w).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    bufs = [torch.empty(w.ncells, dtype=torch.float64).pin_memory().numpy() for _ in range(3)]
    m.run(150)
    m.snapshot_begin(*bufs)
    m.run(250)                              # queued while the snapshot is being copied
    t_snap = m.snapshot_wait()
    for a, b in zip(bufs, mid[:3]):
        np.testing.assert_array_equal(a, b)
    assert t_snap == mid[3]
    for a, b in zip(m.get_state()[:4], end[:4]):
        np.testing.assert_array_equal(a, b)


def test_plain_hll_solver_matches_oracle():
    """swe_params.riemann = SWE_RIEMANN_HLL against the oracle's HLL."""
    w = W.config4(nx=320, ny=80)
    m = B.SweMesh.from_workload(w, riemann=B.RIEMANN_HLL).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    o = OracleSolver.from_workload(w)
    o.set_riemann(True)
    m.run(600)
    assert o.run(600) == 600
    hg = assert_parity(m, o, w)[0]
    # and it is a different scheme: the HLLC run differs where there is shear
    c = B.SweMesh.from_workload(w).bind_device()
    c.set_state(w.h, w.hu, w.hv)
    c.run(600)
    assert np.abs(c.get_state()[0] - hg).max() > 1e-6


def test_two_handles_with_different_shared_memory_needs_interleave():
    """Handles whose tile tables need different amounts of shared memory (random numbering: 3 x the
    edges and halo) keep working when their runs alternate."""
    w = W.config5("0.1M", nsteps=60)
    a = B.SweMesh.from_workload(w, ordering=B.ORDER_IDENTITY, loop_mode=B.LOOP_GRAPH).bind_device()
    b = B.SweMesh.from_workload(w, ordering=B.ORDER_HILBERT, loop_mode=B.LOOP_GRAPH).bind_device()
    assert a.get_tile_info()["smem_bytes"] > 1.5 * b.get_tile_info()["smem_bytes"]
    for m in (a, b):
        m.set_state(w.h, w.hu, w.hv)
    for _ in range(3):
        a.run(10)
        b.run(10)
        b.run(10)
        a.run(10)
    for x, y in zip(a.get_state()[:4], b.get_state()[:4]):
        np.testing.assert_array_equal(x, y)


def test_non_default_parameters_two_inflow_groups_rcm():
    """g, CFL and h_dry away from their defaults, two prescribed-discharge groups (one of them an
    extraction, Q < 0), RCM ordering, persistent loop: every table and constant that carries a
    parameter is exercised against the oracle."""
    w = W.config4(nx=240, ny=60)
    w.g, w.cfl, w.h_dry = 3.71, 0.45, 2e-4            # Mars gravity, cautious CFL, coarse threshold
    # second group: the wet cells of the right edge pump water out instead of draining freely
    tags = w.bc_tags.copy()
    tags[tags == W.BC_TRANSMISSIVE] = W.BC_INFLOW0 + 1
    w.bc_tags = tags
    w.bc_values = {W.BC_INFLOW0: 350.0, W.BC_INFLOW0 + 1: -40.0}
    m, o = run_both(w, 800, ordering=B.ORDER_RCM, loop_mode=B.LOOP_PERSISTENT)
    assert_parity(m, o, w)
    vg, vo = m.get_boundary_volumes(), o.boundary_volumes()
    np.testing.assert_allclose(vg, vo, rtol=1e-10, atol=1e-10)
    t = m.get_state()[3]
    assert vg[W.BC_INFLOW0] == pytest.approx(-350.0 * t, rel=1e-12)
    assert vg[W.BC_INFLOW0 + 1] == pytest.approx(40.0 * t, rel=1e-12)


def test_locally_refined_mesh():
    """SURVEY.md section 8(f) NEXT-3 (second half): a mesh whose inradius varies 32:1 (the paper refines
    around bridge piers).  The time step is set by the few smallest cells, tiles
    cover very different areas, and the Hilbert order still keeps 90 % of the edges inside tiles."""
    w = W.refined_basin()
    m, o = run_both(w, w.nsteps)
    assert_parity(m, o, w)
    geo = o.geometry()
    assert geo["rin"].max() / geo["rin"].min() > 25.0
    assert m.get_tile_info()["edges_per_cell"] < 1.75
    # dt is a min over cells of very different size: it must equal the oracle's to 1e-12 at every
    # stage of the run, not only at the end
    m2 = B.SweMesh.from_workload(w).bind_device()
    m2.set_state(w.h, w.hu, w.hv)
    o2 = OracleSolver.from_workload(w)
    for _ in range(6):
        assert m2.compute_dt() == pytest.approx(o2.compute_dt(), rel=1e-12)
        m2.run(37)
        o2.run(37)


def test_gauges_sample_cells_against_get_state_and_oracle():
    """swe_sample_cells: a gauge record (h, hu, hv at fixed cells) taken at three stages of the wet-dry dam break
    equals swe_get_state at those cells bit for bit and the oracle's state at the usual bar; ids are checked."""
    w = W.config2(nx=300, ny=30)
    m = B.SweMesh.from_workload(w).bind_device()
    o = OracleSolver.from_workload(w)
    m.set_state(w.h, w.hu, w.hv)
    rng = np.random.default_rng(5)
    cells = np.concatenate([[0, w.ncells - 1], rng.choice(w.ncells, 200, replace=False)]).astype(np.int32)
    for stage in range(3):
        m.run(120)
        assert o.run(120) == 120
        gh, ghu, ghv, gt = m.sample_cells(cells)
        h, hu, hv, t, _ = m.get_state()
        np.testing.assert_array_equal(gh, h[cells])
        np.testing.assert_array_equal(ghu, hu[cells])
        np.testing.assert_array_equal(ghv, hv[cells])
        assert gt == t
        ho, huo, hvo, to, _ = o.get_state()
        np.testing.assert_allclose(gh, ho[cells], rtol=RTOL, atol=ATOL)
        np.testing.assert_allclose(ghu, huo[cells], rtol=RTOL, atol=ATOL)
        np.testing.assert_allclose(ghv, hvo[cells], rtol=RTOL, atol=ATOL)
        assert gt == pytest.approx(to, rel=1e-12)
    assert np.count_nonzero(gh > w.h_dry) > 20 and np.count_nonzero(gh <= w.h_dry) > 20     # gauges on both sides of the front
    for bad in ([-1], [w.ncells], []):
        with pytest.raises(B.SweError):
            m.sample_cells(bad)
    with pytest.raises(B.SweError):
        m.sample_cells(np.arange(w.ncells // 2 + 1))
    # single-precision storage on the edge-centric kernels: the same read path
    e = B.SweMesh.from_workload(w, kernel=B.KERNEL_EDGE_TWO_PASS, fp_kind=B.FP_MIXED32).bind_device()
    e.set_state(w.h, w.hu, w.hv)
    e.run(50)
    gh, ghu, ghv, _ = e.sample_cells(cells)
    h, hu, hv = e.get_state()[:3]
    np.testing.assert_array_equal(gh, h[cells])
    np.testing.assert_array_equal(ghu, hu[cells])
    np.testing.assert_array_equal(ghv, hv[cells])


def test_active_tile_counter():
    """swe_stats.active_tile_steps: every tile of an all-wet mesh is active at every step; on the
    wet-dry dam break the dry end of the canal is not, and the count grows as the front advances."""
    w = W.config1()
    m = B.SweMesh.from_workload(w).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    m.run(50)
    assert m.get_stats()["active_tile_steps"] == 50 * m.get_tile_info()["ntiles"]
    w = W.config2(nx=600, ny=60)
    m = B.SweMesh.from_workload(w, loop_mode=B.LOOP_PERSISTENT).bind_device()
    m.set_state(w.h, w.hu, w.hv)
    nt = m.get_tile_info()["ntiles"]
    m.run(100)
    a1 = m.get_stats()["active_tile_steps"]
    m.run(100)
    a2 = m.get_stats()["active_tile_steps"] - a1
    assert 0.4 * 100 * nt < a1 < a2 < 100 * nt
