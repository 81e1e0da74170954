"""CPU-only checks of the C-ABI library: it loads, exports every declared symbol, and its host
mesh builder (no CUDA involved) agrees with the oracle's independent geometry."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle.swe_oracle import OracleSolver
from paper_2010_14416_b200 import binding as B
from paper_2010_14416_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    L = B.load_library()
    header = open(os.path.join(ROOT, "include", "swe.h")).read()
    declared = set(re.findall(r"\b(swe_[a-z_]+)\s*\(", header))
    declared -= {"swe_last_error"} - set(B.SYMBOLS)
    assert declared == set(B.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name


def test_struct_sizes_match_header():
    assert ctypes.sizeof(B.SweParams) == 3 * 8 + 6 * 4
    assert ctypes.sizeof(B.SweStats) == 3 * 8 + 8 * 8
    p = B.SweParams()
    B.load_library().swe_params_default(ctypes.byref(p))
    assert (p.g, p.cfl, p.h_dry, p.ordering, p.loop_mode) == (9.81, 0.9, 1e-6, B.ORDER_HILBERT, B.LOOP_AUTO)


@pytest.mark.parametrize("ordering", [B.ORDER_IDENTITY, B.ORDER_HILBERT, B.ORDER_RCM])
def test_tables_match_oracle_geometry(ordering):
    w = W.config4(nx=60, ny=15)
    m = B.SweMesh.from_workload(w, ordering=ordering)
    t = m.get_tables()
    geo = OracleSolver.from_workload(w).geometry()
    nbr_o = geo["nbr"].copy()
    bnd = nbr_o < 0
    assert ((t["nbr"] < 0) == bnd).all()
    np.testing.assert_array_equal(t["nbr"][~bnd], nbr_o[~bnd])
    # boundary edges carry -tag
    np.testing.assert_array_equal(-t["nbr"][bnd], np.maximum(w.bc_tags[bnd], 1))
    np.testing.assert_allclose(t["normal"][:, :, 0], geo["n1"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(t["normal"][:, :, 1], geo["n2"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(t["length"], geo["len"], rtol=1e-15)
    np.testing.assert_allclose(t["area"], geo["area"], rtol=1e-15)
    np.testing.assert_allclose(t["inradius"], geo["rin"], rtol=1e-15)
    np.testing.assert_allclose(t["cell_z"], geo["z"], rtol=1e-15, atol=1e-15)
    perm = m.get_permutation()
    assert sorted(perm.tolist()) == list(range(w.ncells))
    if ordering == B.ORDER_IDENTITY:
        assert (perm == np.arange(w.ncells)).all()


def _mean_neighbour_distance(w, perm):
    inv = np.empty_like(perm)
    inv[perm] = np.arange(perm.size, dtype=perm.dtype)
    nbr = OracleSolver.from_workload(w).geometry()["nbr"]
    i = np.repeat(np.arange(w.ncells), 3)
    j = nbr.ravel()
    ok = j >= 0
    return np.abs(inv[i[ok]].astype(np.int64) - inv[j[ok]].astype(np.int64)).mean()


def test_locality_orderings_shrink_neighbour_distance():
    """a13: the Hilbert / RCM numbering keeps a cell's neighbours close in memory."""
    w = W.config2(nx=200, ny=20)
    d_id = _mean_neighbour_distance(w, np.arange(w.ncells, dtype=np.int32))
    d_h = _mean_neighbour_distance(w, B.SweMesh.from_workload(w, ordering=B.ORDER_HILBERT).get_permutation())
    d_r = _mean_neighbour_distance(w, B.SweMesh.from_workload(w, ordering=B.ORDER_RCM).get_permutation())
    assert d_id > 1000          # the generator's random permutation scatters neighbours
    assert d_h < 40 and d_r < 80


def test_clockwise_triangles_and_tag_permutation():
    w = W.config4(nx=40, ny=10)
    tris, tags = w.tris.copy(), w.bc_tags.copy()
    flip = np.arange(w.ncells) % 2 == 0
    tris[flip] = tris[flip][:, [0, 2, 1]]
    tags[flip] = tags[flip][:, [2, 1, 0]]
    a = B.SweMesh(w.nodes_xy, w.tris, w.bathymetry, w.manning, w.bc_tags).get_tables()
    b = B.SweMesh(w.nodes_xy, tris, w.bathymetry, w.manning, tags).get_tables()
    # an unflipped cell is unchanged; a flipped cell (v0,v2,v1) is re-oriented to (v0,v1,v2)
    # (nbr holds -tag on boundary edges, so the permuted tags must have landed on the right edges)
    for key in ("nbr", "length", "area", "inradius", "normal", "cell_z"):
        np.testing.assert_array_equal(a[key], b[key])
    assert (a["nbr"] < 0).any() and (a["nbr"] == -W.BC_INFLOW0).any() and (a["nbr"] == -W.BC_TRANSMISSIVE).any()
    # and against the oracle's own orientation fix on the flipped input
    from oracle.swe_oracle import OracleSolver
    geo = OracleSolver(w.nodes_xy, tris, w.bathymetry, w.manning, tags).geometry()
    np.testing.assert_allclose(b["normal"][:, :, 0], geo["n1"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(b["normal"][:, :, 1], geo["n2"], rtol=0, atol=1e-15)
    np.testing.assert_array_equal(np.where(b["nbr"] >= 0, b["nbr"], -1), geo["nbr"])


def test_invalid_input_codes():
    w = W.two_triangles()
    bad = w.tris.copy(); bad[0, 0] = 9
    with pytest.raises(B.SweError) as e:
        B.SweMesh(w.nodes_xy, bad, w.bathymetry, w.manning, w.bc_tags)
    assert e.value.code == -2
    deg = w.tris.copy(); deg[0] = [0, 1, 1]
    with pytest.raises(B.SweError) as e:
        B.SweMesh(w.nodes_xy, deg, w.bathymetry, w.manning, w.bc_tags)
    assert e.value.code == -3
    tri3 = np.vstack([w.tris, [[0, 2, 1]]]).astype(np.int32)
    with pytest.raises(B.SweError) as e:
        B.SweMesh(w.nodes_xy, tri3, w.bathymetry, np.zeros(3), np.ones((3, 3), dtype=np.int8))
    assert e.value.code == -4
    with pytest.raises(B.SweError) as e:
        B.SweMesh(w.nodes_xy, w.tris, w.bathymetry, np.array([0.0, -1.0]), w.bc_tags)
    assert e.value.code == -5
    xy = w.nodes_xy.copy(); xy[1, 0] = np.nan
    with pytest.raises(B.SweError) as e:
        B.SweMesh(xy, w.tris, w.bathymetry, w.manning, w.bc_tags)
    assert e.value.code == -5
    with pytest.raises(B.SweError) as e:
        B.SweMesh(w.nodes_xy, w.tris, w.bathymetry, w.manning, w.bc_tags, block_size=100)
    assert e.value.code == -1


def test_compute_entry_points_fail_loudly_without_a_device():
    """No CPU fallback: unbound handles refuse to compute."""
    w = W.two_triangles()
    m = B.SweMesh.from_workload(w)
    assert m.workspace_bytes() > 0
    for call in (lambda: m.set_state(w.h, w.hu, w.hv), m.compute_dt, m.step, lambda: m.run(3),
                 m.get_state, m.get_stats, m.sync):
        with pytest.raises(B.SweError) as e:
            call()
        assert e.value.code == -6
    with pytest.raises(B.SweError) as e:
        m.set_bc_value(3, 1.0)       # no edge carries tag 3 on this mesh
    assert e.value.code == -11


@pytest.mark.parametrize("ordering", [B.ORDER_IDENTITY, B.ORDER_HILBERT, B.ORDER_RCM])
@pytest.mark.parametrize("block", [64, 192, 256])
def test_tile_tables_cover_every_cell_edge_exactly_once(ordering, block):
    """Tile tables of the step kernel, checked against the ORACLE's neighbour/geometry tables:
    every (cell, local edge) is the a- or b-side of exactly one edge record of its tile, that
    record's other end is the oracle's neighbour (through the halo list if it lives in another
    tile), a is the smaller caller id, the normal is a's outward normal and the tag matches."""
    w = W.config4(nx=50, ny=13)              # ragged last tile, inflow / outflow / wall tags
    m = B.SweMesh.from_workload(w, ordering=ordering, block_size=block)
    X = m.get_tile_tables()
    geo = OracleSolver.from_workload(w).geometry()
    perm = m.get_permutation()
    nt, TC = w.ncells, X["tile_cells"]
    assert TC == block and X["ntiles"] == (nt + TC - 1) // TC
    seen = np.zeros((nt, 3), dtype=np.int32)
    bnum = []
    mask = (1 << 29) - 1
    assert X["tinfo"][:, 0].tolist() == np.concatenate([[0], np.cumsum(X["tinfo"][:, 1])[:-1]]).tolist()
    assert X["tinfo"][:, 1].sum() == X["nedges"] and (X["tinfo"][:, 1].max() + 1) // 2 * 2 == X["max_edges"]   # lists are padded to even length
    for t in range(X["ntiles"]):
        e0, ne, nh = X["tinfo"][t, :3]
        halo = X["tinfo"][t, 4:4 + nh]
        assert nh <= X["max_halo"] and len(set(halo.tolist())) == nh
        assert ((halo < t * TC) | (halo >= (t + 1) * TC)).all()      # halo cells live in other tiles
        assert (X["tinfo"][t, 4 + nh:] == -1).all()

        def internal(pos):
            return t * TC + pos if pos < TC else halo[pos - TC]

        for e in range(e0, e0 + ne):
            a, b = int(X["edge_a"][e]), int(X["edge_b"][e])
            pa, ka = internal(a & mask), a >> 29
            ca = perm[pa]
            n1, n2, L = X["edge_geom"][e]
            assert abs(n1 - geo["n1"][ca, ka]) <= 1e-15 and abs(n2 - geo["n2"][ca, ka]) <= 1e-15
            assert L == pytest.approx(geo["len"][ca, ka], rel=1e-15)
            if (a & mask) < TC:
                seen[ca, ka] += 1
            if b < 0:                                                  # boundary edge
                assert geo["nbr"][ca, ka] < 0 and (-b) & 127 == max(int(w.bc_tags[ca, ka]), 1)
                assert (a & mask) < TC
                bnum.append((-b) >> 7)
                continue
            pb, kb = internal(b & mask), b >> 29
            cb = perm[pb]
            assert geo["nbr"][ca, ka] == cb and geo["nbr"][cb, kb] == ca and ca < cb
            assert (a & mask) < TC or (b & mask) < TC                  # the edge touches this tile
            if (b & mask) < TC:
                seen[cb, kb] += 1
    assert (seen == 1).all()
    assert sorted(bnum) == list(range(int((geo["nbr"] < 0).sum())))   # boundary edges numbered once each
    # locality: a space-filling-curve order keeps most edges inside one tile
    if ordering == B.ORDER_HILBERT and block >= 192:
        assert X["edges_per_cell"] < 1.85
    assert 1.5 <= X["edges_per_cell"] <= 3.0


# ------------------------------------------------------------------ the paper's mesh file (Fig. 4)
def test_mesh_file_reader_hand_written_file():
    """PAPER.md:296-328 Fig. 4: node table "id x y z", connectivity table "id n1 n2 n3 manning",
    counts on their own lines, 1-based ids, ghost-block sections (multi-GPU) ignored.  The
    hand-written 4-node file is the two-triangle mesh of workloads.two_triangles()."""
    import os
    d = B.read_mesh_file(os.path.join(os.path.dirname(__file__), "golden", "fig4_two_triangles.txt"))
    w = W.two_triangles()
    np.testing.assert_array_equal(d["nodes_xy"], w.nodes_xy)
    np.testing.assert_array_equal(d["tris"], w.tris)
    np.testing.assert_array_equal(d["bathymetry"], [0.25, 0.5, 0.75, 1.0])     # rows 3 and 4 are swapped in the file
    np.testing.assert_array_equal(d["manning"], [0.03, 0.05])
    # feeds swe_mesh_create as it is (no tags in the file: walls)
    m = B.SweMesh(d["nodes_xy"], d["tris"], d["bathymetry"], d["manning"], np.zeros((2, 3), dtype=np.int8))
    t = m.get_tables()
    np.testing.assert_allclose(t["area"], [0.5, 0.5], rtol=1e-15)
    np.testing.assert_allclose(t["cell_z"], [0.5, 2.0 / 3.0], rtol=1e-15)


def test_mesh_file_reader_round_trip_and_errors(tmp_path):
    w = W.config4(nx=30, ny=8)
    p = tmp_path / "mesh.txt"
    with open(p, "w") as f:
        f.write("Coordinate table\n%d\n" % w.nnodes)
        for i in range(w.nnodes):
            f.write("%d %.17g %.17g %.17g\n" % (i + 1, w.nodes_xy[i, 0], w.nodes_xy[i, 1], w.bathymetry[i]))
        f.write("Connectivity table\n%d\n" % w.ncells)
        for i in range(w.ncells):
            f.write("%d %d %d %d %.17g\n" % (i + 1, w.tris[i, 0] + 1, w.tris[i, 1] + 1, w.tris[i, 2] + 1, w.manning[i]))
    d = B.read_mesh_file(str(p))
    np.testing.assert_array_equal(d["nodes_xy"], w.nodes_xy)
    np.testing.assert_array_equal(d["bathymetry"], w.bathymetry)
    np.testing.assert_array_equal(d["tris"], w.tris)
    np.testing.assert_array_equal(d["manning"], w.manning)
    with pytest.raises(B.SweError) as e:
        B.read_mesh_file(str(tmp_path / "missing.txt"))
    assert e.value.code == -13
    bad = tmp_path / "bad.txt"
    bad.write_text("Coordinate table\n2\n1 0 0 0\n3 1 0 0\n")          # id 3 of 2
    with pytest.raises(B.SweError) as e:
        B.read_mesh_file(str(bad))
    assert e.value.code == -14 and ":4:" in str(e.value)
    bad.write_text("Coordinate table\n2\n1 0 0 0\n2 1 0 0\nConnectivity table\n1\n1 1 2 5 0.03\n")   # node 5 of 2
    with pytest.raises(B.SweError) as e:
        B.read_mesh_file(str(bad))
    assert e.value.code == -14
    bad.write_text("Coordinate table\n2\n1 0 0 0\n2 1 0 0\nConnectivity table\n2\n1 1 2 2 0.03\n")   # truncated
    with pytest.raises(B.SweError) as e:
        B.read_mesh_file(str(bad))
    assert e.value.code == -14
