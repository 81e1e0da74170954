"""Pins of the oracle's geometry, neighbour tables and one hand-computed update."""
import math
import os

import numpy as np
import pytest

from oracle.swe_oracle import OracleSolver
from paper_2010_14416_b200 import workloads as W

G = 9.81
HERE = os.path.dirname(__file__)


def _golden_shock_flux():
    with open(os.path.join(HERE, "golden", "single_edge_fluxes.txt")) as f:
        for line in f:
            if line.startswith("shock"):
                return [float(x) for x in line.split("|")[2].split()]
    raise AssertionError


def test_two_triangle_geometry():
    w = W.two_triangles()
    geo = OracleSolver.from_workload(w).geometry()
    r2 = math.sqrt(2.0)
    np.testing.assert_array_equal(geo["nbr"], [[-1, -1, 1], [0, -1, -1]])
    np.testing.assert_allclose(geo["area"], [0.5, 0.5], rtol=0, atol=0)
    np.testing.assert_allclose(geo["len"], [[1, 1, r2], [r2, 1, 1]], rtol=1e-15)
    np.testing.assert_allclose(geo["n1"], [[0, 1, -1 / r2], [1 / r2, 0, -1]], atol=1e-15)
    np.testing.assert_allclose(geo["n2"], [[-1, 0, 1 / r2], [-1 / r2, 1, 0]], atol=1e-15)
    np.testing.assert_allclose(geo["rin"], [1.0 / (2.0 + r2)] * 2, rtol=1e-15)


def test_two_triangle_hand_update():
    """Unit square, walls, h = 1 below / 0.5 above the diagonal, one step of size dt.

    Hand computation (eq.(27), :125 wall flux): cell 0 has walls on y = 0
    (n = (0,-1), L = 1) and x = 1 (n = (1,0), L = 1) and the diagonal (n = (-1,1)/sqrt2,
    L = sqrt2) whose Riemann problem is the golden 'shock' row (h = 1 | 0.5 at rest), flux
    (G1, G2, 0) in the edge frame.  |Omega| = 1/2.
    """
    G1, G2, _ = _golden_shock_flux()
    w = W.two_triangles(1.0, 0.5)
    s = OracleSolver.from_workload(w)
    dt = 0.01
    s.step_dt(dt)
    h, hu, hv, _, _ = s.get_state()
    r2 = math.sqrt(2.0)
    pw0 = 0.5 * G * 1.0 ** 2
    pw1 = 0.5 * G * 0.5 ** 2
    # cell 0: sum_k L_k T^-1 G
    m0 = r2 * G1
    fx0 = 1.0 * pw0 * 1.0 + r2 * G2 * (-1 / r2)
    fy0 = 1.0 * pw0 * (-1.0) + r2 * G2 * (1 / r2)
    # cell 1 (h = 0.5) sees the mirrored problem: mass flux -G1, normal momentum flux G2 along
    # its own outward normal (1,-1)/sqrt2; walls on x = 0 (n = (-1,0)) and y = 1 (n = (0,1))
    m1 = -r2 * G1
    fx1 = r2 * G2 * (1 / r2) + pw1 * (-1.0)
    fy1 = r2 * G2 * (-1 / r2) + pw1 * 1.0
    np.testing.assert_allclose(h, [1.0 - dt * 2 * m0, 0.5 - dt * 2 * m1], rtol=1e-13)
    np.testing.assert_allclose(hu, [-dt * 2 * fx0, -dt * 2 * fx1], rtol=1e-12)
    np.testing.assert_allclose(hv, [-dt * 2 * fy0, -dt * 2 * fy1], rtol=1e-12)


def test_neighbours_are_mutual_and_share_two_nodes():
    w = W.config1()
    geo = OracleSolver.from_workload(w).geometry()
    nbr = geo["nbr"]
    nt = w.ncells
    assert (nbr < 0).sum() == 2 * (100 + 10)
    for i in range(0, nt, 7):
        for k in range(3):
            j = nbr[i, k]
            if j < 0:
                continue
            assert i in nbr[j]
            a, b = w.tris[i, k], w.tris[i, (k + 1) % 3]
            assert a in w.tris[j] and b in w.tris[j]
            kk = list(nbr[j]).index(i)
            # outward normals of the two sides are opposite, lengths equal
            assert geo["n1"][j, kk] == pytest.approx(-geo["n1"][i, k], abs=1e-15)
            assert geo["n2"][j, kk] == pytest.approx(-geo["n2"][i, k], abs=1e-15)
            assert geo["len"][j, kk] == geo["len"][i, k]
    # discrete divergence theorem: sum_k L_k n_k = 0 for every closed cell
    np.testing.assert_allclose((geo["len"] * geo["n1"]).sum(1), 0.0, atol=1e-14)
    np.testing.assert_allclose((geo["len"] * geo["n2"]).sum(1), 0.0, atol=1e-14)
    assert geo["area"].sum() == pytest.approx(1000.0, rel=1e-13)


def test_clockwise_input_is_reoriented():
    w = W.config1()
    s_ref = OracleSolver.from_workload(w)
    tris = w.tris.copy()
    tags = w.bc_tags.copy()
    flip = np.arange(w.ncells) % 3 == 0
    tris[flip] = tris[flip][:, [0, 2, 1]]
    tags[flip] = tags[flip][:, [2, 1, 0]]
    s = OracleSolver(w.nodes_xy, tris, w.bathymetry, w.manning, tags, g=w.g, cfl=w.cfl, h_dry=w.h_dry)
    s.set_state(w.h, w.hu, w.hv)
    s.run(20)
    s_ref.run(20)
    a, b = s.get_state(), s_ref.get_state()
    np.testing.assert_allclose(a[0], b[0], rtol=1e-13)
    assert a[3] == pytest.approx(b[3], rel=1e-14)


def test_invalid_meshes_are_rejected():
    w = W.two_triangles()
    bad = w.tris.copy()
    bad[0, 0] = 9
    with pytest.raises(ValueError):
        OracleSolver(w.nodes_xy, bad, w.bathymetry, w.manning, w.bc_tags)
    deg = w.tris.copy()
    deg[0] = [0, 1, 1]
    with pytest.raises(ValueError):
        OracleSolver(w.nodes_xy, deg, w.bathymetry, w.manning, w.bc_tags)
    tri3 = np.vstack([w.tris, [[0, 2, 1]]]).astype(np.int32)   # edge 0-2 now shared by 3 cells
    with pytest.raises(ValueError):
        OracleSolver(w.nodes_xy, tri3, w.bathymetry, np.zeros(3), np.ones((3, 3), dtype=np.int8))


def test_rotation_invariance():
    """PAPER.md:113 eq.(12): the scheme commutes with rotations of the plane."""
    w = W.canal_dam_break(40, 6, seed=11, length=40.0, manning=0.02)
    rng = np.random.default_rng(5)
    w.hu = rng.uniform(-0.3, 0.3, w.ncells)
    w.hv = rng.uniform(-0.3, 0.3, w.ncells)
    ang = 0.7
    wr = W.rotated(w, ang)
    a = OracleSolver.from_workload(w)
    b = OracleSolver.from_workload(wr)
    a.run(60)
    b.run(60)
    ha, hua, hva, ta, _ = a.get_state()
    hb, hub, hvb, tb, _ = b.get_state()
    c, s = math.cos(ang), math.sin(ang)
    assert tb == pytest.approx(ta, rel=1e-12)
    np.testing.assert_allclose(hb, ha, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(hub, c * hua - s * hva, rtol=1e-10, atol=1e-11)
    np.testing.assert_allclose(hvb, s * hua + c * hva, rtol=1e-10, atol=1e-11)


def test_mirror_symmetry():
    """A dam break on a mesh symmetric about y = 0 stays symmetric (h, hu even; hv odd)."""
    w = W.mirrored_canal(manning=0.02)
    s = OracleSolver.from_workload(w)
    s.run(100)
    h, hu, hv, _, _ = s.get_state()
    n = w.ncells // 2
    np.testing.assert_allclose(h[:n], h[n:], rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(hu[:n], hu[n:], rtol=1e-10, atol=1e-11)
    np.testing.assert_allclose(hv[:n], -hv[n:], rtol=1e-10, atol=1e-11)
    assert np.abs(hv).max() > 1e-4   # the jittered mesh does produce transverse flow
