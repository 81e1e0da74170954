"""Pins of the oracle's whole step: invariants, closed forms, analytic dam breaks."""
import math

import numpy as np
import pytest

from oracle.swe_oracle import OracleSolver
from paper_2010_14416_b200 import workloads as W
from tests.analytic import ritter_profile, stoker, stoker_profile

G = 9.81


def _l1(hnum, hexact, area):
    return float(np.sum(np.abs(hnum - hexact) * area) / np.sum(area))


# ------------------------------------------------------------------ well-balancedness
def test_lake_at_rest_variable_bed_with_islands():
    """R-13/R-14: rest over 64 bumps, some emergent, is kept to round-off (config 3 shape)."""
    w = W.config3(nx=120, ny=60, nsteps=300)
    s = OracleSolver.from_workload(w)
    geo = s.geometry()
    dry0 = w.h <= w.h_dry
    assert 0.005 < dry0.mean() < 0.6, "the reduced config must keep emergent islands"
    dt0 = s.compute_dt()
    s.run(300)
    h, hu, hv, _, dt = s.get_state()
    wet = h > w.h_dry
    np.testing.assert_array_equal(~wet, dry0)
    u = np.where(wet, hu / np.where(wet, h, 1.0), 0.0)
    v = np.where(wet, hv / np.where(wet, h, 1.0), 0.0)
    assert np.abs(u).max() < 1e-10 and np.abs(v).max() < 1e-10
    assert np.abs(h[wet] + geo["z"][wet] - 2.0).max() < 1e-12
    assert dt == pytest.approx(dt0, rel=1e-12)
    assert s.stats()["nclamp"] == 0


def test_wrong_source_factor_would_not_be_at_rest():
    """The lake-at-rest pin is sharp: the step's momentum residual comes from cancelling the
    edge pressure g h**^2/2 against eq.(30) with g/2; here we check the two pieces separately
    are O(1), so a lost factor (R-13) or sign could not pass the test above."""
    w = W.config3(nx=40, ny=20)
    flat = W.config3(nx=40, ny=20)
    flat.bathymetry = np.zeros_like(flat.bathymetry)      # same depths, flat bed: not at rest
    s = OracleSolver.from_workload(flat)
    s.run(1)
    _, hu, hv, _, _ = s.get_state()
    assert max(np.abs(hu).max(), np.abs(hv).max()) > 1e-3
    s = OracleSolver.from_workload(w)
    s.run(1)
    _, hu, hv, _, _ = s.get_state()
    assert max(np.abs(hu).max(), np.abs(hv).max()) < 1e-13


def test_flat_bed_rest_to_roundoff():
    """Equal depths on a flat bed: every edge returns exactly (0, g h^2/2, 0) (R-12), so the
    only residual is the closure sum_k L_k n_k = 0 in floating point (a few ulp per step)."""
    w = W.canal_dam_break(30, 5, h_left=0.8, h_right=0.8, manning=0.03, length=30.0)
    s = OracleSolver.from_workload(w)
    s.run(50)
    h, hu, hv, _, _ = s.get_state()
    assert np.abs(h - 0.8).max() < 1e-14
    assert max(np.abs(hu).max(), np.abs(hv).max()) < 1e-14


# ------------------------------------------------------------------ conservation
@pytest.mark.parametrize("hr,mn", [(0.5, 0.0), (0.0, 0.03)])
def test_mass_conservation_closed_box(hr, mn):
    w = W.canal_dam_break(100, 10, h_left=1.0, h_right=hr, manning=mn, seed=20102)
    s = OracleSolver.from_workload(w)
    v0 = s.stats()["volume"]
    s.run(500)
    st = s.stats()
    assert st["nclamp"] == 0
    assert st["volume"] == pytest.approx(v0, rel=1e-12)
    assert st["boundary_volume_out"] == 0.0


def test_inflow_outflow_mass_balance():
    """R-20: d/dt sum h|Omega| = Q_in - outflow, to round-off (river-shaped small domain)."""
    w = W.config4(nx=120, ny=30, nsteps=300)
    s = OracleSolver.from_workload(w)
    v0 = s.stats()["volume"]
    s.run(300)
    st = s.stats()
    h, hu, hv, t, _ = s.get_state()
    assert st["nclamp"] == 0 and t > 0
    assert st["volume"] - v0 == pytest.approx(-st["boundary_volume_out"], rel=1e-9, abs=1e-9 * v0)
    # nothing has reached the outlet yet, so the gain is exactly the prescribed discharge
    right_wet = (W.centroids(w.nodes_xy, w.tris)[:, 0] > 0.98 * w.nodes_xy[:, 0].max()) & (hu > 1e-9)
    if not right_wet.any():
        assert st["volume"] - v0 == pytest.approx(500.0 * t, rel=1e-9)


def _uniform_channel(nx=24, ny=6, h=0.9, u=0.5, length=24.0):
    """Flat frictionless channel flowing in +x: prescribed discharge on the left edge,
    transmissive right edge, walls along the sides."""
    w = W.canal_dam_break(nx, ny, h_left=h, h_right=h, manning=0.0, length=length, seed=31)
    left = np.zeros(w.bc_tags.shape, dtype=bool)
    right = np.zeros(w.bc_tags.shape, dtype=bool)
    for k in range(3):
        xa = w.nodes_xy[w.tris[:, k], 0]
        xb = w.nodes_xy[w.tris[:, (k + 1) % 3], 0]
        left[:, k] = (xa == 0.0) & (xb == 0.0)
        right[:, k] = (xa == length) & (xb == length)
    w.bc_tags[left] = W.BC_INFLOW0
    w.bc_tags[right] = W.BC_TRANSMISSIVE
    width = w.nodes_xy[:, 1].max()
    w.bc_values = {W.BC_INFLOW0: h * u * width}
    w.hu[:] = h * u
    return w


def test_inflow_momentum_flux_keeps_uniform_channel_flow_steady():
    """the prescribed-discharge flux is (Q, Q^2/h_l + g h_l^2/2, 0).  Uniform flow
    (h, u, 0) fed with Q = h u per unit width is a steady state of the equations: every interior
    edge returns the physical flux of the common state (consistency), walls and the free outflow
    return it too, so the inflow edge must return exactly G(U) = (h u, h u^2 + g h^2/2, 0) for the
    3-edge sum of each cell to close (sum_k L_k n_k = 0).  A wrong momentum term (Q^2 h, Q^2/h^2,
    a lost pressure term, a non-zero third component) leaves an O(1) residual in the first column
    of cells."""
    h0, u0 = 0.9, 0.5
    w = _uniform_channel(h=h0, u=u0)
    s = OracleSolver.from_workload(w)
    s.run(40)
    h, hu, hv, t, _ = s.get_state()
    assert t > 0.5
    np.testing.assert_allclose(h, h0, rtol=0, atol=2e-14)
    np.testing.assert_allclose(hu, h0 * u0, rtol=0, atol=2e-14)
    np.testing.assert_allclose(hv, 0.0, rtol=0, atol=2e-14)
    vol = s.boundary_volumes()
    assert vol[W.BC_INFLOW0] == pytest.approx(-vol[W.BC_TRANSMISSIVE], rel=1e-13)


def test_dry_inflow_cell_hand_value():
    """R-20, dry branch: an inflow edge on a dry cell carries the prescribed mass flux and no
    momentum flux (there is no depth to form Q^2/h or g h^2/2 with).  Two dry triangles, bottom
    edge of cell 0 (L = 1, |Omega| = 1/2) fed with Q = 0.3 m^3/s: after dt = 0.1 the cell holds
    h = dt (L/|Omega|) Q/L = 0.06 m, at rest; its neighbour stays dry."""
    w = W.two_triangles(0.0, 0.0)
    w.bc_tags[0, 0] = W.BC_INFLOW0
    w.bc_values = {W.BC_INFLOW0: 0.3}
    s = OracleSolver.from_workload(w)
    s.step_dt(0.1)
    h, hu, hv, _, _ = s.get_state()
    np.testing.assert_allclose(h, [0.06, 0.0], rtol=1e-15, atol=0)
    assert (hu == 0.0).all() and (hv == 0.0).all()
    # next step the cell is wet: G_2 = Q^2/h + g h^2/2 enters with the edge normal (0,-1), so the
    # y-momentum gained is dt (L/|Omega|) (q_n^2/h + g h^2/2) and the x-momentum stays 0 on this
    # edge; the diagonal edge (right side dry) adds its own flux, so only the inflow edge's share
    # is checked, through the boundary volume: -Q (dt1 + dt2)
    s.step_dt(0.01)
    assert s.boundary_volumes()[W.BC_INFLOW0] == pytest.approx(-0.3 * 0.11, rel=1e-14)
    assert np.isfinite(np.concatenate(s.get_state()[:3])).all()


# ------------------------------------------------------------------ friction
def test_friction_closed_form_uniform_flow():
    """eq.(33)-(37): uniform h and q, flat bed, transmissive box: one step gives exactly
    q' = q / (1 + dt c |q|), c = g m^2 h^(-7/3), direction preserved (SURVEY 8(c) pin)."""
    w = W.canal_dam_break(12, 6, h_left=0.9, h_right=0.9, manning=0.035, length=12.0)
    w.bc_tags[w.bc_tags > 0] = W.BC_TRANSMISSIVE
    q = np.array([0.6, -0.35])
    w.hu[:] = q[0]
    w.hv[:] = q[1]
    s = OracleSolver.from_workload(w)
    dt = 0.37
    s.step_dt(dt)
    h, hu, hv, _, _ = s.get_state()
    c = G * 0.035 ** 2 * 0.9 ** (-7.0 / 3.0)
    f = 1.0 / (1.0 + dt * c * np.linalg.norm(q))
    np.testing.assert_allclose(h, 0.9, rtol=1e-13)
    np.testing.assert_allclose(hu, q[0] * f, rtol=1e-12)
    np.testing.assert_allclose(hv, q[1] * f, rtol=1e-12)


def test_zero_manning_is_the_explicit_scheme():
    w0 = W.canal_dam_break(40, 6, manning=0.0, length=40.0, seed=3)
    w1 = W.canal_dam_break(40, 6, manning=1e-30, length=40.0, seed=3)
    a, b = OracleSolver.from_workload(w0), OracleSolver.from_workload(w1)
    a.run(40)
    b.run(40)
    for x, y in zip(a.get_state()[:3], b.get_state()[:3]):
        np.testing.assert_allclose(x, y, rtol=1e-13, atol=1e-15)


def test_friction_decelerates_and_h_column_sign():
    """With friction the dam-break front is slower; momentum magnitude never grows by friction."""
    w0 = W.canal_dam_break(100, 4, h_right=0.0, manning=0.0, seed=5)
    w1 = W.canal_dam_break(100, 4, h_right=0.0, manning=0.05, seed=5)
    a, b = OracleSolver.from_workload(w0), OracleSolver.from_workload(w1)
    a.run(200)
    b.run(200)
    cx = W.centroids(w0.nodes_xy, w0.tris)[:, 0]
    fa = cx[a.get_state()[0] > 1e-3].max()
    fb = cx[b.get_state()[0] > 1e-3].max()
    assert fb < fa


# ------------------------------------------------------------------ time step
def test_dt_closed_form_uniform_state():
    """eq.(15), R-9: dt = CFL R_min / (sqrt(g h) + |V|) on a uniform state."""
    w = W.canal_dam_break(20, 5, h_left=1.7, h_right=1.7, length=20.0)
    w.hu[:] = 1.7 * 0.8
    w.hv[:] = -1.7 * 0.6
    s = OracleSolver.from_workload(w)
    rmin = s.geometry()["rin"].min()
    assert s.compute_dt() == pytest.approx(0.9 * rmin / (math.sqrt(G * 1.7) + 1.0), rel=1e-14)
    # inradius: R = 2 |Omega| / perimeter
    geo = s.geometry()
    np.testing.assert_allclose(geo["rin"], 2 * geo["area"] / geo["len"].sum(1), rtol=1e-15)


def test_all_dry_gives_zero_dt_and_no_steps():
    w = W.canal_dam_break(10, 3, h_left=0.0, h_right=0.0, length=10.0)
    s = OracleSolver.from_workload(w)
    assert s.compute_dt() == 0.0
    assert s.run(5) == 0


# ------------------------------------------------------------------ analytic dam breaks
def _run_until(s, t_end, chunk=10, max_steps=200000):
    """A broken oracle (NaN or collapsing dt) must fail the test, not hang the suite."""
    done = 0
    while s.get_state()[3] < t_end:
        n = s.run(chunk)
        done += n
        t, dt = s.get_state()[3:5]
        assert n == chunk and math.isfinite(t) and math.isfinite(dt) and dt > 0.0, \
            f"oracle stopped advancing at t={t}, dt={dt}"
        assert done < max_steps, f"t_end={t_end} not reached after {done} steps (t={t}, dt={dt})"
    return s.get_state()


@pytest.mark.parametrize("hL,hR,t_end", [(1.0, 0.5, 8.0), (10.0, 1.0, 2.5)])
def test_stoker_convergence(hL, hR, t_end):
    """Wet-wet dam break against the Stoker solution (BASELINE config 1; paper's 10 | 1 case,
    PAPER.md:485-491): L1(h) error decreases with dx at the first-order-scheme rate, plateau
    depth within 1 %."""
    errs = []
    for nx in (100, 200, 400):
        w = W.canal_dam_break(nx, 4, h_left=hL, h_right=hR, seed=20102)
        s = OracleSolver.from_workload(w)
        h, hu, hv, t, _ = _run_until(s, t_end)
        cx = W.centroids(w.nodes_xy, w.tris)[:, 0]
        hex_, _ = stoker_profile((cx - 50.0) / t, hL, hR)
        errs.append(_l1(h, hex_, s.geometry()["area"]))
        if nx == 400:
            p = stoker(hL, hR)
            xi = (cx - 50.0) / t
            plateau = (xi > p["tail"] + 0.25 * (p["shock"] - p["tail"])) & \
                      (xi < p["shock"] - 0.25 * (p["shock"] - p["tail"]))
            assert np.abs(h[plateau] / p["hm"] - 1.0).max() < 0.01
            u = hu[plateau] / h[plateau]
            assert np.abs(u / p["um"] - 1.0).max() < 0.02
            assert s.stats()["nclamp"] == 0
    assert errs[1] < 0.72 * errs[0] and errs[2] < 0.72 * errs[1]
    assert errs[2] < 0.012 * hL


def test_ritter_front_and_profile():
    """Frictionless wet-dry dam break (config 2 variant, m = 0) against Ritter."""
    errs, tips = [], []
    for nx in (200, 400):
        w = W.canal_dam_break(nx, 4, h_left=1.0, h_right=0.0, manning=0.0, seed=20103)
        s = OracleSolver.from_workload(w)
        h, hu, hv, t, _ = _run_until(s, 5.0)
        cx = W.centroids(w.nodes_xy, w.tris)[:, 0]
        hex_, _ = ritter_profile((cx - 50.0) / t, 1.0)
        errs.append(_l1(h, hex_, s.geometry()["area"]))
        # front position: the h = 5 cm contour within 3 %; the thin tip (1 cm contour) is known
        # to lag in first-order schemes and must approach the exact position under refinement
        ratios = []
        for thr in (5e-2, 1e-2):
            front = cx[h > thr].max() - 50.0
            exact = t * (2.0 * math.sqrt(G) - 3.0 * math.sqrt(G * thr))
            ratios.append(front / exact)
        assert ratios[0] == pytest.approx(1.0, abs=0.03)
        assert 0.85 < ratios[1] < 1.0
        tips.append(ratios[1])
        assert s.stats()["nclamp"] == 0
        # upstream of the rarefaction head only numerical diffusion has arrived
        assert np.abs(h[cx < 50.0 - 1.05 * math.sqrt(G) * t - 2.0] - 1.0).max() < 0.01
    assert errs[1] < 0.75 * errs[0]
    assert tips[1] > tips[0]


def test_friction_jacobian_including_h_column_vs_symbolic_derivative():
    """eq.(34)-(37), R-19: J_f is DEFINED as dS_f/dU of eq.(32).  The oracle's step must satisfy
    [I - dt/2 J] dU = dt (b + S_f) with J taken here by symbolic differentiation of eq.(32)
    (sympy), not from the printed matrix (35).  dt*b comes from the same step without friction.
    The d/dh column matters: the same residual with that column zeroed is orders larger."""
    import sympy as sp
    h, qx, qy, gg, mm = sp.symbols("h qx qy g m", positive=True)
    qn = sp.sqrt(qx ** 2 + qy ** 2)
    Sf = sp.Matrix([0, -gg * mm ** 2 * qx * qn / h ** sp.Rational(7, 3),
                    -gg * mm ** 2 * qy * qn / h ** sp.Rational(7, 3)])          # eq.(32)
    Jf = Sf.jacobian([h, qx, qy])
    f_S = sp.lambdify((h, qx, qy, gg, mm), Sf, "numpy")
    f_J = sp.lambdify((h, qx, qy, gg, mm), Jf, "numpy")

    mn = 0.04
    w0 = W.canal_dam_break(30, 4, h_left=1.3, h_right=0.4, manning=0.0, length=30.0, seed=11)
    rng = np.random.default_rng(5)
    w0.hu[:] = w0.h * rng.uniform(0.5, 2.0, w0.ncells)
    w0.hv[:] = w0.h * rng.uniform(-1.0, 1.0, w0.ncells)
    w1 = W.canal_dam_break(30, 4, h_left=1.3, h_right=0.4, manning=mn, length=30.0, seed=11)
    w1.hu[:], w1.hv[:] = w0.hu, w0.hv
    dt = 0.05
    a, b = OracleSolver.from_workload(w0), OracleSolver.from_workload(w1)
    a.step_dt(dt)
    b.step_dt(dt)
    U = np.stack([w0.h, w0.hu, w0.hv], 1)
    dU0 = np.stack(a.get_state()[:3], 1) - U            # dt * b
    dU1 = np.stack(b.get_state()[:3], 1) - U
    assert np.abs(dU0[:, 0]).max() > 1e-3                # depth does change: the h column is exercised
    worst, worst_noh = 0.0, 0.0
    for i in range(w0.ncells):
        S = np.array(f_S(U[i, 0], U[i, 1], U[i, 2], G, mn), dtype=float).ravel()
        J = np.array(f_J(U[i, 0], U[i, 1], U[i, 2], G, mn), dtype=float)
        scale = np.abs(dU0[i]).max() + dt * np.abs(S).max()
        r = (np.eye(3) - 0.5 * dt * J) @ dU1[i] - dU0[i] - dt * S
        worst = max(worst, np.abs(r).max() / scale)
        J[:, 0] = 0.0
        r = (np.eye(3) - 0.5 * dt * J) @ dU1[i] - dU0[i] - dt * S
        worst_noh = max(worst_noh, np.abs(r).max() / scale)
    assert worst < 1e-12
    assert worst_noh > 1e4 * max(worst, 1e-16)


# ------------------------------------------------------------------ boundary diagnostics, run-until
def test_boundary_volumes_per_tag_and_run_until():
    """R-20 / PAPER.md:453: the inflow tag's cumulative volume is exactly -Q t, walls carry none,
    the tags add up to the total, and the volume in the domain changes by minus that total.
    run_until ends on t_end by shortening the last step and otherwise equals run()."""
    w = W.config4(nx=80, ny=20)
    s = OracleSolver.from_workload(w)
    v0 = s.stats()["volume"]
    n = s.run_until(30.0)
    h, hu, hv, t, dt = s.get_state()
    assert t == 30.0 and n == s.stats()["steps"]
    vol = s.boundary_volumes()
    assert vol[W.BC_INFLOW0] == pytest.approx(-500.0 * 30.0, rel=1e-12)
    assert vol[W.BC_WALL] == 0.0 and vol[W.BC_TRANSMISSIVE] > 0.0
    assert vol.sum() == pytest.approx(s.stats()["boundary_volume_out"], rel=1e-12)
    assert s.stats()["volume"] - v0 == pytest.approx(-vol.sum(), rel=1e-9)
    # the same number of plain steps reproduces every step but the shortened last one
    r = OracleSolver.from_workload(w)
    r.run(n - 1)
    r2 = OracleSolver.from_workload(w)
    r2.run_until(1e30, max_steps=n - 1)
    for a, b in zip(r.get_state()[:4], r2.get_state()[:4]):
        np.testing.assert_array_equal(a, b)
    assert r.get_state()[3] < 30.0 <= r.get_state()[3] + r.get_state()[4]


def test_refined_mesh_mass_and_dt_scale():
    """Locally refined basin (inradius ratio > 25): mass is conserved to round-off in the closed
    box, and the CFL step is bounded by the smallest wet cell's R / sqrt(g h) (eq.15, R-9)."""
    w = W.refined_basin(nx=120, ny=60)
    s = OracleSolver.from_workload(w)
    v0 = s.stats()["volume"]
    geo = s.geometry()
    wet = w.h > w.h_dry
    bound = 0.9 * (geo["rin"][wet] / np.sqrt(G * w.h[wet])).min()
    assert s.compute_dt() == pytest.approx(bound, rel=1e-14)       # at rest: lambda = sqrt(g h)
    s.run(300)
    assert s.stats()["volume"] == pytest.approx(v0, rel=1e-12)
    assert s.stats()["nclamp"] == 0


def test_single_precision_storage_stays_within_accumulated_float_roundoff():
    """PAPER.md:424 (configurable floating-point kind), the oracle side of SWE_FP_MIXED32: the state
    is rounded to single precision between the steps and everything else is unchanged.  Pinned by
    what that definition fixes: the stored state is exactly representable in float; each step adds
    at most one float rounding (2^-24 relative) to each of h, u, v, so after n steps of a
    non-amplifying scheme the distance to the double-precision run is at most ~n 2^-24 (here a few
    2^-24 sqrt(n), the roundings being uncorrelated); volume is conserved to the same order."""
    w = W.config1()
    n = 500
    a, b = OracleSolver.from_workload(w), OracleSolver.from_workload(w, storage32=True)
    v0 = b.stats()["volume"]
    assert a.run(n) == n and b.run(n) == n
    ha, hua, hva, ta, _ = a.get_state()
    hb, hub, hvb, tb, _ = b.get_state()
    np.testing.assert_array_equal(hb, hb.astype(np.float32).astype(np.float64))
    u = hub / hb
    np.testing.assert_allclose(u, u.astype(np.float32), rtol=2e-16, atol=0)       # h u with u a float
    eps = 2.0 ** -24
    for x, y in ((ha, hb), (hua, hub), (hva, hvb)):
        d = np.abs(x - y).max()
        assert 0.0 < d < 20.0 * eps * math.sqrt(n)
    assert abs(ta - tb) / ta < 10.0 * eps
    assert abs(b.stats()["volume"] - v0) / v0 < n * eps
