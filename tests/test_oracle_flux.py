"""Pins of the oracle's single-edge HLLC flux (eq.(17)-(26))."""
import math
import os

import numpy as np
import pytest

from oracle.swe_oracle import hllc
from tests.analytic import stoker

G = 9.81
HERE = os.path.dirname(__file__)


def _rows():
    rows = []
    with open(os.path.join(HERE, "golden", "single_edge_fluxes.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, rest = line.split(None, 1)
            a, b, c = rest.split("|")
            rows.append((name, [float(x) for x in a.split()], [float(x) for x in b.split()],
                         [float(x) for x in c.split()]))
    return rows


@pytest.mark.parametrize("row", _rows(), ids=lambda r: r[0])
def test_golden_single_edge(row):
    name, st, dg, fl = row
    Gf, d = hllc(*st)
    got = [d["branch"], d["h0"], d["hs"], d["pL"], d["pR"], d["SL"], d["SR"], d["Sstar"]]
    for want, have in zip(dg, got):
        if not math.isnan(want):
            # printed to 12-13 significant digits (4-5 for the supercritical row)
            tol = 1e-4 if name == "supercrit" else 2e-12
            assert have == pytest.approx(want, rel=tol, abs=tol)
    for want, have in zip(fl, Gf):
        assert have == pytest.approx(want, rel=1e-12, abs=1e-14)


def _phys(h, u, v):
    return np.array([h * u, h * u * u + 0.5 * G * h * h, h * u * v])


def test_consistency_equal_states():
    """G~(U, U) = G(U): any consistent solver -- sub- and super-critical."""
    rng = np.random.default_rng(1)
    for _ in range(200):
        h = rng.uniform(0.01, 5.0)
        u = rng.uniform(-12.0, 12.0)
        v = rng.uniform(-3.0, 3.0)
        Gf, _ = hllc(h, u, v, h, u, v)
        np.testing.assert_allclose(Gf, _phys(h, u, v), rtol=1e-13, atol=1e-13)


def test_rest_equal_states_bitwise():
    """R-12: equal states at rest return (0, g h^2/2, 0) exactly."""
    rng = np.random.default_rng(2)
    for _ in range(100):
        h = rng.uniform(1e-3, 30.0)
        Gf, _ = hllc(h, 0.0, 0.0, h, 0.0, 0.0)
        assert Gf[0] == 0.0 and Gf[2] == 0.0
        assert Gf[1] == 0.5 * G * h * h


def test_supercritical_upwinding():
    """eq.(17): S_L >= 0 returns G(U_L), S_R <= 0 returns G(U_R)."""
    Gf, d = hllc(0.3, 6.0, 0.5, 0.25, 5.5, -0.4)
    assert d["SL"] > 0
    np.testing.assert_array_equal(Gf, _phys(0.3, 6.0, 0.5))
    Gf, d = hllc(0.25, -5.5, 0.4, 0.3, -6.0, -0.5)
    assert d["SR"] < 0
    np.testing.assert_array_equal(Gf, _phys(0.3, -6.0, -0.5))


def test_antisymmetry():
    """Swapping the sides and reversing the normal negates the flux seen from the other cell.

    Mirror of (hL,uL,vL | hR,uR,vR) about the edge: (hR,-uR,-vR | hL,-uL,-vL); then
    G1' = -G1 (bitwise, R-12), G2' = +G2 (momentum flux along the flipped normal), G3' = +G3.
    """
    rng = np.random.default_rng(3)
    for _ in range(300):
        hL, hR = rng.uniform(0.05, 3.0, 2)
        uL, uR = rng.uniform(-4.0, 4.0, 2)
        vL, vR = rng.uniform(-2.0, 2.0, 2)
        if rng.uniform() < 0.15:
            hR = 0.0
        A, _ = hllc(hL, uL, vL, hR, uR, vR)
        B, _ = hllc(hR, -uR, -vR, hL, -uL, -vL)
        assert B[0] == -A[0]
        assert B[1] == pytest.approx(A[1], rel=1e-13, abs=1e-13)
        assert B[2] == pytest.approx(A[2], rel=1e-13, abs=1e-13)


def test_dry_bed_speeds():
    """eq.(26), R-18: right-dry still water gives the Ritter front speed 2 sqrt(g h)."""
    _, d = hllc(1.0, 0.0, 0.0, 0.0, 0.0, 0.0)
    assert d["SR"] == pytest.approx(2.0 * math.sqrt(G), rel=1e-15)
    assert d["SL"] == pytest.approx(-math.sqrt(G), rel=1e-15)
    _, d = hllc(0.0, 0.0, 0.0, 2.0, 0.3, 0.0)
    assert d["SL"] == pytest.approx(0.3 - 2.0 * math.sqrt(2 * G), rel=1e-15)
    assert d["SR"] == pytest.approx(0.3 + math.sqrt(2 * G), rel=1e-15)
    Gf, _ = hllc(0.0, 0.0, 0.0, 5e-7, 0.0, 0.0)
    assert (Gf == 0.0).all()
    # a dry side contributes no tangential momentum: the wet side's v is upwinded (R-16)
    Gf, _ = hllc(1.0, 0.5, 0.25, 0.0, 7.0, 9.0)
    assert Gf[2] == pytest.approx(Gf[0] * 0.25, rel=1e-15)


def test_wave_speed_vs_exact_shock():
    """R-7: with p_k = sqrt(h*(h*+h_k)/2)/h_k the estimate S_R is within 0.2 % of the exact
    Stoker shock speed (the printed, garbled p_k is off by tens of percent)."""
    for hL, hR in [(1.0, 0.5), (10.0, 1.0), (2.0, 1.9)]:
        _, d = hllc(hL, 0.0, 0.0, hR, 0.0, 0.0)
        exact = stoker(hL, hR)
        assert d["SR"] == pytest.approx(exact["shock"], rel=0.06 if hL / hR > 5 else 2e-3)
        assert d["SL"] == pytest.approx(exact["head"], rel=1e-12)


def test_pk_continuity():
    """p_k -> 1 as h* -> h_k (R-7): the wave speed is continuous across h* = h_k."""
    h = 1.3
    eps = 1e-7
    _, a = hllc(h, eps, 0.0, h, -eps, 0.0)     # converging: h* slightly above h
    _, b = hllc(h, -eps, 0.0, h, eps, 0.0)     # diverging: h* slightly below h
    assert a["pL"] == pytest.approx(1.0, abs=1e-6) and b["pL"] == 1.0
    assert a["SR"] == pytest.approx(b["SR"], abs=1e-5)


def test_eq22_clamp_dry_bed_generating_rarefactions():
    """R-6 (eq.22): for strongly diverging states, u_R - u_L >= 2 (a_L + a_R), the exact
    Riemann solution opens a dry bed between two rarefactions whose heads travel at exactly
    u_L - a_L and u_R + a_R (Toro 2001, dry-bed generation), i.e. p_L = p_R = 1 in eq.(19).  The
    bracket of eq.(22) is negative there; squaring it unclamped gives h* = 1.94 > h_k here and a
    spurious "shock" factor p_k = 1.69, so the clamp at 0 is what reproduces the exact speeds."""
    h, uL, uR = 1.0, -15.0, 15.0
    a = math.sqrt(G * h)
    assert uR - uL > 8.0 * a                 # bracket^2 / g > h: the unclamped reading differs
    Gf, d = hllc(h, uL, 0.0, h, uR, 0.0)
    assert d["branch"] == 3 and d["hs"] == 0.0
    assert d["pL"] == 1.0 and d["pR"] == 1.0
    assert d["SL"] == uL - a and d["SR"] == uR + a
    # the same with unequal depths and a tangential velocity; the mass flux is the HLL average (18)
    hL, hR = 0.7, 1.6
    aL, aR = math.sqrt(G * hL), math.sqrt(G * hR)
    Gf, d = hllc(hL, -22.0, 0.3, hR, 21.0, -0.2)
    assert d["branch"] == 3 and d["hs"] == 0.0
    assert d["SL"] == -22.0 - aL and d["SR"] == 21.0 + aR
    SL, SR = d["SL"], d["SR"]
    want = (SR * hL * -22.0 - SL * hR * 21.0 + SL * SR * (hR - hL)) / (SR - SL)
    assert Gf[0] == pytest.approx(want, rel=1e-14)


def test_eq24_continuous_with_eq17_across_SL_zero():
    """R-16 (eq.24): the flux is a continuous function of the states, so as
    S_L -> 0^- the star-region flux must tend to eq.(17)'s G(U_L) = (h u, ., h u v_L): the tangential
    velocity is v_L for S* >= 0.  The inequality as printed (v_L for S* <= 0) would give h u v_R
    here.  Mirror case: S_R -> 0^+ must tend to G(U_R)."""
    h, vL, vR = 1.0, 0.7, -0.4
    a = math.sqrt(G * h)
    for eps in (1e-3, 1e-6, 1e-9):
        u = a * (1.0 - eps)                   # equal depths and normal velocities: S_L = u - a = -eps a
        Gf, d = hllc(h, u, vL, h, u, vR)
        assert -2.0 * eps * a < d["SL"] < 0.0 and d["Sstar"] > 0.0
        assert Gf[0] == pytest.approx(h * u, rel=1e-12)
        assert Gf[2] == pytest.approx(h * u * vL, rel=1e-12)      # printed inequality: h u vR = -1.25
        Gf, d = hllc(h, -u, vL, h, -u, vR)
        assert 0.0 < d["SR"] < 2.0 * eps * a and d["Sstar"] < 0.0
        assert Gf[2] == pytest.approx(-h * u * vR, rel=1e-12)
    # and just on the other side of the switch, eq.(17) itself
    Gf, d = hllc(h, a * (1.0 + 1e-9), vL, h, a * (1.0 + 1e-9), vR)
    assert d["SL"] > 0.0 and Gf[2] == pytest.approx(h * a * vL, rel=1e-8)


def test_stoker_golden_digits():
    rows = {}
    with open(os.path.join(HERE, "golden", "stoker_ritter.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            p = line.split()
            rows[p[0]] = [float(x) for x in p[1:]]
    for key in ("stoker_1_0.5", "stoker_10_1"):
        hL, hR, hm, um, s, head, tail = rows[key]
        e = stoker(hL, hR)
        for want, have in zip((hm, um, s, head, tail),
                              (e["hm"], e["um"], e["shock"], e["head"], e["tail"])):
            assert have == pytest.approx(want, rel=1e-11)
    assert rows["ritter_1"][4] == pytest.approx(2 * math.sqrt(G), rel=1e-12)


# ------------------------------------------------------------------ plain HLL
def test_hll_equals_hllc_for_equal_tangential_velocity():
    """eq.(18) on the third component with v_L = v_R = v gives v times the HLL mass flux, which is
    what eq.(24) gives too; components 1-2 are shared by construction."""
    from oracle.swe_oracle import hll
    for (hL, uL, hR, uR, v) in [(1.0, 0.0, 0.5, 0.0, 0.3), (1.0, -1.0, 1.0, 1.0, -0.7),
                                (0.8, 0.4, 1.3, -0.2, 2.0), (1.0, 0.5, 0.0, 0.0, 0.25)]:
        Gc, _ = hllc(hL, uL, v, hR, uR, v)
        Gh = hll(hL, uL, v, hR, uR, v)
        np.testing.assert_allclose(Gh, Gc, rtol=1e-14, atol=1e-15)


def test_hll_pure_shear_closed_form():
    """Equal depths at rest in the normal direction, tangential velocities v_L != v_R: S_L = -a,
    S_R = a, so eq.(18) gives G_3 = S_R S_L h (v_R - v_L) / (S_R - S_L) = -a h (v_R - v_L) / 2, the
    numerical diffusion of a contact that HLLC removes (its G_3 is G_1 v = 0)."""
    from oracle.swe_oracle import hll
    h, vL, vR = 0.9, 0.4, -1.1
    a = (9.81 * h) ** 0.5
    Gh = hll(h, 0.0, vL, h, 0.0, vR)
    assert Gh[0] == 0.0 and Gh[1] == pytest.approx(0.5 * 9.81 * h * h, rel=1e-15)
    assert Gh[2] == pytest.approx(-a * h * (vR - vL) / 2.0, rel=1e-14)
    Gc, _ = hllc(h, 0.0, vL, h, 0.0, vR)
    assert Gc[2] == 0.0


def test_hll_consistency_and_supercritical():
    from oracle.swe_oracle import hll
    for (h, u, v) in [(0.7, 0.3, -0.2), (0.2, 3.0, 1.0), (0.2, -3.0, 1.0)]:
        np.testing.assert_allclose(hll(h, u, v, h, u, v), _phys(h, u, v), rtol=1e-14, atol=1e-15)
