"""ctypes binding of the CPU oracle (oracle/swe_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module; the product (paper_2010_14416_b200) never does.
"""
from __future__ import annotations

import ctypes as C
import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, ip, i64 = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.c_int64
        L.oracle_create.restype = C.c_void_p
        L.oracle_create.argtypes = [dp, i64, ip, i64, dp, dp, C.POINTER(C.c_int8), C.c_double,
                                    C.c_double, C.c_double, C.POINTER(C.c_int)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_set_inflow.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.oracle_set_inflow.restype = C.c_int
        L.oracle_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.oracle_get_threads.argtypes = [C.c_void_p]
        L.oracle_get_threads.restype = C.c_int
        L.oracle_set_state.argtypes = [C.c_void_p, dp, dp, dp, C.c_double]
        L.oracle_compute_dt.argtypes = [C.c_void_p]
        L.oracle_compute_dt.restype = C.c_double
        L.oracle_run.argtypes = [C.c_void_p, i64]
        L.oracle_run.restype = i64
        L.oracle_step_dt.argtypes = [C.c_void_p, C.c_double]
        L.oracle_run_until.argtypes = [C.c_void_p, C.c_double, i64]
        L.oracle_run_until.restype = i64
        L.oracle_get_boundary_volumes.argtypes = [C.c_void_p, dp]
        L.oracle_get_state.argtypes = [C.c_void_p, dp, dp, dp, dp, dp]
        L.oracle_get_stats.argtypes = [C.c_void_p, dp]
        L.oracle_get_geometry.argtypes = [C.c_void_p, C.POINTER(C.c_int64), dp, dp, dp, dp, dp, dp]
        L.oracle_hllc.argtypes = [C.c_double] * 8 + [dp, dp]
        L.oracle_hll.argtypes = [C.c_double] * 8 + [dp]
        L.oracle_set_riemann.argtypes = [C.c_void_p, C.c_int]
        L.oracle_set_storage32.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def hllc(hL, uL, vL, hR, uR, vR, g=9.81, h_dry=1e-6):
    """Single-edge HLLC flux in the edge frame; returns (G[3], diag dict)."""
    G = np.zeros(3)
    d = np.zeros(8)
    lib().oracle_hllc(g, h_dry, hL, uL, vL, hR, uR, vR, _dp(G), _dp(d))
    names = ["branch", "h0", "hs", "pL", "pR", "SL", "SR", "Sstar"]
    return G, dict(zip(names, d.tolist()))


def hll(hL, uL, vL, hR, uR, vR, g=9.81, h_dry=1e-6):
    """Single-edge plain HLL flux (all three components by eq.17-18) in the edge frame."""
    G = np.zeros(3)
    lib().oracle_hll(g, h_dry, hL, uL, vL, hR, uR, vR, _dp(G))
    return G


class OracleSolver:
    """The scheme of PAPER.md sections 2-3 on a triangular mesh, on the CPU."""

    def __init__(self, nodes_xy, tris, bathymetry, manning, bc_tags, *, g=9.81, cfl=0.9,
                 h_dry=1e-6, threads=None):
        L = lib()
        self._L = L
        xy = np.ascontiguousarray(nodes_xy, dtype=np.float64)
        tr = np.ascontiguousarray(tris, dtype=np.int32)
        zz = np.ascontiguousarray(bathymetry, dtype=np.float64)
        mn = np.ascontiguousarray(manning, dtype=np.float64)
        tg = np.ascontiguousarray(bc_tags, dtype=np.int8)
        self.nt = int(tr.shape[0])
        self.nn = int(xy.shape[0])
        assert xy.shape == (self.nn, 2) and tr.shape == (self.nt, 3)
        assert zz.shape == (self.nn,) and mn.shape == (self.nt,) and tg.shape == (self.nt, 3)
        err = C.c_int(0)
        self._h = L.oracle_create(_dp(xy), self.nn, tr.ctypes.data_as(C.POINTER(C.c_int32)), self.nt,
                                  _dp(zz), _dp(mn), tg.ctypes.data_as(C.POINTER(C.c_int8)),
                                  float(g), float(cfl), float(h_dry), C.byref(err))
        if not self._h:
            raise ValueError(f"oracle_create failed with code {err.value}")
        if threads is not None:
            L.oracle_set_threads(self._h, int(threads))

    @classmethod
    def from_workload(cls, w, threads=None, storage32=False):
        s = cls(w.nodes_xy, w.tris, w.bathymetry, w.manning, w.bc_tags, g=w.g, cfl=w.cfl,
                h_dry=w.h_dry, threads=threads)
        if storage32:
            s.set_storage32()
        for tag, q in w.bc_values.items():
            s.set_inflow(tag, q)
        s.set_state(w.h, w.hu, w.hv)
        return s

    def __del__(self):
        if getattr(self, "_h", None):
            self._L.oracle_destroy(self._h)
            self._h = None

    @property
    def threads(self):
        return self._L.oracle_get_threads(self._h)

    def set_riemann(self, hll):
        """hll=True: plain HLL instead of HLLC."""
        self._L.oracle_set_riemann(self._h, int(bool(hll)))

    def set_storage32(self):
        """State and cell beds kept in single precision between the steps (call before set_state)."""
        self._L.oracle_set_storage32(self._h)

    def set_threads(self, n):
        self._L.oracle_set_threads(self._h, int(n))

    def set_inflow(self, tag, q_total):
        rc = self._L.oracle_set_inflow(self._h, int(tag), float(q_total))
        if rc != 0:
            raise ValueError(f"oracle_set_inflow failed with code {rc}")

    def set_state(self, h, hu, hv, t0=0.0):
        a = [np.ascontiguousarray(x, dtype=np.float64) for x in (h, hu, hv)]
        assert all(x.shape == (self.nt,) for x in a)
        self._L.oracle_set_state(self._h, _dp(a[0]), _dp(a[1]), _dp(a[2]), float(t0))

    def compute_dt(self):
        return self._L.oracle_compute_dt(self._h)

    def run(self, nsteps):
        return self._L.oracle_run(self._h, int(nsteps))

    def run_until(self, t_end, max_steps=1 << 40):
        return self._L.oracle_run_until(self._h, float(t_end), int(max_steps))

    def boundary_volumes(self):
        """Cumulative outward volume (m^3) per boundary tag since set_state, array [128]."""
        v = np.zeros(128)
        self._L.oracle_get_boundary_volumes(self._h, _dp(v))
        return v

    def step_dt(self, dt):
        self._L.oracle_step_dt(self._h, float(dt))

    def get_state(self):
        h, hu, hv = np.empty(self.nt), np.empty(self.nt), np.empty(self.nt)
        t, dt = C.c_double(0), C.c_double(0)
        self._L.oracle_get_state(self._h, _dp(h), _dp(hu), _dp(hv), C.byref(t), C.byref(dt))
        return h, hu, hv, t.value, dt.value

    def stats(self):
        s = np.zeros(5)
        self._L.oracle_get_stats(self._h, _dp(s))
        return dict(volume=s[0], ndry=int(s[1]), nclamp=int(s[2]), steps=int(s[3]),
                    boundary_volume_out=s[4])

    def geometry(self):
        nt = self.nt
        nbr = np.empty((nt, 3), dtype=np.int64)
        n1, n2, ln = np.empty((nt, 3)), np.empty((nt, 3)), np.empty((nt, 3))
        area, rin, z = np.empty(nt), np.empty(nt), np.empty(nt)
        self._L.oracle_get_geometry(self._h, nbr.ctypes.data_as(C.POINTER(C.c_int64)), _dp(n1),
                                    _dp(n2), _dp(ln), _dp(area), _dp(rin), _dp(z))
        return dict(nbr=nbr, n1=n1, n2=n2, len=ln, area=area, rin=rin, z=z)
