"""Thin ctypes binding of libswe_b200 (include/swe.h): argument marshalling only.

PyTorch is used for device memory and the CUDA stream, nothing else: every step of the
hot path runs in the library's own CUDA kernels.  There is no CPU fallback: if the
shared library is missing or CUDA is unavailable the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

ORDER_IDENTITY, ORDER_HILBERT, ORDER_RCM = 0, 1, 2
LOOP_AUTO, LOOP_GRAPH, LOOP_PERSISTENT, LOOP_LAUNCH, LOOP_CLUSTER = 0, 1, 2, 3, 4
RIEMANN_HLLC, RIEMANN_HLL = 0, 1
KERNEL_TILED, KERNEL_EDGE_TWO_PASS = 0, 1
FP64, FP_MIXED32 = 0, 1
LOOP_NAMES = {0: "auto", 1: "graph", 2: "persistent", 3: "launch", 4: "cluster"}
ERR_ALL_DRY = -9

# every symbol include/swe.h declares
SYMBOLS = [
    "swe_params_default", "swe_mesh_create", "swe_mesh_file_read", "swe_mesh_destroy", "swe_mesh_workspace_bytes",
    "swe_mesh_bind_device", "swe_set_bc_value", "swe_set_state", "swe_set_state_device",
    "swe_compute_dt", "swe_step", "swe_run", "swe_run_until", "swe_get_boundary_volumes",
    "swe_snapshot_begin", "swe_snapshot_wait", "swe_sync", "swe_get_state", "swe_get_state_device",
    "swe_get_stats", "swe_get_permutation", "swe_get_tables", "swe_get_tile_info",
    "swe_get_tile_tables", "swe_get_launch_info", "swe_get_step_bytes", "swe_cfl_dt_static", "swe_sample_cells",
    "swe_last_error",
]


class SweParams(C.Structure):
    _fields_ = [("g", C.c_double), ("cfl", C.c_double), ("h_dry", C.c_double),
                ("ordering", C.c_int32), ("block_size", C.c_int32), ("loop_mode", C.c_int32),
                ("riemann", C.c_int32), ("kernel", C.c_int32), ("fp_kind", C.c_int32)]


class SweStats(C.Structure):
    _fields_ = [("volume", C.c_double), ("t", C.c_double), ("dt_last", C.c_double),
                ("steps", C.c_int64), ("n_dry", C.c_int64), ("n_clamped", C.c_int64),
                ("n_nonfinite", C.c_int64), ("active_tile_steps", C.c_int64),
                ("edge_list_fetches", C.c_int64), ("quiet_tile_steps", C.c_int64), ("stolen_tile_steps", C.c_int64)]


class SweError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libswe_b200 error {code}: {msg}")
        self.code = code


_lib = None


def load_library(rebuild_if_stale: bool = True):
    """dlopen the in-tree libswe_b200.so (building it with nvcc first if needed)."""
    global _lib
    if _lib is not None:
        return _lib
    # SWE_B200_LIB: use a prebuilt library instead of (re)building the in-tree one
    path = os.environ.get("SWE_B200_LIB") or (_build.build() if rebuild_if_stale else _build.LIB)
    L = C.CDLL(path)
    dp, i32p, i64 = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.c_int64
    vp = C.c_void_p
    L.swe_params_default.argtypes = [C.POINTER(SweParams)]
    L.swe_mesh_create.argtypes = [dp, i64, i32p, i64, dp, dp, C.POINTER(C.c_int8),
                                  C.POINTER(SweParams), C.POINTER(vp)]
    L.swe_mesh_file_read.argtypes = [C.c_char_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64), dp, dp, i32p, dp]
    L.swe_mesh_destroy.argtypes = [vp]
    L.swe_mesh_workspace_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
    L.swe_mesh_bind_device.argtypes = [vp, vp, C.c_size_t, vp]
    L.swe_set_bc_value.argtypes = [vp, C.c_int, C.c_double]
    L.swe_set_state.argtypes = [vp, dp, dp, dp, C.c_double]
    L.swe_set_state_device.argtypes = [vp, vp, vp, vp, C.c_double]
    L.swe_compute_dt.argtypes = [vp, dp]
    L.swe_step.argtypes = [vp]
    L.swe_run.argtypes = [vp, i64]
    L.swe_run_until.argtypes = [vp, C.c_double, i64, C.POINTER(C.c_int64)]
    L.swe_get_boundary_volumes.argtypes = [vp, dp]
    L.swe_snapshot_begin.argtypes = [vp, dp, dp, dp, dp]
    L.swe_snapshot_wait.argtypes = [vp]
    L.swe_sync.argtypes = [vp]
    L.swe_get_state.argtypes = [vp, dp, dp, dp, dp, dp]
    L.swe_get_state_device.argtypes = [vp, vp, vp, vp]
    L.swe_get_stats.argtypes = [vp, C.POINTER(SweStats)]
    L.swe_sample_cells.argtypes = [vp, i32p, i64, dp, dp, dp, dp]
    L.swe_get_permutation.argtypes = [vp, i32p]
    L.swe_get_tables.argtypes = [vp, i32p, dp, dp, dp, dp, dp]
    L.swe_get_tile_info.argtypes = [vp, i32p, C.POINTER(C.c_int64), C.POINTER(C.c_int64), i32p, i32p,
                                    C.POINTER(C.c_size_t)]
    L.swe_get_tile_tables.argtypes = [vp, i32p, i32p, dp, i32p]
    L.swe_get_launch_info.argtypes = [vp, i32p, i32p, i32p, C.POINTER(C.c_int64)]
    L.swe_get_step_bytes.argtypes = [vp, C.c_double, C.c_double, C.c_double, dp]
    L.swe_cfl_dt_static.argtypes = [vp, vp, vp, vp, i64, C.c_double, C.c_double, C.c_double, vp, vp]
    L.swe_last_error.argtypes = [vp]
    L.swe_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        if name != "swe_last_error":
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def cfl_dt_static(d_h, d_hu, d_hv, d_inradius, n, g, cfl, h_dry, d_dt, stream=None):
    """swe_cfl_dt_static (include/swe.h): the CFL time step with no handle and no allocation; all
    arguments are device addresses (ints, e.g. tensor.data_ptr()); stream = cudaStream_t as int."""
    L = load_library()
    rc = L.swe_cfl_dt_static(d_h, d_hu, d_hv, d_inradius, n, g, cfl, h_dry, d_dt, stream)
    if rc != 0:
        raise SweError(rc, (L.swe_last_error(None) or b"").decode())


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def read_mesh_file(path):
    """Mesh file in the paper's layout (Fig. 4) -> dict of 0-based arrays
    (nodes_xy, bathymetry, tris, manning); the file has no boundary tags."""
    L = load_library()
    nn, nt = C.c_int64(0), C.c_int64(0)
    enc = os.fsencode(path)
    rc = L.swe_mesh_file_read(enc, C.byref(nn), C.byref(nt), None, None, None, None)
    if rc != 0:
        raise SweError(rc, (L.swe_last_error(None) or b"").decode())
    xy, z = np.empty((nn.value, 2)), np.empty(nn.value)
    tris, mn = np.empty((nt.value, 3), dtype=np.int32), np.empty(nt.value)
    rc = L.swe_mesh_file_read(enc, C.byref(nn), C.byref(nt), _dp(xy), _dp(z),
                              tris.ctypes.data_as(C.POINTER(C.c_int32)), _dp(mn))
    if rc != 0:
        raise SweError(rc, (L.swe_last_error(None) or b"").decode())
    return dict(nodes_xy=xy, bathymetry=z, tris=tris, manning=mn)


class SweMesh:
    """One mesh handle.  Methods carry the names of the C entry points without the prefix."""

    def __init__(self, nodes_xy, tris, bathymetry, manning, bc_tags, *, g=9.81, cfl=0.9,
                 h_dry=1e-6, ordering=ORDER_HILBERT, block_size=0, loop_mode=LOOP_AUTO,
                 riemann=RIEMANN_HLLC, kernel=KERNEL_TILED, fp_kind=FP64):
        self._h = None
        L = load_library()
        self._L = L
        xy = np.ascontiguousarray(nodes_xy, dtype=np.float64)
        tr = np.ascontiguousarray(tris, dtype=np.int32)
        zz = np.ascontiguousarray(bathymetry, dtype=np.float64)
        mn = np.ascontiguousarray(manning, dtype=np.float64)
        tg = np.ascontiguousarray(bc_tags, dtype=np.int8)
        self.nn, self.nt = int(xy.shape[0]), int(tr.shape[0])
        if xy.shape != (self.nn, 2) or tr.shape != (self.nt, 3) or zz.shape != (self.nn,) \
                or mn.shape != (self.nt,) or tg.shape != (self.nt, 3):
            raise ValueError("array shapes do not match the mesh sizes")
        p = SweParams()
        L.swe_params_default(C.byref(p))
        p.g, p.cfl, p.h_dry = float(g), float(cfl), float(h_dry)
        p.ordering, p.block_size, p.loop_mode = int(ordering), int(block_size), int(loop_mode)
        p.riemann = int(riemann)
        p.kernel = int(kernel)
        p.fp_kind = int(fp_kind)
        self.params = p
        h = C.c_void_p()
        rc = L.swe_mesh_create(_dp(xy), self.nn, tr.ctypes.data_as(C.POINTER(C.c_int32)), self.nt,
                               _dp(zz), _dp(mn), tg.ctypes.data_as(C.POINTER(C.c_int8)),
                               C.byref(p), C.byref(h))
        if rc != 0:
            raise SweError(rc, (L.swe_last_error(None) or b"").decode())
        self._h = h
        self._workspace = None   # torch tensor keeping the device memory alive
        self._stream = None

    @classmethod
    def from_workload(cls, w, **kw):
        m = cls(w.nodes_xy, w.tris, w.bathymetry, w.manning, w.bc_tags, g=w.g, cfl=w.cfl,
                h_dry=w.h_dry, **kw)
        for tag, q in w.bc_values.items():
            m.set_bc_value(tag, q)
        return m

    def _ck(self, rc):
        if rc != 0:
            raise SweError(rc, (self._L.swe_last_error(self._h) or b"").decode())

    def destroy(self):
        if self._h is not None:
            self._L.swe_mesh_destroy(self._h)
            self._h = None
        self._workspace = None

    __del__ = destroy

    # ---- device plumbing (torch: memory + stream only) ------------------------------------
    def workspace_bytes(self) -> int:
        n = C.c_size_t(0)
        self._ck(self._L.swe_mesh_workspace_bytes(self._h, C.byref(n)))
        return int(n.value)

    def bind_device(self, device="cuda:0", stream=None):
        """Allocate the workspace as a torch tensor on `device` and bind it with a stream."""
        import torch
        if not torch.cuda.is_available():
            raise SweError(-8, "CUDA is not available: libswe_b200 has no CPU fallback")
        dev = torch.device(device)
        torch.cuda.set_device(dev)
        nbytes = self.workspace_bytes()
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
        off = (-ws.data_ptr()) % 256
        self._workspace = ws
        self._stream = stream if stream is not None else torch.cuda.Stream(device=dev)
        self._ck(self._L.swe_mesh_bind_device(self._h, C.c_void_p(ws.data_ptr() + off), nbytes,
                                              C.c_void_p(self._stream.cuda_stream)))
        return self

    @property
    def stream(self):
        return self._stream

    # ---- the C entry points ------------------------------------------------------------------
    def set_bc_value(self, tag, total_discharge):
        self._ck(self._L.swe_set_bc_value(self._h, int(tag), float(total_discharge)))

    def set_state(self, h, hu, hv, t0=0.0):
        a = [np.ascontiguousarray(x, dtype=np.float64) for x in (h, hu, hv)]
        if any(x.shape != (self.nt,) for x in a):
            raise ValueError("state arrays must have shape (nt,)")
        self._ck(self._L.swe_set_state(self._h, _dp(a[0]), _dp(a[1]), _dp(a[2]), float(t0)))

    def set_state_device(self, d_h, d_hu, d_hv, t0=0.0):
        """torch float64 CUDA tensors of shape (nt,), caller numbering."""
        self._ck(self._L.swe_set_state_device(self._h, C.c_void_p(d_h.data_ptr()),
                                              C.c_void_p(d_hu.data_ptr()),
                                              C.c_void_p(d_hv.data_ptr()), float(t0)))

    def compute_dt(self) -> float:
        dt = C.c_double(0.0)
        self._ck(self._L.swe_compute_dt(self._h, C.byref(dt)))
        return dt.value

    def step(self):
        self._ck(self._L.swe_step(self._h))

    def run(self, nsteps):
        self._ck(self._L.swe_run(self._h, int(nsteps)))

    def run_until(self, t_end, max_steps=1 << 40):
        done = C.c_int64(0)
        self._ck(self._L.swe_run_until(self._h, float(t_end), int(max_steps), C.byref(done)))
        return done.value

    def get_boundary_volumes(self):
        v = np.zeros(128, dtype=np.float64)
        self._ck(self._L.swe_get_boundary_volumes(self._h, _dp(v)))
        return v

    def snapshot_begin(self, h, hu, hv):
        """Asynchronous snapshot into the given float64 arrays (pinned for a real overlap)."""
        self._snap_t = C.c_double(0.0)
        self._snap_bufs = (h, hu, hv)      # keep them alive until snapshot_wait
        self._ck(self._L.swe_snapshot_begin(self._h, _dp(h), _dp(hu), _dp(hv), C.byref(self._snap_t)))

    def snapshot_wait(self):
        self._ck(self._L.swe_snapshot_wait(self._h))
        return self._snap_t.value

    def sync(self):
        self._ck(self._L.swe_sync(self._h))

    def get_state(self):
        h, hu, hv = np.empty(self.nt), np.empty(self.nt), np.empty(self.nt)
        t, dt = C.c_double(0), C.c_double(0)
        self._ck(self._L.swe_get_state(self._h, _dp(h), _dp(hu), _dp(hv), C.byref(t), C.byref(dt)))
        return h, hu, hv, t.value, dt.value

    def get_state_into(self, h, hu, hv):
        """Read back into caller-provided (e.g. pinned) numpy arrays; returns (t, dt_next)."""
        t, dt = C.c_double(0), C.c_double(0)
        self._ck(self._L.swe_get_state(self._h, _dp(h), _dp(hu), _dp(hv), C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def get_state_device(self, d_h, d_hu, d_hv):
        self._ck(self._L.swe_get_state_device(self._h, C.c_void_p(d_h.data_ptr()),
                                              C.c_void_p(d_hu.data_ptr()),
                                              C.c_void_p(d_hv.data_ptr())))

    def sample_cells(self, cells):
        """Gauges: (h, hu, hv, t) of the given cells (caller ids) at the current time."""
        cells = np.ascontiguousarray(cells, dtype=np.int32)
        n = cells.size
        h, hu, hv = np.empty(n), np.empty(n), np.empty(n)
        t = C.c_double(0)
        self._ck(self._L.swe_sample_cells(self._h, cells.ctypes.data_as(C.POINTER(C.c_int32)), n, _dp(h), _dp(hu), _dp(hv),
                                          C.byref(t)))
        return h, hu, hv, t.value

    def get_stats(self) -> dict:
        s = SweStats()
        self._ck(self._L.swe_get_stats(self._h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in SweStats._fields_}

    def get_permutation(self):
        perm = np.empty(self.nt, dtype=np.int32)
        self._ck(self._L.swe_get_permutation(self._h, perm.ctypes.data_as(C.POINTER(C.c_int32))))
        return perm

    def get_tables(self) -> dict:
        nt = self.nt
        nbr = np.empty((nt, 3), dtype=np.int32)
        normal, length = np.empty((nt, 3, 2)), np.empty((nt, 3))
        area, rin, z = np.empty(nt), np.empty(nt), np.empty(nt)
        self._ck(self._L.swe_get_tables(self._h, nbr.ctypes.data_as(C.POINTER(C.c_int32)),
                                        _dp(normal), _dp(length), _dp(area), _dp(rin), _dp(z)))
        return dict(nbr=nbr, normal=normal, length=length, area=area, inradius=rin, cell_z=z)

    def get_tile_info(self) -> dict:
        tc, mx, mh = C.c_int32(0), C.c_int32(0), C.c_int32(0)
        nti, ne, sm = C.c_int64(0), C.c_int64(0), C.c_size_t(0)
        self._ck(self._L.swe_get_tile_info(self._h, C.byref(tc), C.byref(nti), C.byref(ne), C.byref(mx),
                                           C.byref(mh), C.byref(sm)))
        return dict(tile_cells=tc.value, ntiles=nti.value, nedges=ne.value, max_edges=mx.value,
                    max_halo=mh.value, smem_bytes=sm.value, edges_per_cell=ne.value / self.nt)

    def get_tile_tables(self) -> dict:
        ti = self.get_tile_info()
        ne, stride = ti["nedges"], 4 + ti["max_halo"]
        a = np.empty(ne, dtype=np.int32)
        b = np.empty(ne, dtype=np.int32)
        geom = np.empty((ne, 3), dtype=np.float64)
        tinfo = np.empty((ti["ntiles"], stride), dtype=np.int32)
        i32p = C.POINTER(C.c_int32)
        self._ck(self._L.swe_get_tile_tables(self._h, a.ctypes.data_as(i32p), b.ctypes.data_as(i32p),
                                             _dp(geom), tinfo.ctypes.data_as(i32p)))
        return dict(edge_a=a, edge_b=b, edge_geom=geom, tinfo=tinfo, **ti)

    def get_step_bytes(self, active_tiles, edge_lists, quiet_tiles=0.0) -> float:
        b = C.c_double(0.0)
        self._ck(self._L.swe_get_step_bytes(self._h, float(active_tiles), float(edge_lists), float(quiet_tiles),
                                            C.byref(b)))
        return b.value

    def get_launch_info(self) -> dict:
        g, b, lm, n = C.c_int32(0), C.c_int32(0), C.c_int32(0), C.c_int64(0)
        self._ck(self._L.swe_get_launch_info(self._h, C.byref(g), C.byref(b), C.byref(lm), C.byref(n)))
        return dict(grid=g.value, block=b.value, loop_mode=LOOP_NAMES[lm.value], kernel_launches=n.value)
