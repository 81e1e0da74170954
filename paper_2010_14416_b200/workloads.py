"""Seeded synthetic workloads (meshes, beds, initial states) shaped like the paper's.

This module is the ONLY thing the CPU oracle's tests and the CUDA path share.  It holds
no arithmetic of the method (no flux, no geometry tables, no time stepping): it only
draws random numbers and lays out plain arrays in the paper's mesh-file format
(node table x, y, z; connectivity table of 3 node ids + Manning coefficient per cell,
PAPER.md:296-328 Fig. 4) plus per-local-edge boundary tags.

The meshes stand in for the paper's dam-break canal on a point-grid triangulation
 and its river domains with inflow / outflow, wet channel, dry land
and per-cell Manning; the real river meshes are not public.
Recipe: nx x ny squares of side dx, interior vertices
jittered uniformly by +-0.2 dx, each square split along a seeded random diagonal,
triangles emitted counter-clockwise, cells renumbered by a seeded random permutation.
RNG: numpy default_rng(seed), consumed in the order jitter -> diagonals -> permutation
-> bed -> Manning.

Local edge k of a triangle joins its vertices k and (k+1) mod 3.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BC_WALL = 1          # solid wall
BC_TRANSMISSIVE = 2  # free outflow, U_R = U_L
BC_INFLOW0 = 3       # first prescribed-discharge group; tags >= 3 are inflow groups


@dataclass
class Workload:
    name: str
    nodes_xy: np.ndarray      # [nn, 2] float64
    tris: np.ndarray          # [nt, 3] int32, CCW
    bathymetry: np.ndarray    # [nn] float64, bed elevation per node
    manning: np.ndarray       # [nt] float64, Manning coefficient per cell
    bc_tags: np.ndarray       # [nt, 3] int8, per local edge; read only on boundary edges
    h: np.ndarray             # [nt] initial depth
    hu: np.ndarray            # [nt] initial x-discharge
    hv: np.ndarray            # [nt] initial y-discharge
    g: float = 9.81
    cfl: float = 0.9
    h_dry: float = 1e-6
    nsteps: int = 0
    bc_values: dict = field(default_factory=dict)   # inflow tag -> total discharge m^3/s
    meta: dict = field(default_factory=dict)

    @property
    def ncells(self) -> int:
        return int(self.tris.shape[0])

    @property
    def nnodes(self) -> int:
        return int(self.nodes_xy.shape[0])


# ----------------------------------------------------------------------------------
# mesh
# ----------------------------------------------------------------------------------
def jittered_triangulation(nx: int, ny: int, dx: float, rng, jitter: float = 0.2,
                           permute: bool = True, x0: float = 0.0, y0: float = 0.0):
    """nx x ny squares -> (nodes_xy, tris, ij) with ij the un-jittered grid index per node."""
    ii, jj = np.meshgrid(np.arange(nx + 1), np.arange(ny + 1), indexing="xy")
    ii = ii.ravel()
    jj = jj.ravel()
    xy = np.empty((ii.size, 2), dtype=np.float64)
    xy[:, 0] = x0 + ii * dx
    xy[:, 1] = y0 + jj * dx
    # draw 1: jitter (for every node, then zeroed on the boundary so the domain stays a box)
    jit = rng.uniform(-jitter * dx, jitter * dx, size=xy.shape)
    interior = (ii > 0) & (ii < nx) & (jj > 0) & (jj < ny)
    xy += jit * interior[:, None]
    # draw 2: diagonals
    diag = rng.integers(0, 2, size=nx * ny).astype(bool)
    si, sj = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    si = si.ravel()
    sj = sj.ravel()
    a = (sj * (nx + 1) + si).astype(np.int32)
    b = a + 1
    d = a + (nx + 1)
    c = d + 1
    # diag False: split a-c -> (a,b,c),(a,c,d) ; diag True: split b-d -> (a,b,d),(b,c,d)
    t0 = np.where(diag[:, None], np.stack([a, b, d], 1), np.stack([a, b, c], 1))
    t1 = np.where(diag[:, None], np.stack([b, c, d], 1), np.stack([a, c, d], 1))
    tris = np.empty((2 * nx * ny, 3), dtype=np.int32)
    tris[0::2] = t0
    tris[1::2] = t1
    # draw 3: cell permutation
    if permute:
        perm = rng.permutation(tris.shape[0])
        tris = np.ascontiguousarray(tris[perm])
    ij = np.stack([ii, jj], 1).astype(np.int32)
    return xy, tris, ij


def box_boundary_tags(tris, ij, nx, ny, left=BC_WALL, right=BC_WALL, bottom=BC_WALL,
                      top=BC_WALL):
    """Per-local-edge tags for the four sides of the box; 0 on interior edges."""
    tags = np.zeros(tris.shape, dtype=np.int8)
    for k in range(3):
        na = tris[:, k]
        nb = tris[:, (k + 1) % 3]
        ia, ja = ij[na, 0], ij[na, 1]
        ib, jb = ij[nb, 0], ij[nb, 1]
        tags[(ia == 0) & (ib == 0), k] = left
        tags[(ia == nx) & (ib == nx), k] = right
        tags[(ja == 0) & (jb == 0), k] = bottom
        tags[(ja == ny) & (jb == ny), k] = top
    return tags


def centroids(nodes_xy, tris):
    return (nodes_xy[tris[:, 0]] + nodes_xy[tris[:, 1]] + nodes_xy[tris[:, 2]]) / 3.0


def cell_mean(node_values, tris):
    """Mean of the three node values of each cell, summed in vertex order 0,1,2."""
    return (node_values[tris[:, 0]] + node_values[tris[:, 1]] + node_values[tris[:, 2]]) / 3.0


# ----------------------------------------------------------------------------------
# BASELINE.json configs
# ----------------------------------------------------------------------------------
def canal_dam_break(nx: int, ny: int, *, h_left=1.0, h_right=0.5, manning=0.0, seed=20101,
                    length=100.0, nsteps=500, cfl=0.9, jitter=0.2, permute=True,
                    name="canal") -> Workload:
    """Dam break in a flat canal length x (length*ny/nx), dam at x = length/2, walls all round.

    Shape of the paper's 1-D dam break; depths from BASELINE.json.
    """
    rng = np.random.default_rng(seed)
    dx = length / nx
    xy, tris, ij = jittered_triangulation(nx, ny, dx, rng, jitter=jitter, permute=permute)
    tags = box_boundary_tags(tris, ij, nx, ny)
    cx = centroids(xy, tris)[:, 0]
    h = np.where(cx < 0.5 * length, h_left, h_right).astype(np.float64)
    nt = tris.shape[0]
    return Workload(name=name, nodes_xy=xy, tris=tris, bathymetry=np.zeros(xy.shape[0]),
                    manning=np.full(nt, float(manning)), bc_tags=tags, h=h,
                    hu=np.zeros(nt), hv=np.zeros(nt), cfl=cfl, nsteps=nsteps,
                    meta=dict(nx=nx, ny=ny, dx=dx, length=length, dam_x=0.5 * length,
                              h_left=h_left, h_right=h_right, seed=seed))


def config1(**kw) -> Workload:
    """BASELINE.json configs[0]: wet-wet dam break, 100x10 squares, 2000 cells, 500 steps."""
    args = dict(nx=100, ny=10, h_left=1.0, h_right=0.5, manning=0.0, seed=20101 + 1,
                nsteps=500, name="config1_wetwet_dambreak")
    args.update(kw)
    return canal_dam_break(**args)


def config2(**kw) -> Workload:
    """BASELINE.json configs[1]: wet-dry dam break, 1000x100 squares, 200k cells, n=0.03."""
    args = dict(nx=1000, ny=100, h_left=1.0, h_right=0.0, manning=0.03, seed=20101 + 2,
                nsteps=2000, name="config2_wetdry_dambreak")
    args.update(kw)
    return canal_dam_break(**args)


def config3(nx=2000, ny=1000, *, seed=20101 + 3, nsteps=1000, nbumps=64, stage=2.0,
            permute=True) -> Workload:
    """BASELINE.json configs[2]: lake at rest over 64 Gaussian bumps, some emergent."""
    rng = np.random.default_rng(seed)
    dx = 1.0
    xy, tris, ij = jittered_triangulation(nx, ny, dx, rng, permute=permute)
    tags = box_boundary_tags(tris, ij, nx, ny)
    # draw 4: bed
    amp = rng.uniform(0.1, 1.5, nbumps)
    wid = rng.uniform(5.0, 50.0, nbumps) * dx
    # widths scale with the domain so reduced-size variants keep the same shape
    wid *= min(1.0, nx / 2000.0)
    # centres: clusters of 4 around uniform cluster centres, so that overlapping bumps rise
    # above the stage (no single bump can: 1.5 m < 2.0 m) and form emergent islands
    ncl = (nbumps + 3) // 4
    ccx = np.repeat(rng.uniform(0.0, nx * dx, ncl), 4)[:nbumps]
    ccy = np.repeat(rng.uniform(0.0, ny * dx, ncl), 4)[:nbumps]
    cxb = ccx + rng.normal(0.0, 0.6, nbumps) * wid
    cyb = ccy + rng.normal(0.0, 0.6, nbumps) * wid
    z = np.zeros(xy.shape[0])
    for A, w, x0, y0 in zip(amp, wid, cxb, cyb):
        r2 = (xy[:, 0] - x0) ** 2 + (xy[:, 1] - y0) ** 2
        z += A * np.exp(-r2 / (2.0 * w * w))
    zc = cell_mean(z, tris)
    h = np.maximum(0.0, stage - zc)
    nt = tris.shape[0]
    return Workload(name="config3_lake_at_rest", nodes_xy=xy, tris=tris, bathymetry=z,
                    manning=np.full(nt, 0.025), bc_tags=tags, h=h, hu=np.zeros(nt),
                    hv=np.zeros(nt), cfl=0.9, nsteps=nsteps,
                    meta=dict(nx=nx, ny=ny, dx=dx, stage=stage, seed=seed))


def _value_noise(x, y, rng, base_cell, octaves=5, persistence=0.5):
    """Fractal value noise in [-1, 1]: seeded lattices, smoothstep-bilinear interpolation."""
    out = np.zeros_like(x)
    amp = 1.0
    tot = 0.0
    cell = base_cell
    x0, y0 = x.min(), y.min()
    for _ in range(octaves):
        gx = int(np.ceil((x.max() - x0) / cell)) + 2
        gy = int(np.ceil((y.max() - y0) / cell)) + 2
        lat = rng.uniform(-1.0, 1.0, size=(gy, gx))
        fx = (x - x0) / cell
        fy = (y - y0) / cell
        ix = np.floor(fx).astype(np.int64)
        iy = np.floor(fy).astype(np.int64)
        tx = fx - ix
        ty = fy - iy
        tx = tx * tx * (3.0 - 2.0 * tx)
        ty = ty * ty * (3.0 - 2.0 * ty)
        v00 = lat[iy, ix]
        v10 = lat[iy, ix + 1]
        v01 = lat[iy + 1, ix]
        v11 = lat[iy + 1, ix + 1]
        out += amp * ((v00 * (1 - tx) + v10 * tx) * (1 - ty) + (v01 * (1 - tx) + v11 * tx) * ty)
        tot += amp
        amp *= persistence
        cell *= 0.5
    return out / tot


def config4(nx=5100, ny=1275, *, seed=20101 + 4, nsteps=2000, discharge=500.0,
            permute=True) -> Workload:
    """BASELINE.json configs[3]: river-like domain, meandering channel in fractal terrain."""
    rng = np.random.default_rng(seed)
    dx = 2.0
    xy, tris, ij = jittered_triangulation(nx, ny, dx, rng, permute=permute)
    Lx, Ly = nx * dx, ny * dx
    x, y = xy[:, 0], xy[:, 1]
    # draw 4: bed
    noise = _value_noise(x, y, rng, base_cell=Lx / 16.0)
    slope = 1e-3 * (Lx - x)
    terrain = slope + 2.0 * noise
    Am, lam = 0.25 * Ly, Lx / 3.0

    def dist_to_centreline(px, py):
        yc = 0.5 * Ly + Am * np.sin(2.0 * np.pi * px / lam)
        dyc = Am * 2.0 * np.pi / lam * np.cos(2.0 * np.pi * px / lam)
        return np.abs(py - yc) / np.sqrt(1.0 + dyc * dyc)

    half_w, bank = 20.0 * dx, 4.0 * dx
    d = dist_to_centreline(x, y)
    s = np.clip((half_w + bank - d) / bank, 0.0, 1.0)
    s = s * s * (3.0 - 2.0 * s)                       # 1 in the channel, 0 on the floodplain
    z = (1.0 - s) * terrain + s * (slope - 3.0)
    # draw 5: Manning per cell
    nt = tris.shape[0]
    manning = rng.uniform(0.02, 0.06, nt)
    # initial stage: channel bed + 2.5 m inside the channel band, dry floodplain
    c = centroids(xy, tris)
    zc = cell_mean(z, tris)
    stage = 1e-3 * (Lx - c[:, 0]) - 3.0 + 2.5
    in_channel = dist_to_centreline(c[:, 0], c[:, 1]) < half_w + bank
    h = np.where(in_channel, np.maximum(0.0, stage - zc), 0.0)
    tags = box_boundary_tags(tris, ij, nx, ny, left=BC_WALL, right=BC_TRANSMISSIVE)
    # inflow on left-edge boundary edges whose cell is initially wet (bed below the stage)
    for k in range(3):
        na, nb = tris[:, k], tris[:, (k + 1) % 3]
        on_left = (ij[na, 0] == 0) & (ij[nb, 0] == 0)
        tags[on_left & (h > 0.0), k] = BC_INFLOW0
    return Workload(name="config4_river", nodes_xy=xy, tris=tris, bathymetry=z,
                    manning=manning, bc_tags=tags, h=h, hu=np.zeros(nt), hv=np.zeros(nt),
                    cfl=0.8, nsteps=nsteps, bc_values={BC_INFLOW0: float(discharge)},
                    meta=dict(nx=nx, ny=ny, dx=dx, seed=seed, discharge=discharge))


# config 5: throughput sweep on the canal wet-dry mesh, nx = 10 ny
SWEEP_NY = {"0.1M": 71, "0.5M": 158, "2M": 316, "8M": 632, "13M": 806, "50M": 1581}


def config5(size: str, **kw) -> Workload:
    ny = SWEEP_NY[size]
    args = dict(nx=10 * ny, ny=ny, h_left=1.0, h_right=0.0, manning=0.03, seed=20101 + 5,
                nsteps=200, name=f"config5_sweep_{size}")
    args.update(kw)
    return canal_dam_break(**args)


# ----------------------------------------------------------------------------------
# locally refined mesh (the paper refines its river meshes around
# bridge piers)
# ----------------------------------------------------------------------------------
def refined_basin(nx=240, ny=120, *, a=0.85, seed=20101 + 6, length=240.0, manning=0.03,
                  nsteps=800) -> Workload:
    """Walled basin whose cell size varies 12:1 (a = 0.85): the jittered triangulation is mapped by
    x' = x + a L/(2 pi) sin(2 pi x / L) (and the same in y), which is monotone for a < 1, so the
    smallest cells sit around the domain centre like a refinement patch.  Two Gaussian bumps on
    the bed, a column of water released next to the fine region, Manning friction."""
    rng = np.random.default_rng(seed)
    dx = length / nx
    xy, tris, ij = jittered_triangulation(nx, ny, dx, rng)
    Lx, Ly = nx * dx, ny * dx
    two_pi = 2.0 * np.pi
    xy = np.stack([xy[:, 0] + a * Lx / two_pi * np.sin(two_pi * xy[:, 0] / Lx + np.pi),
                   xy[:, 1] + a * Ly / two_pi * np.sin(two_pi * xy[:, 1] / Ly + np.pi)], 1)
    tags = box_boundary_tags(tris, ij, nx, ny)
    z = 0.4 * np.exp(-((xy[:, 0] - 0.35 * Lx) ** 2 + (xy[:, 1] - 0.6 * Ly) ** 2) / (2 * (0.06 * Lx) ** 2)) \
        + 0.9 * np.exp(-((xy[:, 0] - 0.7 * Lx) ** 2 + (xy[:, 1] - 0.4 * Ly) ** 2) / (2 * (0.05 * Lx) ** 2))
    c = centroids(xy, tris)
    zc = cell_mean(z, tris)
    r2 = (c[:, 0] - 0.45 * Lx) ** 2 + (c[:, 1] - 0.5 * Ly) ** 2
    stage = np.where(r2 < (0.12 * Lx) ** 2, 1.6, 0.5)
    h = np.maximum(0.0, stage - zc)
    nt = tris.shape[0]
    return Workload(name="refined_basin", nodes_xy=np.ascontiguousarray(xy), tris=tris, bathymetry=z,
                    manning=np.full(nt, float(manning)), bc_tags=tags, h=h, hu=np.zeros(nt),
                    hv=np.zeros(nt), cfl=0.9, nsteps=nsteps,
                    meta=dict(nx=nx, ny=ny, dx=dx, a=a, seed=seed))


# ----------------------------------------------------------------------------------
# small meshes for unit tests
# ----------------------------------------------------------------------------------
def two_triangles(h_lower=1.0, h_upper=0.5) -> Workload:
    """Unit square split on the diagonal (0,0)-(1,1); walls all round; flat bed.

    Cell 0 = (0,0),(1,0),(1,1) (below the diagonal), cell 1 = (0,0),(1,1),(0,1).
    """
    xy = np.array([[0.0, 0.0], [1.0, 0.0], [1.0, 1.0], [0.0, 1.0]])
    tris = np.array([[0, 1, 2], [0, 2, 3]], dtype=np.int32)
    tags = np.array([[BC_WALL, BC_WALL, 0], [0, BC_WALL, BC_WALL]], dtype=np.int8)
    return Workload(name="two_triangles", nodes_xy=xy, tris=tris, bathymetry=np.zeros(4),
                    manning=np.zeros(2), bc_tags=tags, h=np.array([h_lower, h_upper]),
                    hu=np.zeros(2), hv=np.zeros(2), nsteps=1)


def mirrored_canal(nx=40, ny_half=4, *, seed=7, length=40.0, h_left=1.0, h_right=0.5,
                   manning=0.0) -> Workload:
    """Canal whose mesh is the reflection of a jittered half-mesh about y = 0.

    Returns cells ordered so that cell i (upper half) mirrors cell i + nt/2 (lower half).
    """
    rng = np.random.default_rng(seed)
    dx = length / nx
    xy, tris, ij = jittered_triangulation(nx, ny_half, dx, rng, permute=False)
    # un-jitter the axis row (j == 0) stays on y = 0 already (boundary nodes are not moved)
    nn = xy.shape[0]
    on_axis = ij[:, 1] == 0
    mirror_id = np.where(on_axis, np.arange(nn), nn + np.cumsum(~on_axis) - 1).astype(np.int32)
    xy_m = xy[~on_axis].copy()
    xy_m[:, 1] *= -1.0
    xy_all = np.vstack([xy, xy_m])
    tris_m = mirror_id[tris][:, [0, 2, 1]]           # reflection flips orientation
    tris_all = np.vstack([tris, tris_m]).astype(np.int32)
    ij_all = np.vstack([ij, np.stack([ij[~on_axis, 0], -ij[~on_axis, 1]], 1)])
    nt = tris_all.shape[0]
    tags = np.zeros((nt, 3), dtype=np.int8)
    for k in range(3):
        na, nb = tris_all[:, k], tris_all[:, (k + 1) % 3]
        ia, ja, ib, jb = ij_all[na, 0], ij_all[na, 1], ij_all[nb, 0], ij_all[nb, 1]
        bnd = ((ia == 0) & (ib == 0)) | ((ia == nx) & (ib == nx)) | \
              ((ja == ny_half) & (jb == ny_half)) | ((ja == -ny_half) & (jb == -ny_half))
        tags[bnd, k] = BC_WALL
    cx = centroids(xy_all, tris_all)[:, 0]
    h = np.where(cx < 0.5 * length, h_left, h_right).astype(np.float64)
    return Workload(name="mirrored_canal", nodes_xy=xy_all, tris=tris_all,
                    bathymetry=np.zeros(xy_all.shape[0]), manning=np.full(nt, float(manning)),
                    bc_tags=tags, h=h, hu=np.zeros(nt), hv=np.zeros(nt), nsteps=100,
                    meta=dict(nx=nx, ny_half=ny_half, dx=dx, length=length))


def rotated(w: Workload, angle: float) -> Workload:
    """The same workload with mesh and discharge vectors rotated by `angle` about the origin."""
    c, s = np.cos(angle), np.sin(angle)
    R = np.array([[c, -s], [s, c]])
    xy = w.nodes_xy @ R.T
    hu = c * w.hu - s * w.hv
    hv = s * w.hu + c * w.hv
    return Workload(name=w.name + "_rot", nodes_xy=np.ascontiguousarray(xy), tris=w.tris,
                    bathymetry=w.bathymetry, manning=w.manning, bc_tags=w.bc_tags, h=w.h,
                    hu=hu, hv=hv, g=w.g, cfl=w.cfl, h_dry=w.h_dry, nsteps=w.nsteps,
                    bc_values=dict(w.bc_values), meta=dict(w.meta))
