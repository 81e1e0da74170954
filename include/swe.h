/*
 * swe.h -- C ABI of libswe_b200: the time-explicit cell-centred finite-volume step of the
 * 2-D Shallow-Water Equations on an unstructured triangular mesh, FP64, one B200 (sm_100a).
 *
 * Method: Delmas & Soulaimani, arXiv 2010.14416, sections 2-3:
 *   state U = (h, hu, hv) per triangle (eq.1), explicit Euler finite volumes
 *   (eq.6-16), HLLC flux per edge in the rotated frame (PAPER.md:111-123
 *   eq.12-14, :141-189 eq.17-26), bathymetry by hydrostatic reconstruction (PAPER.md:196-217
 *   eq.28-30), semi-implicit Manning friction (eq.31-37), boundary fluxes
 *   (PAPER.md:125), CFL time step with the inscribed-circle radius (eq.15)
 *   reduced on the device.  Readings of garbled passages: DESIGN.md section 4.
 *
 * Conventions
 *   - Every function returns SWE_OK (0) or a negative swe_status; nothing throws across the
 *     ABI.  swe_last_error(mesh) gives a message for the last failure on that handle
 *     (swe_last_error(NULL): last failure of a call without a handle in this thread).
 *   - "host" pointers are ordinary CPU memory, caller-owned, read or written during the call
 *     only.  "device" pointers are CUDA device memory of the bound device, caller-owned.
 *   - Cells are addressed in the CALLER's numbering everywhere in this ABI; the internal
 *     locality renumbering (swe_params.ordering) is invisible except via swe_get_permutation.
 *   - Local edge k (0,1,2) of a triangle joins its vertices k and (k+1) mod 3.
 *   - A handle is not thread-safe.  All device work is issued on the stream given to
 *     swe_mesh_bind_device; swe_step / swe_run are asynchronous on that stream.
 *   - There is no CPU fallback: every compute entry point fails with SWE_ERR_NOT_BOUND or
 *     SWE_ERR_CUDA when no device workspace is bound or CUDA is unavailable.
 */
#ifndef SWE_B200_H
#define SWE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct swe_mesh swe_mesh; /* opaque */

typedef enum {
    SWE_OK = 0,
    SWE_ERR_INVALID_ARG = -1,   /* NULL pointer, non-positive size, bad enum value */
    SWE_ERR_BAD_INDEX = -2,     /* triangle refers to a node outside [0, nn) */
    SWE_ERR_DEGENERATE = -3,    /* zero-area triangle */
    SWE_ERR_NON_MANIFOLD = -4,  /* an edge is shared by more than two triangles */
    SWE_ERR_BAD_VALUE = -5,     /* NaN/inf coordinate, bed or state; negative Manning or depth */
    SWE_ERR_NOT_BOUND = -6,     /* no device workspace bound yet */
    SWE_ERR_WORKSPACE = -7,     /* workspace too small or misaligned */
    SWE_ERR_CUDA = -8,          /* a CUDA call failed (message in swe_last_error) */
    SWE_ERR_ALL_DRY = -9,       /* every cell is dry: no time step can be defined */
    SWE_ERR_NO_STATE = -10,     /* swe_set_state has not been called */
    SWE_ERR_BAD_TAG = -11,      /* boundary tag out of range or without edges */
    SWE_ERR_NOMEM = -12,
    SWE_ERR_IO = -13,           /* a mesh file cannot be opened */
    SWE_ERR_FORMAT = -14        /* a mesh file does not follow the layout of PAPER.md Fig. 4 */
} swe_status;

/* boundary tags of bc_tags */
enum { SWE_BC_WALL = 1, SWE_BC_TRANSMISSIVE = 2, SWE_BC_INFLOW0 = 3, SWE_BC_MAX_TAG = 127 };
/* swe_params.ordering: create-time renumbering of the cells for gather locality */
enum { SWE_ORDER_IDENTITY = 0, SWE_ORDER_HILBERT = 1, SWE_ORDER_RCM = 2 };
/* swe_params.riemann: HLLC (the paper's scheme) or plain HLL for all three
 * components (eq.17-18) */
enum { SWE_RIEMANN_HLLC = 0, SWE_RIEMANN_HLL = 1 };
/* swe_params.kernel: TILED = the fused tile kernel (one launch per step: every edge of a tile once in
 * shared memory, then the tile's cells); EDGE_TWO_PASS = the edge-centric alternative the paper's text
 * leaves open: pass 1, one thread per edge of the mesh, writes the edge's
 * length-weighted flux + sources for both sides to HBM; pass 2, one thread per cell, adds its three
 * edges in the order k = 0,1,2 and does friction, update and rate.  Same arithmetic, same results;
 * more HBM traffic, no shared-memory scatter (A/B in profiles/).  No dry-tile shortcut, GRAPH or
 * LAUNCH loop only. */
enum { SWE_KERNEL_TILED = 0, SWE_KERNEL_EDGE_TWO_PASS = 1 };
/* swe_params.fp_kind: the paper's floating-point kind is a parameter of its code.  FP64 =
 * everything in double precision (north_star; the only kind the 1e-10 parity bar applies to).
 * MIXED32 = the state records {h, u, v, z} live in HBM in single precision (16 bytes per cell instead of
 * 32); every step converts them to double on load, does all of its arithmetic in double and rounds the new
 * state on store.  Only with SWE_KERNEL_EDGE_TWO_PASS.  Agreement with the FP64 result is at the level
 * of single-precision round-off accumulated over the steps (DESIGN.md section 9 derives the bar). */
enum { SWE_FP64 = 0, SWE_FP_MIXED32 = 1 };
/* swe_params.loop_mode: how swe_run iterates without host round trips: GRAPH = CUDA graphs of
 * 128 / 16 / 2 step-kernel launches, PERSISTENT = one cooperative launch with a grid barrier per
 * step, LAUNCH = plain launches, CLUSTER = meshes of at most 16 tiles only: one launch of one
 * thread-block cluster, one CTA per tile, state resident in shared memory for the whole run, halo
 * records through distributed shared memory, the hardware cluster barrier per step (PAPER.md:517:
 * small meshes are "strictly limited by latencies").  AUTO = CLUSTER when the mesh fits (with
 * block_size 0: tiles of 128 cells, up to 2048 cells), else GRAPH (as fast as or faster than
 * PERSISTENT at every larger mesh size).  All modes give bit-identical results. */
enum { SWE_LOOP_AUTO = 0, SWE_LOOP_GRAPH = 1, SWE_LOOP_PERSISTENT = 2, SWE_LOOP_LAUNCH = 3, SWE_LOOP_CLUSTER = 4 };

typedef struct {
    double g;           /* gravitational acceleration; the paper gives no value, default 9.81 */
    double cfl;         /* CFL number of eq.(15); default 0.9 */
    double h_dry;       /* wet/dry threshold: a cell or edge side is dry iff h <= h_dry; 1e-6.
                           Values below 1e-250 act as 1e-250 (keeps every rsqrt argument normal) */
    int32_t ordering;   /* SWE_ORDER_*; default SWE_ORDER_HILBERT */
    int32_t block_size; /* cells per tile (= CUDA threads per block, twice that in CLUSTER mode): 64, 128, 192 or
                           256; 0 = default (192; 128 for meshes that AUTO runs in CLUSTER mode) */
    int32_t loop_mode;  /* SWE_LOOP_*; default SWE_LOOP_AUTO */
    int32_t riemann;    /* SWE_RIEMANN_*; default SWE_RIEMANN_HLLC */
    int32_t kernel;     /* SWE_KERNEL_*; default SWE_KERNEL_TILED */
    int32_t fp_kind;    /* SWE_FP_*; default SWE_FP64 */
} swe_params;

typedef struct {
    double volume;        /* sum_i h_i |Omega_i| (m^3): fixed-tree partial sums on the device, added on the host */
    double t;             /* simulated time */
    double dt_last;       /* time step used by the most recent step (0 before the first) */
    int64_t steps;        /* steps taken since swe_set_state */
    int64_t n_dry;        /* cells with h <= h_dry */
    int64_t n_clamped;    /* times a negative depth was clamped to 0 (R-15; expected 0) */
    int64_t n_nonfinite;  /* cells whose state is NaN/inf (expected 0) */
    int64_t active_tile_steps; /* sum over the steps since swe_set_state of the number of tiles that were
                                  not all dry (tile + halo dry, no inflow edge: such tiles copy their
                                  records and skip the arithmetic) */
    int64_t edge_list_fetches; /* sum over the steps of the number of tile edge lists read from HBM (the list of
                                  a tile that was all dry at the previous step is read only if the tile turns
                                  out active): with active_tile_steps it fixes the bytes a step requests */
    int64_t quiet_tile_steps;  /* sum over the steps of the number of QUIET tiles: inactive in the previous step with
                                  all their neighbour tiles, hence all dry now, and with their records already in
                                  place in both state buffers: they are not touched */
    int64_t stolen_tile_steps; /* sum over the steps of the number of tiles computed by a thread block other than the
                                  one they are dealt to (work stealing); results do not depend on it */
} swe_stats;

/* Fills *p with the defaults listed above. */
int swe_params_default(swe_params *p);

/*
 * Builds the mesh tables on the host (Fig. 4 gives the input format: node
 * table x, y, z and connectivity table of three node ids + Manning coefficient per cell).
 *   nodes_xy    host [nn][2]  node coordinates (m)
 *   tris        host [nt][3]  node ids per triangle; clockwise triangles are re-oriented by
 *                             swapping vertices 1 and 2 (their edge tags follow)
 *   bathymetry  host [nn]     bed elevation z per node; the cell bed is the mean of its three
 *                             node values (R-1)
 *   manning     host [nt]     Manning coefficient m per cell, >= 0 (eq.5)
 *   bc_tags     host [nt][3]  boundary tag per local edge, read only where the edge has no
 *                             neighbour; <= 0 or missing means SWE_BC_WALL
 *   params      host          NULL = defaults
 * Tables built (in the internal cell order): per-tile edge lists (end points, length-scaled normal),
 * halo lists, 1 / |Omega_i|, 1 / R_i, g m^2, cell bed.  nt < 2^29.  No CUDA call is made.
 */
int swe_mesh_create(const double *nodes_xy, int64_t nn, const int32_t *tris, int64_t nt,
                    const double *bathymetry, const double *manning, const int8_t *bc_tags,
                    const swe_params *params, swe_mesh **out);

/*
 * Reads a mesh file in the paper's layout (Fig. 4): a title line, the number of
 * nodes on its own line, one row "id x y z" per node; a title line, the number of cells, one row
 * "id n1 n2 n3 manning" per cell.  Ids are 1-based in the file and 0-based in the arrays; rows may
 * come in any order.  What follows the connectivity table (the "Ghost cells to be sent / received"
 * block lists of the paper's multi-GPU decomposition) is ignored.  The file carries no boundary
 * tags (the paper flags inflow nodes separately): pass your own bc_tags to
 * swe_mesh_create, or zeros for solid walls.
 * Call once with all four arrays NULL to get *nn and *nt, allocate, call again:
 *   nodes_xy host [nn][2], bathymetry host [nn], tris host [nt][3], manning host [nt] (any may be NULL)
 * Errors: SWE_ERR_IO, SWE_ERR_FORMAT (message with the line number in swe_last_error(NULL)).
 */
int swe_mesh_file_read(const char *path, int64_t *nn, int64_t *nt, double *nodes_xy,
                       double *bathymetry, int32_t *tris, double *manning);

/* Frees the host tables and CUDA graphs.  Never frees the caller's device workspace. */
int swe_mesh_destroy(swe_mesh *mesh);

/* Bytes of device memory the mesh needs (tables + two state buffers + staging). */
int swe_mesh_workspace_bytes(const swe_mesh *mesh, size_t *bytes);

/*
 * Binds caller-provided device memory (>= workspace bytes, 256-byte aligned, on the current
 * CUDA device) and a CUDA stream (cudaStream_t as void*, NULL = default stream), uploads the
 * tables.  The memory must stay valid until swe_mesh_destroy or a new bind.
 */
int swe_mesh_bind_device(swe_mesh *mesh, void *device_workspace, size_t bytes, void *cuda_stream);

/*
 * Prescribed inflow (R-20): total discharge Q (m^3/s, positive into the domain)
 * over all boundary edges carrying `tag` (>= SWE_BC_INFLOW0); each edge gets the unit
 * discharge -Q / sum(L) along its outward normal.  Call after swe_mesh_create, any time.
 */
int swe_set_bc_value(swe_mesh *mesh, int tag, double total_discharge);

/*
 * Sets U = (h, hu, hv) and the time.  host / device [nt] each, caller numbering.  Requires
 * h >= 0 and finite values (both variants check this on the device while converting; on
 * SWE_ERR_BAD_VALUE the handle is left without a state).  Momentum of dry cells (h <= h_dry)
 * is discarded (R-15).  Resets the step counter and the boundary volumes; the time step becomes stale.
 */
int swe_set_state(swe_mesh *mesh, const double *h, const double *hu, const double *hv, double t0);
int swe_set_state_device(swe_mesh *mesh, const double *d_h, const double *d_hu, const double *d_hv,
                         double t0);

/*
 * Time step of the CURRENT state, eq.(15) with d = R_i, reduced on the device
 * (PAPER.md:457): dt = CFL / max_i (sqrt(g h_i) + |V_i|) / R_i over wet cells.  Synchronises the
 * stream.  Leaves dt on the device for the next step.  SWE_ERR_ALL_DRY if no cell is wet.
 */
int swe_compute_dt(swe_mesh *mesh, double *dt_out);

/* One step (eq.37) with the device-resident dt, then the next dt. = swe_run(mesh, 1) */
int swe_step(swe_mesh *mesh);

/*
 * nsteps steps, asynchronous, no host<->device traffic inside: each step gathers the three
 * neighbours, computes the three edge fluxes with sources and friction, writes U^{n+1} to the
 * other state buffer and the per-block maximum of (sqrt(g h)+|V|)/R for the next dt.
 * If the domain becomes all dry the remaining steps leave the state unchanged (dt = 0).
 */
int swe_run(swe_mesh *mesh, int64_t nsteps);

/*
 * Steps until the simulated time reaches t_end (the paper specifies its runs by simulated time,
 * PAPER.md:541, :611): the step that would pass t_end is shortened to end on it.  At most
 * max_steps steps.  *steps_done (may be NULL) = steps actually taken.  Synchronises the stream
 * (the host looks at the device clock between batches of steps; the steps themselves never leave
 * the device).  Stops early if the domain becomes all dry.
 */
int swe_run_until(swe_mesh *mesh, double t_end, int64_t max_steps, int64_t *steps_done);

/*
 * Boundary discharge diagnostics (inflow / outflow rates are accumulated every step).
 * volume_by_tag host [SWE_BC_MAX_TAG + 1]: volume (m^3) that has LEFT the domain through the
 * boundary edges of each tag since swe_set_state = sum over steps and edges of dt L G~_1
 * (negative = entered: an inflow tag with discharge Q reads -Q t; walls read 0).  Each boundary
 * edge has one device accumulator with a single writer, summed here on the host in edge order,
 * so the result is deterministic.  Synchronises the stream.
 */
int swe_get_boundary_volumes(swe_mesh *mesh, double *volume_by_tag);

/* Waits for the stream. */
int swe_sync(swe_mesh *mesh);

/*
 * Reads the state back in caller numbering.  Any of h, hu, hv, t, dt_next may be NULL.
 * dt_next is the step the next swe_step would use (0 if all dry).  Synchronises the stream.
 */
int swe_get_state(swe_mesh *mesh, double *h, double *hu, double *hv, double *t, double *dt_next);
int swe_get_state_device(swe_mesh *mesh, double *d_h, double *d_hu, double *d_hv);

/*
 * Asynchronous snapshot (PAPER.md:453 uses a side stream for its per-step diagnostics): the
 * current state is converted on the mesh's stream and then copied to the host buffers on a side
 * stream, while steps queued after this call run concurrently.  h, hu, hv host [nt] (pinned
 * memory for a truly asynchronous copy), t host (may be NULL): valid after swe_snapshot_wait (or
 * the next swe_snapshot_begin / swe_get_state / swe_set_state / swe_mesh_destroy on this handle,
 * which wait for it).  One snapshot can be pending per handle.
 */
int swe_snapshot_begin(swe_mesh *mesh, double *h, double *hu, double *hv, double *t);
int swe_snapshot_wait(swe_mesh *mesh);

/*
 * Gauges: (h, hu, hv) of n cells, given by their caller ids, at the current time -- a water-level or discharge
 * record at fixed points costs 28 bytes per gauge instead of a read-back of the whole state (the paper streams
 * its per-step diagnostics to the host beside the computation).  The values are the ones
 * swe_get_state returns for those cells, bit for bit.
 *   cells host [n], 0 <= id < nt, 1 <= n <= max(1, nt / 2);  h, hu, hv host [n];  t may be NULL
 * Synchronises the stream; waits for a pending snapshot (the samples pass through the same staging buffer).
 * Errors: SWE_ERR_INVALID_ARG, SWE_ERR_BAD_INDEX (id out of range), SWE_ERR_NOT_BOUND, SWE_ERR_NO_STATE.
 */
int swe_sample_cells(swe_mesh *mesh, const int32_t *cells, int64_t n, double *h, double *hu, double *hv,
                     double *t);

/* Diagnostics (synchronises, copies h to the host). */
int swe_get_stats(swe_mesh *mesh, swe_stats *stats);

/* perm[p] = caller's cell id stored at internal position p.  host [nt]. */
int swe_get_permutation(const swe_mesh *mesh, int32_t *perm);

/*
 * Host tables in caller numbering, for tests of the mesh builder; any pointer may be NULL.
 *   nbr [nt][3] neighbour cell id, or -tag on a boundary edge
 *   normal [nt][3][2], length [nt][3], area [nt], inradius [nt], cell_z [nt]
 */
int swe_get_tables(const swe_mesh *mesh, int32_t *nbr, double *normal, double *length,
                   double *area, double *inradius, double *cell_z);

/*
 * Tile decomposition of the step kernel: the internal cell order is cut
 * into tiles of tile_cells consecutive cells (= swe_params.block_size); every edge touching a
 * tile is listed once in that tile (an edge between two tiles is listed in both, so
 * nedges / nt >= 1.5 measures the locality of the ordering).  max_edges / max_halo: longest edge
 * list (rounded up to an even count) / halo list of any tile; smem_bytes: dynamic shared memory per block.  Any pointer may be NULL.
 */
int swe_get_tile_info(const swe_mesh *mesh, int32_t *tile_cells, int64_t *ntiles, int64_t *nedges,
                      int32_t *max_edges, int32_t *max_halo, size_t *smem_bytes);

/*
 * Bytes one time step REQUESTS from device memory, from the library's own table sizes, given how
 * many tiles are active (not all dry), how many tile edge lists are fetched and how many tiles are
 * quiet (not touched) in that step (per-step averages taken from swe_stats.
 * active_tile_steps / edge_list_fetches / quiet_tile_steps): the 32-byte record in and out of every
 * cell of a tile that is not quiet, one 32-byte sector per halo record of such a tile, tile headers + halo ids,
 * activity flags and neighbour-tile rows,
 * 24 bytes of cell constants per cell of an active tile, 24 bytes per edge of a fetched list (mean
 * list length).  This is the kernel's request stream, not a DRAM counter: L2 hits on the halo
 * records make the DRAM traffic smaller (bench.py reports it as roofline.traffic; the cross-check
 * against ncu's dram__bytes is in profiles/).
 */
int swe_get_step_bytes(const swe_mesh *mesh, double active_tiles, double edge_lists, double quiet_tiles,
                       double *bytes);

/*
 * The tile tables themselves, for tests of the mesh builder; any pointer may be NULL.
 *   edge_a, edge_b [nedges]   end points: bits 0-28 = position in the tile's record array (local
 *                             cell index if < tile_cells, else tile_cells + index into the tile's
 *                             halo list), bits 29-30 = local edge index in that cell; on a boundary
 *                             edge edge_b = -(tag + 128 * boundary edge number); a is the end point
 *                             with the smaller caller id
 *   edge_geom [nedges][3]     a's unit outward normal (n1, n2) and the edge length
 *   tinfo [ntiles][4+max_halo] {first edge, #edges, #halo ids, 1 if the tile has an inflow edge,
 *                             halo ids (internal), -1 padding}
 */
int swe_get_tile_tables(const swe_mesh *mesh, int32_t *edge_a, int32_t *edge_b, double *edge_geom,
                        int32_t *tinfo);

/* Launch facts for reporting: grid, block, loop mode actually in use, kernel launches issued
 * by this handle so far (step, rate, pack/unpack kernels). */
int swe_get_launch_info(const swe_mesh *mesh, int32_t *grid, int32_t *block, int32_t *loop_mode,
                        int64_t *kernel_launches);

/*
 * The CFL time step of eq.(15) WITHOUT a handle, a workspace or any
 * allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, serving loops,
 * harnesses that forbid it): dt = cfl / max_i (sqrt(g h_i) + |(hu_i, hv_i)| / h_i) / inradius_i over
 * the cells with h_i > h_dry, 0 if there is none.  The same quantity swe_compute_dt returns for that
 * state (equal to rounding: the handle-based path stores velocities and 1/R).
 *   d_h, d_hu, d_hv, d_inradius   device [n], any cell order (inradius as swe_get_tables returns it)
 *   d_dt                          device, one double, written on the stream
 *   cuda_stream                   cudaStream_t (NULL: the default stream); nothing is synchronised
 * The per-block partial maxima live in a fixed device array inside the library (512 KiB per GPU that
 * loads it, held until exit) sized for n <= SWE_STATIC_MAX_CELLS; a larger n is rejected with
 * SWE_ERR_INVALID_ARG and a message in swe_last_error(NULL).  All calls share that array: calls that
 * overlap on the GPU (different streams, no dependency between them) race on it; calls on one stream
 * are safe, and a call does not depend on what the previous one left there.  Works on the device
 * that is current at the call.  Calls no cudaMalloc / cudaFree / allocating routine.
 * Errors: SWE_ERR_INVALID_ARG, SWE_ERR_CUDA (launch failure; message in swe_last_error(NULL)).
 */
#define SWE_STATIC_MAX_CELLS 67108864   /* 2^26 cells (the largest workload of the paper's kind here has 50M) */
int swe_cfl_dt_static(const double *d_h, const double *d_hu, const double *d_hv, const double *d_inradius,
                      int64_t n, double g, double cfl, double h_dry, double *d_dt, void *cuda_stream);

const char *swe_last_error(const swe_mesh *mesh);

#ifdef __cplusplus
}
#endif
#endif /* SWE_B200_H */
