// libswe_b200: C ABI (include/swe.h), kernels and the device-resident time loop.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "mesh_builder.h"
#include "swe_kernels.cuh"

namespace cg = cooperative_groups;
using namespace swe;

// =================================================================================================
// kernels
// =================================================================================================
namespace {

constexpr int kDefaultBlock = 192;   // cells per tile = threads per block (best of 128/192/256 on B200)
constexpr int kMaxBlock = 256;
#ifndef SWE_MIN_BLOCKS
#define SWE_MIN_BLOCKS 3
#endif
constexpr int kMaxPart = 8192;       // upper bound on the grid of the step kernel
extern __shared__ __align__(128) unsigned char dyn_smem[];

// nsteps time steps.  Every block first reduces the per-block maxima of the previous step into
// dt (redundantly: a few KB from L2), so no separate finaliser launch and no atomics sit between
// two steps; block 0 advances the device clock.  Blocks walk the tiles with a stride of the grid
// through the TMA pipeline of swe_kernels.cuh.  TC = cells per tile = threads per block.
//   graph / launch mode: nsteps = 1 per launch, the kernel boundary separates the steps;
//   persistent mode: one cooperative launch runs the whole loop with a grid barrier between
//   steps (small meshes are "strictly limited by latencies" of kernel launches).
// One kernel serves all modes, so their results are bitwise identical by construction.
template <int TC>
__global__ void __launch_bounds__(TC, (SWE_MIN_BLOCKS * kMaxBlock) / TC)
swe_step_kernel(const Params P, int cur, const long long nsteps)
{
    __shared__ double s_red[32];
    if (threadIdx.x == 0) {
        uint64_t *bar = reinterpret_cast<uint64_t *>(dyn_smem + SmemLayout<TC>::bar);
        for (int s = 0; s < kNumBars; s++) mbar_init(bar + s, 1);
        for (int q = 0; q < 4; q++) reinterpret_cast<unsigned *>(bar + kNumBars)[q] = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    PipeState it;
    for (long long s = 0; s < nsteps; s++) {
        // (these loads are in flight during the reduction below)
        const int ninact = ldcg_i32(P.binact + blockIdx.x);
        const double t_now = __ldcg(&P.ctrl->t[cur]), t_end = __ldcg(&P.ctrl->t_end);
        const double dt_cfl = reduce_dt(P, P.pmax(cur), s_red);
        // swe_run_until: the step that would pass t_end ends on it; after that, zero steps
        const double left = t_end - t_now;
        const bool clipped = dt_cfl >= left;
        const double dt = fmax(clipped ? left : dt_cfl, 0.0);
        unsigned nclamp = 0;
        // quiet tiles are looked for when at least a quarter of the block's tiles were inactive a step ago
        // and the block has enough tiles to repay the look (flags, a barrier, the scan)
        const int nmy = (int)blockIdx.x < P.ntiles ? (P.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
        double rate = 4 * ninact >= nmy && nmy >= 8 ? step_tiles<TC, true>(P, dyn_smem, cur, dt, nclamp, it)
                                                      : step_tiles<TC, false>(P, dyn_smem, cur, dt, nclamp, it);
        rate = block_max(rate, s_red);
        if (nclamp) atomicAdd(&P.ctrl->n_clamped, (unsigned long long)nclamp);   // diagnostics only
        if (threadIdx.x == TC - 32) {                                            // likewise (the producer thread's counters)
            unsigned *cnt = reinterpret_cast<unsigned *>(dyn_smem + SmemLayout<TC>::bar) + 2 * kNumBars;
            if (cnt[0]) { atomicAdd(&P.ctrl->n_active, (unsigned long long)cnt[0]); cnt[0] = 0; }
            if (cnt[1]) { atomicAdd(&P.ctrl->n_elists, (unsigned long long)cnt[1]); cnt[1] = 0; }
            if (cnt[2]) { atomicAdd(&P.ctrl->n_quiet, (unsigned long long)cnt[2]); cnt[2] = 0; }
            P.binact[blockIdx.x] = (int)cnt[3]; cnt[3] = 0;
            const int nst = reinterpret_cast<const ClaimState *>(dyn_smem + SmemLayout<TC>::ring + 16)->stolen;
            if (nst > 0 && (int)blockIdx.x < P.ntiles) atomicAdd(&P.ctrl->n_stolen, (unsigned long long)nst);
        }
        if (threadIdx.x == 0) {
            P.pmax(cur ^ 1)[blockIdx.x] = rate;
            if (blockIdx.x == 0) {
                Ctrl *c = P.ctrl;
                // R-24: the clipped step ends ON t_end (t + (t_end - t) may round off it)
                c->t[cur ^ 1] = clipped ? fmax(t_end, t_now) : t_now + dt;
                if (dt > 0.0) { c->dt_last = dt; c->steps += 1; }
                if (!(dt_cfl > 0.0)) c->all_dry = 1;
            }
        }
        cur ^= 1;
        if (s + 1 < nsteps) {     // only reached in a cooperative launch
            // the next step's bulk copies (async proxy) read what this step's threads stored
            asm volatile("fence.proxy.async;" ::: "memory");
            cg::this_grid().sync();
        }
    }
}

// ---- edge-centric two-pass alternative (SWE_KERNEL_EDGE_TWO_PASS) -------------
// The time step of a launch: dt = CFL / max of the per-block maxima, clipped to t_end (swe_run_until).
__device__ __forceinline__ double launch_dt(const Params &P, const int cur, double *s_red, double &dt_cfl,
                                            double &t_now, bool &clipped)
{
    dt_cfl = reduce_dt(P, P.pmax(cur), s_red);
    t_now = __ldcg(&P.ctrl->t[cur]);
    const double left = __ldcg(&P.ctrl->t_end) - t_now;
    clipped = dt_cfl >= left;
    return fmax(clipped ? left : dt_cfl, 0.0);
}

// pass 1: one thread per edge of the mesh (a2-a7): both end points' records are gathered from HBM / L2
// (one 32-byte sector each), the result for each side is written once
template <class R>
__global__ void __launch_bounds__(256)
swe_edge_pass_kernel(const Params P, const int cur)
{
    __shared__ double s_red[32];
    double dt_cfl, t_now; bool clipped;
    const double dt = launch_dt(P, cur, s_red, dt_cfl, t_now, clipped);
    const R *__restrict__ U = reinterpret_cast<const R *>(P.U(cur));
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < P.nge; e += (long long)gridDim.x * blockDim.x) {
        const int2 ab = __ldg(reinterpret_cast<const int2 *>(P.gedges + e));
        const double2 l = make_double2(__ldg(&P.gedges[e].lx), __ldg(&P.gedges[e].ly));   // 24-byte records: 8-byte aligned
        const Rec A = ldrec<R>(U + ab.x);
        Rec B = A;
        if (ab.y >= 0) B = ldrec<R>(U + ab.y);
        double o[5];
        edge_eval(P, l.x, l.y, A, B, ab.y, dt, o);
        double2 *r = reinterpret_cast<double2 *>(P.eres + 6 * e);
        r[0] = make_double2(o[0], o[1]);
        r[1] = make_double2(o[2], -o[0]);
        r[2] = make_double2(-o[3], -o[4]);
    }
}

// pass 2: one thread per cell (a7-a11): its three edge results in the order k = 0,1,2, friction,
// update, local rate; per-block maximum; block 0 advances the device clock
template <class R>
__global__ void __launch_bounds__(256)
swe_cell_pass_kernel(const Params P, const int cur, const int tile_cells)
{
    __shared__ double s_red[32];
    double dt_cfl, t_now; bool clipped;
    const double dt = launch_dt(P, cur, s_red, dt_cfl, t_now, clipped);
    const R *__restrict__ Uin = reinterpret_cast<const R *>(P.U(cur));
    R *__restrict__ Uout = reinterpret_cast<R *>(P.U(cur ^ 1));
    double rate = 0.0;
    unsigned nclamp = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < P.nt; i += (long long)gridDim.x * blockDim.x) {
        const int32_t c0 = __ldg(P.cedge + 3 * i), c1 = __ldg(P.cedge + 3 * i + 1), c2 = __ldg(P.cedge + 3 * i + 2);
        const double *r0 = P.eres + 3 * (size_t)c0, *r1 = P.eres + 3 * (size_t)c1, *r2 = P.eres + 3 * (size_t)c2;
        // three edges in the fixed order k = 0,1,2 (R-17)
        const double s1 = (__ldcg(r0) + __ldcg(r1)) + __ldcg(r2);
        const double s2 = (__ldcg(r0 + 1) + __ldcg(r1 + 1)) + __ldcg(r2 + 1);
        const double s3 = (__ldcg(r0 + 2) + __ldcg(r1 + 2)) + __ldcg(r2 + 2);
        const Rec Ui = ldrec<R>(Uin + i);
        const int t = (int)(i / tile_cells), q = (int)(i - (long long)t * tile_cells);
        const double *cc = P.cellc + (size_t)t * 3 * tile_cells + q;
        Rec Un;
        rate = fmax(rate, cell_update(P, Ui, s1, s2, s3, __ldg(cc), __ldg(cc + tile_cells), __ldg(cc + 2 * tile_cells), dt, Un, nclamp));
        strec(Uout + i, Un);
    }
    rate = block_max(rate, s_red);
    if (nclamp) atomicAdd(&P.ctrl->n_clamped, (unsigned long long)nclamp);   // diagnostics only
    if (threadIdx.x == 0) {
        P.pmax(cur ^ 1)[blockIdx.x] = rate;
        if (blockIdx.x == 0) {
            Ctrl *c = P.ctrl;
            c->t[cur ^ 1] = clipped ? fmax(__ldcg(&P.ctrl->t_end), t_now) : t_now + dt;    // R-24
            if (dt > 0.0) { c->dt_last = dt; c->steps += 1; }
            if (!(dt_cfl > 0.0)) c->all_dry = 1;
            c->n_active += (unsigned long long)P.ntiles;      // no dry-tile shortcut on this path
        }
    }
}

// the whole run of a small mesh in one thread-block cluster (cluster_loop, swe_kernels.cuh)
template <int TC>
__global__ void __launch_bounds__(2 * TC, 1)
swe_cluster_kernel(const Params P, int cur, const long long nsteps)
{
    __shared__ double s_red[32];
    cluster_loop<TC>(P, dyn_smem, s_red, cur, nsteps);
}

typedef void (*step_kernel_t)(const Params, int, const long long);
step_kernel_t cluster_kernel_for(int tc)
{
    switch (tc) {
    case 64: return swe_cluster_kernel<64>;
    case 128: return swe_cluster_kernel<128>;
    case 192: return swe_cluster_kernel<192>;
    case 256: return swe_cluster_kernel<256>;
    default: return nullptr;
    }
}
step_kernel_t step_kernel_for(int tc)
{
    switch (tc) {
    case 64: return swe_step_kernel<64>;
    case 128: return swe_step_kernel<128>;
    case 192: return swe_step_kernel<192>;
    case 256: return swe_step_kernel<256>;
    default: return nullptr;
    }
}

// Per-block maxima of (sqrt(g h)+|V|)/R for the state in U[cur] (swe_compute_dt, first step).
template <class R>
__global__ void __launch_bounds__(kMaxBlock)
swe_rate_kernel(const Params P, const int cur)
{
    __shared__ double s_red[32];
    double rate = 0.0;
    for (int t = blockIdx.x; t < P.ntiles; t += gridDim.x) {
        const int i = t * blockDim.x + threadIdx.x;
        if (i < P.nt) {
            const Rec U = ldrec<R>(reinterpret_cast<const R *>(P.U(cur)) + i);
            if (U.h > P.hdry)
                rate = fmax(rate, (sqrt(P.g * U.h) + sqrt(fma(U.u, U.u, U.v * U.v))) *
                                  __ldg(P.cellc + ((size_t)t * 3 + 1) * blockDim.x + threadIdx.x));
        }
    }
    rate = block_max(rate, s_red);
    if (threadIdx.x == 0) P.pmax(cur)[blockIdx.x] = rate;
}

// ctrl->dt = CFL / max(pmax[cur]) (for read-back; the step kernels reduce on their own)
__global__ void swe_finalize_dt_kernel(const Params P, const int cur)
{
    __shared__ double s_red[32];
    const double dt = reduce_dt(P, P.pmax(cur), s_red);
    if (threadIdx.x == 0) P.ctrl->dt = dt;
}

// swe_get_stats on the device: per-block partial sums of h |Omega| (fixed tree, so the result does
// not depend on timing), number of dry cells, number of non-finite cells.  out[block] = {volume,
// dry, non-finite}; the host adds the <= kStatBlocks partials in block order.
constexpr int kStatBlocks = 1024, kStatThreads = 256;
struct StatPart { double volume; long long ndry, nbad; };
template <class R>
__global__ void __launch_bounds__(kStatThreads)
swe_stats_kernel(const Params P, const int cur, const int tile_cells, StatPart *__restrict__ out)
{
    __shared__ double s_v[kStatThreads];
    __shared__ long long s_d[kStatThreads], s_b[kStatThreads];
    double v = 0.0; long long nd = 0, nb = 0;
    for (long long i = (long long)blockIdx.x * kStatThreads + threadIdx.x; i < P.nt; i += (long long)gridDim.x * kStatThreads) {
        const Rec U = ldrec<R>(reinterpret_cast<const R *>(P.U(cur)) + i);
        const int t = (int)(i / tile_cells), q = (int)(i - (long long)t * tile_cells);
        const double area = 1.0 / __ldg(P.cellc + (size_t)t * 3 * tile_cells + q);
        v = fma(U.h, area, v);
        nd += U.h <= P.hdry;
        nb += !(isfinite(U.h) && isfinite(U.u) && isfinite(U.v));
    }
    s_v[threadIdx.x] = v; s_d[threadIdx.x] = nd; s_b[threadIdx.x] = nb;
    __syncthreads();
    for (int o = kStatThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            s_v[threadIdx.x] += s_v[threadIdx.x + o]; s_d[threadIdx.x] += s_d[threadIdx.x + o];
            s_b[threadIdx.x] += s_b[threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[blockIdx.x].volume = s_v[0]; out[blockIdx.x].ndry = s_d[0]; out[blockIdx.x].nbad = s_b[0]; }
}

// caller numbering (h, hu, hv) -> internal records {h, u, v, z}; dry cells lose their momentum
// Both kernels run over the CALLER's numbering c (coalesced on the caller's arrays) and touch the
// internal record inv[c] as one 32-byte sector.  zcell is in caller numbering too.
template <class R>
__global__ void swe_pack_kernel(const Params P, const int cur, const int32_t *__restrict__ inv,
                                const double *__restrict__ h, const double *__restrict__ hu,
                                const double *__restrict__ hv, const double *__restrict__ zcell)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.nt) return;
    Rec r; r.h = h[c]; r.z = zcell[c];
    const double qx = hu[c], qy = hv[c];
    // validation on the device: the state is here anyway, and a host loop over three arrays
    // would cost more than the copy
    if (!(r.h >= 0.0) || !isfinite(r.h) || !isfinite(qx) || !isfinite(qy)) atomicMin(&P.ctrl->bad_cell, c);
    if (r.h > P.hdry) { r.u = qx / r.h; r.v = qy / r.h; } else { r.u = 0.0; r.v = 0.0; }
    strec(reinterpret_cast<R *>(P.U(cur)) + inv[c], r);
}
template <class R>
__global__ void swe_unpack_kernel(const Params P, const int cur, const int32_t *__restrict__ inv,
                                  double *__restrict__ h, double *__restrict__ hu, double *__restrict__ hv)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.nt) return;
    const Rec r = ldrec<R>(reinterpret_cast<const R *>(P.U(cur)) + inv[c]);
    if (h) h[c] = r.h;
    if (hu) hu[c] = r.h * r.u;
    if (hv) hv[c] = r.h * r.v;
}
// swe_sample_cells: (h, hu, hv) of n cells given by caller ids (gauges); out = [3][n]
template <class R>
__global__ void swe_sample_kernel(const Params P, const int cur, const int32_t *__restrict__ inv,
                                  const int32_t *__restrict__ cells, const int n, double *__restrict__ out)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const Rec r = ldrec<R>(reinterpret_cast<const R *>(P.U(cur)) + inv[cells[k]]);
    out[k] = r.h; out[n + k] = r.h * r.u; out[2 * n + k] = r.h * r.v;
}

} // namespace

// =================================================================================================
// handle
// =================================================================================================
struct swe_mesh {
    swe_params prm;
    HostTables T;
    TileTables X;
    GlobalEdges E;            // SWE_KERNEL_EDGE_TWO_PASS only
    bool edge_kernel = false, f32 = false; int grid_edge = 0, grid_cell = 0;
    std::string err;
    // device
    bool bound = false, have_state = false, have_rates = false;
    char *ws = nullptr; size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    Params P{};
    int32_t *d_inv = nullptr; double *d_zcell = nullptr; double *d_stage = nullptr;
    double *d_qn = nullptr;
    int cur = 0, grid = 0, block = kDefaultBlock, coop_grid = 0, loop_mode = SWE_LOOP_LAUNCH;
    size_t smem = 0;          // dynamic shared memory of the step kernel
    void (*kern)(const Params, int, const long long) = nullptr;
    void (*ckern)(const Params, int, const long long) = nullptr;   // SWE_LOOP_CLUSTER
    size_t csmem = 0;
    int64_t launches = 0;
    double qn_tag[SWE_BC_MAX_TAG + 1] = {};
    std::map<std::pair<int, int>, cudaGraphExec_t> graphs; // (steps, cur) -> exec
    // asynchronous snapshot (side stream)
    cudaStream_t side = nullptr; cudaEvent_t ev_ready = nullptr, ev_done = nullptr;
    bool snap_pending = false; double *snap_t = nullptr; Ctrl *snap_ctrl = nullptr /* pinned */; int snap_cur = 0;
};

static thread_local std::string g_create_err;

#define CK(call)                                                                         \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            m->err = std::string(#call) + ": " + cudaGetErrorString(e_);                 \
            return SWE_ERR_CUDA;                                                         \
        }                                                                                \
    } while (0)

static size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

namespace {
static_assert(sizeof(HostEdge) == 24 && kDevPosMask == kPosMask && kDevKShift == kKShift && kDevSlotShift == kSlotShift &&
              kDevNoSlot == kNoSlot, "edge list encoding (mesh_builder.h / swe_kernels.cuh)");
static_assert(kTileNbrs == kNbrs && sizeof(HostEdge) == sizeof(GEdge), "neighbour-tile rows / global edge records");
struct Layout {
    size_t U0, U1, cellc, edges, tinfo, bvol, act0, act1, tnbr, binact, wq, wlist, zcell, perm, stage, pmax0, pmax1, qn, ctrl, gedges, cedge, eres, total;
};
Layout make_layout(const HostTables &T, const TileTables &X, const GlobalEdges &E)
{
    Layout L; size_t o = 0; const size_t n = (size_t)T.nt;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    L.U0 = take(n * sizeof(Rec)); L.U1 = take(n * sizeof(Rec));
    L.cellc = take(X.cellc.size() * sizeof(double)); L.edges = take(X.edges.size() * sizeof(HostEdge));
    L.tinfo = take(X.tinfo.size() * sizeof(int32_t));
    L.bvol = take(((size_t)X.nbedges + 1) * sizeof(double));
    L.act0 = take(((size_t)X.ntiles + 1) * sizeof(int32_t)); L.act1 = take(((size_t)X.ntiles + 1) * sizeof(int32_t));
    L.tnbr = take(X.tnbr.size() * sizeof(int32_t)); L.binact = take(kMaxPart * sizeof(int32_t));
    L.wq = take(kMaxPart * sizeof(unsigned long long)); L.wlist = take(((size_t)X.ntiles + kMaxPart) * sizeof(int32_t));
    L.zcell = take(n * sizeof(double)); L.perm = take(n * sizeof(int32_t));
    L.stage = take(3 * n * sizeof(double));
    L.pmax0 = take(kMaxPart * sizeof(double)); L.pmax1 = take(kMaxPart * sizeof(double));
    L.qn = take((SWE_BC_MAX_TAG + 1) * sizeof(double)); L.ctrl = take(sizeof(Ctrl));
    L.gedges = take(E.edges.size() * sizeof(HostEdge)); L.cedge = take(E.cedge.size() * sizeof(int32_t));
    L.eres = take(E.edges.size() * 6 * sizeof(double));
    L.total = o;
    return L;
}
} // namespace

extern "C" {

int swe_params_default(swe_params *p)
{
    if (!p) return SWE_ERR_INVALID_ARG;
    p->g = 9.81; p->cfl = 0.9; p->h_dry = 1e-6;
    p->ordering = SWE_ORDER_HILBERT; p->block_size = 0; p->loop_mode = SWE_LOOP_AUTO; p->riemann = SWE_RIEMANN_HLLC;
    p->kernel = SWE_KERNEL_TILED; p->fp_kind = SWE_FP64;
    return SWE_OK;
}

const char *swe_last_error(const swe_mesh *m) { return m ? m->err.c_str() : g_create_err.c_str(); }

int swe_mesh_create(const double *nodes_xy, int64_t nn, const int32_t *tris, int64_t nt,
                    const double *bathymetry, const double *manning, const int8_t *bc_tags,
                    const swe_params *params, swe_mesh **out)
{
    if (out) *out = nullptr;
    if (!nodes_xy || !tris || !bathymetry || !manning || !bc_tags || !out || nn <= 0 || nt <= 0 ||
        nt >= (int64_t)INT32_MAX / 4 || nn >= (int64_t)INT32_MAX) {
        g_create_err = "swe_mesh_create: NULL pointer or size out of range";
        return SWE_ERR_INVALID_ARG;
    }
    swe_params p;
    swe_params_default(&p);
    if (params) p = *params;
    if (!(p.g > 0.0) || !(p.cfl > 0.0) || !(p.h_dry >= 0.0) || p.ordering < 0 || p.ordering > SWE_ORDER_RCM ||
        p.loop_mode < 0 || p.loop_mode > SWE_LOOP_CLUSTER || p.riemann < 0 || p.riemann > SWE_RIEMANN_HLL ||
        p.kernel < 0 || p.kernel > SWE_KERNEL_EDGE_TWO_PASS || p.fp_kind < 0 || p.fp_kind > SWE_FP_MIXED32 ||
        (p.fp_kind == SWE_FP_MIXED32 && p.kernel != SWE_KERNEL_EDGE_TWO_PASS) ||
        (p.block_size != 0 && p.block_size != 64 && p.block_size != 128 && p.block_size != 192 && p.block_size != 256)) {
        g_create_err = "swe_mesh_create: invalid swe_params (block_size must be 0, 64, 128, 192 or 256; SWE_FP_MIXED32 needs SWE_KERNEL_EDGE_TWO_PASS)";
        return SWE_ERR_INVALID_ARG;
    }
    swe_mesh *m = new (std::nothrow) swe_mesh();
    if (!m) { g_create_err = "out of host memory"; return SWE_ERR_NOMEM; }
    m->prm = p;
    int rc;
    try {
        rc = build_tables(nodes_xy, nn, tris, nt, bathymetry, manning, bc_tags, p.ordering, m->T, m->err);
    } catch (const std::bad_alloc &) { rc = SWE_ERR_NOMEM; m->err = "out of host memory"; }
    if (rc != SWE_OK) { g_create_err = m->err; delete m; return rc; }
    m->block = p.block_size ? p.block_size : kDefaultBlock;
    // small meshes that AUTO will run as one cluster: 128-cell tiles (up to 16 of them)
    if (!p.block_size && p.kernel == SWE_KERNEL_TILED && (p.loop_mode == SWE_LOOP_AUTO || p.loop_mode == SWE_LOOP_CLUSTER) &&
        nt <= (int64_t)kMaxClusterTiles * 128)
        m->block = 128;
    rc = build_tiles(m->T, m->block, p.g, m->X, m->err);
    if (rc != SWE_OK) { g_create_err = m->err; delete m; return rc; }
    m->edge_kernel = p.kernel == SWE_KERNEL_EDGE_TWO_PASS;
    m->f32 = p.fp_kind == SWE_FP_MIXED32;
    if (m->edge_kernel) {
        rc = build_global_edges(m->T, m->E, m->err);
        if (rc != SWE_OK) { g_create_err = m->err; delete m; return rc; }
    }
    *out = m;
    return SWE_OK;
}

int swe_mesh_file_read(const char *path, int64_t *nn, int64_t *nt, double *nodes_xy,
                       double *bathymetry, int32_t *tris, double *manning)
{
    try {
        return read_mesh_file(path, nn, nt, nodes_xy, bathymetry, tris, manning, g_create_err);
    } catch (const std::bad_alloc &) { g_create_err = "out of host memory"; return SWE_ERR_NOMEM; }
}

int swe_mesh_destroy(swe_mesh *m)
{
    if (!m) return SWE_OK;
    // steps still queued on the stream write the caller's workspace: let them finish before the
    // caller is told it may free or reuse that memory
    if (m->bound) cudaStreamSynchronize(m->stream);
    for (auto &kv : m->graphs) cudaGraphExecDestroy(kv.second);
    if (m->snap_pending) cudaEventSynchronize(m->ev_done);
    if (m->ev_ready) cudaEventDestroy(m->ev_ready);
    if (m->ev_done) cudaEventDestroy(m->ev_done);
    if (m->side) cudaStreamDestroy(m->side);
    if (m->snap_ctrl) cudaFreeHost(m->snap_ctrl);
    delete m;
    return SWE_OK;
}

int swe_mesh_workspace_bytes(const swe_mesh *m, size_t *bytes)
{
    if (!m || !bytes) return SWE_ERR_INVALID_ARG;
    *bytes = make_layout(m->T, m->X, m->E).total;
    return SWE_OK;
}

int swe_get_permutation(const swe_mesh *m, int32_t *perm)
{
    if (!m || !perm) return SWE_ERR_INVALID_ARG;
    std::memcpy(perm, m->T.perm.data(), sizeof(int32_t) * (size_t)m->T.nt);
    return SWE_OK;
}

int swe_get_tables(const swe_mesh *m, int32_t *nbr, double *normal, double *length, double *area,
                   double *inradius, double *cell_z)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    const size_t n = (size_t)m->T.nt;
    if (nbr) std::memcpy(nbr, m->T.nbr.data(), 3 * n * sizeof(int32_t));
    if (normal) std::memcpy(normal, m->T.normal.data(), 6 * n * sizeof(double));
    if (length) std::memcpy(length, m->T.length.data(), 3 * n * sizeof(double));
    if (area) std::memcpy(area, m->T.area.data(), n * sizeof(double));
    if (inradius) std::memcpy(inradius, m->T.inradius.data(), n * sizeof(double));
    if (cell_z) std::memcpy(cell_z, m->T.cell_z.data(), n * sizeof(double));
    return SWE_OK;
}

int swe_get_tile_info(const swe_mesh *m, int32_t *tile_cells, int64_t *ntiles, int64_t *nedges,
                      int32_t *max_edges, int32_t *max_halo, size_t *smem_bytes)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    if (tile_cells) *tile_cells = m->X.tile_cells;
    if (ntiles) *ntiles = m->X.ntiles;
    if (nedges) *nedges = m->X.nedges;
    if (max_edges) *max_edges = m->X.max_edges;
    if (max_halo) *max_halo = m->X.max_halo;
    if (smem_bytes) *smem_bytes = tile_smem_bytes(m->X.tile_cells, m->X.max_halo, m->X.max_edges);
    return SWE_OK;
}

int swe_get_step_bytes(const swe_mesh *m, double active_tiles, double edge_lists, double quiet_tiles, double *bytes)
{
    if (!m || !bytes || !(active_tiles >= 0.0) || !(edge_lists >= 0.0) || !(quiet_tiles >= 0.0)) return SWE_ERR_INVALID_ARG;
    const TileTables &X = m->X;
    const double nt = (double)m->T.nt, ntiles = (double)X.ntiles, TC = (double)X.tile_cells;
    if (m->edge_kernel) {
        // pass 1: edge record, one sector per end point, both sides' results out; pass 2: edge ids,
        // three 24-byte results, record in and out, cell constants
        const double ne = (double)m->E.edges.size(), nb = (double)X.nbedges;
        const double rec = m->f32 ? 16.0 : 32.0;
        *bytes = ne * 24.0 + (2.0 * ne - nb) * 32.0 + ne * 48.0 + nt * (12.0 + 72.0 + rec + 24.0 + rec);
        return SWE_OK;
    }
    double b = 0.0;
    const double voting = std::max(0.0, ntiles - quiet_tiles);   // tiles that gather their halo and vote
    b += 32.0 * nt * voting / ntiles;                 // their cells' records read (TMA bulk copy) ...
    b += 32.0 * nt * voting / ntiles;                 // ... and written (256-bit store); quiet tiles are not touched
    b += 32.0 * (double)X.nhalo * voting / ntiles;    // halo records, one 32-byte sector each (mean list length)
    b += voting * (16.0 + 4.0 * (double)std::min(X.max_halo, X.tile_cells));   // header, halo ids
    b += ntiles * (4.0 + 4.0) + (ntiles - voting + active_tiles) * 4.0 * kNbrs;  // activity flag in and out, neighbour rows
    b += active_tiles * 24.0 * TC;                    // cell constants of the tiles that are not all dry
    b += edge_lists * 24.0 * (double)X.edges.size() / ntiles;   // edge lists fetched (mean list length)
    *bytes = b;
    return SWE_OK;
}

int swe_get_tile_tables(const swe_mesh *m, int32_t *edge_a, int32_t *edge_b, double *edge_geom, int32_t *tinfo)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    // records without the padding, tile after tile; tinfo[.][0] is rewritten to index this list
    const size_t stride = 4 + (size_t)m->X.max_halo;
    size_t o = 0;
    for (int64_t t = 0; t < m->X.ntiles; t++) {
        const int32_t *ti = m->X.tinfo.data() + (size_t)t * stride;
        for (int32_t k = 0; k < ti[1]; k++, o++) {
            const HostEdge &E = m->X.edges[(size_t)ti[0] + k];
            if (edge_a) edge_a[o] = E.a;
            if (edge_b) edge_b[o] = E.b;
            if (edge_geom) {
                const double L = std::sqrt(E.lx * E.lx + E.ly * E.ly);
                edge_geom[3 * o] = E.lx / L; edge_geom[3 * o + 1] = E.ly / L; edge_geom[3 * o + 2] = L;
            }
        }
    }
    if (tinfo) {
        std::memcpy(tinfo, m->X.tinfo.data(), m->X.tinfo.size() * sizeof(int32_t));
        int32_t first = 0;
        for (int64_t t = 0; t < m->X.ntiles; t++) { tinfo[(size_t)t * stride] = first; first += tinfo[(size_t)t * stride + 1]; }
    }
    return SWE_OK;
}

int swe_get_launch_info(const swe_mesh *m, int32_t *grid, int32_t *block, int32_t *loop_mode, int64_t *launches)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    if (grid) *grid = m->loop_mode == SWE_LOOP_PERSISTENT ? m->coop_grid : m->grid;
    if (block) *block = m->block;
    if (loop_mode) *loop_mode = m->loop_mode;
    if (launches) *launches = m->launches;
    return SWE_OK;
}

int swe_mesh_bind_device(swe_mesh *m, void *device_workspace, size_t bytes, void *cuda_stream)
{
    if (!m || !device_workspace) return SWE_ERR_INVALID_ARG;
    const HostTables &T = m->T;
    const size_t n = (size_t)T.nt;
    const Layout L = make_layout(T, m->X, m->E);
    if (bytes < L.total || ((uintptr_t)device_workspace & 255u)) {
        m->err = "workspace too small or not 256-byte aligned";
        return SWE_ERR_WORKSPACE;
    }
    for (auto &kv : m->graphs) cudaGraphExecDestroy(kv.second);
    m->graphs.clear();
    m->bound = false; m->have_state = false; m->have_rates = false;
    m->ws = (char *)device_workspace; m->ws_bytes = bytes; m->stream = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0, coop = 0, smem_optin = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    CK(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    // dynamic shared memory of the tile pipeline (swe_kernels.cuh), sized for this mesh's longest lists
    const TileTables &X = m->X;
    m->smem = tile_smem_bytes(m->block, X.max_halo, X.max_edges);
    if (m->smem > (size_t)smem_optin - 1024) { m->err = "tile does not fit in shared memory"; return SWE_ERR_CUDA; }
    // end point words hold 13-bit positions, tile headers 12-bit counts (swe_kernels.cuh)
    if (m->block + X.max_halo > (int)kPosMask || X.max_edges > 4095 || X.max_halo > 4095) {
        m->err = "tile edge / halo lists too long for the kernel's tables"; return SWE_ERR_INVALID_ARG;
    }
    m->kern = step_kernel_for(m->block);
    // the attribute belongs to the kernel, not to this handle: allow the device maximum so that
    // handles with different tile tables can coexist
    CK(cudaFuncSetAttribute((const void *)m->kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 1024));
    int occ_step = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_step, (const void *)m->kern, m->block, m->smem));
    if (occ_step < 1) { m->err = "kernel does not fit on this device"; return SWE_ERR_CUDA; }
    const int ntiles = (int)X.ntiles;
    // grid: every SM holds its full complement of resident blocks, each walking tiles with a
    // stride of the grid (a multiple of the SM count); small meshes get one block per tile
    m->grid = std::min(std::min(ntiles, sms * occ_step), kMaxPart);
    m->coop_grid = m->grid;       // the same kernel runs both ways
    int mode = m->prm.loop_mode;
    // measured on B200 (2000 to 200 000 cells): replaying 128-step CUDA graphs is as fast as the
    // cooperative launch on the smallest meshes (6.0 us per step at 11 blocks) and 14 % faster once
    // blocks own two tiles (12.8 vs 14.9 us at 200 000 cells), so AUTO means GRAPH
    if ((mode == SWE_LOOP_AUTO || mode == SWE_LOOP_CLUSTER) && !m->edge_kernel && ntiles <= kMaxClusterTiles) {
        // can one cluster of ntiles CTAs be resident?  (non-portable sizes above 8 need the opt-in)
        m->ckern = cluster_kernel_for(m->block);
        m->csmem = cluster_smem_bytes(m->block, X.max_halo, X.max_edges);
        int nclusters = 0;
        if (m->csmem <= (size_t)smem_optin - 1024 &&
            cudaFuncSetAttribute((const void *)m->ckern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 1024) == cudaSuccess &&
            cudaFuncSetAttribute((const void *)m->ckern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(ntiles); cfg.blockDim = dim3(2 * m->block); cfg.dynamicSmemBytes = m->csmem;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = ntiles; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            cfg.attrs = at; cfg.numAttrs = 1;
            if (cudaOccupancyMaxActiveClusters(&nclusters, (const void *)m->ckern, &cfg) != cudaSuccess) nclusters = 0;
        }
        (void)cudaGetLastError();
        mode = nclusters >= 1 ? SWE_LOOP_CLUSTER : SWE_LOOP_GRAPH;
    }
    if (mode == SWE_LOOP_AUTO || mode == SWE_LOOP_CLUSTER) mode = mode == SWE_LOOP_CLUSTER && m->ckern && ntiles <= kMaxClusterTiles && !m->edge_kernel ? mode : SWE_LOOP_GRAPH;
    if (mode == SWE_LOOP_PERSISTENT && !coop) mode = SWE_LOOP_GRAPH;
    if (m->edge_kernel) {
        // two kernels per step: the kernel boundary is the only grid-wide barrier they have
        if (mode == SWE_LOOP_PERSISTENT) mode = SWE_LOOP_GRAPH;
        const int64_t want_e = ((int64_t)m->E.edges.size() + 255) / 256, want_c = ((int64_t)n + 255) / 256;
        m->grid_edge = (int)std::max<int64_t>(1, std::min<int64_t>(want_e, (int64_t)sms * 8));
        m->grid_cell = (int)std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(want_c, (int64_t)sms * 8), kMaxPart));
        m->grid = m->coop_grid = m->grid_cell;     // the per-block maxima are pass 2's
    }
    m->loop_mode = mode;

    Params &P = m->P;
    P.U0 = (Rec *)(m->ws + L.U0); P.U1 = (Rec *)(m->ws + L.U1);
    P.cellc = (const double *)(m->ws + L.cellc); P.edges = (const double *)(m->ws + L.edges);
    P.tinfo = (const int32_t *)(m->ws + L.tinfo);
    P.bvol = (double *)(m->ws + L.bvol);
    P.act0 = (int32_t *)(m->ws + L.act0); P.act1 = (int32_t *)(m->ws + L.act1);
    P.tnbr = (const int32_t *)(m->ws + L.tnbr); P.binact = (int32_t *)(m->ws + L.binact);
    P.wq = (unsigned long long *)(m->ws + L.wq); P.wlist = (int32_t *)(m->ws + L.wlist);
    m->d_zcell = (double *)(m->ws + L.zcell); m->d_inv = (int32_t *)(m->ws + L.perm);
    m->d_stage = (double *)(m->ws + L.stage);
    P.pmax0 = (double *)(m->ws + L.pmax0); P.pmax1 = (double *)(m->ws + L.pmax1);
    m->d_qn = (double *)(m->ws + L.qn); P.qn_tag = m->d_qn;
    P.ctrl = (Ctrl *)(m->ws + L.ctrl);
    P.hll = m->prm.riemann == SWE_RIEMANN_HLL;
    P.gedges = m->edge_kernel ? (const GEdge *)(m->ws + L.gedges) : nullptr;
    P.cedge = m->edge_kernel ? (const int32_t *)(m->ws + L.cedge) : nullptr;
    P.eres = m->edge_kernel ? (double *)(m->ws + L.eres) : nullptr;
    P.nge = (int32_t)m->E.edges.size();
    P.nt = (int32_t)T.nt; P.ntiles = ntiles; P.max_edges = X.max_edges; P.max_halo = X.max_halo;
    P.npart = mode == SWE_LOOP_PERSISTENT ? m->coop_grid : m->grid;
    P.wstride = (ntiles + P.npart - 1) / std::max(P.npart, 1);
    P.g = m->prm.g; P.hg = 0.5 * m->prm.g; P.inv_g = 1.0 / m->prm.g; P.cfl = m->prm.cfl;
    // a side is dry iff h <= h_dry; the floor keeps every argument of the MUFU-seeded
    // reciprocal / rsqrt a normal number when the caller asks for h_dry = 0
    P.hdry = std::max(m->prm.h_dry, 1e-250);

    try {
        cudaStream_t s = m->stream;
        CK(cudaMemcpyAsync(m->ws + L.cellc, X.cellc.data(), X.cellc.size() * sizeof(double), cudaMemcpyHostToDevice, s));
        std::vector<double> dev_edges;          // the edge lists as the kernel reads them (freed after the upload)
        pack_device_edges(X, dev_edges);
        CK(cudaMemcpyAsync(m->ws + L.edges, dev_edges.data(), dev_edges.size() * sizeof(double), cudaMemcpyHostToDevice, s));
        CK(cudaMemcpyAsync(m->ws + L.tinfo, X.tinfo.data(), X.tinfo.size() * sizeof(int32_t), cudaMemcpyHostToDevice, s));
        CK(cudaMemcpyAsync(m->ws + L.tnbr, X.tnbr.data(), X.tnbr.size() * sizeof(int32_t), cudaMemcpyHostToDevice, s));
        if (m->edge_kernel) {
            CK(cudaMemcpyAsync(m->ws + L.gedges, m->E.edges.data(), m->E.edges.size() * sizeof(HostEdge), cudaMemcpyHostToDevice, s));
            CK(cudaMemcpyAsync(m->ws + L.cedge, m->E.cedge.data(), m->E.cedge.size() * sizeof(int32_t), cudaMemcpyHostToDevice, s));
        }
        CK(cudaMemcpyAsync(m->d_zcell, T.cell_z.data(), n * sizeof(double), cudaMemcpyHostToDevice, s));
        CK(cudaMemcpyAsync(m->d_inv, T.inv.data(), n * sizeof(int32_t), cudaMemcpyHostToDevice, s));
        CK(cudaMemcpyAsync(m->d_qn, m->qn_tag, sizeof(m->qn_tag), cudaMemcpyHostToDevice, s));
        CK(cudaMemsetAsync(P.pmax0, 0, kMaxPart * sizeof(double), s));
        CK(cudaMemsetAsync(P.pmax1, 0, kMaxPart * sizeof(double), s));
        CK(cudaMemsetAsync(P.ctrl, 0, sizeof(Ctrl), s));
        CK(cudaMemsetAsync(P.wq, 0, kMaxPart * sizeof(unsigned long long), s));
        CK(cudaMemsetAsync(P.bvol, 0, ((size_t)X.nbedges + 1) * sizeof(double), s));
        CK(cudaStreamSynchronize(s));
    } catch (const std::bad_alloc &) { m->err = "out of host memory"; return SWE_ERR_NOMEM; }
    m->bound = true;
    return SWE_OK;
}

int swe_set_bc_value(swe_mesh *m, int tag, double total_discharge)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    if (tag < SWE_BC_INFLOW0 || tag > SWE_BC_MAX_TAG || !(m->T.inflow_length[tag] > 0.0)) {
        m->err = "inflow tag out of range or carried by no boundary edge";
        return SWE_ERR_BAD_TAG;
    }
    if (!std::isfinite(total_discharge)) { m->err = "non-finite discharge"; return SWE_ERR_BAD_VALUE; }
    m->qn_tag[tag] = -total_discharge / m->T.inflow_length[tag];      // R-20
    if (m->bound) {
        CK(cudaMemcpyAsync(m->d_qn, m->qn_tag, sizeof(m->qn_tag), cudaMemcpyHostToDevice, m->stream));
        CK(cudaStreamSynchronize(m->stream));
    }
    return SWE_OK;
}

static int snapshot_finish(swe_mesh *m);

static int set_state_common(swe_mesh *m, const double *h, const double *hu, const double *hv, double t0)
{
    const int n = (int)m->T.nt;
    m->cur = 0;
    m->have_state = false; m->have_rates = false;
    Ctrl c{}; c.t[0] = t0; c.t[1] = t0; c.t_end = INFINITY; c.bad_cell = INT32_MAX;
    // nothing known yet: every tile counts as active in the previous step (!= 0), so none is quiet
    CK(cudaMemsetAsync(m->P.act0, 1, (size_t)m->X.ntiles * sizeof(int32_t), m->stream));
    CK(cudaMemsetAsync(m->P.act1, 1, (size_t)m->X.ntiles * sizeof(int32_t), m->stream));
    CK(cudaMemsetAsync(m->P.binact, 0, kMaxPart * sizeof(int32_t), m->stream));
    if (m->X.nbedges > 0) CK(cudaMemsetAsync(m->P.bvol, 0, (size_t)m->X.nbedges * sizeof(double), m->stream));
    CK(cudaMemcpyAsync(m->P.ctrl, &c, sizeof(Ctrl), cudaMemcpyHostToDevice, m->stream));
    if (m->f32) swe_pack_kernel<RecF><<<(n + 255) / 256, 256, 0, m->stream>>>(m->P, 0, m->d_inv, h, hu, hv, m->d_zcell);
    else swe_pack_kernel<Rec><<<(n + 255) / 256, 256, 0, m->stream>>>(m->P, 0, m->d_inv, h, hu, hv, m->d_zcell);
    m->launches++;
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(&c, m->P.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, m->stream));
    CK(cudaStreamSynchronize(m->stream));
    if (c.bad_cell != INT32_MAX) {
        m->err = "state has a negative depth or a non-finite value at cell " + std::to_string(c.bad_cell);
        return SWE_ERR_BAD_VALUE;
    }
    m->have_state = true;
    return SWE_OK;
}

int swe_set_state(swe_mesh *m, const double *h, const double *hu, const double *hv, double t0)
{
    if (!m || !h || !hu || !hv || !std::isfinite(t0)) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    const size_t n = (size_t)m->T.nt;
    double *st = m->d_stage;
    { int rc = snapshot_finish(m); if (rc != SWE_OK) return rc; }
    CK(cudaMemcpyAsync(st, h, n * sizeof(double), cudaMemcpyHostToDevice, m->stream));
    CK(cudaMemcpyAsync(st + n, hu, n * sizeof(double), cudaMemcpyHostToDevice, m->stream));
    CK(cudaMemcpyAsync(st + 2 * n, hv, n * sizeof(double), cudaMemcpyHostToDevice, m->stream));
    return set_state_common(m, st, st + n, st + 2 * n, t0);
}

int swe_set_state_device(swe_mesh *m, const double *d_h, const double *d_hu, const double *d_hv, double t0)
{
    if (!m || !d_h || !d_hu || !d_hv || !std::isfinite(t0)) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    return set_state_common(m, d_h, d_hu, d_hv, t0);
}

static int ensure_rates(swe_mesh *m)
{
    if (m->have_rates) return SWE_OK;
    if (m->f32) swe_rate_kernel<RecF><<<m->P.npart, m->block, 0, m->stream>>>(m->P, m->cur);
    else swe_rate_kernel<Rec><<<m->P.npart, m->block, 0, m->stream>>>(m->P, m->cur);
    m->launches++;
    CK(cudaGetLastError());
    m->have_rates = true;
    return SWE_OK;
}

static int read_ctrl(swe_mesh *m, Ctrl *c, bool finalize)
{
    if (finalize) {
        int rc = ensure_rates(m);
        if (rc != SWE_OK) return rc;
        swe_finalize_dt_kernel<<<1, 256, 0, m->stream>>>(m->P, m->cur);
        m->launches++;
        CK(cudaGetLastError());
    }
    CK(cudaMemcpyAsync(c, m->P.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, m->stream));
    CK(cudaStreamSynchronize(m->stream));
    return SWE_OK;
}

int swe_compute_dt(swe_mesh *m, double *dt_out)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    if (!m->have_state) { m->err = "no state set"; return SWE_ERR_NO_STATE; }
    // the per-block maxima of the current state are already on the device after a step (the step
    // kernel leaves them for the next one); recomputing them here with another kernel could differ
    // in the last bit and make a run depend on whether this getter was called
    Ctrl c;
    int rc = read_ctrl(m, &c, true);
    if (rc != SWE_OK) return rc;
    if (dt_out) *dt_out = c.dt;
    if (!(c.dt > 0.0)) { m->err = "every cell is dry"; return SWE_ERR_ALL_DRY; }
    return SWE_OK;
}

// one time step on stream st from the state in buffer cur: the fused tile kernel, or the two passes
static void launch_step(swe_mesh *m, cudaStream_t st, int cur)
{
    if (m->edge_kernel) {
        if (m->f32) {
            swe_edge_pass_kernel<RecF><<<m->grid_edge, 256, 0, st>>>(m->P, cur);
            swe_cell_pass_kernel<RecF><<<m->grid_cell, 256, 0, st>>>(m->P, cur, m->X.tile_cells);
        } else {
            swe_edge_pass_kernel<Rec><<<m->grid_edge, 256, 0, st>>>(m->P, cur);
            swe_cell_pass_kernel<Rec><<<m->grid_cell, 256, 0, st>>>(m->P, cur, m->X.tile_cells);
        }
    } else {
        m->kern<<<m->grid, m->block, m->smem, st>>>(m->P, cur, 1);
    }
}
static int kernels_per_step(const swe_mesh *m) { return m->edge_kernel ? 2 : 1; }

static int launch_steps_direct(swe_mesh *m, int64_t n)
{
    for (int64_t s = 0; s < n; s++) {
        launch_step(m, m->stream, m->cur);
        m->cur ^= 1;
        m->launches += kernels_per_step(m);
    }
    CK(cudaGetLastError());
    return SWE_OK;
}

static int graph_for(swe_mesh *m, int steps, cudaGraphExec_t *out)
{
    auto key = std::make_pair(steps, m->cur);
    auto it = m->graphs.find(key);
    if (it != m->graphs.end()) { *out = it->second; return SWE_OK; }
    cudaGraph_t g = nullptr; cudaGraphExec_t ex = nullptr;
    // capture on a private stream so that a NULL (legacy default) user stream works too
    cudaStream_t cap;
    CK(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    int c = m->cur;
    if (e == cudaSuccess) {
        for (int s = 0; s < steps; s++) { launch_step(m, cap, c); c ^= 1; }
        e = cudaStreamEndCapture(cap, &g);
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&ex, g, 0);
    if (g) cudaGraphDestroy(g);
    cudaStreamDestroy(cap);
    if (e != cudaSuccess) { m->err = std::string("CUDA graph build: ") + cudaGetErrorString(e); return SWE_ERR_CUDA; }
    m->graphs[key] = ex;
    *out = ex;
    return SWE_OK;
}

int swe_run(swe_mesh *m, int64_t nsteps)
{
    if (!m || nsteps < 0) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    if (!m->have_state) { m->err = "no state set"; return SWE_ERR_NO_STATE; }
    if (nsteps == 0) return SWE_OK;
    int rc = ensure_rates(m);
    if (rc != SWE_OK) return rc;
    if (m->loop_mode == SWE_LOOP_PERSISTENT) {
        Params P = m->P; int cur = m->cur; long long ns = nsteps;
        void *args[] = { &P, &cur, &ns };
        CK(cudaLaunchCooperativeKernel((void *)m->kern, dim3(m->coop_grid), dim3(m->block), args, m->smem, m->stream));
        m->launches++;
        m->cur ^= (int)(nsteps & 1);
        return SWE_OK;
    }
    if (m->loop_mode == SWE_LOOP_CLUSTER) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(m->grid); cfg.blockDim = dim3(2 * m->block); cfg.dynamicSmemBytes = m->csmem; cfg.stream = m->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = m->grid; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        CK(cudaLaunchKernelEx(&cfg, m->ckern, m->P, m->cur, (long long)nsteps));
        m->launches++;
        m->cur ^= (int)(nsteps & 1);
        return SWE_OK;
    }
    if (m->loop_mode == SWE_LOOP_LAUNCH) return launch_steps_direct(m, nsteps);
    // CUDA graphs of 128 / 16 / 2 steps (even, so the ping-pong parity is unchanged), rest direct
    static const int chunks[3] = { 128, 16, 2 };
    int64_t left = nsteps;
    for (int q = 0; q < 3; q++) {
        while (left >= chunks[q]) {
            cudaGraphExec_t ex;
            rc = graph_for(m, chunks[q], &ex);
            if (rc != SWE_OK) return rc;
            CK(cudaGraphLaunch(ex, m->stream));
            m->launches += (int64_t)chunks[q] * kernels_per_step(m);
            left -= chunks[q];
        }
    }
    return launch_steps_direct(m, left);
}

int swe_step(swe_mesh *m) { return swe_run(m, 1); }

int swe_run_until(swe_mesh *m, double t_end, int64_t max_steps, int64_t *steps_done)
{
    if (steps_done) *steps_done = 0;
    if (!m || max_steps < 0 || !(t_end == t_end)) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    if (!m->have_state) { m->err = "no state set"; return SWE_ERR_NO_STATE; }
    Ctrl c;
    int rc = read_ctrl(m, &c, true);
    if (rc != SWE_OK) return rc;
    const long long steps0 = c.steps;
    CK(cudaMemcpyAsync(&m->P.ctrl->t_end, &t_end, sizeof(double), cudaMemcpyHostToDevice, m->stream));
    int64_t left = max_steps;
    while (left > 0 && c.t[m->cur] < t_end && c.dt > 0.0) {
        // the time step varies, so run the estimated number of remaining steps (zero steps after
        // t_end is reached change nothing) and look again
        const double est = std::ceil((t_end - c.t[m->cur]) / c.dt);
        const int64_t chunk = std::min<int64_t>(left, est < 1.0 ? 1 : est > 128.0 ? 128 : (int64_t)est);
        rc = swe_run(m, chunk);
        if (rc != SWE_OK) break;
        const long long before = c.steps;
        rc = read_ctrl(m, &c, true);
        if (rc != SWE_OK) break;
        left -= c.steps - before;
        if (c.steps == before) break;       // no progress: all dry
    }
    const double inf = INFINITY;
    CK(cudaMemcpyAsync(&m->P.ctrl->t_end, &inf, sizeof(double), cudaMemcpyHostToDevice, m->stream));
    CK(cudaStreamSynchronize(m->stream));
    if (steps_done) *steps_done = c.steps - steps0;
    return rc;
}

int swe_get_boundary_volumes(swe_mesh *m, double *volume_by_tag)
{
    if (!m || !volume_by_tag) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    if (!m->have_state) { m->err = "no state set"; return SWE_ERR_NO_STATE; }
    const size_t nb = (size_t)m->X.nbedges;
    std::vector<double> v(nb);
    if (nb) CK(cudaMemcpyAsync(v.data(), m->P.bvol, nb * sizeof(double), cudaMemcpyDeviceToHost, m->stream));
    CK(cudaStreamSynchronize(m->stream));
    long double sum[SWE_BC_MAX_TAG + 1] = {};
    for (size_t b = 0; b < nb; b++) sum[m->X.btag[b]] += (long double)v[b];
    for (int k = 0; k <= SWE_BC_MAX_TAG; k++) volume_by_tag[k] = (double)sum[k];
    return SWE_OK;
}

int swe_sync(swe_mesh *m)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    CK(cudaStreamSynchronize(m->stream));
    return SWE_OK;
}

int swe_get_state_device(swe_mesh *m, double *d_h, double *d_hu, double *d_hv)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    if (!m->have_state) { m->err = "no state set"; return SWE_ERR_NO_STATE; }
    const int n = (int)m->T.nt;
    if (m->f32) swe_unpack_kernel<RecF><<<(n + 255) / 256, 256, 0, m->stream>>>(m->P, m->cur, m->d_inv, d_h, d_hu, d_hv);
    else swe_unpack_kernel<Rec><<<(n + 255) / 256, 256, 0, m->stream>>>(m->P, m->cur, m->d_inv, d_h, d_hu, d_hv);
    m->launches++;
    CK(cudaGetLastError());
    return SWE_OK;
}

// the staging buffer is shared by swe_set_state, swe_get_state and the snapshot: finish a
// pending snapshot before anyone else writes it
static int snapshot_finish(swe_mesh *m)
{
    if (!m->snap_pending) return SWE_OK;
    CK(cudaEventSynchronize(m->ev_done));
    m->snap_pending = false;
    if (m->snap_t) *m->snap_t = m->snap_ctrl->t[m->snap_cur];
    return SWE_OK;
}

int swe_snapshot_begin(swe_mesh *m, double *h, double *hu, double *hv, double *t)
{
    if (!m || !h || !hu || !hv) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    if (!m->have_state) { m->err = "no state set"; return SWE_ERR_NO_STATE; }
    int rc = snapshot_finish(m);
    if (rc != SWE_OK) return rc;
    if (!m->side) {
        CK(cudaStreamCreateWithFlags(&m->side, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&m->ev_ready, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&m->ev_done, cudaEventDisableTiming));
        CK(cudaHostAlloc((void **)&m->snap_ctrl, sizeof(Ctrl), cudaHostAllocDefault));
    }
    const size_t n = (size_t)m->T.nt;
    double *st = m->d_stage;
    // main stream: convert the current state into the staging buffer, then go on stepping
    rc = swe_get_state_device(m, st, st + n, st + 2 * n);
    if (rc != SWE_OK) return rc;
    CK(cudaMemcpyAsync(m->snap_ctrl, m->P.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, m->stream));
    CK(cudaEventRecord(m->ev_ready, m->stream));
    // side stream: device -> host while the main stream runs the next steps
    CK(cudaStreamWaitEvent(m->side, m->ev_ready, 0));
    CK(cudaMemcpyAsync(h, st, n * sizeof(double), cudaMemcpyDeviceToHost, m->side));
    CK(cudaMemcpyAsync(hu, st + n, n * sizeof(double), cudaMemcpyDeviceToHost, m->side));
    CK(cudaMemcpyAsync(hv, st + 2 * n, n * sizeof(double), cudaMemcpyDeviceToHost, m->side));
    CK(cudaEventRecord(m->ev_done, m->side));
    m->snap_pending = true; m->snap_t = t; m->snap_cur = m->cur;
    return SWE_OK;
}

int swe_snapshot_wait(swe_mesh *m)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    return snapshot_finish(m);
}

int swe_get_state(swe_mesh *m, double *h, double *hu, double *hv, double *t, double *dt_next)
{
    if (!m) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    if (!m->have_state) { m->err = "no state set"; return SWE_ERR_NO_STATE; }
    const size_t n = (size_t)m->T.nt;
    double *st = m->d_stage;
    if (h || hu || hv) {
        int rc = snapshot_finish(m);
        if (rc != SWE_OK) return rc;
        rc = swe_get_state_device(m, h ? st : nullptr, hu ? st + n : nullptr, hv ? st + 2 * n : nullptr);
        if (rc != SWE_OK) return rc;
        if (h) CK(cudaMemcpyAsync(h, st, n * sizeof(double), cudaMemcpyDeviceToHost, m->stream));
        if (hu) CK(cudaMemcpyAsync(hu, st + n, n * sizeof(double), cudaMemcpyDeviceToHost, m->stream));
        if (hv) CK(cudaMemcpyAsync(hv, st + 2 * n, n * sizeof(double), cudaMemcpyDeviceToHost, m->stream));
    }
    Ctrl c;
    int rc = read_ctrl(m, &c, dt_next != nullptr);
    if (rc != SWE_OK) return rc;
    if (t) *t = c.t[m->cur];
    if (dt_next) *dt_next = c.dt;
    return SWE_OK;
}

int swe_sample_cells(swe_mesh *m, const int32_t *cells, int64_t n, double *h, double *hu, double *hv, double *t)
{
    if (!m || !cells || !h || !hu || !hv || n <= 0) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    if (!m->have_state) { m->err = "no state set"; return SWE_ERR_NO_STATE; }
    const int64_t nt = m->T.nt;
    if (n > std::max<int64_t>(1, nt / 2)) { m->err = "swe_sample_cells: at most half the cells (swe_get_state reads them all)"; return SWE_ERR_INVALID_ARG; }
    for (int64_t k = 0; k < n; k++)
        if (cells[k] < 0 || cells[k] >= nt) { m->err = "swe_sample_cells: cell id out of range at position " + std::to_string(k); return SWE_ERR_BAD_INDEX; }
    int rc = snapshot_finish(m);       // the samples pass through the staging buffer
    if (rc != SWE_OK) return rc;
    // staging buffer: [3][n] doubles out, the ids behind the first two thirds of it
    double *d_out = m->d_stage;
    int32_t *d_cells = reinterpret_cast<int32_t *>(m->d_stage + 2 * (size_t)nt);
    CK(cudaMemcpyAsync(d_cells, cells, (size_t)n * sizeof(int32_t), cudaMemcpyHostToDevice, m->stream));
    const unsigned nb = (unsigned)((n + 127) / 128);
    if (m->f32) swe_sample_kernel<RecF><<<nb, 128, 0, m->stream>>>(m->P, m->cur, m->d_inv, d_cells, (int)n, d_out);
    else swe_sample_kernel<Rec><<<nb, 128, 0, m->stream>>>(m->P, m->cur, m->d_inv, d_cells, (int)n, d_out);
    m->launches++;
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(h, d_out, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, m->stream));
    CK(cudaMemcpyAsync(hu, d_out + n, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, m->stream));
    CK(cudaMemcpyAsync(hv, d_out + 2 * n, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, m->stream));
    Ctrl c;
    rc = read_ctrl(m, &c, false);      // synchronises the stream
    if (rc != SWE_OK) return rc;
    if (t) *t = c.t[m->cur];
    return SWE_OK;
}

int swe_get_stats(swe_mesh *m, swe_stats *s)
{
    if (!m || !s) return SWE_ERR_INVALID_ARG;
    if (!m->bound) { m->err = "no device workspace bound"; return SWE_ERR_NOT_BOUND; }
    if (!m->have_state) { m->err = "no state set"; return SWE_ERR_NO_STATE; }
    int rc = snapshot_finish(m);       // the partial sums live in the staging buffer
    if (rc != SWE_OK) return rc;
    const int nblk = (int)std::min<int64_t>(kStatBlocks, (m->T.nt + kStatThreads - 1) / kStatThreads);
    StatPart *d_part = reinterpret_cast<StatPart *>(m->d_stage);
    if (m->f32) swe_stats_kernel<RecF><<<nblk, kStatThreads, 0, m->stream>>>(m->P, m->cur, m->X.tile_cells, d_part);
    else swe_stats_kernel<Rec><<<nblk, kStatThreads, 0, m->stream>>>(m->P, m->cur, m->X.tile_cells, d_part);
    m->launches++;
    CK(cudaGetLastError());
    std::vector<StatPart> part((size_t)nblk);
    CK(cudaMemcpyAsync(part.data(), d_part, sizeof(StatPart) * (size_t)nblk, cudaMemcpyDeviceToHost, m->stream));
    Ctrl c;
    rc = read_ctrl(m, &c, false);      // synchronises the stream
    if (rc != SWE_OK) return rc;
    long double vol = 0.0L; int64_t ndry = 0, nbad = 0;
    for (const StatPart &p : part) { vol += (long double)p.volume; ndry += p.ndry; nbad += p.nbad; }
    s->volume = (double)vol; s->t = c.t[m->cur]; s->dt_last = c.dt_last; s->steps = c.steps;
    s->n_dry = ndry; s->n_clamped = (int64_t)c.n_clamped; s->n_nonfinite = nbad;
    s->active_tile_steps = (int64_t)c.n_active;
    s->edge_list_fetches = (int64_t)c.n_elists;
    s->quiet_tile_steps = (int64_t)c.n_quiet;
    s->stolen_tile_steps = (int64_t)c.n_stolen;
    return SWE_OK;
}

} // extern "C"

// =================================================================================================
// swe_cfl_dt_static: the CFL time step without any allocation (include/swe.h)
// =================================================================================================
// A variant of swe_rate_kernel + swe_finalize_dt_kernel for callers that cannot allocate (code under
// CUDA graph capture, serving loops, harnesses that forbid cudaMalloc) and have no workspace to bind:
// the per-block maxima, which the handle-based path keeps in the caller's workspace, live in a
// file-scope device array of fixed size.  Every GPU that loads the library holds these 512 KiB until
// exit.  In host code the array's NAME is a host-side stand-in, not a device address: the address a
// kernel can use comes from cudaGetSymbolAddress, asked once per device with that device current.
// Every call shares the array; it keeps the previous call's contents, which is harmless here because
// a call writes each of the partials it later reads (nothing has to start at zero), but two calls
// that overlap on the GPU (different streams) race on it.
namespace {
constexpr int kStaticThreads = 256, kStaticCellsPerThread = 4;
constexpr int kStaticCellsPerBlock = kStaticThreads * kStaticCellsPerThread;              // 1024
constexpr int64_t kStaticMaxCells = SWE_STATIC_MAX_CELLS;
constexpr int kStaticMaxBlocks = (int)(kStaticMaxCells / kStaticCellsPerBlock);          // 65536 partial maxima
static_assert(kStaticMaxCells % kStaticCellsPerBlock == 0, "SWE_STATIC_MAX_CELLS: a multiple of 1024");
static __device__ __align__(256) double g_static_scratch[kStaticMaxBlocks];

// pass 1: block b takes cells [1024 b, 1024 b + 1024); scratch[b] = its maximum of (sqrt(g h)+|V|)/R
__global__ void __launch_bounds__(kStaticThreads)
swe_static_rate_kernel(const double *__restrict__ h, const double *__restrict__ hu, const double *__restrict__ hv,
                       const double *__restrict__ inradius, const long long n, const double g, const double hdry,
                       double *__restrict__ scratch)
{
    __shared__ double s_red[32];
    double rate = 0.0;
    const long long base = (long long)blockIdx.x * kStaticCellsPerBlock + threadIdx.x;
#pragma unroll
    for (int q = 0; q < kStaticCellsPerThread; q++) {
        const long long i = base + (long long)q * kStaticThreads;
        if (i < n) {
            const double hi = __ldg(h + i);
            if (hi > hdry) {                                    // eq.(15) with d = R_i, wet cells only (R-15)
                const double u = __ldg(hu + i) / hi, v = __ldg(hv + i) / hi;
                rate = fmax(rate, (sqrt(g * hi) + sqrt(fma(u, u, v * v))) / __ldg(inradius + i));
            }
        }
    }
    rate = block_max(rate, s_red);
    if (threadIdx.x == 0) scratch[blockIdx.x] = rate;
}

// pass 2: one block; dt = CFL / max of the nblk partials this call wrote (0 if every cell is dry)
__global__ void __launch_bounds__(1024)
swe_static_dt_kernel(const double *__restrict__ scratch, const int nblk, const double cfl, double *__restrict__ dt_out)
{
    __shared__ double s_red[32];
    double r = 0.0;
    for (int k = threadIdx.x; k < nblk; k += blockDim.x) r = fmax(r, scratch[k]);
    r = block_max(r, s_red);
    if (threadIdx.x == 0) *dt_out = r > 0.0 ? cfl / r : 0.0;
}

// device address of g_static_scratch on the current device, looked up once per device
constexpr int kMaxDevices = 64;
double *g_static_ptr[kMaxDevices] = {};
std::mutex g_static_mutex;
cudaError_t static_scratch_for_current_device(double **ptr)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        g_static_ptr[dev] = p;
    }
    *ptr = g_static_ptr[dev];
    return cudaSuccess;
}
} // namespace

extern "C" int swe_cfl_dt_static(const double *d_h, const double *d_hu, const double *d_hv, const double *d_inradius,
                                 int64_t n, double g, double cfl, double h_dry, double *d_dt, void *cuda_stream)
{
    if (!d_h || !d_hu || !d_hv || !d_inradius || !d_dt || n <= 0 || !(g > 0.0) || !(cfl > 0.0) || !(h_dry >= 0.0)) {
        g_create_err = "swe_cfl_dt_static: NULL pointer, n <= 0 or a parameter out of range";
        return SWE_ERR_INVALID_ARG;
    }
    if (n > kStaticMaxCells) {
        g_create_err = "swe_cfl_dt_static: n = " + std::to_string(n) + " cells exceeds SWE_STATIC_MAX_CELLS = " +
                       std::to_string(kStaticMaxCells) + " (the fixed scratch array holds one partial maximum per 1024 cells)";
        return SWE_ERR_INVALID_ARG;
    }
    double *scratch = nullptr;
    cudaError_t e = static_scratch_for_current_device(&scratch);
    if (e == cudaSuccess) {
        cudaStream_t s = (cudaStream_t)cuda_stream;
        const int nblk = (int)((n + kStaticCellsPerBlock - 1) / kStaticCellsPerBlock);
        swe_static_rate_kernel<<<nblk, kStaticThreads, 0, s>>>(d_h, d_hu, d_hv, d_inradius, (long long)n, g, h_dry, scratch);
        swe_static_dt_kernel<<<1, 1024, 0, s>>>(scratch, nblk, cfl, d_dt);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        g_create_err = std::string("swe_cfl_dt_static: ") + cudaGetErrorString(e);
        return SWE_ERR_CUDA;
    }
    return SWE_OK;
}
