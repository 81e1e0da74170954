// Device code of libswe_b200: the fused, tiled, edge-once SWE step for sm_100a (FP64).
//
// The cells are numbered along a space-filling curve (mesh_builder.cpp) and cut into tiles of
// blockDim.x consecutive cells.  One thread block processes one tile at a time:
//
//   phase 0  every thread loads its own cell's state record (one 256-bit load) into shared
//            memory and registers, its cell-table record, and the first edge record it will
//            evaluate; edge end points that live in another tile are gathered from global
//            memory right away so that their latency overlaps the barrier
//   phase 1  (edge-parallel) every edge that touches the tile is evaluated ONCE: hydrostatic
//            reconstruction, rotation, HLLC flux, rotation back, both sides' bathymetry source;
//            five doubles per edge go to shared memory (a1-a7 of SURVEY.md section 8(a))
//   phase 2  (cell-parallel) every cell sums its three edges in the fixed order k = 0,1,2,
//            applies the semi-implicit friction and the update, writes its new record with
//            one 256-bit store and contributes (sqrt(g h)+|V|)/R of the NEW state to the block
//            maximum (a7-a11)
//
// The per-block maxima (warp shuffles + shared memory, no atomics) are reduced to dt by every
// block at the start of the next step.  PAPER.md sections 2-3 and :457.
//
// State record in HBM: {h, u, v, z} as one 32-byte sector, so a gather is exactly one sector
// whatever the ordering (LDG.E.256 on sm_100a).  Velocities (not discharges) are stored so
// that the edge phase needs no division; the caller still sees (h, hu, hv) (pack/unpack).
//
// Arithmetic: FP64 throughout.  Division and square root are the FP64 pipe's dominant cost on
// wet meshes (profiles/r01_v1_README.md), so the kernels use the MUFU seeds (rcp/rsqrt.approx)
// with a third-order correction (error ~1 ulp, no special-case handling: every argument is a
// normal positive number by construction) instead of the IEEE-rounded sequences.
// section 7 derives why this stays inside the 1e-10 parity bar.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace swe {

struct __align__(32) Rec { double h, u, v, z; };

// One edge of a tile.  a is always a cell; b is a cell or -tag on a boundary edge.  (n1,n2) is
// a's unit outward normal on this edge (so b's is its negative).  a is the end point with the
// smaller CALLER id, which makes the result independent of the renumbering (R-17).
struct __align__(32) EdgeRec { int32_t a, b; double n1, n2, len; };

// Per-cell constants.  slot k (16 bits): bits 0-14 = index of local edge k in the tile's edge
// list, bit 15 = 1 if this cell is the edge's b side.
struct __align__(32) CellRec { uint32_t slots01, slots2; double inv_area, inv_R, gm2; };

struct Ctrl {                 // device-resident loop state
    double t;                 // simulated time
    double dt;                // step the next update will use (valid after a finalise)
    double dt_last;           // step used by the latest update
    long long steps;
    unsigned long long n_clamped;
    int all_dry;              // set when a step found no wet cell
    int pad;
};

struct Params {
    Rec *U0, *U1;             // ping-pong state, internal order
    const CellRec *cells;     // [nt]
    const EdgeRec *edges;     // [estart[ntiles]] tile after tile
    const int32_t *estart;    // [ntiles + 1]
    const double *qn_tag;     // [128] unit discharge along the outward normal per inflow tag
    double *pmax0, *pmax1;    // [npart] per-block max rate of state U0 / U1
    Ctrl *ctrl;
    int32_t nt, ntiles, npart, max_edges;
    double g, inv_g, cfl, hdry;
    // selected with a ternary so the kernel parameter block is never indexed dynamically
    __host__ __device__ __forceinline__ Rec *U(int c) const { return c ? U1 : U0; }
    __host__ __device__ __forceinline__ double *pmax(int c) const { return c ? pmax1 : pmax0; }
};

// ---- 256-bit access --------------------------------------------------------------------------
template <bool kReadOnlyPath>
__device__ __forceinline__ Rec load_rec(const Rec *p)
{
    Rec r;
    if (kReadOnlyPath)   // state is constant for the whole launch
        asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
                     : "=d"(r.h), "=d"(r.u), "=d"(r.v), "=d"(r.z) : "l"(p));
    else                 // persistent loop: other blocks rewrote it before the grid barrier
        asm volatile("ld.global.cg.v4.f64 {%0,%1,%2,%3}, [%4];"
                     : "=d"(r.h), "=d"(r.u), "=d"(r.v), "=d"(r.z) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void store_rec(Rec *p, const Rec &r)
{
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "d"(r.h), "d"(r.u), "d"(r.v), "d"(r.z) : "memory");
}
__device__ __forceinline__ EdgeRec load_edge(const EdgeRec *p)
{
    EdgeRec e; double ab;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(ab), "=d"(e.n1), "=d"(e.n2), "=d"(e.len) : "l"(p));
    const long long w = __double_as_longlong(ab);
    e.a = (int32_t)(w & 0xffffffffll); e.b = (int32_t)(w >> 32);
    return e;
}
__device__ __forceinline__ CellRec load_cell(const CellRec *p)
{
    CellRec c; double s;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(s), "=d"(c.inv_area), "=d"(c.inv_R), "=d"(c.gm2) : "l"(p));
    const long long w = __double_as_longlong(s);
    c.slots01 = (uint32_t)(w & 0xffffffffll); c.slots2 = (uint32_t)((unsigned long long)w >> 32);
    return c;
}

// ---- MUFU-seeded FP64 reciprocal / rsqrt / rcbrt ---------------------------------------------
// Arguments are finite, normal and positive at every call site (depths above the wet/dry
// threshold, sums of celerities, S_R - S_L in the star region, determinants >= 1).
// Seed relative error e0 <= ~2^-20; the corrections below leave O(e0^3) + rounding (~1 ulp).
__device__ __forceinline__ double fast_rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);          // x y = 1 - e
    const double t = fma(e, e, e);             // e + e^2
    return fma(y, t, y);                       // y (1 + e + e^2)
}
__device__ __forceinline__ double fast_rsqrt(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double e = fma(-t, y, 1.0);          // x y^2 = 1 - e
    const double p = fma(e, 0.375, 0.5) * e;   // e/2 + 3 e^2/8
    return fma(y, p, y);
}
// x^(-1/3) for x in [2^-96, 2^96] (fp32 seed); callers fall back to rcbrt() outside.
__device__ __forceinline__ double fast_rcbrt(double x)
{
    const float xf = (float)x;
    const double y = (double)exp2f(-0.333333343f * __log2f(xf));
    const double y3 = (y * y) * y;
    const double e = fma(-x, y3, 1.0);         // x y^3 = 1 - e
    const double p = fma(e, 2.0 / 9.0, 1.0 / 3.0) * e;
    return fma(y, p, y);
}

// ---- block reduction (max), deterministic, no atomics ----------------------------------------
__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
// Result valid in every thread.  s_red: >= 32 doubles of shared memory.
__device__ __forceinline__ double block_max(double v, double *s_red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    v = warp_max(v);
    __syncthreads();                 // protect s_red against the previous use
    if (lane == 0) s_red[wid] = v;
    __syncthreads();
    double r = lane < nw ? s_red[lane] : 0.0;
    return warp_max(r);
}

// dt = CFL / max over the per-block maxima, eq.(15) and :457; 0 if all dry.
__device__ __forceinline__ double reduce_dt(const Params &P, const double *pmax, double *s_red)
{
    double r = 0.0;
    for (int k = threadIdx.x; k < P.npart; k += blockDim.x) r = fmax(r, __ldcg(pmax + k));
    r = block_max(r, s_red);
    return r > 0.0 ? P.cfl / r : 0.0;
}

// ---- HLLC flux in the edge frame, eq.(17)-(26) --------------------------------
// Inputs: reconstructed depths, normal/tangential velocities.  Output (G0,G1,G2) = mass, normal
// and tangential momentum flux.  Same expression trees as the oracle's step list (DESIGN.md
// section 4) except that a_k = sqrt(g h_k) and 1/h_k both come from one rsqrt(g h_k), and that
// a_k p_k of eq.(19)-(20) is formed as sqrt(g h* (h*+h_k) / (2 h_k)) (one square root, R-7).
__device__ __forceinline__ void hllc_flux(const double g, const double inv_g, const double hdry,
                                          double hL, double uL, double vL, double hR, double uR,
                                          double vR, double &G0, double &G1, double &G2)
{
    const bool dL = hL <= hdry, dR = hR <= hdry;           // R-15
    G0 = 0.0; G1 = 0.0; G2 = 0.0;
    if (dL && dR) return;
    double SL, SR;
    if (dL) {                                               // eq.(26) line 1
        hL = 0.0; uL = 0.0; vL = 0.0;
        const double ghR = g * hR, aR = ghR * fast_rsqrt(ghR);
        SL = uR - 2.0 * aR; SR = uR + aR;
    } else if (dR) {                                        // eq.(26) line 2 (R-18)
        hR = 0.0; uR = 0.0; vR = 0.0;
        const double ghL = g * hL, aL = ghL * fast_rsqrt(ghL);
        SL = uL - aL; SR = uL + 2.0 * aL;
    } else {
        const double ghL = g * hL, ghR = g * hR;
        const double rL = fast_rsqrt(ghL), rR = fast_rsqrt(ghR);
        const double aL = ghL * rL, aR = ghR * rR;
        const double hs_sum = hL + hR, as_sum = aR + aL;
        const double h0 = 0.5 * hs_sum - (uR - uL) * hs_sum * (0.25 * fast_rcp(as_sum)); // eq.(21)
        double hs;
        if (h0 <= fmin(hL, hR)) {                           // rarefaction, eq.(22), R-6
            const double w = fmax(0.5 * as_sum + 0.25 * (uL - uR), 0.0);
            hs = w * w * inv_g;
        } else {                                            // shock, eq.(23)
            const double k0 = 0.5 * g * fast_rcp(h0);       // g / (2 h0)
            const double xL = k0 * (h0 + hL) * (g * rL * rL);   // g (h0+hL) / (2 h0 hL)
            const double xR = k0 * (h0 + hR) * (g * rR * rR);
            const double gL = xL * fast_rsqrt(xL), gR = xR * fast_rsqrt(xR);
            hs = ((hL * gL + hR * gR) + (uL - uR)) * fast_rcp(gL + gR);
        }
        SL = uL - aL; SR = uR + aR;                         // eq.(19) with p_k = 1
        if (hs > hL) {                                      // eq.(20), R-7
            const double x = 0.5 * g * hs * (hs + hL) * (g * rL * rL);
            SL = uL - x * fast_rsqrt(x);
        }
        if (hs > hR) {
            const double x = 0.5 * g * hs * (hs + hR) * (g * rR * rR);
            SR = uR + x * fast_rsqrt(x);
        }
    }
    const double qL = hL * uL, qR = hR * uR;
    const double GL1 = qL * uL + 0.5 * g * hL * hL, GR1 = qR * uR + 0.5 * g * hR * hR;
    if (SL >= 0.0) { G0 = qL; G1 = GL1; G2 = qL * vL; return; }                  // eq.(17), R-11
    if (SR <= 0.0) { G0 = qR; G1 = GR1; G2 = qR * vR; return; }
    const double inv = fast_rcp(SR - SL);
    G0 = ((SR * qL - SL * qR) + SR * SL * (hR - hL)) * inv;                      // eq.(18)
    G1 = GL1 + SL * (SR * (qR - qL) - (GR1 - GL1)) * inv;                        // eq.(18), R-12
    // eq.(24)-(26), R-16: the tangential velocity is upwinded by the sign of S*.  The numerator
    // of eq.(25) equals -(SR-SL) G0 and its denominator is negative, so sign(S*) = sign(G0);
    // in the dry-bed cases eq.(26) sets S* = SL (left dry) or SR (right dry), the same sign.
    G2 = G0 * (G0 >= 0.0 ? vL : vR);
}

// ---- one edge: a2-a7 of SURVEY.md section 8(a) -------------------------------------------------
// o[0] = L G0, (o[1], o[2]) = L (F - sb_a n), (o[3], o[4]) = L (F - sb_b n) with F = T^-1 G~ in
// the frame of a's outward normal n.  Side a subtracts (o0,o1,o2)/|Omega_a|, side b adds
// (o0,o3,o4)/|Omega_b| (its outward normal is -n).
__device__ __forceinline__ void edge_eval(const Params &P, const EdgeRec &er, const Rec &A,
                                          const Rec &B, double o[5])
{
    const double g = P.g, hdry = P.hdry;
    const double n1 = er.n1, n2 = er.n2;
    const double uL = A.u * n1 + A.v * n2, vL = A.v * n1 - A.u * n2;             // eq.(12)
    double G0, G1, G2, sba = 0.0, sbb = 0.0;
    if (er.b >= 0) {
        // a2: hydrostatic reconstruction, eq.(28), R-14
        const double zf = fmax(A.z, B.z);
        const double hL = fmax(0.0, A.h + (A.z - zf));
        const double hR = fmax(0.0, B.h + (B.z - zf));
        const double uR = B.u * n1 + B.v * n2, vR = B.v * n1 - B.u * n2;
        hllc_flux(g, P.inv_g, hdry, hL, uL, vL, hR, uR, vR, G0, G1, G2);
        // bathymetry source eq.(30) with g/2 (R-13), one value per side
        sba = 0.5 * g * (hL * hL - A.h * A.h);
        sbb = 0.5 * g * (hR * hR - B.h * B.h);
    } else {                                    // a6: boundary edge
        const int tag = -er.b;
        const double hL = A.h;
        const double pr = 0.5 * g * hL * hL;
        if (tag == SWE_BC_WALL) { G0 = 0.0; G1 = pr; G2 = 0.0; }                 // R-4
        else if (tag == SWE_BC_TRANSMISSIVE) {                                    // R-21
            if (hL > hdry) { G0 = hL * uL; G1 = G0 * uL + pr; G2 = G0 * vL; }
            else { G0 = 0.0; G1 = 0.0; G2 = 0.0; }
        } else {                                                                  // R-20
            const double qn = __ldg(P.qn_tag + tag);
            G0 = qn; G2 = 0.0;
            G1 = hL > hdry ? qn * qn * fast_rcp(hL) + pr : 0.0;
        }
    }
    // a7: rotate back (T^-1) and scale by the edge length
    const double L = er.len;
    const double Fx = G1 * n1 - G2 * n2, Fy = G1 * n2 + G2 * n1;
    o[0] = L * G0;
    o[1] = L * (Fx - sba * n1); o[2] = L * (Fy - sba * n2);
    o[3] = L * (Fx - sbb * n1); o[4] = L * (Fy - sbb * n2);
}

// ---- one cell: a7-a10, eq.(37), PAPER.md:250 ---------------------------------------------------
// so = the tile's edge outputs in shared memory (SoA, stride ME).  Returns the local rate
// (sqrt(g h') + |V'|) / R_i of the new state (0 if dry), eq.(15).
__device__ __forceinline__ double cell_update(const Params &P, const Rec &Ui, const CellRec &ct,
                                              const double *so, const int ME, const double dt,
                                              Rec &Un, unsigned &nclamp)
{
    const double g = P.g, hdry = P.hdry;
    const double hi = Ui.h, ui = Ui.u, vi = Ui.v;
    // three edges in the fixed order k = 0,1,2 (R-17)
    double s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const uint32_t w = k == 0 ? ct.slots01 : k == 1 ? ct.slots01 >> 16 : ct.slots2;
        const int e = (int)(w & 0x7fffu);
        const bool bside = (w & 0x8000u) != 0;
        const double *q = so + e;
        const double o0 = q[0];
        const double ox = q[(bside ? 3 : 1) * ME], oy = q[(bside ? 4 : 2) * ME];
        if (bside) { s1 -= o0; s2 -= ox; s3 -= oy; } else { s1 += o0; s2 += ox; s3 += oy; }
    }
    const double b1 = -ct.inv_area * s1, b2 = -ct.inv_area * s2, b3 = -ct.inv_area * s3;
    // a8: semi-implicit friction, eq.(32)-(37), R-19
    const double qx = hi * ui, qy = hi * vi;
    const double dh = dt * b1;
    double r2 = dt * b2, r3 = dt * b3, dqx, dqy;
    const double qq2 = qx * qx + qy * qy;
    if (hi > hdry && ct.gm2 > 0.0 && qq2 > 1e-200) {
        const double rq = fast_rsqrt(qq2), qq = qq2 * rq;
        const double c3 = (hi > 1e-28 && hi < 1e28) ? fast_rcbrt(hi) : rcbrt(hi);   // h^(-1/3)
        const double c32 = c3 * c3, rh = c32 * c3;              // h^(-2/3), 1/h
        const double cfr = ct.gm2 * (rh * rh) * c3;             // g m^2 / h^(7/3)
        const double S2 = -cfr * qx * qq, S3 = -cfr * qy * qq;
        const double k73 = (7.0 / 3.0) * cfr * qq * rh;
        const double J21 = k73 * qx, J31 = k73 * qy;
        const double J22 = -cfr * (qq + qx * qx * rq), J33 = -cfr * (qq + qy * qy * rq);
        const double J23 = -cfr * qx * qy * rq;
        const double hdt = 0.5 * dt;
        r2 += dt * S2 + hdt * J21 * dh;
        r3 += dt * S3 + hdt * J31 * dh;
        const double a22 = 1.0 - hdt * J22, a33 = 1.0 - hdt * J33, a23 = -hdt * J23;
        const double rdet = fast_rcp(a22 * a33 - a23 * a23);
        dqx = (r2 * a33 - a23 * r3) * rdet;
        dqy = (a22 * r3 - a23 * r2) * rdet;
    } else { dqx = r2; dqy = r3; }
    // a9: update, dry handling (R-15)
    double hn = hi + dh;
    const double qxn = qx + dqx, qyn = qy + dqy;
    if (hn < 0.0) { hn = 0.0; nclamp++; }
    Un.h = hn; Un.z = Ui.z;
    double rate = 0.0;
    if (hn > hdry) {
        const double rhn = fast_rcp(hn);
        Un.u = qxn * rhn; Un.v = qyn * rhn;
        // a10: local rate of the new state, eq.(15) with d = R_i
        const double ghn = g * hn, a = ghn * fast_rsqrt(ghn);
        const double v2 = Un.u * Un.u + Un.v * Un.v;
        const double vm = v2 > 1e-200 ? v2 * fast_rsqrt(v2) : 0.0;
        rate = (a + vm) * ct.inv_R;
    } else { Un.u = 0.0; Un.v = 0.0; }
    return rate;
}

// ---- one tile ------------------------------------------------------------------------------------
// smem: Rec srec[blockDim.x] followed by double so[5][ME].  Two block barriers per tile; the
// caller needs none between tiles (srec is read only before the second barrier, so is written
// only after the next tile's first barrier).
template <bool kReadOnlyPath>
__device__ __forceinline__ double process_tile(const Params &P, const Rec *__restrict__ Uin,
                                               Rec *__restrict__ Uout, const int tile,
                                               const double dt, unsigned &nclamp,
                                               unsigned char *smem)
{
    const int TC = blockDim.x, tid = threadIdx.x, ME = P.max_edges;
    const int base = tile * TC, i = base + tid;
    const bool active = i < P.nt;
    Rec *srec = reinterpret_cast<Rec *>(smem);
    double *so = reinterpret_cast<double *>(smem + (size_t)TC * sizeof(Rec));
    const int e0 = __ldg(P.estart + tile), ne = __ldg(P.estart + tile + 1) - e0;
    // ---- phase 0
    Rec Ui; CellRec ct;
    if (active) {
        Ui = load_rec<kReadOnlyPath>(Uin + i);
        ct = load_cell(P.cells + i);
    }
    EdgeRec er; Rec A, B;
    bool offA = false, offB = false;
    if (tid < ne) {
        er = load_edge(P.edges + e0 + tid);
        offA = (unsigned)(er.a - base) >= (unsigned)TC;
        offB = er.b >= 0 && (unsigned)(er.b - base) >= (unsigned)TC;
        if (offA) A = load_rec<kReadOnlyPath>(Uin + er.a);
        if (offB) B = load_rec<kReadOnlyPath>(Uin + er.b);
    }
    if (active) srec[tid] = Ui;
    __syncthreads();
    // ---- phase 1: every edge of the tile once
    for (int e = tid; e < ne; e += TC) {
        if (e != tid) {
            er = load_edge(P.edges + e0 + e);
            offA = (unsigned)(er.a - base) >= (unsigned)TC;
            offB = er.b >= 0 && (unsigned)(er.b - base) >= (unsigned)TC;
            if (offA) A = load_rec<kReadOnlyPath>(Uin + er.a);
            if (offB) B = load_rec<kReadOnlyPath>(Uin + er.b);
        }
        if (!offA) A = srec[er.a - base];
        if (er.b >= 0 && !offB) B = srec[er.b - base];
        double o[5];
        edge_eval(P, er, A, B, o);
#pragma unroll
        for (int c = 0; c < 5; c++) so[c * ME + e] = o[c];
    }
    __syncthreads();
    // ---- phase 2: every cell of the tile
    double rate = 0.0;
    if (active) {
        Rec Un;
        rate = cell_update(P, Ui, ct, so, ME, dt, Un, nclamp);
        store_rec(Uout + i, Un);
    }
    return rate;
}

} // namespace swe
