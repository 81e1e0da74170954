// Device code of libswe_b200: the fused, tiled, edge-once SWE step for sm_100a (FP64).
//
// The cells are numbered along a space-filling curve (mesh_builder.cpp) and cut into tiles of
// blockDim.x consecutive cells.  A thread block walks tiles through a software pipeline:
//
//   stage    one elected thread issues TMA bulk copies (cp.async.bulk, mbarrier complete_tx)
//            for the tile's CONTIGUOUS streams: the state records of its cells, its edge list,
//            its info block (halo ids).  The copies for tile n+1 are in flight while tile n is
//            computed; nothing passes through registers.  Halo records and cell constants come
//            by per-thread cp.async.  A tile whose cells and halo are all dry (and that has no
//            inflow edge) copies its records and skips everything else; the edge list of a tile
//            that was like that at the previous step is not even requested.
//   phase 1  (edge-parallel) every edge that touches the tile is evaluated ONCE: hydrostatic
//            reconstruction, rotation, HLLC flux, rotation back, both sides' bathymetry source;
//            the signed, length-weighted result goes to the (cell, local edge) slots of its end
//            points in shared memory (a1-a7 of SURVEY.md section 8(a)).  End points in another
//            tile are the only gathers from global memory (one 32-byte sector each).
//   phase 2  (cell-parallel) every cell sums its three slots in the fixed order k = 0,1,2,
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
// with a third-order correction (measured max error 1.1-1.5e-16, no special-case handling:
// every argument is a normal positive number by construction) instead of the IEEE-rounded
// sequences.  DESIGN.md section 7 derives why this stays inside the 1e-10 parity bar.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace swe {

struct __align__(32) Rec { double h, u, v, z; };

// One edge of a tile (24 bytes).  a is always a cell; b is a cell, or -(tag + 128 * boundary edge
// number) on a boundary edge.  (lx, ly) = edge length times a's unit outward normal (so b's is
// its negative): the unit normal and the length come from one rsqrt(lx^2 + ly^2), and the
// length-weighted flux needs neither.  a is the end point with the smaller CALLER id, which
// makes the result independent of the renumbering (R-17).
// Bits 0-28 of a and b: position in the tile's shared-memory record array (< tile size: the
// tile's own cell with that local index; >= tile size: entry of the tile's halo list);
// bits 29-30: the local edge index k of this edge in that cell.
struct __align__(8) EdgeRec { int32_t a, b; double lx, ly; };
constexpr int kIdBits = 29;
constexpr int32_t kIdMask = (1 << kIdBits) - 1;

struct Ctrl {                 // device-resident loop state
    double t[2];              // simulated time of the state in U0 / U1 (ping-pong like the state: every
                              // block reads t[cur] while block 0 writes t[cur ^ 1])
    double dt;                // step the next update will use (valid after a finalise)
    double dt_last;           // step used by the latest update
    double t_end;             // the step that would pass t_end ends on it (swe_run_until); +inf otherwise
    long long steps;
    unsigned long long n_clamped;
    unsigned long long n_active;  // tiles that were not all dry, summed over the steps (diagnostics)
    int all_dry;              // set when a step found no wet cell
    int bad_cell;             // smallest caller id with a negative depth or a non-finite value (swe_set_state)
};

struct Params {
    Rec *U0, *U1;             // ping-pong state, internal order
    const double *cellc;      // [ntiles][3][tile] per tile: 1/|Omega|, 1/R, g m^2 (SoA, padded)
    const EdgeRec *edges;     // [estart[ntiles]] tile after tile
    const int32_t *tinfo;     // [ntiles][4 + max_halo] per-tile info block, see "the tile pipeline"
    const double *qn_tag;     // [128] unit discharge along the outward normal per inflow tag
    double *bvol;             // [boundary edges] cumulative outward volume through each boundary edge
    int4 *hint;               // [ntiles] .x = 1 if the tile was active (not all dry) at the previous step
                              // (16-byte entries: fetched with cp.async.cg, which bypasses L1)
    double *pmax0, *pmax1;    // [npart] per-block max rate of state U0 / U1
    Ctrl *ctrl;
    int32_t nt, ntiles, npart, max_edges, max_halo;
    int32_t hll;              // 1: plain HLL for the tangential momentum too (SWE_RIEMANN_HLL)
    double g, hg, inv_g, cfl, hdry;   // hg = g/2
    // selected with a ternary so the kernel parameter block is never indexed dynamically
    __host__ __device__ __forceinline__ Rec *U(int c) const { return c ? U1 : U0; }
    __host__ __device__ __forceinline__ double *pmax(int c) const { return c ? pmax1 : pmax0; }
};

// ---- 256-bit access --------------------------------------------------------------------------
// Gather of a record of another tile: L2-coherent (.cg), because in the persistent loop other
// blocks rewrote the state before the grid barrier; L1 would add nothing (each such record is
// used about once per tile).
__device__ __forceinline__ Rec load_rec(const Rec *p)
{
    Rec r;
    asm volatile("ld.global.cg.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(r.h), "=d"(r.u), "=d"(r.v), "=d"(r.z) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void store_rec(Rec *p, const Rec &r)
{
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "d"(r.h), "d"(r.u), "d"(r.v), "d"(r.z) : "memory");
}
// ---- MUFU-seeded FP64 reciprocal / rsqrt / rcbrt ---------------------------------------------
// Arguments are finite, normal and positive at every call site (depths above the wet/dry
// threshold, sums of celerities, S_R - S_L in the star region, determinants >= 1).
// Seed relative error e0 <= ~2^-20; the corrections below leave O(e0^3) + rounding: measured
// max relative error 1.1e-16 (rcp), 1.4e-16 (rsqrt), 1.5e-16 (rcbrt) over 2^-60..2^60.
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
// section 4) except that
//   - a_k = sqrt(g h_k) and 1/h_k both come from one rsqrt(g h_k);
//   - a_k p_k of eq.(19)-(20) is formed as sqrt(g m (m+h_k) / (2 h_k)) with m = max(h*, h_k):
//     one square root, and no branch because the formula gives a_k at m = h_k (R-7 continuity).
// hg = g/2.
__device__ __forceinline__ void hllc_flux(const double g, const double hg, const double inv_g,
                                          const double hdry, double hL, double uL, double vL,
                                          double hR, double uR, double vR, const double pL,
                                          const double pR, const bool hll, double &G0, double &G1,
                                          double &G2)
{
    const bool dL = hL <= hdry, dR = hR <= hdry;           // R-15
    G0 = 0.0; G1 = 0.0; G2 = 0.0;
    if (dL && dR) return;
    double SL, SR, GL1 = pL, GR1 = pR;                      // pressure parts g h^2 / 2
    if (dL) {                                               // eq.(26) line 1
        hL = 0.0; uL = 0.0; vL = 0.0; GL1 = 0.0;
        const double ghR = g * hR, aR = ghR * fast_rsqrt(ghR);
        SL = uR - 2.0 * aR; SR = uR + aR;
    } else if (dR) {                                        // eq.(26) line 2 (R-18)
        hR = 0.0; uR = 0.0; vR = 0.0; GR1 = 0.0;
        const double ghL = g * hL, aL = ghL * fast_rsqrt(ghL);
        SL = uL - aL; SR = uL + 2.0 * aL;
    } else {
        const double ghL = g * hL, ghR = g * hR;
        const double rL = fast_rsqrt(ghL), rR = fast_rsqrt(ghR);
        const double aL = ghL * rL, aR = ghR * rR;
        const double ihL = g * (rL * rL), ihR = g * (rR * rR);          // 1/h_k
        const double hsum = hL + hR, asum = aR + aL, du = uL - uR;
        const double h0 = fma(du * hsum, 0.25 * fast_rcp(asum), 0.5 * hsum);   // eq.(21)
        double hs;
        if (h0 <= fmin(hL, hR)) {                           // rarefaction, eq.(22), R-6
            const double w = fmax(fma(0.25, du, 0.5 * asum), 0.0);
            hs = w * w * inv_g;
        } else {                                            // shock, eq.(23)
            const double k0 = hg * fast_rcp(h0);            // g / (2 h0)
            const double xL = k0 * (h0 + hL) * ihL;         // g (h0+hL) / (2 h0 hL)
            const double xR = k0 * (h0 + hR) * ihR;
            const double gL = xL * fast_rsqrt(xL), gR = xR * fast_rsqrt(xR);
            hs = ((hL * gL + hR * gR) + du) * fast_rcp(gL + gR);
        }
        // eq.(19)-(20), R-7
        const double mL = fmax(hs, hL), mR = fmax(hs, hR);
        const double yL = hg * mL * (mL + hL) * ihL, yR = hg * mR * (mR + hR) * ihR;
        SL = uL - yL * fast_rsqrt(yL);
        SR = uR + yR * fast_rsqrt(yR);
    }
    const double qL = hL * uL, qR = hR * uR;
    GL1 = fma(qL, uL, GL1); GR1 = fma(qR, uR, GR1);
    if (SL >= 0.0) { G0 = qL; G1 = GL1; G2 = qL * vL; return; }                  // eq.(17), R-11
    if (SR <= 0.0) { G0 = qR; G1 = GR1; G2 = qR * vR; return; }
    const double inv = fast_rcp(SR - SL);
    G0 = ((SR * qL - SL * qR) + SR * SL * (hR - hL)) * inv;                      // eq.(18)
    G1 = GL1 + SL * (SR * (qR - qL) - (GR1 - GL1)) * inv;                        // eq.(18), R-12
    // eq.(24)-(26), R-16: the tangential velocity is upwinded by the sign of S*.  The numerator
    // of eq.(25) equals -(SR-SL) G0 and its denominator is negative, so sign(S*) = sign(G0);
    // in the dry-bed cases eq.(26) sets S* = SL (left dry) or SR (right dry), the same sign.
    G2 = G0 * (G0 >= 0.0 ? vL : vR);
    // plain HLL: eq.(18) for the third component too
    if (hll) G2 = ((SR * (qL * vL) - SL * (qR * vR)) + SR * SL * (hR * vR - hL * vL)) * inv;
}

// ---- one edge: a2-a7 of SURVEY.md section 8(a) -------------------------------------------------
// o[0] = L G0, (o[1], o[2]) = L (F - sb_a n), (o[3], o[4]) = L (F - sb_b n) with F = T^-1 G~ in
// the frame of a's outward normal n.  Side a subtracts (o0,o1,o2)/|Omega_a|, side b adds
// (o0,o3,o4)/|Omega_b| (its outward normal is -n).
__device__ __forceinline__ void edge_eval(const Params &P, const EdgeRec &er, const Rec &A,
                                          const Rec &B, const double dt, double o[5])
{
    const double g = P.g, hg = P.hg, hdry = P.hdry;
    const double lx = er.lx, ly = er.ly;
    const double L2 = fma(lx, lx, ly * ly), rl = fast_rsqrt(L2);
    const double n1 = lx * rl, n2 = ly * rl;                                    // unit outward normal of a
    const double uL = fma(A.u, n1, A.v * n2), vL = fma(A.v, n1, -(A.u * n2));    // eq.(12)
    double G0, G1, G2, sba = 0.0, sbb = 0.0;
    if (er.b >= 0) {
        // a2: hydrostatic reconstruction, eq.(28), R-14
        const double zf = fmax(A.z, B.z);
        const double hL = fmax(0.0, A.h + (A.z - zf));
        const double hR = fmax(0.0, B.h + (B.z - zf));
        const double uR = fma(B.u, n1, B.v * n2), vR = fma(B.v, n1, -(B.u * n2));
        const double hL2 = hL * hL, hR2 = hR * hR;
        hllc_flux(g, hg, P.inv_g, hdry, hL, uL, vL, hR, uR, vR, hg * hL2, hg * hR2, P.hll != 0, G0, G1, G2);
        // bathymetry source eq.(30) with g/2 (R-13), one value per side
        sba = hg * (hL2 - A.h * A.h);
        sbb = hg * (hR2 - B.h * B.h);
    } else {                                    // a6: boundary edge
        const int tag = (-er.b) & 127;
        const double hL = A.h;
        const double pr = hg * hL * hL;
        if (tag == SWE_BC_WALL) { G0 = 0.0; G1 = pr; G2 = 0.0; }                 // R-4
        else if (tag == SWE_BC_TRANSMISSIVE) {                                    // R-21
            if (hL > hdry) { G0 = hL * uL; G1 = G0 * uL + pr; G2 = G0 * vL; }
            else { G0 = 0.0; G1 = 0.0; G2 = 0.0; }
        } else {                                                                  // R-20
            const double qn = __ldg(P.qn_tag + tag);
            G0 = qn; G2 = 0.0;
            G1 = hL > hdry ? qn * qn * fast_rcp(hL) + pr : 0.0;
        }
        // boundary diagnostics: volume that left through this edge so far.  One
        // writer per edge, so the sum is deterministic; walls carry no mass.
        if (tag != SWE_BC_WALL) P.bvol[(-er.b) >> 7] += G0 * (L2 * rl) * dt;
    }
    // a7: rotate back (T^-1) and scale by the edge length: L (G1 n - G2 t) = G1 l - G2 l_perp
    const double LFx = G1 * lx - G2 * ly, LFy = G1 * ly + G2 * lx;
    o[0] = (L2 * rl) * G0;
    o[1] = fma(-sba, lx, LFx); o[2] = fma(-sba, ly, LFy);
    o[3] = fma(-sbb, lx, LFx); o[4] = fma(-sbb, ly, LFy);
}

// ---- one cell: a7-a10, eq.(37), PAPER.md:250 ---------------------------------------------------
// (s1,s2,s3) = sum over the three edges of the signed, length-weighted flux + source.  Returns
// the local rate (sqrt(g h') + |V'|) / R_i of the new state (0 if dry), eq.(15).
__device__ __forceinline__ double cell_update(const Params &P, const Rec &Ui, const double s1,
                                              const double s2, const double s3,
                                              const double inv_area, const double inv_R,
                                              const double gm2, const double dt, Rec &Un,
                                              unsigned &nclamp)
{
    const double g = P.g, hdry = P.hdry;
    const double hi = Ui.h, ui = Ui.u, vi = Ui.v;
    const double b1 = -inv_area * s1, b2 = -inv_area * s2, b3 = -inv_area * s3;
    // a8: semi-implicit friction, eq.(32)-(37), R-19
    const double qx = hi * ui, qy = hi * vi;
    const double dh = dt * b1;
    double r2 = dt * b2, r3 = dt * b3, dqx, dqy;
    const double qq2 = qx * qx + qy * qy;
    if (hi > hdry && gm2 > 0.0 && qq2 > 1e-200) {
        const double rq = fast_rsqrt(qq2), qq = qq2 * rq;
        const double c3 = (hi > 1e-28 && hi < 1e28) ? fast_rcbrt(hi) : rcbrt(hi);   // h^(-1/3)
        const double c32 = c3 * c3, rh = c32 * c3;              // h^(-2/3), 1/h
        const double cfr = gm2 * (rh * rh) * c3;                // g m^2 / h^(7/3)
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
        // a zero step (t_end reached, swe_run_until) must not change a bit: (h u) / h is not u
        if (dt == 0.0) { Un.u = ui; Un.v = vi; }
        // a10: local rate of the new state, eq.(15) with d = R_i
        const double ghn = g * hn, a = ghn * fast_rsqrt(ghn);
        const double v2 = Un.u * Un.u + Un.v * Un.v;
        const double vm = v2 > 1e-200 ? v2 * fast_rsqrt(v2) : 0.0;
        rate = (a + vm) * inv_R;
    } else { Un.u = 0.0; Un.v = 0.0; }
    return rate;
}

// ---- TMA bulk copy + mbarrier (sm_90+/sm_100a) ---------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                 :: "r"(smem_u32(bar)), "r"(parity) : "memory");
}
// bytes: multiple of 16; src and dst 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// per-thread asynchronous copies (LDGSTS): no registers, completion by cp.async.wait_group
__device__ __forceinline__ void cp_async16(void *dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async8(void *dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory");
}

// ---- the tile pipeline -----------------------------------------------------------------------------
// Per-tile info block in global memory (P.tinfo, fixed stride 4 + MH int32, MH = P.max_halo):
//   [0] first edge of the tile in P.edges   [1] number of edges   [2] number of halo ids
//   [3] 1 if an inflow edge touches it      [4..] halo ids (internal cell ids), padded with -1
// Shared memory of one block (dynamic); TC = blockDim.x, ME = P.max_edges:
//   double  so[3][3 TC + 5]        (local edge k)(component, cell) flux slots of the tile's cells; the 5
//                                  doubles of padding put the three slots of one cell in different banks
//                                  (two edges of a cell are usually evaluated by adjacent lanes)
//   Rec     srec[2][TC + MH]       state records of the tile's cells, then of its halo cells
//   EdgeRec sedge[2][ME]           the tile's edge list (24-byte records, ME even)
//   double  scell[3][TC]           1/|Omega|, 1/R, g m^2
//   int32   sinfo[3][4 + MH]       info blocks (three tiles deep)
//   uint64  bar[7]                 rec[2], info[3], edge[2]
//   int32   eflag[2]               was the edge list of the tile in stage s requested?
//   int4    shint[4]               P.hint entries of the next tiles (cp.async by the producer thread)
// Schedule for the block's n-th tile (s = n & 1), all copies asynchronous and one tile ahead
// (measured: with the edge list issued only after the edge phase, blocks spent 26 % of their
// time waiting for it):
//   top      wait: own halo gathers, records and edge list of tile n; barrier (= the dry vote)
//            issue: records of tile n+1 (bulk) -> srec[s^1]; edge list of tile n+1 (bulk) ->
//                   sedge[s^1]; info block of tile n+2 (bulk); cell constants of tile n
//                   (cp.async); halo gathers of tile n+1 (cp.async, its info block landed one
//                   tile ago) -> srec[s^1][TC..]
//   phase 1  edges: shared memory only
//   mid      barrier
//   phase 2  cells
constexpr int kInfoHdr = 4;
template <int TC> struct SlotLayout { static constexpr int plane = 3 * TC + 5; static constexpr int doubles = 3 * plane + 4; };
constexpr int kNumBars = 7;
__host__ __device__ __forceinline__ size_t tile_smem_bytes(int TC, int MH, int ME)
{
    return ((size_t)TC * 9 + 28) * sizeof(double) + 2 * (size_t)(TC + MH) * sizeof(Rec) +
           2 * (size_t)ME * sizeof(EdgeRec) + (size_t)TC * 3 * sizeof(double) +
           3 * (size_t)(kInfoHdr + MH) * sizeof(int32_t) + kNumBars * sizeof(uint64_t) + 32 + 4 * sizeof(int4);
}
template <int TC> struct TilePipe {
    double *so; Rec *srec0; EdgeRec *sedge0; double *scell; int32_t *sinfo0; uint64_t *bar;
    int edge_stride;
    __device__ __forceinline__ EdgeRec *sedge(int s) const { return sedge0 + s * edge_stride; }
    int rec_stride, info_stride;
    __device__ __forceinline__ Rec *srec(int s) const { return srec0 + s * rec_stride; }
    __device__ __forceinline__ int32_t *sinfo(int j) const { return sinfo0 + j * info_stride; }
    __device__ __forceinline__ uint64_t *rbar(int s) const { return bar + s; }
    __device__ __forceinline__ uint64_t *ibar(int j) const { return bar + 2 + j; }
    __device__ __forceinline__ uint64_t *ebar(int s) const { return bar + 5 + s; }
    // eflag[s]: bit 0 = an edge-list copy into sedge[s] was issued for the tile that uses stage s,
    // bit 1 = parity to wait for on ebar(s); ecnt[s] (producer only) = completed copies into stage s
    __device__ __forceinline__ volatile int32_t *eflag() const { return reinterpret_cast<volatile int32_t *>(bar + kNumBars); }
    // ring of hints fetched ahead by the producer thread
    __device__ __forceinline__ volatile int32_t *ecnt() const { return reinterpret_cast<volatile int32_t *>(bar + kNumBars) + 2; }
    // nact (producer only): active tiles of this block in the current step
    __device__ __forceinline__ volatile int32_t *nact() const { return reinterpret_cast<volatile int32_t *>(bar + kNumBars) + 4; }
    __device__ __forceinline__ int4 *shint(unsigned m) const { return reinterpret_cast<int4 *>(bar + kNumBars + 3) + (m & 3u); }
};
template <int TC> __device__ __forceinline__ TilePipe<TC> make_pipe(const Params &P, unsigned char *smem)
{
    TilePipe<TC> p;
    p.rec_stride = TC + P.max_halo; p.info_stride = kInfoHdr + P.max_halo;
    p.so = reinterpret_cast<double *>(smem);                 smem += ((size_t)TC * 9 + 28) * sizeof(double);
    p.srec0 = reinterpret_cast<Rec *>(smem);                 smem += 2 * (size_t)p.rec_stride * sizeof(Rec);
    p.sedge0 = reinterpret_cast<EdgeRec *>(smem);            smem += 2 * (size_t)P.max_edges * sizeof(EdgeRec);
    p.edge_stride = P.max_edges;
    p.scell = reinterpret_cast<double *>(smem);              smem += (size_t)TC * 3 * sizeof(double);
    p.sinfo0 = reinterpret_cast<int32_t *>(smem);            smem += 3 * (size_t)p.info_stride * sizeof(int32_t);
    p.bar = reinterpret_cast<uint64_t *>(smem);
    return p;
}

// single-thread issue helpers
template <int TC> __device__ __forceinline__ void issue_recs(const Params &P, const TilePipe<TC> &pp,
                                                             const Rec *Uin, const int tile, const int s)
{
    const int base = tile * TC, nc = min(TC, P.nt - base);
    mbar_expect_tx(pp.rbar(s), (unsigned)nc * sizeof(Rec));
    bulk_g2s(pp.srec(s), Uin + base, (unsigned)nc * sizeof(Rec), pp.rbar(s));
}
template <int TC> __device__ __forceinline__ void issue_edges(const Params &P, const TilePipe<TC> &pp,
                                                              const int e0, const int ne, const int s)
{
    const unsigned bytes = (unsigned)((ne + 1) & ~1) * sizeof(EdgeRec);      // lists are padded to 16 bytes
    mbar_expect_tx(pp.ebar(s), bytes);
    bulk_g2s(pp.sedge(s), P.edges + e0, bytes, pp.ebar(s));
}
template <int TC> __device__ __forceinline__ void issue_info(const Params &P, const TilePipe<TC> &pp,
                                                             const int tile, const int j)
{
    const unsigned bytes = (unsigned)pp.info_stride * sizeof(int32_t);
    mbar_expect_tx(pp.ibar(j), bytes);
    bulk_g2s(pp.sinfo(j), P.tinfo + (size_t)tile * pp.info_stride, bytes, pp.ibar(j));
}
// all threads: gather the halo records listed in info block j into srec[s][TC..]
template <int TC> __device__ __forceinline__ void gather_halo(const TilePipe<TC> &pp, const Rec *Uin,
                                                              const int j, const int s)
{
    const int32_t *info = pp.sinfo(j);
    const int nh = info[2];
    Rec *dst = pp.srec(s) + TC;
    for (int q = TC - 1 - (int)threadIdx.x; q < nh; q += TC) {        // last warps first: they have slack
        const char *src = reinterpret_cast<const char *>(Uin + info[kInfoHdr + q]);
        cp_async16(reinterpret_cast<char *>(dst + q), src);
        cp_async16(reinterpret_cast<char *>(dst + q) + 16, src + 16);
    }
}

// Pipeline state carried across the steps of a persistent launch: tiles pushed through so far
// (fixes buffers and barrier parities).  The edge barriers complete a phase only when a list was
// requested, so their parity is kept by the producer thread in shared memory (ecnt) and published
// with the request flag: eflag[s] = requested | parity << 1.
struct PipeState { unsigned n = 0; };

// All the tiles of this block for one time step.
// Returns this thread's maximum rate contribution.
template <int TC>
__device__ __forceinline__ double step_tiles(const Params &P, const TilePipe<TC> &pp,
                                             const Rec *__restrict__ Uin, Rec *__restrict__ Uout,
                                             const double dt, unsigned &nclamp, PipeState &ps)
{
    const int tid = threadIdx.x, G = gridDim.x;
    double rate = 0.0;
    unsigned n = ps.n;
    int tile = blockIdx.x;
    if (tile >= P.ntiles) return 0.0;
    // ---- prologue: everything tile n needs, and the info block of tile n+1
    // the copies are issued by lane 0 of the LAST warp: the edge loop gives the first warps one more
    // iteration than the last ones (ne ~ 1.66 TC), so the last warp has the slack (measured: with
    // thread 0 as producer warp 0 reached the mid barrier ~1000 cycles late)
    const bool producer = tid == TC - 32;
    // Edge lists are 40 of the ~105 bytes a cell costs and an all-dry tile never reads its list, so
    // the list of the NEXT tile is requested only if that tile was active at the previous step
    // (P.hint, read one tile early); a tile that turns out active without its list (the wet front
    // reached it) fetches it on the spot.
    if (producer) {
        issue_info(P, pp, tile, n % 3);
        issue_recs(P, pp, Uin, tile, n & 1);
        const int32_t *gi = P.tinfo + (size_t)tile * pp.info_stride;
        issue_edges(P, pp, __ldg(gi), __ldg(gi + 1), n & 1);      // the step's first tile: always
        pp.eflag()[n & 1] = 1 | ((pp.ecnt()[n & 1] & 1) << 1);
        if (tile + G < P.ntiles) {
            issue_info(P, pp, tile + G, (n + 1) % 3);
            cp_async16(pp.shint(n + 1), P.hint + tile + G);           // lands before the first barrier
        }
    }
    mbar_wait(pp.ibar(n % 3), (n / 3) & 1u);
    gather_halo(pp, Uin, n % 3, n & 1);
    cp_async_commit();
    double *const so = pp.so;
    for (; tile < P.ntiles; tile += G, n++) {
        const int s = n & 1;
        const int base = tile * TC;
        const bool have_next = tile + G < P.ntiles;
        // ---- top
        cp_async_wait<0>();                               // own halo gathers of this tile
        mbar_wait(pp.rbar(s), (n >> 1) & 1u);
        const Rec *const srec = pp.srec(s);
        const EdgeRec *const sedge = pp.sedge(s);
        const int32_t *const info = pp.sinfo(n % 3);
        const int ne = info[1], nh = info[2];
        // is anything wet in the tile or its halo?  Each thread looks at its own record and at
        // the halo records it gathered itself, so the vote can BE the tile's first barrier.
        const int i = base + tid;
        bool wet = i < P.nt && srec[tid].h > P.hdry;
        if (!wet)       // a wet own cell already decides the vote
            for (int q = TC - 1 - tid; q < nh; q += TC) wet |= srec[TC + q].h > P.hdry;
        // barrier: everyone has left the previous tile; everyone's gathers are visible
        // (the warp vote only tells the compiler that the outcome is warp-uniform)
        const bool active = __any_sync(0xffffffffu, __syncthreads_or(wet) || info[3] != 0);
        if (producer && have_next) {
            issue_recs(P, pp, Uin, tile + G, s ^ 1);
            if (tile + 2 * G < P.ntiles) issue_info(P, pp, tile + 2 * G, (n + 2) % 3);
        }
        if (active && i < P.nt) {
            const double *src = P.cellc + (size_t)tile * 3 * TC + tid;
            double *dst = pp.scell + tid;
            cp_async8(dst, src); cp_async8(dst + TC, src + TC); cp_async8(dst + 2 * TC, src + 2 * TC);
        }
        cp_async_commit();
        if (have_next) {
            mbar_wait(pp.ibar((n + 1) % 3), ((n + 1) / 3) & 1u);
            if (producer) {
                const int hint_next = pp.shint(n + 1)->x;            // requested one tile ago
                pp.eflag()[s ^ 1] = (hint_next != 0) | ((pp.ecnt()[s ^ 1] & 1) << 1);
                if (hint_next) {
                    const int32_t *ni = pp.sinfo((n + 1) % 3);
                    issue_edges(P, pp, ni[0], ni[1], s ^ 1);
                }
                if (tile + 2 * G < P.ntiles) cp_async16(pp.shint(n + 2), P.hint + tile + 2 * G);
            }
            gather_halo(pp, Uin, (n + 1) % 3, s ^ 1);
        }
        cp_async_commit();
        if (producer) { P.hint[tile].x = active; if (active) *pp.nact() = *pp.nact() + 1; }
        // this tile's edge list: requested one tile ago (flag written before the barrier above),
        // or fetched now if the tile is active without it
        {
            const int f = pp.eflag()[s];
            const bool requested = (f & 1) != 0;
            if (!requested && active && producer) issue_edges(P, pp, info[0], ne, s);
            if (requested || active) {
                mbar_wait(pp.ebar(s), (unsigned)f >> 1);
                if (producer) pp.ecnt()[s] = pp.ecnt()[s] + 1;
            }
        }
        if (!active) {
            // Every cell of the tile and every neighbour is dry and no discharge is prescribed:
            // all fluxes vanish, h' = h + 0, and dry cells carry u = v = 0 already (R-15), so the
            // step leaves the records unchanged bit for bit.  The copy still moves them.
            if (i < P.nt) store_rec(Uout + i, srec[tid]);
        } else {
            // ---- phase 1: every edge of the tile once, shared memory only
            for (int e = tid; e < ne; e += TC) {
                const EdgeRec er = sedge[e];
                const int ia = er.a & kIdMask, ka = er.a >> kIdBits;
                const Rec A = srec[ia];
                Rec B;
                int ib = TC, kb = 0;
                if (er.b >= 0) { ib = er.b & kIdMask; kb = er.b >> kIdBits; B = srec[ib]; }
                double o[5];
                edge_eval(P, er, A, B, dt, o);
                if (ia < TC) {
                    double *q = so + ka * SlotLayout<TC>::plane + ia;
                    q[0] = o[0]; q[TC] = o[1]; q[2 * TC] = o[2];
                }
                if (ib < TC) {
                    double *q = so + kb * SlotLayout<TC>::plane + ib;
                    q[0] = -o[0]; q[TC] = -o[3]; q[2 * TC] = -o[4];
                }
            }
            cp_async_wait<1>();                               // this tile's cell constants
            __syncthreads();
            // ---- phase 2: every cell of the tile
            if (i < P.nt) {
                const Rec Ui = srec[tid];
                const double *sc = pp.scell + tid;
                const double *q = so + tid;
                // three edges in the fixed order k = 0,1,2 (R-17)
                constexpr int PL = SlotLayout<TC>::plane;
                const double s1 = (q[0] + q[PL]) + q[2 * PL];
                const double s2 = (q[TC] + q[PL + TC]) + q[2 * PL + TC];
                const double s3 = (q[2 * TC] + q[PL + 2 * TC]) + q[2 * PL + 2 * TC];
                Rec Un;
                rate = fmax(rate, cell_update(P, Ui, s1, s2, s3, sc[0], sc[TC], sc[2 * TC], dt, Un, nclamp));
                store_rec(Uout + i, Un);
            }
        }
    }
    cp_async_wait<0>();
    ps.n = n;
    return rate;
}

} // namespace swe
