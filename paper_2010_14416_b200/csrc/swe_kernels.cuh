// Device code of libswe_b200: the fused, tiled, edge-once SWE step for sm_100a (FP64).
//
// The cells are numbered along a space-filling curve (mesh_builder.cpp) and cut into tiles of
// blockDim.x consecutive cells.  A thread block walks tiles through a software pipeline:
//
//   stage    one elected thread issues TMA bulk copies (cp.async.bulk, mbarrier complete_tx)
//            for the tile's CONTIGUOUS streams: the state records of its cells, its edge list,
//            its cell constants.  The copies for tile n+1 are in flight while tile n is
//            computed; nothing passes through registers.  Halo records (end points in other
//            tiles) come by per-thread cp.async, one 32-byte sector each; the tile header, the
//            halo id and the activity hint a thread needs travel in its registers, loaded two
//            tiles ahead.  A tile whose cells and halo are all dry (and that has no inflow edge)
//            copies its records and skips everything else; the edge list of a tile that was
//            like that at the previous step is not even requested; and a tile that was like
//            that together with all its neighbour tiles ("quiet") never enters the pipeline and
//            is not touched at all: the previous step copied its records unchanged, so both state
//            buffers hold them already.  A block that runs out of tiles takes some from the
//            lists of others ("work stealing").
//   phase 1  (edge-parallel) every edge that touches the tile is evaluated ONCE: hydrostatic
//            reconstruction, rotation, HLLC flux, rotation back, both sides' bathymetry source;
//            the signed, length-weighted result goes to the (cell, local edge) slots of its end
//            points in shared memory (a1-a7 of SURVEY.md section 8(a)).
//   phase 2  (cell-parallel) every cell sums its three slots in the fixed order k = 0,1,2,
//            applies the semi-implicit friction and the update, writes its new record with
//            one 256-bit store and contributes (sqrt(g h)+|V|)/R of the NEW state to the block
//            maximum (a7-a11)
//
// The per-block maxima (warp shuffles + shared memory, no atomics) are reduced to dt by every
// block at the start of the next step.  PAPER.md sections 2-3 and :457.
//
// State record in HBM: {h, u, v, z} as one 32-byte sector, so a gather is exactly one sector
// whatever the ordering.  Velocities (not discharges) are stored so that the edge phase needs
// no division; the caller still sees (h, hu, hv) (pack/unpack).
//
// Arithmetic: FP64 throughout.  On a wet mesh the kernel is bound by instruction issue and the
// FP64 pipe, not by HBM (profiles/), so the code is written for few instructions: MUFU seeds
// (rcp/rsqrt.approx) with a third-order correction (measured max error 1.1-1.5e-16; every
// argument is a normal positive number by construction) instead of the IEEE-rounded division /
// square-root sequences, compare-and-select instead of fmax/fmin (no NaN can reach them), end
// point words that hold ready-made shared-memory indices, vector shared-memory accesses.
// DESIGN.md section 7 derives why this stays inside the 1e-10 parity bar.  The library is compiled
// with --fmad=false and every fused multiply-add is written out as fma(): the arithmetic is then
// fixed by the source, so the tile kernel, the cluster loop and the edge-centric kernels, which all
// instantiate edge_eval / cell_update, produce identical bits.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace swe {

struct __align__(32) Rec { double h, u, v, z; };

// Edge list of one tile as the kernel reads it (built by pack_device_edges, mesh_builder.cpp),
// nep = number of edges rounded up to even:
//   uint2   ab[nep]    end point words of a and b
//   double2 lxy[nep]   edge length times a's unit outward normal (b's is its negative): the unit
//                      normal and the length come from one rsqrt(lx^2 + ly^2)
// a is the end point with the smaller CALLER id, which makes the result independent of the
// renumbering (R-17).  End point word: bits 0-12 position in the tile's shared-memory record
// array (< tile size: the tile's own cell with that local index; >= tile size: entry of the
// tile's halo list); bits 13-14 the local edge index k of this edge in that cell; bits 16-30 the
// flux slot k * (tile size + 1) + position of a cell of the tile, kNoSlot for a halo cell.  On a
// boundary edge b = -(tag + 128 * boundary edge number) (negative).
constexpr uint32_t kPosMask = 0x1FFFu;
constexpr int kKShift = 13, kSlotShift = 16;
constexpr uint32_t kNoSlot = 0x7FFFu;

struct __align__(8) GEdge { int32_t a, b; double lx, ly; };     // 24 bytes (= HostEdge, mesh_builder.h)

struct Ctrl {                 // device-resident loop state
    double t[2];              // simulated time of the state in U0 / U1 (ping-pong like the state: every
                              // block reads t[cur] while block 0 writes t[cur ^ 1])
    double dt;                // step the next update will use (valid after a finalise)
    double dt_last;           // step used by the latest update
    double t_end;             // the step that would pass t_end ends on it (swe_run_until); +inf otherwise
    long long steps;
    unsigned long long n_clamped;
    unsigned long long n_active;  // tiles that were not all dry, summed over the steps (diagnostics)
    unsigned long long n_elists;  // edge lists fetched, summed over the steps (diagnostics)
    unsigned long long n_quiet;   // quiet tiles (left untouched), summed over the steps (diagnostics)
    unsigned long long n_stolen;  // tiles computed by a block other than their owner, summed over the steps (diagnostics)
    int all_dry;              // set when a step found no wet cell
    int bad_cell;             // smallest caller id with a negative depth or a non-finite value (swe_set_state)
};

struct Params {
    Rec *U0, *U1;             // ping-pong state, internal order
    const double *cellc;      // [ntiles][3][tile] per tile: 1/|Omega|, 1/R, g m^2 (SoA, padded)
    const double *edges;      // per-tile edge lists, tile after tile; 3 doubles (24 bytes) per edge
    const int32_t *tinfo;     // [ntiles][4 + max_halo] per-tile header + halo ids, see "the tile pipeline"
    const double *qn_tag;     // [128] unit discharge along the outward normal per inflow tag
    double *bvol;             // [boundary edges] cumulative outward volume through each boundary edge
    int32_t *act0, *act1;     // [ntiles] 1 if the tile was active (not all dry) in the step that produced U0 / U1
    const int32_t *tnbr;      // [ntiles][kNbrs] tiles owning each tile's halo cells (-1 padding; [0] = -2: never quiet)
    int32_t *binact;          // [npart] inactive tiles each block walked through in the previous step
    unsigned long long *wq;   // [npart] work word of each block's tile list: head / tail claims, see "work stealing"
    int32_t *wlist;           // [npart][wstride] tiles of each block's list that are not quiet (published when quiet tiles were looked for)
    int32_t wstride;          // = ceil(ntiles / npart)
    double *pmax0, *pmax1;    // [npart] per-block max rate of state U0 / U1
    Ctrl *ctrl;
    // edge-centric two-pass kernels only (SWE_KERNEL_EDGE_TWO_PASS; NULL otherwise)
    const GEdge *gedges;      // [nge] every edge of the mesh once: internal cell ids of a and b, (lx, ly)
    const int32_t *cedge;     // [nt][3] 2 * edge + side for local edge k of internal cell p
    double *eres;             // [nge][2][3] pass-1 results: side a (o0,o1,o2), side b (-o0,-o3,-o4)
    int32_t nge;
    int32_t nt, ntiles, npart, max_edges, max_halo;
    int32_t hll;              // 1: plain HLL for the tangential momentum too (SWE_RIEMANN_HLL)
    double g, hg, inv_g, cfl, hdry;   // hg = g/2
    // selected with a ternary so the kernel parameter block is never indexed dynamically
    __host__ __device__ __forceinline__ Rec *U(int c) const { return c ? U1 : U0; }
    __host__ __device__ __forceinline__ double *pmax(int c) const { return c ? pmax1 : pmax0; }
    __host__ __device__ __forceinline__ int32_t *act(int c) const { return c ? act1 : act0; }
};

// ---- 256-bit access --------------------------------------------------------------------------
// L2-coherent (.cg): in the persistent loop other blocks rewrote the state before the grid barrier.
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
// ---- state storage kinds (the paper's floating-point kind is configurable) ----------
// Rec  : FP64 records, 32 bytes (the default, everything in this file).
// RecF : FP32 records {h, u, v, z}, 16 bytes (SWE_FP_MIXED32): the state lives in HBM in single
//        precision, every step converts to FP64 on load, computes in FP64 and rounds on store.
//        Only the edge-centric two-pass kernels take this kind (templated on the record type).
struct __align__(16) RecF { float h, u, v, z; };
template <class R> __device__ __forceinline__ Rec ldrec(const R *p);
template <> __device__ __forceinline__ Rec ldrec<Rec>(const Rec *p) { return load_rec(p); }
template <> __device__ __forceinline__ Rec ldrec<RecF>(const RecF *p)
{
    float4 v;
    asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
    Rec r; r.h = v.x; r.u = v.y; r.v = v.z; r.z = v.w;
    return r;
}
__device__ __forceinline__ void strec(Rec *p, const Rec &r) { store_rec(p, r); }
__device__ __forceinline__ void strec(RecF *p, const Rec &r)
{
    asm volatile("st.global.v4.f32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "f"((float)r.h), "f"((float)r.u), "f"((float)r.v), "f"((float)r.z) : "memory");
}

__device__ __forceinline__ int32_t ldcg_i32(const int32_t *p)
{
    int32_t v;
    asm volatile("ld.global.cg.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// max / min of two numbers that are never NaN: one compare and one select (fmax / fmin carry a
// NaN-quieting sequence of ~8 instructions in FP64)
// (written in PTX: the compiler turns "a > b ? a : b" back into fmax)
__device__ __forceinline__ double dmax(double a, double b)
{
    double r;
    asm("{\n\t.reg .pred p;\n\tsetp.gt.f64 p, %1, %2;\n\tselp.f64 %0, %1, %2, p;\n\t}" : "=d"(r) : "d"(a), "d"(b));
    return r;
}
__device__ __forceinline__ double dmin(double a, double b)
{
    double r;
    asm("{\n\t.reg .pred p;\n\tsetp.lt.f64 p, %1, %2;\n\tselp.f64 %0, %1, %2, p;\n\t}" : "=d"(r) : "d"(a), "d"(b));
    return r;
}

// ---- shared memory through 32-bit addresses ---------------------------------------------------
// The hot loops address shared memory with one 32-bit register per array (generic pointers cost
// the conversion sequence again at every access).  Loads are volatile so that they stay between
// the barriers they were written between.
__device__ __forceinline__ double lds_f64(uint32_t a)
{
    double x;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(x) : "r"(a));
    return x;
}
__device__ __forceinline__ double2 lds_v2f64(uint32_t a)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ uint2 lds_v2u32(uint32_t a)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts_f64(uint32_t a, double x)
{
    asm volatile("st.shared.f64 [%0], %1;" :: "r"(a), "d"(x) : "memory");
}
__device__ __forceinline__ void sts_v2f64(uint32_t a, double x, double y)
{
    asm volatile("st.shared.v2.f64 [%0], {%1,%2};" :: "r"(a), "d"(x), "d"(y) : "memory");
}

// ---- MUFU-seeded FP64 reciprocal / rsqrt / sqrt / rcbrt --------------------------------------
// Arguments are finite, normal and positive at every call site (depths above the wet/dry
// threshold, sums of celerities, S_R - S_L in the star region, determinants >= 1).
// Seed relative error e0 <= ~2^-20; the corrections below leave O(e0^3) + rounding: measured
// max relative error 1.1e-16 (rcp), 1.4e-16 (rsqrt, sqrt), 1.5e-16 (rcbrt) over 2^-60..2^60.
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
// sqrt(x) alone: one instruction fewer than x * fast_rsqrt(x), same error
__device__ __forceinline__ double fast_sqrt(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double s = x * y;                    // sqrt(x) (1 - e)^(1/2)
    const double e = fma(-s, y, 1.0);
    const double p = fma(e, 0.375, 0.5);
    return fma(s * e, p, s);
}
// both 1/sqrt(x) (r) and sqrt(x) (returned)
__device__ __forceinline__ double fast_sqrt_rsqrt(double x, double &r)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double s = x * y;
    const double e = fma(-s, y, 1.0);
    const double p = fma(e, 0.375, 0.5) * e;
    r = fma(y, p, y);
    return fma(s, p, s);
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
// Inputs: reconstructed depths, normal/tangential velocities, pressure parts pL = g hL^2/2.
// Output (G0,G1,G2) = mass, normal and tangential momentum flux.  Same expression trees as the
// oracle's step list except that
//   - a_k = sqrt(g h_k) and 1/h_k both come from one rsqrt(g h_k);
//   - a_k p_k of eq.(19)-(20) is formed as sqrt(g m (m+h_k) / (2 h_k)) with m = max(h*, h_k):
//     one square root, and no branch because the formula gives a_k at m = h_k (R-7 continuity).
// hg = g/2.  The wave speeds of the three regimes (both wet; eq.(26) left dry; right dry) are
// the only part that branches; the flux itself is selected, not branched on.
__device__ __forceinline__ void hllc_flux(const double g, const double hg, const double inv_g,
                                          const double hdry, const double hL, const double uL,
                                          const double vL, const double hR, const double uR,
                                          const double vR, const double pL, const double pR,
                                          const bool hll, double &G0, double &G1, double &G2)
{
    const bool wL = hL > hdry, wR = hR > hdry;              // R-15
    double SL, SR, qL, qR, GL1, GR1, dh;
    if (wL && wR) {
        const double ghL = g * hL, ghR = g * hR;
        double rL, rR;
        const double aL = fast_sqrt_rsqrt(ghL, rL), aR = fast_sqrt_rsqrt(ghR, rR);
        const double ihL = g * (rL * rL), ihR = g * (rR * rR);          // 1/h_k
        const double hsum = hL + hR, asum = aR + aL, du = uL - uR;
        const double h0 = fma(du * hsum, 0.25 * fast_rcp(asum), 0.5 * hsum);   // eq.(21)
        double hs;
        if ((h0 <= hL) & (h0 <= hR)) {                      // rarefaction, eq.(22), R-6
            const double w = dmax(fma(0.25, du, 0.5 * asum), 0.0);
            hs = w * w * inv_g;
        } else {                                            // shock, eq.(23)
            const double k0 = hg * fast_rcp(h0);            // g / (2 h0)
            const double xL = k0 * (h0 + hL) * ihL;         // g (h0+hL) / (2 h0 hL)
            const double xR = k0 * (h0 + hR) * ihR;
            const double gL = fast_sqrt(xL), gR = fast_sqrt(xR);
            hs = (fma(hL, gL, hR * gR) + du) * fast_rcp(gL + gR);
        }
        // eq.(19)-(20), R-7
        const double mL = dmax(hs, hL), mR = dmax(hs, hR);
        const double yL = hg * mL * (mL + hL) * ihL, yR = hg * mR * (mR + hR) * ihR;
        SL = uL - fast_sqrt(yL);
        SR = uR + fast_sqrt(yR);
        qL = hL * uL; qR = hR * uR;
        GL1 = fma(qL, uL, pL); GR1 = fma(qR, uR, pR);
        dh = hR - hL;
    } else if (wR) {                                        // eq.(26) line 1: left side dry
        const double aR = fast_sqrt(g * hR);
        SL = fma(-2.0, aR, uR); SR = uR + aR;
        qL = 0.0; GL1 = 0.0; qR = hR * uR; GR1 = fma(qR, uR, pR); dh = hR;
    } else if (wL) {                                        // eq.(26) line 2 (R-18): right side dry
        const double aL = fast_sqrt(g * hL);
        SL = uL - aL; SR = fma(2.0, aL, uL);
        qR = 0.0; GR1 = 0.0; qL = hL * uL; GL1 = fma(qL, uL, pL); dh = -hL;
    } else {
        G0 = 0.0; G1 = 0.0; G2 = 0.0;
        return;
    }
    // a dry side has no tangential velocity either (R-15)
    const double tL = wL ? vL : 0.0, tR = wR ? vR : 0.0;
    // eq.(18) in the star region; eq.(17), R-11: S_L >= 0 first, then S_R <= 0 (selected below)
    const double inv = fast_rcp(SR - SL);
    const double SS = SR * SL;
    const double G0s = fma(SS, dh, fma(SR, qL, -(SL * qR))) * inv;
    const double G1s = fma(SL * inv, fma(SR, qR - qL, -(GR1 - GL1)), GL1);      // R-12
    const bool supL = SL >= 0.0, supR = SR <= 0.0;
    G0 = supL ? qL : (supR ? qR : G0s);
    G1 = supL ? GL1 : (supR ? GR1 : G1s);
    // eq.(24)-(26), R-16: the tangential velocity is upwinded by the sign of S*.  The numerator
    // of eq.(25) equals -(SR-SL) G0 and its denominator is negative, so sign(S*) = sign(G0);
    // in the dry-bed cases eq.(26) sets S* = SL (left dry) or SR (right dry), the same sign; and
    // in the supercritical cases G0 = qL > 0 / qR < 0 picks the upwind side as eq.(17) does.
    G2 = G0 * (G0 >= 0.0 ? tL : tR);
    if (hll) {       // plain HLL: eq.(18) for the third component too
        const double G2s = fma(SS, fma(hR, tR, -(hL * tL)), fma(SR, qL * tL, -(SL * (qR * tR)))) * inv;
        G2 = supL ? qL * tL : (supR ? qR * tR : G2s);
    }
}

// ---- one edge: a2-a7 of SURVEY.md section 8(a) -------------------------------------------------
// (lx, ly) = edge length times the unit outward normal n of end point a.  bword >= 0: interior edge
// with end points A and B; bword < 0: boundary edge of A, -bword = tag + 128 * boundary edge number.
// o[0] = L G0, (o[1], o[2]) = L (F - sb_a n), (o[3], o[4]) = L (F - sb_b n) with F = T^-1 G~ in the
// frame of n.  Side a subtracts (o0,o1,o2)/|Omega_a|, side b adds (o0,o3,o4)/|Omega_b| (its outward
// normal is -n).  Shared by the tiled step kernel and the edge-centric two-pass kernels.
__device__ __forceinline__ void edge_eval(const Params &P, const double lx, const double ly, const Rec &A,
                                          const Rec &B, const int32_t bword, const double dt, double o[5])
{
    const double g = P.g, hg = P.hg, hdry = P.hdry;
    const double L2 = fma(lx, lx, ly * ly);
    double rl;
    const double L = fast_sqrt_rsqrt(L2, rl);
    const double n1 = lx * rl, n2 = ly * rl;                                  // unit outward normal of a
    const double uL = fma(A.u, n1, A.v * n2), vL = fma(A.v, n1, -(A.u * n2));   // eq.(12)
    double G0, G1, G2, sba = 0.0, sbb = 0.0;
    if (bword >= 0) {
        // a2: hydrostatic reconstruction, eq.(28), R-14
        const double zf = dmax(A.z, B.z);
        const double hL = dmax(0.0, A.h + (A.z - zf));
        const double hR = dmax(0.0, B.h + (B.z - zf));
        const double uR = fma(B.u, n1, B.v * n2), vR = fma(B.v, n1, -(B.u * n2));
        const double hL2 = hL * hL, hR2 = hR * hR;
        hllc_flux(g, hg, P.inv_g, hdry, hL, uL, vL, hR, uR, vR, hg * hL2, hg * hR2, P.hll != 0, G0, G1, G2);
        // bathymetry source eq.(30) with g/2 (R-13), one value per side
        sba = hg * fma(-A.h, A.h, hL2);
        sbb = hg * fma(-B.h, B.h, hR2);
    } else {                                    // a6: boundary edge
        const int bw = -bword, tag = bw & 127;
        const double hL = A.h;
        const double pr = hg * hL * hL;
        if (tag == SWE_BC_WALL) { G0 = 0.0; G1 = pr; G2 = 0.0; }                 // R-4
        else if (tag == SWE_BC_TRANSMISSIVE) {                                    // R-21
            if (hL > hdry) { G0 = hL * uL; G1 = fma(G0, uL, pr); G2 = G0 * vL; }
            else { G0 = 0.0; G1 = 0.0; G2 = 0.0; }
        } else {                                                                  // R-20
            const double qn = __ldg(P.qn_tag + tag);
            G0 = qn; G2 = 0.0;
            G1 = hL > hdry ? fma(qn * qn, fast_rcp(hL), pr) : 0.0;
        }
        // boundary diagnostics: volume that left through this edge so far.  One
        // writer per edge, so the sum is deterministic; walls carry no mass.
        if (tag != SWE_BC_WALL) P.bvol[bw >> 7] = fma(G0 * L, dt, P.bvol[bw >> 7]);
    }
    // a7: rotate back (T^-1) and scale by the edge length: L (G1 n - G2 t) = G1 l - G2 l_perp
    const double LFx = fma(G1, lx, -(G2 * ly)), LFy = fma(G1, ly, G2 * lx);
    o[0] = L * G0;
    o[1] = fma(-sba, lx, LFx); o[2] = fma(-sba, ly, LFy);
    o[3] = fma(-sbb, lx, LFx); o[4] = fma(-sbb, ly, LFy);
}

// ---- one cell: a7-a10, eq.(37), PAPER.md:250 ---------------------------------------------------
// (s1,s2,s3) = sum over the three edges of the signed, length-weighted flux + source.  Returns
// the local rate (sqrt(g h') + |V'|) / R_i of the new state (0 if dry), eq.(15).
//
// Friction, eq.(32)-(37), R-19.  With c = g m^2 / h^(7/3), Q = |q|, D = dt c / 2 the 2x2 block of
// I - dt/2 J_f is A = (1 + D Q) I + (D/Q) q q^T, whose inverse is known in closed form
// (det A = (1 + D Q)(1 + 2 D Q)); the right-hand side dt (b + S_f) + dt/2 J_21,31 dh is
// dt b + q E with E = c Q dt (7/6 dh/h - 1).  The oracle solves the printed system by Cramer's
// rule; the two agree to rounding.
__device__ __forceinline__ double cell_update(const Params &P, const Rec &Ui, const double s1,
                                              const double s2, const double s3,
                                              const double inv_area, const double inv_R,
                                              const double gm2, const double dt, Rec &Un,
                                              unsigned &nclamp)
{
    const double g = P.g, hdry = P.hdry;
    const double hi = Ui.h, ui = Ui.u, vi = Ui.v;
    const double ndt = -dt * inv_area;
    const double dh = ndt * s1;
    double dqx = ndt * s2, dqy = ndt * s3;                  // dt b
    const double qx = hi * ui, qy = hi * vi;
    const double qq2 = fma(qx, qx, qy * qy);
    if (hi > hdry && gm2 > 0.0 && qq2 > 1e-200) {           // a8
        double rq;
        const double Q = fast_sqrt_rsqrt(qq2, rq);
        const double c3 = (hi > 1e-28 && hi < 1e28) ? fast_rcbrt(hi) : rcbrt(hi);   // h^(-1/3)
        const double rh = (c3 * c3) * c3;                       // 1/h
        const double cQ = gm2 * (rh * rh) * c3 * Q;             // g m^2 |q| / h^(7/3)
        const double E = cQ * (dt * fma(7.0 / 6.0, dh * rh, -1.0));
        const double r2 = fma(qx, E, dqx), r3 = fma(qy, E, dqy);
        const double DQ = 0.5 * dt * cQ;                        // D Q
        const double al = 1.0 + DQ;
        const double inv = fast_rcp(al * fma(2.0, DQ, 1.0));    // 1 / det
        const double bw = (DQ * (rq * rq)) * fma(qy, r2, -(qx * r3));   // (D/Q) (q x r)
        dqx = fma(bw, qy, al * r2) * inv;
        dqy = fma(-bw, qx, al * r3) * inv;
    }
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
        const double a = fast_sqrt(g * hn);
        const double v2 = fma(Un.u, Un.u, Un.v * Un.v);
        const double vm = v2 > 1e-200 ? fast_sqrt(v2) : 0.0;
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
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory");
}

// ---- the tile pipeline -----------------------------------------------------------------------------
// Per-tile info block in global memory (P.tinfo, fixed stride 4 + MH int32, MH = P.max_halo):
//   [0] first edge of the tile in P.edges   [1] number of edges   [2] number of halo ids
//   [3] 1 if an inflow edge touches it      [4..] halo ids (internal cell ids), padded with -1
// Shared memory of one block (dynamic); TC = blockDim.x, ME = P.max_edges (even):
//   double2 so01[3][TC + 1]        (mass, x-momentum) flux slot of (local edge k, cell); the extra
//   double  so2 [3][TC + 1]        entry per k staggers the banks of a cell's three slots
//   double  scell[3][TC]           1/|Omega|, 1/R, g m^2
//   uint64  bar[5]                 rec[2], edge[2], cell constants
//   uint32  count[4]               the producer thread's counters
//   int32   ring[4], claim[8]      tiles of the coming pipeline stages; the producer thread's claim state
//   uint32  sq[128]                quiet flags of the block's tiles
//   Rec     srec[2][TC + MH]       state records of the tile's cells, then of its halo cells
//   uint2 + double2  sedge[2][ME]  the tile's edge list (24 bytes per edge)
// Schedule for the block's n-th pipeline stage, i.e. its n-th tile that is not quiet (s = n & 1), all
// copies asynchronous and one stage ahead:
//   top      wait: own halo gathers, records of tile n; barrier (= the dry vote)
//            issue: records of tile n+1 (bulk) -> srec[s^1]; edge list of tile n+1 (bulk) ->
//                   sedge[s^1] if that tile was active a step ago; cell constants of tile n
//                   (bulk); halo gathers of tile n+1 (cp.async, ids in registers)
//            load:  header, halo id, hint of tile n+2 into registers
//            wait:  edge list of tile n
//   phase 1  edges: shared memory only
//   mid      barrier; wait: cell constants
//   phase 2  cells
constexpr int kInfoHdr = 4;
constexpr int kNumBars = 5;
constexpr int kMaxSeq = 4096;             // tiles of a block's sequence that can be flagged quiet (the rest vote)
constexpr int kNbrs = 16;                 // = kTileNbrs (mesh_builder.h)
template <int TC> struct SmemLayout {
    static constexpr int PLC = TC + 1;
    static constexpr int so01 = 0;
    static constexpr int so2 = so01 + 3 * PLC * 16;
    static constexpr int scell = (so2 + 3 * PLC * 8 + 15) & ~15;
    static constexpr int bar = scell + 3 * TC * 8;
    static constexpr int ring = bar + kNumBars * 8 + 16;                 // after four diagnostic counters
    static constexpr int sq = ring + 48;                                 // after the ring and the claim state
    static constexpr int srec = (sq + kMaxSeq / 8 + 31) & ~31;
};
__host__ __device__ __forceinline__ size_t tile_smem_bytes(int TC, int MH, int ME)
{
    const size_t PLC = (size_t)TC + 1;
    size_t o = 3 * PLC * 16;
    o = (o + 3 * PLC * 8 + 15) & ~(size_t)15;
    o += 3 * (size_t)TC * 8;
    o = (o + kNumBars * 8 + 16 + 48 + 4096 / 8 + 31) & ~(size_t)31;      // barriers, counters, ring + claim state, quiet flags (kMaxSeq bits)
    o += 2 * (size_t)(TC + MH) * sizeof(Rec);
    o += 2 * (size_t)ME * 24;
    return o;
}

// Pipeline state carried across the steps of a persistent launch: tiles pushed through so far
// (fixes the record buffers and their barrier parity) and the parities of the barriers that do
// not complete a phase at every tile (edge lists: one bit per stage; cell constants).
struct PipeState { unsigned n = 0, epar = 0, cpar = 0; };

// ---- quiet tiles -------------------------------------------------------------------------------------
// P.act(c)[t] = 1 if tile t was active (not all dry) in the step that produced the state in U(c).  A
// tile that was inactive in the previous step, and whose halo cells all belong to tiles that were
// inactive in the previous step too, is QUIET: none of its cells and none of its halo cells has
// changed since they were seen dry, so it is all dry now, and its update is the identity whatever
// its neighbours do in this step.  And the identity is already in place: the previous step, in which
// the tile was inactive, wrote U(cur)[tile] = U(cur^1)[tile] bit for bit, and nothing has written
// U(cur^1)[tile] since, so the buffer this step writes holds the tile's records already.  A quiet
// tile therefore costs one flag (act(cur^1)[t] = 0) and no traffic on the state: no halo gather, no
// vote, no copy -- the paper's river domains are mostly dry land, and that part
// of the mesh now costs nothing per step.
// Tiles with an inflow edge or with more than kTileNbrs neighbour tiles are never quiet (tnbr[0] = -2).
// The block's tiles are tile(j) = blockIdx.x + j gridDim.x; bit j of sq[] says tile(j) is quiet.

// one flag per tile of the block's sequence, evaluated by one thread each (17 words from L2)
template <int TC>
__device__ __forceinline__ void quiet_flags(const Params &P, const int32_t *__restrict__ act_prev, unsigned *sq, const int nmy)
{
    const int tid = threadIdx.x, G = gridDim.x, lim = min(nmy, kMaxSeq);
    for (int j0 = 0; j0 < lim; j0 += TC) {
        const int j = j0 + tid;
        int v = 1;
        if (j < lim) {
            const int t = blockIdx.x + j * G;
            v = ldcg_i32(act_prev + t);
            if (v == 0) {
                const int4 *row = reinterpret_cast<const int4 *>(P.tnbr + (size_t)t * kNbrs);
#pragma unroll
                for (int q = 0; q < kNbrs / 4; q++) {
                    const int4 r = __ldg(row + q);
                    v |= r.x == -2;
                    if (r.x >= 0) v |= ldcg_i32(act_prev + r.x);
                    if (r.y >= 0) v |= ldcg_i32(act_prev + r.y);
                    if (r.z >= 0) v |= ldcg_i32(act_prev + r.z);
                    if (r.w >= 0) v |= ldcg_i32(act_prev + r.w);
                }
            }
        }
        const unsigned m = __ballot_sync(0xffffffffu, v == 0);
        if ((tid & 31) == 0 && j < ((lim + 31) & ~31)) sq[j >> 5] = m;
    }
}
__device__ __forceinline__ int next_nonquiet(const unsigned *sq, int j, const int nmy)
{
    const int lim = min(nmy, kMaxSeq);
    while (j < lim) {
        const unsigned w = ~sq[j >> 5] & (0xffffffffu << (j & 31));
        if (w) return min((j & ~31) + __ffs(w) - 1, nmy);
        j = (j | 31) + 1;
    }
    return min(j, nmy);
}
// ---- work stealing ---------------------------------------------------------------------------------
// Block b OWNS the tiles tile(j) = b + j gridDim.x; the ones that are not quiet form its list, in the order
// of j.  The blocks of an SM do not advance at the same pace (the warp schedulers favour some warp
// slots: measured, the four blocks of an SM finished their equal shares 115 to 155 us after the launch),
// and the wet part of a mesh is not spread evenly, so a block that has emptied its list takes tiles
// from the lists of others.  P.wq[b] is the list's work word: bits 0-30 head = entries the owner has
// claimed from the front (atomicAdd 1), bit 31 set if the list is spelled out in P.wlist (quiet tiles
// were looked for; otherwise entry k is tile b + k gridDim.x), bits 32-63 tail (signed) = end of the
// unclaimed part, which a thief lowers (atomicAdd -2^32) to claim entry tail - 1.  Either claim is good
// iff head < tail in the word the atomic returned; both counters move one way only, so no entry is given
// out twice, and the owner goes on until a claim of its own fails, so every word ends a step exhausted
// (head >= tail) and a thief that reads a word its owner has not yet set up for this step finds nothing.
// The results do not depend on which block computes a tile (per-cell arithmetic, maxima, single-writer
// boundary accumulators), so they are the same bits with or without stealing.
// All of it is done by the block's producer thread while its warp waits for the longer edge loops of
// the first warps; the tile of the stage after the next one goes to the others through a ring.
// Lists are shared only on meshes with at least kStealMinTiles tiles per block: below that a step is
// one or two passes through the pipeline per block and probing from the prologue would only add latency.
struct ClaimState {
    int src;       // list being consumed: own block first, then victims; -1: nothing left anywhere
    int jc;        // own list: next position of the block's sequence to look at
    int pre;       // own claims already contained in the initial work word
    int fails;     // probe rounds that found no victim since the last good claim
    int stolen;    // tiles taken from other blocks' lists in this step (diagnostics)
    int pad[3];
};
constexpr unsigned long long kTailOne = 1ull << 32;
constexpr unsigned kListBit = 0x80000000u;
#ifndef SWE_PROBE_ROUNDS
#define SWE_PROBE_ROUNDS 2
#endif
constexpr int kProbe = 8, kProbeRounds = SWE_PROBE_ROUNDS;
#ifndef SWE_STEAL_MIN_TILES
#define SWE_STEAL_MIN_TILES 8
#endif
constexpr int kStealMinTiles = SWE_STEAL_MIN_TILES;   // tiles per block (mesh / grid) from which lists are shared

template <bool QUIET>
__device__ __noinline__ int claim_tile(unsigned long long *const wq, const int32_t *const wlist, const int wstride,
                                       ClaimState *cs, const unsigned *sq, const int nmy)
{   // (the kernel parameters by value: a reference would put the whole parameter block on the stack)
    const int b = blockIdx.x, G = gridDim.x;
    if (cs->src == b) {
        const int j = QUIET ? next_nonquiet(sq, cs->jc, nmy) : min(cs->jc, nmy);
        if (j < nmy) {
            cs->jc = j + 1;
            bool ok = true;
            if (cs->pre > 0) cs->pre--;
            else {
                const unsigned long long old = atomicAdd(wq + b, 1ull);
                ok = (int)((unsigned)old & ~kListBit) < (int)(unsigned)(old >> 32);
            }
            if (ok) return b + j * G;
        }
        cs->src = -2;                       // own list finished, or the rest of it was taken: look for a victim
    }
    if (cs->src == -1) return -1;
    for (;;) {
        if (cs->src >= 0) {
            const int v = cs->src;
            const unsigned long long old = atomicAdd(wq + v, 0ull - kTailOne);
            const int h = (int)((unsigned)old & ~kListBit), t = (int)(unsigned)(old >> 32);
            if (h < t) {
                cs->fails = 0; cs->stolen++;
                if (!((unsigned)old & kListBit)) return v + (t - 1) * G;
                __threadfence();            // the list was published before the word
                return ldcg_i32(wlist + (size_t)v * wstride + (t - 1));
            }
            cs->src = -2;
        }
        if (cs->fails >= kProbeRounds) { cs->src = -1; return -1; }
        // a handful of candidates per round: the blocks that share this block's SM when blocks are dealt
        // round-robin (b + G/4, ...), its neighbours, a few scattered ones; the one furthest behind wins
        int best = -1, best_rem = 0;
        const unsigned salt = (unsigned)b * 2654435761u + (unsigned)cs->fails * 40503u + (unsigned)cs->jc * 9973u;
        int cand[kProbe];
        unsigned long long w[kProbe];
#pragma unroll
        for (int q = 0; q < kProbe; q++) {
            int v;
            if (cs->fails == 0 && q < 3) v = b + (q + 1) * (G >> 2);
            else if (cs->fails == 0 && q < 5) v = b + (q == 3 ? 1 : G - 1);
            else v = (int)((salt + (unsigned)q * 2246822519u) >> 8);
            cand[q] = (int)((unsigned)v % (unsigned)G);
            asm volatile("ld.global.cg.u64 %0, [%1];" : "=l"(w[q]) : "l"(wq + cand[q]) : "memory");
        }
#pragma unroll
        for (int q = 0; q < kProbe; q++) {
            const int rem = (int)(unsigned)(w[q] >> 32) - (int)((unsigned)w[q] & ~kListBit);
            if (cand[q] != b && rem > best_rem) { best_rem = rem; best = cand[q]; }
        }
        cs->jc++;                           // (free once the own list is done: varies the scattered candidates)
        if (best < 0) cs->fails++;
        else cs->src = best;
    }
}

// All the tiles of this block for one time step.
// Returns this thread's maximum rate contribution.
// QUIET: look for quiet tiles first and leave them alone (chosen per block and step when a good
// share of the block's tiles was inactive in the previous step; the results are the same either way,
// an all-dry tile that is not treated as quiet is found by the vote and copied).
template <int TC, bool QUIET>
__device__ __forceinline__ double step_tiles(const Params &P, unsigned char *smem, const int cur,
                                             const double dt, unsigned &nclamp, PipeState &ps)
{
    // state and activity flags of this step: read side cur, written side cur ^ 1.  The pointers are
    // re-derived from the kernel parameters where they are used (registers are what limits the tile loop)
#define Uin (static_cast<const Rec *>(P.U(cur)))
#define Uout (P.U(cur ^ 1))
#define act_prev (static_cast<const int32_t *>(P.act(cur)))
#define act_next (P.act(cur ^ 1))
    typedef SmemLayout<TC> SL;
    constexpr int PLC = SL::PLC;
    double2 *const so01 = reinterpret_cast<double2 *>(smem + SL::so01);
    double *const so2 = reinterpret_cast<double *>(smem + SL::so2);
    const double *const scell = reinterpret_cast<const double *>(smem + SL::scell);
    uint64_t *const bar = reinterpret_cast<uint64_t *>(smem + SL::bar);      // rec 0,1; edge 2,3; cell 4
    // kept by the producer thread: [0] active tiles, [1] edge lists fetched, [2] quiet tiles, [3] inactive tiles
    volatile unsigned *const scount = reinterpret_cast<volatile unsigned *>(bar + kNumBars);
    unsigned *const sq = reinterpret_cast<unsigned *>(smem + SL::sq);        // quiet flags of the block's tiles
    Rec *const srec0 = reinterpret_cast<Rec *>(smem + SL::srec);
    const int rstride = TC + P.max_halo;
    unsigned char *const sedge0 = reinterpret_cast<unsigned char *>(srec0 + 2 * rstride);
    const int estride = P.max_edges * 24;
    const int istride = kInfoHdr + P.max_halo;
    const int tid = threadIdx.x, G = gridDim.x;
    const double hdry = P.hdry;
    double rate = 0.0;
    if ((int)blockIdx.x >= P.ntiles) return 0.0;
    const int nmy = (P.ntiles - (int)blockIdx.x + G - 1) / G;       // tiles of this block: tile(j) = blockIdx.x + j G
    unsigned n = ps.n, epar = ps.epar, cpar = ps.cpar;
    // the copies are issued by lane 0 of the LAST warp: the edge loop gives the first warps one more
    // iteration than the last ones (ne ~ 1.66 TC), so the last warp has the slack
    const bool producer = tid == TC - 32;

    auto issue_recs = [&](int t, int s) {
        const int base = t * TC, nc = min(TC, P.nt - base);
        mbar_expect_tx(bar + s, (unsigned)nc * sizeof(Rec));
        bulk_g2s(srec0 + s * rstride, Uin + base, (unsigned)nc * sizeof(Rec), bar + s);
    };
    auto issue_edges = [&](int e0, int ne, int s) {
        const unsigned bytes = (unsigned)((ne + 1) & ~1) * 24u;        // lists are padded to an even length
        mbar_expect_tx(bar + 2 + s, bytes);
        bulk_g2s(sedge0 + s * estride, P.edges + 3 * (size_t)e0, bytes, bar + 2 + s);
        scount[1]++;
    };
    auto issue_cellc = [&](int t) {
        mbar_expect_tx(bar + 4, 3u * TC * 8u);
        bulk_g2s(smem + SL::scell, P.cellc + (size_t)t * 3 * TC, 3u * TC * 8u, bar + 4);
    };
    // halo records of tile t into srec[s][TC..]: thread q fetches halo cell q (id in a register);
    // lists longer than the tile (poor orderings only) are finished from the table
    auto gather_halo = [&](int t, int nh, int hid, int s) {
        Rec *dst = srec0 + s * rstride + TC;
        if (tid < nh) {
            const char *src = reinterpret_cast<const char *>(Uin + hid);
            cp_async16(reinterpret_cast<char *>(dst + tid), src);
            cp_async16(reinterpret_cast<char *>(dst + tid) + 16, src + 16);
        }
        for (int q = tid + TC; q < nh; q += TC) {
            const char *src = reinterpret_cast<const char *>(Uin + __ldg(P.tinfo + (size_t)t * istride + kInfoHdr + q));
            cp_async16(reinterpret_cast<char *>(dst + q), src);
            cp_async16(reinterpret_cast<char *>(dst + q) + 16, src + 16);
        }
    };
    auto load_hdr = [&](int t) { return __ldg(reinterpret_cast<const int4 *>(P.tinfo + (size_t)t * istride)); };
    auto hdr_ne = [](int4 h) { return h.y; };
    auto hdr_nh = [](int4 h) { return h.z; };
    auto load_hid = [&](int t) { return tid < P.max_halo ? __ldg(P.tinfo + (size_t)t * istride + kInfoHdr + tid) : -1; };
    auto tile_of = [&](int j) { return (int)blockIdx.x + j * G; };

    // ---- this block's list: the tiles of its sequence that are not quiet
    int *const sring = reinterpret_cast<int *>(smem + SL::ring);
    ClaimState *const cs = reinterpret_cast<ClaimState *>(smem + SL::ring + 16);
    int len = nmy;
    if constexpr (QUIET) {
        quiet_flags<TC>(P, act_prev, sq, nmy);
        __syncthreads();
        // spell the list out for thieves: entry k = the k-th tile of the sequence that is not quiet
        const int lim = min(nmy, kMaxSeq);
        int32_t *const wl = P.wlist + (size_t)blockIdx.x * P.wstride;
        int nq_all = 0;
        for (int w = 0; w < (lim + 31) >> 5; w++) nq_all += __popc(sq[w]);
        len = nmy - nq_all;
        for (int j = tid; j < nmy; j += TC) {
            int nq = nq_all;
            bool quiet = false;
            if (j < lim) {
                nq = 0;
                for (int w = 0; w < (j >> 5); w++) nq += __popc(sq[w]);
                const unsigned word = sq[j >> 5];
                nq += __popc(word & ((1u << (j & 31)) - 1u));
                quiet = (word >> (j & 31)) & 1u;
            }
            if (!quiet) wl[j - nq] = (int)blockIdx.x + j * G;
            else act_next[(int)blockIdx.x + j * G] = 0;    // all a quiet tile costs: its records are in place already
        }
        if (producer) { scount[2] += (unsigned)nq_all; scount[3] += (unsigned)nq_all; }
        __threadfence();
        __syncthreads();
    }
    if (producer) {
        // Meshes with only a few tiles per block are bound by the latency of one pass through the pipeline,
        // and probing others' lists from the prologue would add to it: there the lists stay private (the
        // whole list is pre-claimed, nobody probes; the criterion is the same for every block of the grid).
        const bool steal = P.wstride >= kStealMinTiles;
        const int pre = steal ? min(len, 2) : len;
        if (steal) P.wq[blockIdx.x] = ((unsigned long long)(unsigned)len << 32) | (QUIET ? kListBit : 0u) | (unsigned)pre;
        cs->src = blockIdx.x; cs->jc = 0; cs->pre = pre; cs->fails = steal ? 0 : kProbeRounds; cs->stolen = 0;
    }
    // the first two stages (a block with a shorter list of its own takes from others right away)
    if (producer) {
        sring[0] = claim_tile<QUIET>(P.wq, P.wlist, P.wstride, cs, sq, nmy);
        sring[1] = claim_tile<QUIET>(P.wq, P.wlist, P.wstride, cs, sq, nmy);
    }
    __syncthreads();
    int tile0 = sring[0], tile1 = sring[1];              // this pipeline stage, the next one
    if (tile0 < 0) return 0.0;                           // nothing but quiet tiles here and nothing to take elsewhere
    // ---- prologue: everything tile0 needs; header, halo id and hint of tile1
    int4 hdr0 = load_hdr(tile0), hdr1 = make_int4(0, 0, 0, 0);
    int hid0 = load_hid(tile0), hid1 = -1, hint1 = 0;
    bool req0 = true;                    // was this tile's edge list requested?  The step's first pipeline stage: always
    if (producer) {
        issue_recs(tile0, n & 1);
        issue_edges(hdr0.x, hdr_ne(hdr0), n & 1);
    }
    if (tile1 >= 0) { hdr1 = load_hdr(tile1); hid1 = load_hid(tile1); hint1 = ldcg_i32(act_prev + tile1); }
    gather_halo(tile0, hdr_nh(hdr0), hid0, n & 1);
    cp_async_commit();
    for (unsigned q = 0;; q++) {                          // q: stage of this step (n runs on across the steps of a launch)
        const int s = n & 1;
        const int tile = tile0;
        const int base = tile * TC;
        const bool have_next = tile1 >= 0;
        const int ne = hdr_ne(hdr0), nh = hdr_nh(hdr0);
        // ---- top
        cp_async_wait<0>();                               // own halo gathers of this tile
        mbar_wait(bar + s, (n >> 1) & 1u);
        const Rec *const srec = srec0 + s * rstride;
        // is anything wet in the tile or its halo?  Each thread looks at its own record and at
        // the halo record it gathered itself, so the vote can BE the tile's first barrier.
        const int i = base + tid;
        bool wet = i < P.nt && srec[tid].h > hdry;
        if (tid < nh) wet |= srec[TC + tid].h > hdry;
        for (int k = tid + TC; k < nh; k += TC) wet |= srec[TC + k].h > hdry;
        // barrier: everyone has left the previous tile; everyone's gathers are visible
        const bool active = __syncthreads_or(wet) || hdr0.w != 0;
        if (producer) {
            if (have_next) {
                issue_recs(tile1, s ^ 1);
                // Edge lists are 40 of the ~105 bytes a cell costs and an all-dry tile never reads its
                // list, so the list of the NEXT tile is requested only if that tile was active at the
                // previous step; a tile that turns out active without its list (the wet front reached
                // it) fetches it on the spot, below.
                if (hint1) issue_edges(hdr1.x, hdr_ne(hdr1), s ^ 1);
            }
            if (active) issue_cellc(tile);
            act_next[tile] = active;
            scount[0] += active; scount[3] += !active;
        }
        if (have_next) gather_halo(tile1, hdr_nh(hdr1), hid1, s ^ 1);
        cp_async_commit();
        // this tile's edge list: requested one tile ago, or fetched now if the tile is active without it
        if (!req0 && active && producer) issue_edges(hdr0.x, ne, s);
        if (req0 || active) {
            mbar_wait(bar + 2 + s, (epar >> s) & 1u);
            epar ^= 1u << s;
        }
        if (!active) {
            // Every cell of the tile and every neighbour is dry and no discharge is prescribed:
            // all fluxes vanish, h' = h + 0, and dry cells carry u = v = 0 already (R-15), so the
            // step leaves the records unchanged bit for bit.  The copy still moves them.
            if (i < P.nt) store_rec(Uout + i, srec[tid]);
            if (producer) sring[(q + 2) & 3] = have_next ? claim_tile<QUIET>(P.wq, P.wlist, P.wstride, cs, sq, nmy) : -1;
            __syncthreads();
        } else {
            // ---- phase 1: every edge of the tile once, shared memory only (a2-a7)
            const unsigned char *const se = sedge0 + s * estride;
            const uint2 *const sab = reinterpret_cast<const uint2 *>(se);
            const double2 *const slxy = reinterpret_cast<const double2 *>(se + ((ne + 1) & ~1) * 8);
            for (int e = tid; e < ne; e += TC) {
                const uint2 ab = sab[e];
                const double2 l = slxy[e];
                const Rec A = srec[ab.x & kPosMask];
                // (a boundary edge reads A again: B is not used there, and selecting the index costs one
                // instruction where copying the record costs eight)
                const Rec B = srec[((int32_t)ab.y >= 0 ? ab.y : ab.x) & kPosMask];
                double o[5];
                edge_eval(P, l.x, l.y, A, B, (int32_t)ab.y, dt, o);
                // b's slot gets the negated values (its outward normal is -n)
                const unsigned sa = ab.x >> kSlotShift;
                if (sa != kNoSlot) {
                    so01[sa] = make_double2(o[0], o[1]);
                    so2[sa] = o[2];
                }
                const unsigned sb = ab.y >> kSlotShift;      // boundary words have bit 31 set: > kNoSlot
                if (sb < kNoSlot) {
                    so01[sb] = make_double2(-o[0], -o[3]);
                    so2[sb] = -o[4];
                }
            }
            // the tile of the stage after the next one: claimed while the first warps finish their edges
            if (producer) sring[(q + 2) & 3] = have_next ? claim_tile<QUIET>(P.wq, P.wlist, P.wstride, cs, sq, nmy) : -1;
            __syncthreads();
        }
        // the stage after the next one: its header, halo id and hint into registers
        const int tile2 = sring[(q + 2) & 3];
        int4 hdr2 = make_int4(0, 0, 0, 0);
        int hid2 = -1, hint2 = 0;
        if (tile2 >= 0) { hdr2 = load_hdr(tile2); hid2 = load_hid(tile2); hint2 = ldcg_i32(act_prev + tile2); }
        if (active) {
            mbar_wait(bar + 4, cpar);                          // this tile's cell constants
            cpar ^= 1u;
            // ---- phase 2: every cell of the tile (a7-a10)
            if (i < P.nt) {
                const Rec Ui = srec[tid];
                // three edges in the fixed order k = 0,1,2 (R-17)
                const double2 f0 = so01[tid], f1 = so01[PLC + tid], f2 = so01[2 * PLC + tid];
                const double s1 = (f0.x + f1.x) + f2.x;
                const double s2 = (f0.y + f1.y) + f2.y;
                const double s3 = (so2[tid] + so2[PLC + tid]) + so2[2 * PLC + tid];
                Rec Un;
                rate = dmax(rate, cell_update(P, Ui, s1, s2, s3, scell[tid], scell[TC + tid], scell[2 * TC + tid], dt, Un, nclamp));
                store_rec(Uout + i, Un);
            }
        }
        if (!have_next) break;
        n++;
        tile0 = tile1; tile1 = tile2;
        hdr0 = hdr1; hid0 = hid1; req0 = hint1 != 0;
        hdr1 = hdr2; hid1 = hid2; hint1 = hint2;
    }
    cp_async_wait<0>();
    ps.n = n + 1; ps.epar = epar; ps.cpar = cpar;
    return rate;
#undef Uin
#undef Uout
#undef act_prev
#undef act_next
}

// ---- small meshes: the whole time loop in ONE thread-block cluster ---------------------------------
// small meshes are "strictly limited by latencies" of kernel launches.  A mesh of at
// most 16 tiles runs swe_run(nsteps) as one launch of one cluster, one CTA per tile: the tile's state
// (double-buffered), edge list and cell constants stay in its shared memory for the whole run; halo
// records are read from the owning CTA's shared memory (distributed shared memory); the per-tile
// maximum rate is stored into every CTA's shared memory, so the next dt needs no global memory; and
// the step boundary is the hardware cluster barrier instead of a kernel boundary or a grid barrier.
// NT = 2 TC threads per CTA, so the ~1.66 TC edges of a tile take ONE pass of the edge loop.
// Same edge_eval / cell_update, same edge orientation and summation order as the tile kernel: the
// results are bit-identical to the other loop modes.
constexpr int kMaxClusterTiles = 16;
template <int TC> struct ClusterLayout {
    static constexpr int PLC = TC + 1;
    static constexpr int so01 = 0;
    static constexpr int so2 = so01 + 3 * PLC * 16;
    static constexpr int scell = (so2 + 3 * PLC * 8 + 15) & ~15;
    static constexpr int smax = scell + 3 * TC * 8;
    static constexpr int srec = (smax + 2 * kMaxClusterTiles * 8 + 31) & ~31;
};
__host__ __device__ __forceinline__ size_t cluster_smem_bytes(int TC, int MH, int ME)
{
    const size_t PLC = (size_t)TC + 1;
    size_t o = 3 * PLC * 16;
    o = (o + 3 * PLC * 8 + 15) & ~(size_t)15;
    o += 3 * (size_t)TC * 8 + 2 * kMaxClusterTiles * 8;
    o = (o + 31) & ~(size_t)31;
    return o + 2 * (size_t)(TC + MH) * sizeof(Rec) + (size_t)ME * 24;
}

template <int TC>
__device__ __forceinline__ void cluster_loop(const Params &P, unsigned char *smem, double *s_red, int cur,
                                             const long long nsteps)
{
    namespace cg = cooperative_groups;
    typedef ClusterLayout<TC> CL;
    constexpr int PLC = CL::PLC, NT = 2 * TC;
    cg::cluster_group cluster = cg::this_cluster();
    double2 *const so01 = reinterpret_cast<double2 *>(smem + CL::so01);
    double *const so2 = reinterpret_cast<double *>(smem + CL::so2);
    double *const scell = reinterpret_cast<double *>(smem + CL::scell);
    double *const smax = reinterpret_cast<double *>(smem + CL::smax);           // [2][kMaxClusterTiles]
    Rec *const srec0 = reinterpret_cast<Rec *>(smem + CL::srec);
    const int rstride = TC + P.max_halo;
    unsigned char *const sedge = reinterpret_cast<unsigned char *>(srec0 + 2 * rstride);
    const int tid = threadIdx.x, tile = blockIdx.x, ntiles = P.ntiles;
    const int istride = kInfoHdr + P.max_halo;
    const int32_t *info = P.tinfo + (size_t)tile * istride;
    const int e0 = __ldg(info), ne = __ldg(info + 1), nh = __ldg(info + 2), inflow = __ldg(info + 3);
    const int nep = (ne + 1) & ~1;
    const int base = tile * TC, i = base + tid;
    const double hdry = P.hdry;
    // ---- everything the tile needs, once per launch
    for (int q = tid; q < 3 * nep; q += NT) reinterpret_cast<double *>(sedge)[q] = __ldg(P.edges + 3 * (size_t)e0 + q);
    for (int q = tid; q < 3 * TC; q += NT) scell[q] = __ldg(P.cellc + (size_t)tile * 3 * TC + q);
    if (tid < TC) {
        Rec r; r.h = 0.0; r.u = 0.0; r.v = 0.0; r.z = 0.0;
        if (i < P.nt) r = load_rec(P.U(cur) + i);
        srec0[tid] = r;
    }
    // halo record q of this tile lives in CTA (id / TC) at local index (id % TC)
    const Rec *hsrc = nullptr;
    if (tid < nh) {
        const int id = __ldg(info + kInfoHdr + tid);
        hsrc = cluster.map_shared_rank(srec0, (unsigned)(id / TC)) + id % TC;
    }
    double t_now = __ldcg(&P.ctrl->t[cur]);
    const double t_end = __ldcg(&P.ctrl->t_end);
    double dt_cfl = reduce_dt(P, P.pmax(cur), s_red);          // first step: from the rates swe_run left in HBM
    cluster.sync();                                             // every tile's state is resident
    double rate = 0.0, dt_last = 0.0;
    unsigned nclamp = 0, nactive = 0;
    long long steps = 0;
    bool all_dry = false;
    const uint2 *const sab = reinterpret_cast<const uint2 *>(sedge);
    const double2 *const slxy = reinterpret_cast<const double2 *>(sedge + nep * 8);
    for (long long s = 0; s < nsteps; s++) {
        const int p = (int)(s & 1);
        Rec *const srec = srec0 + p * rstride, *const snew = srec0 + (p ^ 1) * rstride;
        if (s > 0) {                                            // a11: every CTA holds every tile's maximum
            double r = 0.0;
            for (int k = 0; k < ntiles; k++) r = fmax(r, smax[p * kMaxClusterTiles + k]);
            dt_cfl = r > 0.0 ? P.cfl / r : 0.0;
        }
        const double left = t_end - t_now;
        const bool clipped = dt_cfl >= left;
        const double dt = fmax(clipped ? left : dt_cfl, 0.0);
        // a1: halo records from their owners' shared memory
        bool wet = tid < TC && srec[tid < TC ? tid : 0].h > hdry;
        if (tid < nh) { const Rec r = hsrc[p * rstride]; srec[TC + tid] = r; wet |= r.h > hdry; }
        for (int q = tid + NT; q < nh; q += NT) {               // lists longer than the block (poor orderings)
            const int id = __ldg(info + kInfoHdr + q);
            const Rec r = *(cluster.map_shared_rank(srec0, (unsigned)(id / TC)) + id % TC + p * rstride);
            srec[TC + q] = r; wet |= r.h > hdry;
        }
        const bool active = __syncthreads_or(wet) || inflow != 0;
        rate = 0.0;
        if (!active) {
            if (tid < TC) snew[tid] = srec[tid];                // all dry: the update is the identity
        } else {
            for (int e = tid; e < ne; e += NT) {                // phase 1 (a2-a7)
                const uint2 ab = sab[e];
                const double2 l = slxy[e];
                const Rec A = srec[ab.x & kPosMask];
                const Rec B = srec[((int32_t)ab.y >= 0 ? ab.y : ab.x) & kPosMask];
                double o[5];
                edge_eval(P, l.x, l.y, A, B, (int32_t)ab.y, dt, o);
                const unsigned sa = ab.x >> kSlotShift;
                if (sa != kNoSlot) { so01[sa] = make_double2(o[0], o[1]); so2[sa] = o[2]; }
                const unsigned sb = ab.y >> kSlotShift;
                if (sb < kNoSlot) { so01[sb] = make_double2(-o[0], -o[3]); so2[sb] = -o[4]; }
            }
            __syncthreads();
            if (tid < TC && i < P.nt) {                         // phase 2 (a7-a10)
                const Rec Ui = srec[tid];
                const double2 f0 = so01[tid], f1 = so01[PLC + tid], f2 = so01[2 * PLC + tid];
                const double s1 = (f0.x + f1.x) + f2.x;
                const double s2 = (f0.y + f1.y) + f2.y;
                const double s3 = (so2[tid] + so2[PLC + tid]) + so2[2 * PLC + tid];
                Rec Un;
                rate = cell_update(P, Ui, s1, s2, s3, scell[tid], scell[TC + tid], scell[2 * TC + tid], dt, Un, nclamp);
                snew[tid] = Un;
            }
        }
        rate = block_max(rate, s_red);
        // this tile's maximum into every CTA's table for the next step (distributed shared memory)
        if (tid < ntiles) cluster.map_shared_rank(smax, (unsigned)tid)[(p ^ 1) * kMaxClusterTiles + tile] = rate;
        nactive += active;
        t_now = clipped ? fmax(t_end, t_now) : t_now + dt;      // R-24
        if (dt > 0.0) { dt_last = dt; steps++; }
        if (!(dt_cfl > 0.0)) all_dry = true;
        cluster.sync();                                         // the step boundary
    }
    // ---- back to HBM: state, per-tile maximum, device clock, counters
    const int fin = cur ^ (int)(nsteps & 1);
    if (tid < TC && i < P.nt) store_rec(P.U(fin) + i, srec0[(int)(nsteps & 1) * rstride + tid]);
    if (tid == 0) {
        P.pmax(fin)[tile] = rate;
        if (nactive) atomicAdd(&P.ctrl->n_active, (unsigned long long)nactive);
        if (tile == 0) {
            Ctrl *c = P.ctrl;
            c->t[fin] = t_now;
            if (steps) { c->dt_last = dt_last; c->steps += steps; }
            if (all_dry) c->all_dry = 1;
        }
    }
    if (nclamp) atomicAdd(&P.ctrl->n_clamped, (unsigned long long)nclamp);
}

} // namespace swe
