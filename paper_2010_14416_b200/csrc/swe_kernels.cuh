// Device code of libswe_b200: the fused cell-centric SWE step for sm_100a (FP64).
//
// One thread owns one triangle.  It gathers its three neighbours' records through the
// (locality-renumbered) index table, evaluates the three HLLC edge fluxes with hydrostatic
// reconstruction, the bathymetry source and the semi-implicit Manning friction, writes the new
// record to the other state buffer, and contributes (sqrt(g h)+|V|)/R of the NEW state to a
// per-block maximum (warp shuffles + shared memory, no atomics) from which the next launch (or
// the next iteration of the persistent loop) derives dt.  PAPER.md sections 2-3 and :457.
//
// State record in HBM: {h, u, v, z} as one 32-byte sector, so a neighbour gather is exactly one
// sector whatever the ordering, read with one 256-bit load (LDG.E.ENL2.256 on sm_100a).
// Velocities (not discharges) are stored so that the three neighbour gathers need no division;
// the caller still sees (h, hu, hv) (pack/unpack kernels).
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace swe {

struct __align__(32) Rec { double h, u, v, z; };

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
    const int32_t *nbr;       // [3][nt] neighbour (internal id) or -tag
    const double2 *nrm;       // [3][nt] unit outward normal
    const double *coef;       // [3][nt] L_ij / |Omega_i|
    const double2 *cellp;     // [nt] {1/R_i, g m_i^2}
    const double *qn_tag;     // [128] unit discharge along the outward normal per inflow tag
    double *pmax0, *pmax1;    // [npart] per-block max rate of state U0 / U1
    Ctrl *ctrl;
    int32_t nt, npart;
    double g, cfl, hdry;
    // selected with a ternary so the kernel parameter block is never indexed dynamically
    __host__ __device__ __forceinline__ Rec *U(int c) const { return c ? U1 : U0; }
    __host__ __device__ __forceinline__ double *pmax(int c) const { return c ? pmax1 : pmax0; }
};

// ---- 256-bit record access -----------------------------------------------------------------
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
// and tangential momentum flux.
__device__ __forceinline__ void hllc_flux(const double g, const double hdry, double hL, double uL,
                                          double vL, double hR, double uR, double vR, double &G0,
                                          double &G1, double &G2)
{
    const bool dL = hL <= hdry, dR = hR <= hdry;           // R-15
    if (dL && dR) { G0 = 0.0; G1 = 0.0; G2 = 0.0; return; }
    double SL, SR;
    if (dL) {                                               // eq.(26) line 1
        hL = 0.0; uL = 0.0; vL = 0.0;
        const double aR = sqrt(g * hR);
        SL = uR - 2.0 * aR; SR = uR + aR;
    } else if (dR) {                                        // eq.(26) line 2 (R-18)
        hR = 0.0; uR = 0.0; vR = 0.0;
        const double aL = sqrt(g * hL);
        SL = uL - aL; SR = uL + 2.0 * aL;
    } else {
        const double aL = sqrt(g * hL), aR = sqrt(g * hR);
        const double hs_sum = hL + hR, as_sum = aR + aL;
        const double h0 = 0.5 * hs_sum - (uR - uL) * hs_sum / (4.0 * as_sum);   // eq.(21)
        double hs;
        if (h0 <= fmin(hL, hR)) {                           // rarefaction, eq.(22), R-6
            const double w = fmax(0.5 * as_sum + 0.25 * (uL - uR), 0.0);
            hs = w * w / g;
        } else {                                            // shock, eq.(23)
            const double gL = sqrt(g * (h0 + hL) / (2.0 * h0 * hL));
            const double gR = sqrt(g * (h0 + hR) / (2.0 * h0 * hR));
            hs = ((hL * gL + hR * gR) + (uL - uR)) / (gL + gR);
        }
        const double pL = hs > hL ? sqrt(0.5 * hs * (hs + hL)) / hL : 1.0;      // eq.(20), R-7
        const double pR = hs > hR ? sqrt(0.5 * hs * (hs + hR)) / hR : 1.0;
        SL = uL - aL * pL; SR = uR + aR * pR;               // eq.(19)
    }
    const double qL = hL * uL, qR = hR * uR;
    const double GL1 = qL * uL + 0.5 * g * hL * hL, GR1 = qR * uR + 0.5 * g * hR * hR;
    if (SL >= 0.0) { G0 = qL; G1 = GL1; G2 = qL * vL; return; }                  // eq.(17), R-11
    if (SR <= 0.0) { G0 = qR; G1 = GR1; G2 = qR * vR; return; }
    const double inv = 1.0 / (SR - SL);
    G0 = ((SR * qL - SL * qR) + SR * SL * (hR - hL)) * inv;                      // eq.(18)
    G1 = GL1 + SL * (SR * (qR - qL) - (GR1 - GL1)) * inv;                        // eq.(18), R-12
    // eq.(24)-(26), R-16: the tangential velocity is upwinded by the sign of S*.  The numerator
    // of eq.(25) equals -(SR-SL) G0 and its denominator is negative, so sign(S*) = sign(G0);
    // in the dry-bed cases eq.(26) sets S* = SL (left dry) or SR (right dry), the same sign.
    G2 = G0 * (G0 >= 0.0 ? vL : vR);
}

// ---- one cell: eq.(37), PAPER.md:250 ----------------------------------------------------------
// Returns the local rate (sqrt(g h') + |V'|) / R_i of the new state (0 if dry), eq.(15).
template <bool kReadOnlyPath>
__device__ __forceinline__ double update_cell(const Params &P, const Rec *__restrict__ Uin,
                                              Rec *__restrict__ Uout, const int i, const double dt,
                                              unsigned &nclamp)
{
    const int N = P.nt;
    const double g = P.g, hdry = P.hdry;
    // ---- a1: gather (all loads issued before any arithmetic)
    const Rec Ui = load_rec<kReadOnlyPath>(Uin + i);
    int nb[3];
#pragma unroll
    for (int k = 0; k < 3; k++) nb[k] = __ldg(P.nbr + (size_t)k * N + i);
    Rec Uj[3];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        if (nb[k] >= 0) Uj[k] = load_rec<kReadOnlyPath>(Uin + nb[k]);
        else { Uj[k].h = 0.0; Uj[k].u = 0.0; Uj[k].v = 0.0; Uj[k].z = 0.0; }
    }
    double2 nr[3]; double cf[3];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        nr[k] = __ldg(P.nrm + (size_t)k * N + i);
        cf[k] = __ldg(P.coef + (size_t)k * N + i);
    }
    const double2 cp = __ldg(P.cellp + i);

    const double hi = Ui.h, ui = Ui.u, vi = Ui.v, zi = Ui.z;
    const bool wet = hi > hdry;
    double b1 = 0.0, b2 = 0.0, b3 = 0.0;
#pragma unroll
    for (int k = 0; k < 3; k++) {               // fixed order, R-17
        const double n1 = nr[k].x, n2 = nr[k].y;
        const double uL = ui * n1 + vi * n2, vL = vi * n1 - ui * n2;             // eq.(12)
        double G0, G1, G2, hL;
        if (nb[k] >= 0) {
            // a2: hydrostatic reconstruction, eq.(28), R-14
            const double zf = fmax(zi, Uj[k].z);
            hL = fmax(0.0, hi + (zi - zf));
            const double hR = fmax(0.0, Uj[k].h + (Uj[k].z - zf));
            const double uR = Uj[k].u * n1 + Uj[k].v * n2, vR = Uj[k].v * n1 - Uj[k].u * n2;
            hllc_flux(g, hdry, hL, uL, vL, hR, uR, vR, G0, G1, G2);
        } else {                                // a6: boundary edge
            const int tag = -nb[k];
            hL = hi;
            const double pr = 0.5 * g * hL * hL;
            if (tag == SWE_BC_WALL) { G0 = 0.0; G1 = pr; G2 = 0.0; }             // R-4
            else if (tag == SWE_BC_TRANSMISSIVE) {                                // R-21
                if (hL > hdry) { G0 = hL * uL; G1 = G0 * uL + pr; G2 = G0 * vL; }
                else { G0 = 0.0; G1 = 0.0; G2 = 0.0; }
            } else {                                                              // R-20
                const double qn = __ldg(P.qn_tag + tag);
                G0 = qn; G2 = 0.0;
                G1 = hL > hdry ? qn * qn / hL + pr : 0.0;
            }
        }
        // a7: rotate back (T^-1), bathymetry source eq.(30) with g/2 (R-13), accumulate
        const double sb = 0.5 * g * (hL * hL - hi * hi);
        const double Fn = G1 - sb;
        const double c = cf[k];
        b1 -= c * G0;
        b2 -= c * (Fn * n1 - G2 * n2);
        b3 -= c * (Fn * n2 + G2 * n1);
    }
    // a8: semi-implicit friction, eq.(32)-(37), R-19
    const double qx = hi * ui, qy = hi * vi;
    const double dh = dt * b1;
    double r2 = dt * b2, r3 = dt * b3, dqx, dqy;
    const double qq2 = qx * qx + qy * qy;
    if (wet && cp.y > 0.0 && qq2 > 0.0) {
        const double qq = sqrt(qq2);
        const double rh = 1.0 / hi;
        const double cfr = cp.y * rcbrt(hi) * rh * rh;          // g m^2 / h^(7/3)
        const double rq = 1.0 / qq;
        const double S2 = -cfr * qx * qq, S3 = -cfr * qy * qq;
        const double k73 = (7.0 / 3.0) * cfr * qq * rh;
        const double J21 = k73 * qx, J31 = k73 * qy;
        const double J22 = -cfr * (qq + qx * qx * rq), J33 = -cfr * (qq + qy * qy * rq);
        const double J23 = -cfr * qx * qy * rq;
        const double hdt = 0.5 * dt;
        r2 += dt * S2 + hdt * J21 * dh;
        r3 += dt * S3 + hdt * J31 * dh;
        const double a22 = 1.0 - hdt * J22, a33 = 1.0 - hdt * J33, a23 = -hdt * J23;
        const double rdet = 1.0 / (a22 * a33 - a23 * a23);
        dqx = (r2 * a33 - a23 * r3) * rdet;
        dqy = (a22 * r3 - a23 * r2) * rdet;
    } else { dqx = r2; dqy = r3; }
    // a9: update, dry handling (R-15)
    double hn = hi + dh;
    const double qxn = qx + dqx, qyn = qy + dqy;
    if (hn < 0.0) { hn = 0.0; nclamp++; }
    Rec Un; Un.h = hn; Un.z = zi;
    double rate = 0.0;
    if (hn > hdry) {
        const double rhn = 1.0 / hn;
        Un.u = qxn * rhn; Un.v = qyn * rhn;
        // a10: local rate of the new state, eq.(15) with d = R_i
        rate = (sqrt(g * hn) + sqrt(Un.u * Un.u + Un.v * Un.v)) * cp.x;
    } else { Un.u = 0.0; Un.v = 0.0; }
    store_rec(Uout + i, Un);
    return rate;
}

} // namespace swe
