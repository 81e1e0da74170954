/*
 * swe_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU FP64 implementation of the time-explicit
 * cell-centred finite-volume step of the 2-D Shallow-Water Equations on a triangular
 * mesh, written from the paper (Delmas & Soulaimani, arXiv 2010.14416; PAPER.md) in
 * the paper's order and notation.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may use it.  It shares no code,
 * header, table or helper with the CUDA library (paper_2010_14416_b200/csrc): it has
 * its own neighbour builder, its own geometry and its own solver.
 *
 * Arithmetic rules: double only, compiled -O2 -ffp-contract=off, no fast-math,
 * sqrt()/cbrt() from libm, one independent loop iteration per cell, the three edge
 * contributions added in the fixed order k = 0, 1, 2.  OpenMP over cells only (results
 * do not depend on the thread count: cells are independent and max is exact).
 *
 * Readings of silent / garbled passages are the R-numbers of DESIGN.md section 4.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   oracle_hll         : equals HLLC for equal tangential velocities; pure shear closed form
 *                        -a h (v_R - v_L) / 2 (HLLC: 0); consistency
 *   oracle_hllc        : hand-computed single-edge values (tests/golden/), consistency
 *                        G(U,U) = physical flux, supercritical upwinding, antisymmetry
 *   geometry/neighbours: 2-triangle hand-computed update, rotation invariance
 *   bathymetry source  : lake at rest over a variable bed incl. emergent cells
 *   friction           : closed form q/(1 + dt c |q|) for uniform flow; m = 0 identity;
 *                        the whole Jacobian incl. its d/dh column against the symbolic
 *                        derivative of eq. (32) (its definition, eq. 34) on a non-uniform state
 *   whole step         : Stoker and Ritter dam-break solutions, mass conservation,
 *                        mirror symmetry
 *   boundary volumes   : inflow tag = -Q t exactly, walls 0, tags add up to the total, volume
 *                        change = -sum; run_until: ends on t_end, equals run() before the last step
 *   dt                 : closed form CFL * R_min / (sqrt(g h) + |V|) on a uniform state
 *   inflow flux        : uniform channel flow fed with Q = h u stays steady (momentum term
 *                        Q^2/h + g h^2/2); dry inflow cell hand value
 *   eq.(22) clamp R-6  : dry-bed-generating rarefactions: S_L = u_L - a_L, S_R = u_R + a_R exactly
 *   eq.(24) R-16       : continuity of G_3 with eq.(17) as S_L -> 0-, S_R -> 0+
 *   unpinned conventions: R-1 cell bed = mean of node beds, R-2 g = 9.81.
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define BC_WALL 1
#define BC_TRANSMISSIVE 2
#define BC_INFLOW0 3
#define MAX_TAGS 128

typedef struct {
    int64_t nn, nt;
    double g, cfl, hdry;
    /* geometry, per cell and local edge k (edge k joins vertices k and (k+1)%3) */
    int32_t *tri;      /* [nt][3] CCW */
    int8_t *tag;       /* [nt][3] boundary tag of edge k (after CCW fix) */
    int64_t *nbr;      /* [nt][3] neighbour cell or -1 on the boundary */
    double *n1, *n2;   /* [nt][3] unit outward normal */
    double *len;       /* [nt][3] L_ij */
    double *area;      /* [nt] |Omega_i| */
    double *rin;       /* [nt] inscribed-circle radius R_i */
    double *z;         /* [nt] cell bed (R-1) */
    double *manning;   /* [nt] */
    double qn_tag[MAX_TAGS]; /* unit discharge along the outward normal per inflow tag (R-20) */
    /* state */
    double *h, *hu, *hv, *h2, *hu2, *hv2;
    double t, dt;
    int dt_valid;
    int64_t steps, nclamp;
    long double bnd_volume_out; /* cumulative sum over boundary edges of G1 * L * dt */
    /* boundary diagnostics (inflow / outflow rates are computed every step) */
    int64_t nb;            /* number of boundary edges */
    int32_t *bidx;         /* [nt][3] index of the boundary edge, -1 on interior edges */
    int32_t *btag;         /* [nb] tag of each boundary edge */
    double *bstep;         /* [nb] G1 * L * dt of the current step */
    long double bvol_tag[MAX_TAGS]; /* cumulative outward volume per tag */
    int nthreads;
    int hll;               /* 0: HLLC third component (eq.24), 1: plain HLL for all three (eq.17-18) */
    int storage32;         /* 1: the state {h, u, v} and the cell bed are kept in single precision between the steps
                              (PAPER.md:424 configurable floating-point kind; arithmetic stays double) */
} oracle_mesh;

/* ---------------------------------------------------------------------------------
 * HLLC flux of the 1-D Riemann problem in the edge frame, eq.(17)-(26).
 * Inputs are the (reconstructed) depths and the normal / tangential velocities of the
 * two sides.  Output G[3] = (mass, normal momentum, tangential momentum) flux.
 * diag (may be NULL): {branch, h0, hs, pL, pR, SL, SR, Sstar}; branch 0 both dry,
 * 1 left dry, 2 right dry, 3 rarefaction (eq.22), 4 shock (eq.23).
 * -------------------------------------------------------------------------------*/
static void hllc(double g, double hdry, double hL, double uL, double vL, double hR, double uR,
                 double vR, double G[3], double *diag, int hll)
{
    double SL, SR, Ss, h0 = 0.0, hs = 0.0, pL = 1.0, pR = 1.0;
    int branch;
    int dL = hL <= hdry, dR = hR <= hdry; /* R-15: a side is dry iff h <= h_dry */
    if (dL && dR) {
        G[0] = G[1] = G[2] = 0.0;
        if (diag) { memset(diag, 0, 8 * sizeof(double)); }
        return;
    }
    if (dL) { /* eq.(26) line 1: h_L = 0 */
        hL = uL = vL = 0.0;
        double aR = sqrt(g * hR);
        SL = uR - 2.0 * aR; SR = uR + aR; Ss = SL;
        branch = 1;
    } else if (dR) { /* eq.(26) line 2 (R-18: h_R = 0) */
        hR = uR = vR = 0.0;
        double aL = sqrt(g * hL);
        SL = uL - aL; SR = uL + 2.0 * aL; Ss = SR;
        branch = 2;
    } else {
        double aL = sqrt(g * hL), aR = sqrt(g * hR);
        /* eq.(21) (R-8: the velocities are the normal velocities) */
        h0 = (hL + hR) / 2.0 - (uR - uL) * (hL + hR) / (4.0 * (aR + aL));
        double hmin = hL < hR ? hL : hR;
        if (h0 <= hmin) { /* rarefaction, eq.(22); R-6: bracket clamped at 0 */
            double w = (aR + aL) / 2.0 + (uL - uR) / 4.0;
            if (w < 0.0) w = 0.0;
            hs = w * w / g;
            branch = 3;
        } else { /* shock, eq.(23) */
            double gL = sqrt(g * (h0 + hL) / (2.0 * h0 * hL));
            double gR = sqrt(g * (h0 + hR) / (2.0 * h0 * hR));
            hs = ((hL * gL + hR * gR) + (uL - uR)) / (gL + gR);
            branch = 4;
        }
        /* eq.(20) (R-7: p_k = sqrt(h*(h*+h_k)/2)/h_k) */
        pL = hs > hL ? sqrt(0.5 * hs * (hs + hL)) / hL : 1.0;
        pR = hs > hR ? sqrt(0.5 * hs * (hs + hR)) / hR : 1.0;
        /* eq.(19) */
        SL = uL - aL * pL;
        SR = uR + aR * pR;
        /* eq.(25) */
        Ss = (SL * hR * (uR - SR) - SR * hL * (uL - SL)) / (hR * (uR - SR) - hL * (uL - SL));
    }
    if (diag) {
        diag[0] = branch; diag[1] = h0; diag[2] = hs; diag[3] = pL; diag[4] = pR;
        diag[5] = SL; diag[6] = SR; diag[7] = Ss;
    }
    /* physical flux of the rotated state, R-3: (h u_n, h u_n^2 + g h^2/2, h u_n u_t) */
    double GL0 = hL * uL, GL1 = hL * uL * uL + 0.5 * g * hL * hL, GL2 = hL * uL * vL;
    double GR0 = hR * uR, GR1 = hR * uR * uR + 0.5 * g * hR * hR, GR2 = hR * uR * vR;
    if (SL >= 0.0) { G[0] = GL0; G[1] = GL1; G[2] = GL2; return; } /* eq.(17), R-11 */
    if (SR <= 0.0) { G[0] = GR0; G[1] = GR1; G[2] = GR2; return; }
    /* eq.(18); mass as printed, momentum in the algebraically identical difference form (R-12) */
    G[0] = ((SR * GL0 - SL * GR0) + SR * SL * (hR - hL)) / (SR - SL);
    G[1] = GL1 + SL * (SR * (hR * uR - hL * uL) - (GR1 - GL1)) / (SR - SL);
    if (hll) { /* plain HLL: eq.(18) for the third component too */
        G[2] = ((SR * GL2 - SL * GR2) + SR * SL * (hR * vR - hL * vL)) / (SR - SL);
        return;
    }
    /* eq.(24), R-16: tangential velocity upwinded by the sign of S* */
    G[2] = G[0] * (Ss >= 0.0 ? vL : vR);
}

void oracle_hllc(double g, double hdry, double hL, double uL, double vL, double hR, double uR,
                 double vR, double *G, double *diag)
{
    hllc(g, hdry, hL, uL, vL, hR, uR, vR, G, diag, 0);
}

void oracle_hll(double g, double hdry, double hL, double uL, double vL, double hR, double uR,
                double vR, double *G)
{
    hllc(g, hdry, hL, uL, vL, hR, uR, vR, G, NULL, 1);
}

/* ---------------------------------------------------------------------------------
 * Mesh set-up: orientation, neighbours, geometry.
 * -------------------------------------------------------------------------------*/
typedef struct { uint64_t key; int64_t ck; } edge_rec;

static int edge_cmp(const void *a, const void *b)
{
    const edge_rec *x = (const edge_rec *)a, *y = (const edge_rec *)b;
    if (x->key < y->key) return -1;
    if (x->key > y->key) return 1;
    return (x->ck > y->ck) - (x->ck < y->ck);
}

void oracle_destroy(oracle_mesh *m)
{
    if (!m) return;
    free(m->tri); free(m->tag); free(m->nbr); free(m->n1); free(m->n2); free(m->len);
    free(m->area); free(m->rin); free(m->z); free(m->manning);
    free(m->h); free(m->hu); free(m->hv); free(m->h2); free(m->hu2); free(m->hv2);
    free(m->bidx); free(m->btag); free(m->bstep);
    free(m);
}

/* Returns NULL and writes a code to *err on invalid input:
 * -1 node index out of range, -2 degenerate triangle, -3 edge shared by more than two
 * cells, -4 non-finite coordinate / bed / negative Manning, -5 out of memory. */
oracle_mesh *oracle_create(const double *nodes_xy, int64_t nn, const int32_t *tris, int64_t nt,
                           const double *node_z, const double *manning, const int8_t *bc_tags,
                           double g, double cfl, double hdry, int *err)
{
    *err = 0;
    oracle_mesh *m = (oracle_mesh *)calloc(1, sizeof(oracle_mesh));
    if (!m) { *err = -5; return NULL; }
    m->nn = nn; m->nt = nt; m->g = g; m->cfl = cfl; m->hdry = hdry;
    m->tri = (int32_t *)malloc(sizeof(int32_t) * 3 * nt);
    m->tag = (int8_t *)malloc(3 * nt);
    m->nbr = (int64_t *)malloc(sizeof(int64_t) * 3 * nt);
    m->n1 = (double *)malloc(sizeof(double) * 3 * nt);
    m->n2 = (double *)malloc(sizeof(double) * 3 * nt);
    m->len = (double *)malloc(sizeof(double) * 3 * nt);
    m->area = (double *)malloc(sizeof(double) * nt);
    m->rin = (double *)malloc(sizeof(double) * nt);
    m->z = (double *)malloc(sizeof(double) * nt);
    m->manning = (double *)malloc(sizeof(double) * nt);
    m->h = (double *)calloc(nt, sizeof(double)); m->hu = (double *)calloc(nt, sizeof(double));
    m->hv = (double *)calloc(nt, sizeof(double)); m->h2 = (double *)calloc(nt, sizeof(double));
    m->hu2 = (double *)calloc(nt, sizeof(double)); m->hv2 = (double *)calloc(nt, sizeof(double));
    edge_rec *er = (edge_rec *)malloc(sizeof(edge_rec) * 3 * nt);
    if (!m->tri || !m->tag || !m->nbr || !m->n1 || !m->n2 || !m->len || !m->area || !m->rin ||
        !m->z || !m->manning || !m->h || !m->hu || !m->hv || !m->h2 || !m->hu2 || !m->hv2 || !er) {
        *err = -5; free(er); oracle_destroy(m); return NULL;
    }
#ifdef _OPENMP
    m->nthreads = omp_get_max_threads();
#else
    m->nthreads = 1;
#endif
    for (int64_t i = 0; i < nn; i++) {
        if (!isfinite(nodes_xy[2 * i]) || !isfinite(nodes_xy[2 * i + 1]) || !isfinite(node_z[i])) {
            *err = -4; free(er); oracle_destroy(m); return NULL;
        }
    }
    for (int64_t i = 0; i < nt; i++) {
        int32_t v[3] = { tris[3 * i], tris[3 * i + 1], tris[3 * i + 2] };
        int8_t tg[3] = { bc_tags[3 * i], bc_tags[3 * i + 1], bc_tags[3 * i + 2] };
        for (int k = 0; k < 3; k++)
            if (v[k] < 0 || v[k] >= nn) { *err = -1; free(er); oracle_destroy(m); return NULL; }
        if (!(manning[i] >= 0.0) || !isfinite(manning[i])) { *err = -4; free(er); oracle_destroy(m); return NULL; }
        double x0 = nodes_xy[2 * v[0]], y0 = nodes_xy[2 * v[0] + 1];
        double x1 = nodes_xy[2 * v[1]], y1 = nodes_xy[2 * v[1] + 1];
        double x2 = nodes_xy[2 * v[2]], y2 = nodes_xy[2 * v[2] + 1];
        double A = 0.5 * ((x1 - x0) * (y2 - y0) - (x2 - x0) * (y1 - y0));
        if (A < 0.0) { /* clockwise: swap vertices 1 and 2; edge k of (v0,v2,v1) is old edge 2-k */
            int32_t tv = v[1]; v[1] = v[2]; v[2] = tv;
            int8_t tt = tg[0]; tg[0] = tg[2]; tg[2] = tt;
            double tx = x1, ty = y1; x1 = x2; y1 = y2; x2 = tx; y2 = ty;
            A = 0.5 * ((x1 - x0) * (y2 - y0) - (x2 - x0) * (y1 - y0));
        }
        if (!(A > 0.0)) { *err = -2; free(er); oracle_destroy(m); return NULL; }
        double xs[4] = { x0, x1, x2, x0 }, ys[4] = { y0, y1, y2, y0 };
        double per = 0.0;
        for (int k = 0; k < 3; k++) {
            double ex = xs[k + 1] - xs[k], ey = ys[k + 1] - ys[k];
            double L = sqrt(ex * ex + ey * ey);
            m->len[3 * i + k] = L;
            m->n1[3 * i + k] = ey / L;   /* outward normal of a CCW triangle */
            m->n2[3 * i + k] = -ex / L;
            per += L;
            m->tri[3 * i + k] = v[k];
            m->tag[3 * i + k] = tg[k];
            int32_t a = v[k], b = v[(k + 1) % 3];
            uint64_t lo = (uint64_t)(a < b ? a : b), hi = (uint64_t)(a < b ? b : a);
            er[3 * i + k].key = lo * (uint64_t)nn + hi;
            er[3 * i + k].ck = 3 * i + k;
        }
        m->area[i] = A;
        m->rin[i] = 2.0 * A / per;
        m->z[i] = (node_z[v[0]] + node_z[v[1]] + node_z[v[2]]) / 3.0; /* R-1 */
        m->manning[i] = manning[i];
    }
    /* neighbours: sort the (min,max) node pairs, equal keys are the two sides of an edge */
    qsort(er, (size_t)(3 * nt), sizeof(edge_rec), edge_cmp);
    for (int64_t e = 0; e < 3 * nt;) {
        int64_t f = e + 1;
        while (f < 3 * nt && er[f].key == er[e].key) f++;
        if (f - e > 2) { *err = -3; free(er); oracle_destroy(m); return NULL; }
        if (f - e == 2) {
            m->nbr[er[e].ck] = er[e + 1].ck / 3;
            m->nbr[er[e + 1].ck] = er[e].ck / 3;
        } else {
            m->nbr[er[e].ck] = -1;
            if (m->tag[er[e].ck] <= 0) m->tag[er[e].ck] = BC_WALL; /* untagged boundary = wall */
        }
        e = f;
    }
    free(er);
    for (int k = 0; k < MAX_TAGS; k++) { m->qn_tag[k] = 0.0; m->bvol_tag[k] = 0.0L; }
    /* number the boundary edges in (cell, local edge) order */
    m->bidx = (int32_t *)malloc(sizeof(int32_t) * 3 * nt);
    if (!m->bidx) { *err = -5; oracle_destroy(m); return NULL; }
    m->nb = 0;
    for (int64_t e = 0; e < 3 * nt; e++) m->bidx[e] = m->nbr[e] < 0 ? (int32_t)m->nb++ : -1;
    m->btag = (int32_t *)malloc(sizeof(int32_t) * (m->nb > 0 ? m->nb : 1));
    m->bstep = (double *)calloc((size_t)(m->nb > 0 ? m->nb : 1), sizeof(double));
    if (!m->btag || !m->bstep) { *err = -5; oracle_destroy(m); return NULL; }
    for (int64_t e = 0; e < 3 * nt; e++) if (m->bidx[e] >= 0) m->btag[m->bidx[e]] = m->tag[e];
    return m;
}

/* R-20: total discharge Q (m^3/s, positive into the domain) on a tag group becomes the unit
 * discharge along the outward normal q_n = -Q / sum of the group's edge lengths. */
int oracle_set_inflow(oracle_mesh *m, int tag, double Q_total)
{
    if (tag < BC_INFLOW0 || tag >= MAX_TAGS) return -1;
    long double Lsum = 0.0L;
    for (int64_t e = 0; e < 3 * m->nt; e++)
        if (m->nbr[e] < 0 && m->tag[e] == tag) Lsum += m->len[e];
    if (!(Lsum > 0.0L)) return -2;
    m->qn_tag[tag] = -Q_total / (double)Lsum;
    return 0;
}

/* Single-precision storage (the library's SWE_FP_MIXED32): what is kept between two steps is
 * float(h), float(u), float(v) with u = hu / h of the unrounded new state, and float(z); each step
 * starts from h, h u, h v of those and computes in double as usual. */
static void round_state(oracle_mesh *m)
{
    for (int64_t i = 0; i < m->nt; i++) {
        const double h = m->h[i];
        double u = 0.0, v = 0.0;
        if (h > m->hdry) { u = (double)(float)(m->hu[i] / h); v = (double)(float)(m->hv[i] / h); }
        const double hr = (double)(float)h;
        m->h[i] = hr; m->hu[i] = hr * u; m->hv[i] = hr * v;
    }
}
/* call before oracle_set_state; cannot be switched off again (the cell beds are rounded in place) */
void oracle_set_storage32(oracle_mesh *m)
{
    m->storage32 = 1;
    for (int64_t i = 0; i < m->nt; i++) m->z[i] = (double)(float)m->z[i];
}

void oracle_set_threads(oracle_mesh *m, int n) { m->nthreads = n > 0 ? n : 1; }
void oracle_set_riemann(oracle_mesh *m, int hll) { m->hll = hll != 0; }
int oracle_get_threads(const oracle_mesh *m) { return m->nthreads; }

void oracle_set_state(oracle_mesh *m, const double *h, const double *hu, const double *hv, double t0)
{
    memcpy(m->h, h, sizeof(double) * m->nt);
    memcpy(m->hu, hu, sizeof(double) * m->nt);
    memcpy(m->hv, hv, sizeof(double) * m->nt);
    /* R-15: a dry cell (h <= h_dry) carries no momentum */
    for (int64_t i = 0; i < m->nt; i++)
        if (m->h[i] <= m->hdry) { m->hu[i] = 0.0; m->hv[i] = 0.0; }
    if (m->storage32) round_state(m);
    m->t = t0; m->dt_valid = 0; m->steps = 0; m->nclamp = 0; m->bnd_volume_out = 0.0L;
    for (int k = 0; k < MAX_TAGS; k++) m->bvol_tag[k] = 0.0L;
}

/* CFL time step from the current state, eq.(15), R-9:
 * dt = CFL / max_i (sqrt(g h_i) + sqrt(u_i^2 + v_i^2)) / R_i ; dry cells contribute 0.
 * Returns 0 (and leaves dt = 0) when every cell is dry (R-10). */
double oracle_compute_dt(oracle_mesh *m)
{
    double rmax = 0.0;
#pragma omp parallel for reduction(max : rmax) num_threads(m->nthreads) schedule(static)
    for (int64_t i = 0; i < m->nt; i++) {
        double h = m->h[i];
        if (h > m->hdry) {
            double u = m->hu[i] / h, v = m->hv[i] / h;
            double r = (sqrt(m->g * h) + sqrt(u * u + v * v)) / m->rin[i];
            if (r > rmax) rmax = r;
        }
    }
    m->dt = rmax > 0.0 ? m->cfl / rmax : 0.0;
    m->dt_valid = 1;
    return m->dt;
}

/* One explicit step U^n -> U^{n+1} with the given dt, eq.(37). */
static void step(oracle_mesh *m, double dt)
{
    const double g = m->g, hdry = m->hdry;
    int64_t nclamp = 0;
    long double bvol = 0.0L;
#pragma omp parallel for reduction(+ : nclamp, bvol) num_threads(m->nthreads) schedule(static)
    for (int64_t i = 0; i < m->nt; i++) {
        const double hi = m->h[i], qx = m->hu[i], qy = m->hv[i], zi = m->z[i];
        const int wet = hi > hdry; /* R-15 */
        const double ui = wet ? qx / hi : 0.0, vi = wet ? qy / hi : 0.0;
        double b1 = 0.0, b2 = 0.0, b3 = 0.0;
        for (int k = 0; k < 3; k++) { /* fixed order, R-17 */
            const double n1 = m->n1[3 * i + k], n2 = m->n2[3 * i + k];
            const int64_t j = m->nbr[3 * i + k];
            double G[3], hL;
            /* rotate the cell velocity into the edge frame, eq.(12) */
            const double uL = ui * n1 + vi * n2, vL = -ui * n2 + vi * n1;
            if (j >= 0) {
                /* hydrostatic reconstruction, eq.(28), R-14 */
                const double hj = m->h[j], zj = m->z[j];
                const int wetj = hj > hdry;
                const double uj = wetj ? m->hu[j] / hj : 0.0, vj = wetj ? m->hv[j] / hj : 0.0;
                const double zf = zi > zj ? zi : zj;
                hL = hi + (zi - zf); if (hL < 0.0) hL = 0.0;
                double hR = hj + (zj - zf); if (hR < 0.0) hR = 0.0;
                const double uR = uj * n1 + vj * n2, vR = -uj * n2 + vj * n1;
                hllc(g, hdry, hL, uL, vL, hR, uR, vR, G, NULL, m->hll);
            } else { /* boundary edge */
                const int tag = m->tag[3 * i + k];
                hL = hi;
                if (tag == BC_WALL) { /* R-4: pressure term g h^2/2 only */
                    G[0] = 0.0; G[1] = 0.5 * g * hL * hL; G[2] = 0.0;
                } else if (tag == BC_TRANSMISSIVE) { /* R-21: U_R = U_L gives the physical flux */
                    if (hL > hdry) {
                        G[0] = hL * uL; G[1] = hL * uL * uL + 0.5 * g * hL * hL; G[2] = hL * uL * vL;
                    } else { G[0] = G[1] = G[2] = 0.0; }
                } else { /* prescribed discharge, R-20 */
                    const double qn = m->qn_tag[tag];
                    G[0] = qn; G[2] = 0.0;
                    G[1] = hL > hdry ? qn * qn / hL + 0.5 * g * hL * hL : 0.0;
                }
                bvol += (long double)(G[0] * m->len[3 * i + k] * dt);
                m->bstep[m->bidx[3 * i + k]] = G[0] * m->len[3 * i + k] * dt;
            }
            /* rotate back with T^-1, eq.(12) */
            const double Fx = G[1] * n1 - G[2] * n2, Fy = G[1] * n2 + G[2] * n1;
            /* bathymetry source, eq.(30) with the factor 1/2 (R-13) */
            const double sb = 0.5 * g * (hL * hL - hi * hi);
            const double c = m->len[3 * i + k] / m->area[i];
            b1 += -c * G[0];
            b2 += -c * (Fx - sb * n1);
            b3 += -c * (Fy - sb * n2);
        }
        /* friction: S_f(U_i) and its Jacobian, eq.(32), :242 eq.(35), R-19 */
        double S2 = 0.0, S3 = 0.0, J21 = 0.0, J22 = 0.0, J23 = 0.0, J31 = 0.0, J32 = 0.0, J33 = 0.0;
        const double mn = m->manning[i];
        const double qq = sqrt(qx * qx + qy * qy);
        if (wet && mn > 0.0 && qq > 0.0) {
            const double cf = g * mn * mn / (hi * hi * cbrt(hi)); /* g m^2 / h^(7/3) */
            S2 = -cf * qx * qq; S3 = -cf * qy * qq;
            J21 = (7.0 / 3.0) * cf * qx * qq / hi; J22 = -cf * (qq + qx * qx / qq); J23 = -cf * qx * qy / qq;
            J31 = (7.0 / 3.0) * cf * qy * qq / hi; J32 = J23; J33 = -cf * (qq + qy * qy / qq);
        }
        /* [I - dt/2 J] dU = dt (b + S_f), eq.(37): row 1 explicit, rows 2-3 by Cramer's rule */
        const double dh = dt * b1;
        const double r2 = dt * (b2 + S2) + 0.5 * dt * J21 * dh;
        const double r3 = dt * (b3 + S3) + 0.5 * dt * J31 * dh;
        const double a22 = 1.0 - 0.5 * dt * J22, a23 = -0.5 * dt * J23;
        const double a32 = -0.5 * dt * J32, a33 = 1.0 - 0.5 * dt * J33;
        const double det = a22 * a33 - a23 * a32;
        const double dqx = (r2 * a33 - a23 * r3) / det;
        const double dqy = (a22 * r3 - a32 * r2) / det;
        double hn = hi + dh, qxn = qx + dqx, qyn = qy + dqy;
        if (hn < 0.0) { hn = 0.0; nclamp++; }    /* R-15: must never fire */
        if (hn <= hdry) { qxn = 0.0; qyn = 0.0; } /* R-15: no momentum in dry cells */
        m->h2[i] = hn; m->hu2[i] = qxn; m->hv2[i] = qyn;
    }
    double *t;
    t = m->h; m->h = m->h2; m->h2 = t;
    t = m->hu; m->hu = m->hu2; m->hu2 = t;
    t = m->hv; m->hv = m->hv2; m->hv2 = t;
    if (m->storage32) round_state(m);
    m->nclamp += nclamp;
    m->bnd_volume_out += bvol;
    for (int64_t b = 0; b < m->nb; b++) m->bvol_tag[m->btag[b]] += (long double)m->bstep[b];
    m->t += dt;
    m->steps++;
}

/* nsteps steps; each uses the dt of the state it starts from and leaves the next dt ready
 * ("As soon as the new solution has been updated, the new time step's
 * computation can begin").  Stops early if every cell is dry.  Returns steps done. */
int64_t oracle_run(oracle_mesh *m, int64_t nsteps)
{
    int64_t done = 0;
    if (!m->dt_valid) oracle_compute_dt(m);
    for (; done < nsteps; done++) {
        if (!(m->dt > 0.0)) break;
        step(m, m->dt);
        oracle_compute_dt(m);
    }
    return done;
}

/* Steps until t >= t_end: the step that would pass t_end is shortened to end on it (the paper's
 * runs are specified by simulated time).  At most max_steps.  Returns steps done. */
int64_t oracle_run_until(oracle_mesh *m, double t_end, int64_t max_steps)
{
    int64_t done = 0;
    if (!m->dt_valid) oracle_compute_dt(m);
    while (done < max_steps && m->t < t_end) {
        if (!(m->dt > 0.0) || !isfinite(m->dt)) break;
        double dt = m->dt;
        const int last = t_end - m->t <= dt;
        if (last) dt = t_end - m->t;
        if (!(m->t + dt > m->t)) break; /* a collapsed dt (blow-up) makes no progress: stop, do not spin */
        step(m, dt);
        if (last) m->t = t_end;         /* R-24: the clipped step ends ON t_end (t + (t_end - t) may round off it) */
        oracle_compute_dt(m);
        done++;
    }
    return done;
}

/* vol[MAX_TAGS]: cumulative volume (m^3) that left the domain through the boundary edges of
 * each tag since oracle_set_state (negative = entered). */
void oracle_get_boundary_volumes(const oracle_mesh *m, double *vol)
{
    for (int k = 0; k < MAX_TAGS; k++) vol[k] = (double)m->bvol_tag[k];
}

/* One step with an imposed dt (tests of the closed forms). */
void oracle_step_dt(oracle_mesh *m, double dt) { step(m, dt); m->dt_valid = 0; }

void oracle_get_state(const oracle_mesh *m, double *h, double *hu, double *hv, double *t, double *dt)
{
    if (h) memcpy(h, m->h, sizeof(double) * m->nt);
    if (hu) memcpy(hu, m->hu, sizeof(double) * m->nt);
    if (hv) memcpy(hv, m->hv, sizeof(double) * m->nt);
    if (t) *t = m->t;
    if (dt) *dt = m->dt_valid ? m->dt : -1.0;
}

/* stats[0] = total volume sum h_i |Omega_i|, [1] = #dry cells, [2] = #negative-depth clamps,
 * [3] = steps done, [4] = cumulative volume that left through boundary edges. */
void oracle_get_stats(const oracle_mesh *m, double *stats)
{
    long double vol = 0.0L;
    int64_t ndry = 0;
    for (int64_t i = 0; i < m->nt; i++) {
        vol += (long double)m->h[i] * (long double)m->area[i];
        if (m->h[i] <= m->hdry) ndry++;
    }
    stats[0] = (double)vol; stats[1] = (double)ndry; stats[2] = (double)m->nclamp;
    stats[3] = (double)m->steps; stats[4] = (double)m->bnd_volume_out;
}

/* geometry read-back for the tests: any pointer may be NULL */
void oracle_get_geometry(const oracle_mesh *m, int64_t *nbr, double *n1, double *n2, double *len,
                         double *area, double *rin, double *z)
{
    if (nbr) memcpy(nbr, m->nbr, sizeof(int64_t) * 3 * m->nt);
    if (n1) memcpy(n1, m->n1, sizeof(double) * 3 * m->nt);
    if (n2) memcpy(n2, m->n2, sizeof(double) * 3 * m->nt);
    if (len) memcpy(len, m->len, sizeof(double) * 3 * m->nt);
    if (area) memcpy(area, m->area, sizeof(double) * m->nt);
    if (rin) memcpy(rin, m->rin, sizeof(double) * m->nt);
    if (z) memcpy(z, m->z, sizeof(double) * m->nt);
}
