// Host-side mesh builder: orientation, edge matching, geometry, locality renumbering.
// Input format follows the paper's mesh file (Fig. 4); the renumbering is the
// single-GPU descendant of the paper's "renumber for contiguous access" idea.
#include "mesh_builder.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <numeric>
#include <atomic>
#include <new>
#include <thread>

namespace swe {

namespace {

// Static partition of [0, n) over the host threads (at most 16); fn(begin, end, thread).  The
// results never depend on the number of threads: every loop below writes disjoint outputs.
template <class F> void parallel_for(int64_t n, F fn, int64_t grain = 65536)
{
    int nthr = (int)std::min<int64_t>(std::min<unsigned>(std::max(1u, std::thread::hardware_concurrency()), 16u),
                                      std::max<int64_t>(1, n / grain));
    if (nthr <= 1) { fn((int64_t)0, n, 0); return; }
    std::vector<std::thread> pool;
    std::atomic<bool> failed(false);
    const int64_t chunk = (n + nthr - 1) / nthr;
    for (int t = 0; t < nthr; t++) {
        const int64_t b = std::min<int64_t>(n, t * chunk), e = std::min<int64_t>(n, b + chunk);
        pool.emplace_back([=, &fn, &failed] { try { fn(b, e, t); } catch (...) { failed = true; } });
    }
    for (auto &th : pool) th.join();
    if (failed) throw std::bad_alloc();      // the only thing these loops can throw
}
constexpr int kMaxHostThreads = 16;

// Hilbert index of (x, y) on a 2^order x 2^order grid (classic rotate-and-flip walk).
inline uint64_t hilbert_d(uint32_t x, uint32_t y, int order)
{
    uint64_t d = 0;
    for (uint32_t s = 1u << (order - 1); s > 0; s >>= 1) {
        uint32_t rx = (x & s) ? 1u : 0u, ry = (y & s) ? 1u : 0u;
        d += (uint64_t)s * s * ((3u * rx) ^ ry);
        if (ry == 0) {
            if (rx == 1) { x = s - 1 - (x & (s - 1)); y = s - 1 - (y & (s - 1)); }
            else { x &= (s - 1); y &= (s - 1); }
            std::swap(x, y);
        } else { x &= (s - 1); y &= (s - 1); }
    }
    return d;
}

void order_hilbert(HostTables &T)
{
    const int64_t nt = T.nt;
    // bounding box of the centroids: per-thread extrema, combined in thread order
    double bx[kMaxHostThreads][4];
    for (auto &r : bx) { r[0] = r[2] = 1e300; r[1] = r[3] = -1e300; }
    parallel_for(nt, [&](int64_t b, int64_t e, int thr) {
        double x0 = 1e300, x1 = -1e300, y0 = 1e300, y1 = -1e300;
        for (int64_t i = b; i < e; i++) {
            x0 = std::min(x0, T.cx[i]); x1 = std::max(x1, T.cx[i]);
            y0 = std::min(y0, T.cy[i]); y1 = std::max(y1, T.cy[i]);
        }
        bx[thr][0] = x0; bx[thr][1] = x1; bx[thr][2] = y0; bx[thr][3] = y1;
    });
    double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300;
    for (auto &r : bx) { xmin = std::min(xmin, r[0]); xmax = std::max(xmax, r[1]); ymin = std::min(ymin, r[2]); ymax = std::max(ymax, r[3]); }
    // 17 bits per axis (square curve cells, so a 10:1 canal still has 2^13.7 of them across): the
    // 34-bit curve index and the caller id (< 2^29) share one 64-bit key
    const int order = 17, idbits = kHostIdBits;
    const double ext = std::max(std::max(xmax - xmin, ymax - ymin), 1e-300);
    const double scale = (double)((1u << order) - 1) / ext;
    std::vector<uint64_t> key((size_t)nt), tmp((size_t)nt);
    parallel_for(nt, [&](int64_t b, int64_t e, int) {
        for (int64_t i = b; i < e; i++) {
            uint32_t qx = (uint32_t)((T.cx[i] - xmin) * scale), qy = (uint32_t)((T.cy[i] - ymin) * scale);
            key[(size_t)i] = (hilbert_d(qx, qy, order) << idbits) | (uint64_t)i;
        }
    });
    // stable LSD radix sort on the curve index, 8 bits per pass, on the host threads: every thread
    // counts and then scatters its own contiguous chunk, offsets by (digit, thread), so the result is
    // the unique stable order whatever the number of threads.  The low bits are the caller id in
    // ascending order to begin with, so ties stay broken by caller id: deterministic
    std::vector<size_t> hist((size_t)kMaxHostThreads * 256);
    for (int shift = idbits; shift < idbits + 2 * order; shift += 8) {
        std::fill(hist.begin(), hist.end(), 0);
        parallel_for(nt, [&](int64_t b, int64_t e, int thr) {
            size_t *h = hist.data() + (size_t)thr * 256;
            for (int64_t i = b; i < e; i++) h[(key[(size_t)i] >> shift) & 0xff]++;
        });
        size_t run = 0;
        for (int d = 0; d < 256; d++)
            for (int t = 0; t < kMaxHostThreads; t++) { const size_t c = hist[(size_t)t * 256 + d]; hist[(size_t)t * 256 + d] = run; run += c; }
        parallel_for(nt, [&](int64_t b, int64_t e, int thr) {
            size_t *h = hist.data() + (size_t)thr * 256;
            for (int64_t i = b; i < e; i++) tmp[h[(key[(size_t)i] >> shift) & 0xff]++] = key[(size_t)i];
        });
        key.swap(tmp);
    }
    parallel_for(nt, [&](int64_t b, int64_t e, int) {
        for (int64_t p = b; p < e; p++) T.perm[(size_t)p] = (int32_t)(key[(size_t)p] & (((uint64_t)1 << idbits) - 1));
    });
}

// Reverse Cuthill-McKee on the dual graph (cells adjacent through an edge; degree <= 3).
void order_rcm(HostTables &T)
{
    const int64_t nt = T.nt;
    std::vector<int32_t> order; order.reserve((size_t)nt);
    std::vector<uint8_t> seen((size_t)nt, 0);
    auto degree = [&](int32_t c) {
        int d = 0;
        for (int k = 0; k < 3; k++) d += T.nbr[3 * (size_t)c + k] >= 0;
        return d;
    };
    auto bfs = [&](int32_t start, std::vector<int32_t> &out, std::vector<uint8_t> &mark) {
        size_t head = out.size();
        out.push_back(start); mark[(size_t)start] = 1;
        while (head < out.size()) {
            int32_t c = out[head++];
            int32_t nb[3]; int n = 0;
            for (int k = 0; k < 3; k++) {
                int32_t j = T.nbr[3 * (size_t)c + k];
                if (j >= 0 && !mark[(size_t)j]) { mark[(size_t)j] = 1; nb[n++] = j; }
            }
            std::sort(nb, nb + n, [&](int32_t a, int32_t b) {
                int da = degree(a), db = degree(b);
                return da != db ? da < db : a < b;
            });
            for (int q = 0; q < n; q++) out.push_back(nb[q]);
        }
    };
    std::vector<uint8_t> tmpmark;
    for (int64_t s = 0; s < nt; s++) {
        if (seen[(size_t)s]) continue;
        // pseudo-peripheral start: last cell of a BFS from s, restricted to s's component
        tmpmark = seen;
        std::vector<int32_t> probe;
        bfs((int32_t)s, probe, tmpmark);
        int32_t start = probe.back();
        bfs(start, order, seen);
    }
    for (int64_t p = 0; p < nt; p++) T.perm[(size_t)p] = order[(size_t)(nt - 1 - p)];
}

} // namespace

int build_tables(const double *nodes_xy, int64_t nn, const int32_t *tris, int64_t nt,
                 const double *bathymetry, const double *manning, const int8_t *bc_tags,
                 int ordering, HostTables &T, std::string &err)
{
    char msg[256];
    T.nn = nn; T.nt = nt;
    try {
        T.nbr.assign(3 * (size_t)nt, 0);
        T.normal.resize(6 * (size_t)nt); T.length.resize(3 * (size_t)nt);
        T.area.resize((size_t)nt); T.inradius.resize((size_t)nt); T.cell_z.resize((size_t)nt);
        T.manning.resize((size_t)nt); T.cx.resize((size_t)nt); T.cy.resize((size_t)nt);
        T.perm.resize((size_t)nt); T.inv.resize((size_t)nt);
    } catch (const std::bad_alloc &) { err = "out of host memory"; return SWE_ERR_NOMEM; }

    for (int64_t i = 0; i < nn; i++) {
        if (!std::isfinite(nodes_xy[2 * i]) || !std::isfinite(nodes_xy[2 * i + 1]) ||
            !std::isfinite(bathymetry[i])) {
            snprintf(msg, sizeof msg, "node %lld has a non-finite coordinate or bed", (long long)i);
            err = msg; return SWE_ERR_BAD_VALUE;
        }
    }
    // ---- orientation + geometry; vertices after the CCW fix kept for edge matching
    std::vector<int32_t> vtx(3 * (size_t)nt);
    std::vector<int8_t> tag(3 * (size_t)nt);
    // first offending triangle per thread: {index, status}; the smallest index is reported
    int64_t bad_i[kMaxHostThreads]; int bad_rc[kMaxHostThreads];
    for (int t = 0; t < kMaxHostThreads; t++) { bad_i[t] = INT64_MAX; bad_rc[t] = SWE_OK; }
    parallel_for(nt, [&](int64_t begin, int64_t end, int thr) {
    for (int64_t i = begin; i < end; i++) {
        int32_t v0 = tris[3 * i], v1 = tris[3 * i + 1], v2 = tris[3 * i + 2];
        int8_t t0 = bc_tags[3 * i], t1 = bc_tags[3 * i + 1], t2 = bc_tags[3 * i + 2];
        if (v0 < 0 || v0 >= nn || v1 < 0 || v1 >= nn || v2 < 0 || v2 >= nn) {
            bad_i[thr] = i; bad_rc[thr] = SWE_ERR_BAD_INDEX; return;
        }
        if (!(manning[i] >= 0.0) || !std::isfinite(manning[i])) {
            bad_i[thr] = i; bad_rc[thr] = SWE_ERR_BAD_VALUE; return;
        }
        double ax = nodes_xy[2 * (size_t)v0], ay = nodes_xy[2 * (size_t)v0 + 1];
        double bx = nodes_xy[2 * (size_t)v1], by = nodes_xy[2 * (size_t)v1 + 1];
        double cx = nodes_xy[2 * (size_t)v2], cy = nodes_xy[2 * (size_t)v2 + 1];
        double twiceA = (bx - ax) * (cy - ay) - (cx - ax) * (by - ay);
        if (twiceA < 0.0) { // clockwise: (v0, v2, v1); new edges 0,1,2 are old edges 2,1,0
            std::swap(v1, v2); std::swap(bx, cx); std::swap(by, cy); std::swap(t0, t2);
            twiceA = (bx - ax) * (cy - ay) - (cx - ax) * (by - ay);
        }
        if (!(twiceA > 0.0)) { bad_i[thr] = i; bad_rc[thr] = SWE_ERR_DEGENERATE; return; }
        const double px[4] = { ax, bx, cx, ax }, py[4] = { ay, by, cy, ay };
        double perimeter = 0.0;
        for (int k = 0; k < 3; k++) {
            const double ex = px[k + 1] - px[k], ey = py[k + 1] - py[k];
            const double L = std::sqrt(ex * ex + ey * ey);
            T.length[3 * (size_t)i + k] = L;
            T.normal[6 * (size_t)i + 2 * k] = ey / L;      // CCW triangle: outward = edge rotated by -90 deg
            T.normal[6 * (size_t)i + 2 * k + 1] = -ex / L;
            perimeter += L;
        }
        const double A = 0.5 * twiceA;
        T.area[(size_t)i] = A;
        T.inradius[(size_t)i] = 2.0 * A / perimeter;
        T.cell_z[(size_t)i] = (bathymetry[v0] + bathymetry[v1] + bathymetry[v2]) / 3.0;
        T.manning[(size_t)i] = manning[i];
        T.cx[(size_t)i] = (ax + bx + cx) / 3.0; T.cy[(size_t)i] = (ay + by + cy) / 3.0;
        vtx[3 * (size_t)i] = v0; vtx[3 * (size_t)i + 1] = v1; vtx[3 * (size_t)i + 2] = v2;
        tag[3 * (size_t)i] = t0; tag[3 * (size_t)i + 1] = t1; tag[3 * (size_t)i + 2] = t2;
    }
    });
    {
        int worst = 0;
        for (int t = 1; t < kMaxHostThreads; t++) if (bad_i[t] < bad_i[worst]) worst = t;
        if (bad_rc[worst] != SWE_OK) {
            const long long i = (long long)bad_i[worst];
            if (bad_rc[worst] == SWE_ERR_BAD_INDEX)
                snprintf(msg, sizeof msg, "triangle %lld refers to a node outside [0, %lld)", i, (long long)nn);
            else if (bad_rc[worst] == SWE_ERR_BAD_VALUE)
                snprintf(msg, sizeof msg, "cell %lld has a negative or non-finite Manning coefficient", i);
            else
                snprintf(msg, sizeof msg, "triangle %lld has zero area", i);
            err = msg; return bad_rc[worst];
        }
    }
    // ---- edge matching: bucket the 3 nt half-edges by their smaller node id (counting sort),
    //      then pair equal larger ids inside each (tiny) bucket
    {
        const size_t ne = 3 * (size_t)nt;
        std::vector<int64_t> start((size_t)nn + 1, 0);
        auto lo_of = [&](size_t e) {
            int32_t a = vtx[e], b = vtx[(e / 3) * 3 + (e % 3 + 1) % 3];
            return a < b ? a : b;
        };
        auto hi_of = [&](size_t e) {
            int32_t a = vtx[e], b = vtx[(e / 3) * 3 + (e % 3 + 1) % 3];
            return a < b ? b : a;
        };
        for (size_t e = 0; e < ne; e++) start[(size_t)lo_of(e) + 1]++;
        for (int64_t n = 0; n < nn; n++) start[(size_t)n + 1] += start[(size_t)n];
        std::vector<int64_t> fill(start.begin(), start.end() - 1);
        std::vector<int64_t> slot(ne);
        for (size_t e = 0; e < ne; e++) slot[(size_t)fill[(size_t)lo_of(e)]++] = (int64_t)e;
        std::fill(T.nbr.begin(), T.nbr.end(), INT32_MIN);
        int64_t bad_n[kMaxHostThreads], bad_hi[kMaxHostThreads];
        for (int t = 0; t < kMaxHostThreads; t++) { bad_n[t] = INT64_MAX; bad_hi[t] = 0; }
        parallel_for(nn, [&](int64_t nbegin, int64_t nend, int thr) {
        for (int64_t n = nbegin; n < nend; n++) {
            for (int64_t a = start[(size_t)n]; a < start[(size_t)n + 1]; a++) {
                const size_t ea = (size_t)slot[(size_t)a];
                int matches = 0;
                for (int64_t b = start[(size_t)n]; b < start[(size_t)n + 1]; b++) {
                    if (b == a) continue;
                    const size_t eb = (size_t)slot[(size_t)b];
                    if (hi_of(eb) == hi_of(ea)) {
                        matches++;
                        T.nbr[ea] = (int32_t)(eb / 3);
                    }
                }
                if (matches > 1) { bad_n[thr] = n; bad_hi[thr] = hi_of(ea); return; }
                if (matches == 0) {
                    int t = tag[ea];
                    if (t <= 0) t = SWE_BC_WALL; // untagged boundary edge
                    T.nbr[ea] = -t;
                }
            }
        }
        });
        int worst = 0;
        for (int t = 1; t < kMaxHostThreads; t++) if (bad_n[t] < bad_n[worst]) worst = t;
        if (bad_n[worst] != INT64_MAX) {
            snprintf(msg, sizeof msg, "edge (%d,%d) is shared by more than two triangles", (int)bad_n[worst], (int)bad_hi[worst]);
            err = msg; return SWE_ERR_NON_MANIFOLD;
        }
        // total boundary length per tag, summed in (cell, local edge) order whatever the threads did
        for (size_t e = 0; e < ne; e++) if (T.nbr[e] < 0) T.inflow_length[-T.nbr[e]] += T.length[e];
    }
    // ---- locality renumbering of the cells (edge order inside each cell is preserved, R-17)
    if (ordering == SWE_ORDER_HILBERT) order_hilbert(T);
    else if (ordering == SWE_ORDER_RCM) order_rcm(T);
    else std::iota(T.perm.begin(), T.perm.end(), 0);
    for (int64_t p = 0; p < nt; p++) T.inv[(size_t)T.perm[(size_t)p]] = (int32_t)p;
    return SWE_OK;
}

// ---- global edge list of the edge-centric two-pass kernels ----------------------------------------
int build_global_edges(const HostTables &T, GlobalEdges &E, std::string &err)
{
    const int64_t nt = T.nt;
    try {
        E.edges.clear(); E.edges.reserve((size_t)nt * 3 / 2 + 1024);
        E.cedge.assign(3 * (size_t)nt, -1);
        std::vector<int32_t> bnum(3 * (size_t)nt, -1);          // boundary edges in (caller cell, local edge) order
        int32_t nb = 0;
        for (size_t e = 0; e < 3 * (size_t)nt; e++) if (T.nbr[e] < 0) bnum[e] = nb++;
        for (int64_t p = 0; p < nt; p++) {
            const int32_t c = T.perm[(size_t)p];
            for (int k = 0; k < 3; k++) {
                const int32_t j = T.nbr[3 * (size_t)c + k];
                const double L = T.length[3 * (size_t)c + k];
                const double *nk = &T.normal[6 * (size_t)c + 2 * k];
                if (E.edges.size() >= (size_t)1 << 30) { err = "too many edges"; return SWE_ERR_INVALID_ARG; }
                const int32_t id = (int32_t)E.edges.size();
                if (j < 0) {
                    E.edges.push_back({ (int32_t)p, -((-j) + 128 * bnum[3 * (size_t)c + k]), L * nk[0], L * nk[1] });
                    E.cedge[3 * (size_t)p + k] = 2 * id;
                    continue;
                }
                const int64_t pj = T.inv[(size_t)j];
                if (pj < p) continue;                            // emitted when pj was visited
                int kj = -1;
                for (int q = 0; q < 3; q++) if (T.nbr[3 * (size_t)j + q] == c) kj = q;
                if (kj < 0) { err = "inconsistent neighbour table"; return SWE_ERR_NON_MANIFOLD; }
                if (c < j) {                                     // a = smaller caller id (R-17)
                    E.edges.push_back({ (int32_t)p, (int32_t)pj, L * nk[0], L * nk[1] });
                    E.cedge[3 * (size_t)p + k] = 2 * id; E.cedge[3 * (size_t)pj + kj] = 2 * id + 1;
                } else {
                    const double Lj = T.length[3 * (size_t)j + kj];
                    E.edges.push_back({ (int32_t)pj, (int32_t)p, Lj * T.normal[6 * (size_t)j + 2 * kj],
                                        Lj * T.normal[6 * (size_t)j + 2 * kj + 1] });
                    E.cedge[3 * (size_t)pj + kj] = 2 * id; E.cedge[3 * (size_t)p + k] = 2 * id + 1;
                }
            }
        }
    } catch (const std::bad_alloc &) { err = "out of host memory"; return SWE_ERR_NOMEM; }
    return SWE_OK;
}

// ---- the paper's mesh file (Fig. 4) ---------------------------------------------
namespace {
// splits a line into numeric tokens; returns false if a token is not a number (a title line)
bool numeric_tokens(const char *line, std::vector<double> &tok)
{
    tok.clear();
    const char *p = line;
    for (;;) {
        while (*p == ' ' || *p == '\t' || *p == '\r' || *p == '\n' || *p == ',' || *p == '|') p++;
        if (!*p) return true;
        char *end = nullptr;
        const double v = std::strtod(p, &end);
        if (end == p) return false;
        if (*end && *end != ' ' && *end != '\t' && *end != '\r' && *end != '\n' && *end != ',' && *end != '|') return false;
        tok.push_back(v);
        p = end;
    }
}
} // namespace

int read_mesh_file(const char *path, int64_t *nn_out, int64_t *nt_out, double *nodes_xy, double *bathymetry,
                   int32_t *tris, double *manning, std::string &err)
{
    if (!path || !nn_out || !nt_out) { err = "read_mesh_file: NULL argument"; return SWE_ERR_INVALID_ARG; }
    FILE *f = std::fopen(path, "r");
    if (!f) { err = std::string("cannot open mesh file ") + path; return SWE_ERR_IO; }
    const bool fill = nodes_xy || bathymetry || tris || manning;
    std::vector<char> buf(1 << 16);
    std::vector<double> tok;
    std::vector<unsigned char> seen;
    int64_t count[2] = { -1, -1 }, rows = 0, lineno = 0;
    int table = -1;                 // 0 node table, 1 connectivity table; -1 before the first count
    int rc = SWE_OK;
    auto fail = [&](const std::string &what) {
        err = std::string(path) + ":" + std::to_string(lineno) + ": " + what; rc = SWE_ERR_FORMAT;
    };
    while (rc == SWE_OK && std::fgets(buf.data(), (int)buf.size(), f)) {
        lineno++;
        if (!numeric_tokens(buf.data(), tok)) {                // a title line
            if (table == 1 && rows == count[1]) break;          // "Ghost cells ...": the rest is multi-GPU
            if (table >= 0 && rows < count[table]) { fail("text inside a table"); break; }
            continue;
        }
        if (tok.empty()) continue;
        if (table < 0 || (rows == count[table] && table == 0)) {   // the count line that opens a table
            if (tok.size() != 1 || tok[0] < 1.0 || tok[0] != std::floor(tok[0]) || tok[0] >= 2147483647.0) {
                fail("expected the number of rows on its own line"); break;
            }
            table++; count[table] = (int64_t)tok[0]; rows = 0;
            if (fill) seen.assign((size_t)count[table], 0);
            continue;
        }
        if (rows == count[table]) break;                        // numbers after the connectivity table: ghost lists
        const size_t want = table == 0 ? 4 : 5;
        if (tok.size() != want) { fail(table == 0 ? "a node row is: id x y z" : "a cell row is: id n1 n2 n3 manning"); break; }
        const double idd = tok[0];
        if (idd < 1.0 || idd > (double)count[table] || idd != std::floor(idd)) { fail("row id out of range (ids are 1-based)"); break; }
        const size_t i = (size_t)idd - 1;
        if (fill) {
            if (seen[i]) { fail("row id appears twice"); break; }
            seen[i] = 1;
            if (table == 0) {
                if (nodes_xy) { nodes_xy[2 * i] = tok[1]; nodes_xy[2 * i + 1] = tok[2]; }
                if (bathymetry) bathymetry[i] = tok[3];
            } else {
                for (int k = 0; k < 3; k++) {
                    const double v = tok[1 + k];
                    if (v < 1.0 || v > (double)count[0] || v != std::floor(v)) { fail("node id out of range (ids are 1-based)"); break; }
                    if (tris) tris[3 * i + k] = (int32_t)v - 1;
                }
                if (manning) manning[i] = tok[4];
            }
        }
        rows++;
    }
    std::fclose(f);
    if (rc != SWE_OK) return rc;
    if (count[0] < 0 || count[1] < 0 || rows != count[1]) {
        err = std::string(path) + ": truncated (node table, then connectivity table expected)";
        return SWE_ERR_FORMAT;
    }
    *nn_out = count[0]; *nt_out = count[1];
    return SWE_OK;
}

void pack_device_edges(const TileTables &X, std::vector<double> &out)
{
    out.assign(3 * X.edges.size(), 0.0);
    const int32_t TC = X.tile_cells;
    const int32_t mask = (1 << kHostIdBits) - 1;
    auto word = [TC, mask](int32_t v) -> uint32_t {
        if (v < 0) return (uint32_t)v;                         // boundary: -(tag + 128 * boundary edge number)
        const uint32_t pos = (uint32_t)(v & mask), k = (uint32_t)v >> kHostIdBits;
        const uint32_t slot = pos < (uint32_t)TC ? k * (uint32_t)(TC + 1) + pos : kDevNoSlot;
        return pos | (k << kDevKShift) | (slot << kDevSlotShift);
    };
    parallel_for(X.ntiles, [&](int64_t tb, int64_t te, int) {
        for (int64_t t = tb; t < te; t++) {
            const size_t e0 = (size_t)X.estart[(size_t)t], nep = (size_t)X.estart[(size_t)t + 1] - e0;
            uint32_t *ab = reinterpret_cast<uint32_t *>(out.data() + 3 * e0);
            double *lxy = out.data() + 3 * e0 + nep;
            for (size_t e = 0; e < nep; e++) {
                const HostEdge &E = X.edges[e0 + e];
                ab[2 * e] = word(E.a); ab[2 * e + 1] = word(E.b);
                lxy[2 * e] = E.lx; lxy[2 * e + 1] = E.ly;
            }
        }
    }, 256);
}

// ---- tile tables: each tile's unique edge list and its cells' constants -------------------------
int build_tiles(const HostTables &T, int tile_cells, double g, TileTables &X, std::string &err)
{
    const int64_t nt = T.nt;
    const int TC = tile_cells;
    if (TC < 32 || TC > 1024) { err = "tile size out of range"; return SWE_ERR_INVALID_ARG; }
    if (nt >= ((int64_t)1 << kHostIdBits)) { err = "more than 2^29 cells"; return SWE_ERR_INVALID_ARG; }
    try {
        X.tile_cells = TC;
        X.ntiles = (nt + TC - 1) / TC;
        X.estart.assign((size_t)X.ntiles + 1, 0);
        std::vector<int32_t> hstart((size_t)X.ntiles + 1, 0), halo, ecount((size_t)X.ntiles, 0);
        X.nedges = 0;
        X.max_halo = 0;
        X.cellc.assign((size_t)X.ntiles * 3 * TC, 1.0);
        X.edges.clear();
        X.max_edges = 0;
        auto local_edge_towards = [&](int32_t c, int32_t other) {   // k with nbr(c,k) == other
            for (int k = 0; k < 3; k++) if (T.nbr[3 * (size_t)c + k] == other) return k;
            return -1;
        };
        auto enc = [](int64_t p, int k) { return (int32_t)(p | ((int64_t)k << kHostIdBits)); };
        // boundary edges numbered in (caller cell, local edge) order
        std::vector<int32_t> bnum(3 * (size_t)nt, -1);
        X.nbedges = 0; X.btag.clear();
        for (size_t e = 0; e < 3 * (size_t)nt; e++)
            if (T.nbr[e] < 0) { bnum[e] = (int32_t)X.nbedges++; X.btag.push_back(-T.nbr[e]); }
        if (X.nbedges >= ((int64_t)1 << 24)) { err = "more than 2^24 boundary edges"; return SWE_ERR_INVALID_ARG; }
        // The tiles are independent: every host thread builds the lists of a contiguous range of
        // tiles into its own vectors, which are then laid end to end in tile order, so the tables do
        // not depend on the number of threads.
        struct Chunk { int64_t tb = 0, te = 0; std::vector<HostEdge> edges; std::vector<int32_t> halo; bool bad = false; };
        std::vector<Chunk> chunks(kMaxHostThreads);
        std::vector<int32_t> epad((size_t)X.ntiles, 0), hcount((size_t)X.ntiles, 0);
        parallel_for(X.ntiles, [&](int64_t tb, int64_t te, int thr) {
            Chunk &C = chunks[(size_t)thr];
            C.tb = tb; C.te = te;
            C.edges.reserve((size_t)(te - tb) * TC * 7 / 4 + 1024);
            // off-tile cell -> halo slot of the current tile: open addressing, stamped by tile
            const size_t hmask = 8191;                      // > 4 x (3 x 1024 cells) never needed: 3 TC <= 3072
            std::vector<int64_t> hkey(hmask + 1, -1); std::vector<int32_t> hslot(hmask + 1, 0), hstamp(hmask + 1, -1);
            for (int64_t t = tb; t < te; t++) {
                const int64_t base = t * TC, nc = std::min<int64_t>(TC, nt - base);
                const size_t first = C.edges.size(), hfirst = C.halo.size();
                // position of internal cell pj in the tile's record array
                auto pos = [&](int64_t pj) -> int64_t {
                    if (pj >= base && pj < base + TC) return pj - base;
                    size_t k = (size_t)((uint64_t)pj * 0x9E3779B97F4A7C15ull >> 40) & hmask;
                    while (hstamp[k] == (int32_t)t && hkey[k] != pj) k = (k + 1) & hmask;
                    if (hstamp[k] != (int32_t)t) {
                        hstamp[k] = (int32_t)t; hkey[k] = pj;
                        hslot[k] = (int32_t)(C.halo.size() - hfirst);
                        C.halo.push_back((int32_t)pj);
                    }
                    return TC + hslot[k];
                };
                double *cc = X.cellc.data() + (size_t)t * 3 * TC;
                for (int64_t q = 0; q < TC; q++) cc[2 * TC + q] = 0.0;
                for (int64_t q = 0; q < nc; q++) {
                    const int64_t p = base + q;
                    const int32_t c = T.perm[(size_t)p];
                    for (int k = 0; k < 3; k++) {
                        const int32_t j = T.nbr[3 * (size_t)c + k];
                        const double *nk = &T.normal[6 * (size_t)c + 2 * k];
                        if (j < 0) {                                   // boundary edge: a = this cell
                            const double L = T.length[3 * (size_t)c + k];
                            C.edges.push_back({ enc(q, k), -((-j) + 128 * bnum[3 * (size_t)c + k]), L * nk[0], L * nk[1] });
                            continue;
                        }
                        const int64_t pj = T.inv[(size_t)j];
                        const bool in_tile = pj >= base && pj < base + nc;
                        if (in_tile && pj < p) continue;               // emitted when pj was visited
                        const int kj = local_edge_towards(j, c);
                        if (kj < 0) { C.bad = true; return; }
                        if (c < j) {                                   // a = smaller caller id (R-17)
                            const double L = T.length[3 * (size_t)c + k];
                            C.edges.push_back({ enc(q, k), enc(pos(pj), kj), L * nk[0], L * nk[1] });
                        } else {
                            const double L = T.length[3 * (size_t)j + kj];
                            C.edges.push_back({ enc(pos(pj), kj), enc(q, k), L * T.normal[6 * (size_t)j + 2 * kj],
                                                L * T.normal[6 * (size_t)j + 2 * kj + 1] });
                        }
                    }
                    cc[q] = 1.0 / T.area[(size_t)c];
                    cc[TC + q] = 1.0 / T.inradius[(size_t)c];
                    cc[2 * TC + q] = g * T.manning[(size_t)c] * T.manning[(size_t)c];
                }
                const size_t cnt = C.edges.size() - first;
                ecount[(size_t)t] = (int32_t)cnt;
                if (cnt & 1) C.edges.push_back({ 0, 0, 0.0, 0.0 });       // pad to 16-byte granules
                epad[(size_t)t] = (int32_t)(C.edges.size() - first);
                hcount[(size_t)t] = (int32_t)(C.halo.size() - hfirst);
            }
        }, 256);
        for (const Chunk &C : chunks) if (C.bad) { err = "inconsistent neighbour table"; return SWE_ERR_NON_MANIFOLD; }
        {
            int64_t etot = 0, htot = 0;
            for (int64_t t = 0; t < X.ntiles; t++) {
                X.estart[(size_t)t] = (int32_t)etot; hstart[(size_t)t] = (int32_t)htot;
                etot += epad[(size_t)t]; htot += hcount[(size_t)t];
                X.nedges += ecount[(size_t)t];
                X.max_edges = std::max(X.max_edges, epad[(size_t)t]);
                X.max_halo = std::max(X.max_halo, hcount[(size_t)t]);
            }
            if (etot > (int64_t)INT32_MAX) { err = "too many edges"; return SWE_ERR_INVALID_ARG; }
            if (htot > (int64_t)INT32_MAX) { err = "too many halo cells"; return SWE_ERR_INVALID_ARG; }
            X.estart[(size_t)X.ntiles] = (int32_t)etot; hstart[(size_t)X.ntiles] = (int32_t)htot;
            X.nhalo = htot;
            X.edges.resize((size_t)etot); halo.resize((size_t)htot);
            std::vector<std::thread> pool;
            for (Chunk &C : chunks) {
                if (C.te <= C.tb) continue;
                pool.emplace_back([&X, &halo, &hstart, &C] {
                    std::copy(C.edges.begin(), C.edges.end(), X.edges.begin() + X.estart[(size_t)C.tb]);
                    std::copy(C.halo.begin(), C.halo.end(), halo.begin() + hstart[(size_t)C.tb]);
                    std::vector<HostEdge>().swap(C.edges);
                });
            }
            for (auto &th : pool) th.join();
        }
        // fixed-stride info blocks (16-byte granules for the bulk copy)
        X.max_halo = (X.max_halo + 3) / 4 * 4;
        const size_t stride = 4 + (size_t)X.max_halo;
        X.tinfo.assign((size_t)X.ntiles * stride, -1);
        for (int64_t t = 0; t < X.ntiles; t++) {
            int32_t *ti = X.tinfo.data() + (size_t)t * stride;
            const int32_t nh = hstart[(size_t)t + 1] - hstart[(size_t)t];
            ti[0] = X.estart[(size_t)t]; ti[1] = ecount[(size_t)t];
            ti[2] = nh; ti[3] = 0;
            for (int32_t e = X.estart[(size_t)t]; e < X.estart[(size_t)t] + ecount[(size_t)t]; e++)
                if (X.edges[(size_t)e].b < 0 && ((-X.edges[(size_t)e].b) & 127) >= SWE_BC_INFLOW0) ti[3] = 1;  // prescribed discharge
            std::copy(halo.begin() + hstart[(size_t)t], halo.begin() + hstart[(size_t)t + 1], ti + 4);
        }
        // the tiles that own each tile's halo cells (distinct, in order of first appearance)
        X.tnbr.assign((size_t)X.ntiles * kTileNbrs, -1);
        parallel_for(X.ntiles, [&](int64_t tb, int64_t te, int) {
            for (int64_t t = tb; t < te; t++) {
                int32_t *row = X.tnbr.data() + (size_t)t * kTileNbrs;
                int cnt = 0; bool never = X.tinfo[(size_t)t * stride + 3] != 0;       // prescribed discharge
                for (int32_t h = hstart[(size_t)t]; h < hstart[(size_t)t + 1] && !never; h++) {
                    const int32_t owner = halo[(size_t)h] / TC;
                    bool seen = false;
                    for (int q = 0; q < cnt; q++) seen |= row[q] == owner;
                    if (seen) continue;
                    if (cnt == kTileNbrs) { never = true; break; }
                    row[cnt++] = owner;
                }
                if (never) { std::fill(row, row + kTileNbrs, -1); row[0] = -2; }
            }
        }, 1024);
    } catch (const std::bad_alloc &) { err = "out of host memory"; return SWE_ERR_NOMEM; }
    return SWE_OK;
}

} // namespace swe
