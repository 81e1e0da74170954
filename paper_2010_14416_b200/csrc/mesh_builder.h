// Host-side mesh tables of libswe_b200 (no CUDA here).  See include/swe.h for the contract.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/swe.h"

namespace swe {

// Tables in the CALLER's cell numbering, as built from the paper's mesh format
// (Fig. 4).  Edge k of cell i joins vertices k and (k+1)%3 after the
// counter-clockwise fix.
struct HostTables {
    int64_t nn = 0, nt = 0;
    std::vector<int32_t> nbr;     // [nt][3] neighbour cell, or -tag on a boundary edge
    std::vector<double> normal;   // [nt][3][2] unit outward normal
    std::vector<double> length;   // [nt][3] L_ij
    std::vector<double> area;     // [nt] |Omega_i|
    std::vector<double> inradius; // [nt] R_i
    std::vector<double> cell_z;   // [nt] cell bed, mean of the node beds (R-1)
    std::vector<double> manning;  // [nt]
    std::vector<double> cx, cy;   // [nt] centroids (ordering only)
    std::vector<int32_t> perm;    // [nt] perm[p] = caller id at internal position p
    std::vector<int32_t> inv;     // [nt] inverse of perm
    double inflow_length[SWE_BC_MAX_TAG + 1] = {}; // sum of edge lengths per tag
};

// Tile tables of the step kernel (swe_kernels.cuh), in the INTERNAL cell numbering: the cells
// are cut into tiles of tile_cells consecutive cells; every edge that touches a tile appears
// once in that tile's edge list (an edge between two tiles appears in both lists).
// Edge end points: bits 0-28 = position in the tile's record array (local cell index if
// < tile_cells, else tile_cells + index into the tile's halo list), bits 29-30 = the edge's local
// index k in that cell.  On a boundary edge b = -(tag + 128 * boundary edge number), the boundary
// edges being numbered in (caller cell, local edge) order.  a is the end point with the smaller
// CALLER id.
// (lx, ly) = edge length times a's unit outward normal.  Lists are padded to an even number of
// records (a zero record) so that every tile's list starts and ends on a 16-byte boundary.
struct HostEdge { int32_t a, b; double lx, ly; };                               // 24 bytes
constexpr int kHostIdBits = 29;
constexpr int kTileNbrs = 16;
struct TileTables {
    int32_t tile_cells = 0;
    int64_t ntiles = 0;
    int32_t max_edges = 0;             // longest (padded) edge list of any tile
    int64_t nedges = 0;                // edge records without the padding
    int32_t max_halo = 0;              // longest halo list of any tile, rounded up to a multiple of 4
    int64_t nhalo = 0;                 // halo entries of all tiles together
    // [ntiles][kTileNbrs] the tiles that own this tile's halo cells, padded with -1; tnbr[t][0] = -2 if
    // the tile has more than kTileNbrs such neighbours or an inflow edge ("never quiet", swe_kernels.cuh)
    std::vector<int32_t> tnbr;
    // [ntiles][4 + max_halo]: {first edge, #edges, #halo ids, 1 if the tile has an inflow edge else 0,
    // halo ids (internal cell ids of the tile's off-tile end points) padded with -1}
    std::vector<int32_t> tinfo;
    int64_t nbedges = 0;               // number of boundary edges
    std::vector<int32_t> btag;         // [nbedges] tag of each boundary edge
    std::vector<int32_t> estart;       // [ntiles + 1] offsets into edges
    std::vector<HostEdge> edges;
    std::vector<double> cellc;         // [ntiles][3][tile_cells]: 1/|Omega|, 1/R, g m^2 (padded with 1, 1, 0)
};

// The edge lists in the layout the step kernel reads (swe_kernels.cuh): per tile, nep = its padded
// edge count, first nep (a, b) word pairs, then nep (lx, ly) pairs; 3 doubles per edge in all, so
// estart still indexes it.  End point word: bits 0-12 position, bits 13-14 local edge k, bits 16-30
// flux slot k * (tile_cells + 1) + position for a cell of the tile, kDevNoSlot for a halo cell;
// boundary words (negative) are kept.
constexpr uint32_t kDevPosMask = 0x1FFFu, kDevNoSlot = 0x7FFFu;
constexpr int kDevKShift = 13, kDevSlotShift = 16;
void pack_device_edges(const TileTables &X, std::vector<double> &out);

// Tables of the edge-centric two-pass kernels (SWE_KERNEL_EDGE_TWO_PASS): every edge of the mesh once,
// in the order in which the internal cell numbering meets it.  a, b = INTERNAL cell ids of the end
// points (a = the end point with the smaller caller id, like in the tile tables; on a boundary edge
// b = -(tag + 128 * boundary edge number) with the same edge numbering); (lx, ly) = edge length times
// a's unit outward normal.  cedge[3 p + k] = 2 * edge + side (side 1: cell p is end point b) for local
// edge k of internal cell p.
struct GlobalEdges {
    std::vector<HostEdge> edges;
    std::vector<int32_t> cedge;
};
int build_global_edges(const HostTables &T, GlobalEdges &E, std::string &err);

// Reader for the paper's mesh-file layout (Fig. 4): a node table (a title line, the
// node count on its own line, rows "id x y z") and a connectivity table (title, cell count, rows
// "id n1 n2 n3 manning"), ids 1-based; anything after the connectivity rows (the "Ghost cells to be
// sent / received" block lists of the multi-GPU decomposition) is ignored.  With all array pointers
// NULL only the counts are returned.  Returns SWE_OK or a negative swe_status with a message in err.
int read_mesh_file(const char *path, int64_t *nn, int64_t *nt, double *nodes_xy, double *bathymetry,
                   int32_t *tris, double *manning, std::string &err);

// Returns SWE_OK or a negative swe_status with a message in err.
int build_tiles(const HostTables &T, int tile_cells, double g, TileTables &X, std::string &err);

// Returns SWE_OK or a negative swe_status with a message in err.
int build_tables(const double *nodes_xy, int64_t nn, const int32_t *tris, int64_t nt,
                 const double *bathymetry, const double *manning, const int8_t *bc_tags,
                 int ordering, HostTables &T, std::string &err);

} // namespace swe
