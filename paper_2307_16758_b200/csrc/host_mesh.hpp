// host_mesh.hpp -- host-side mesh set-up of the B200 shallow-water library (not timed, not the
// hot path): topology and geometry of SURVEY.md Appendix A.1, space-filling-curve renumbering,
// zone decomposition of Appendix A.12.  Plain C++17; compiled with -ffp-contract=off so the
// geometry is the literal IEEE evaluation of the formulas of A.1.
#pragma once
#include <cstdint>
#include <functional>
#include <string>
#include <vector>

namespace swe {

constexpr int32_t NB_OUTSIDE = INT32_MIN;  // c2c marker: neighbour not stored in this (zoned) mesh

// Arrays of one mesh in DEVICE numbering (the un-zoned mesh after renumbering, or the
// concatenation of all zones' local meshes).  Interior edges come first, boundary edges last.
struct MeshArrays {
    int64_t nc = 0, ne = 0, ne_int = 0;
    // per cell
    std::vector<int32_t> cell_user;          // user id of the cell
    std::vector<int32_t> c2c;                // 4*nc: 3 neighbours (>=0 cell, -1-e boundary edge e,
                                             //       NB_OUTSIDE) + ghost layer (0 = owned)
    std::vector<int32_t> c2e;                // 4*nc: e (cell is the L-cell) or ~e (R-cell), + layer
    std::vector<double> zc, area, rin;       // cell bed, |Omega_i|, in-radius
    std::vector<double> w[3];                // 2*nc each: least-squares weights (wx,wy) of side k
    std::vector<double> r[3];                // 2*nc each: r_{i,k} = m_e - c_i
    std::vector<float> rres;                 // 2*nc: r_{i,2} + (r_{i,0} + r_{i,1}) in single precision (the device
                                             //       stores r_0, r_1 and this instead of r_2: swe_kernels.cuh stencil_r2)
    std::vector<double> dupw;                // 4*nc: |x_i - x_upw| for side 0,1,2 (multislope MUSCL), pad
    // per edge
    std::vector<int32_t> elr;                // 2*ne: L cell, R cell (-1 on the boundary)
    std::vector<double> en;                  // 2*ne: unit normal, outward of L
    std::vector<double> elen, edx;           // length, WAF Delta-x
    std::vector<double> ed;                  // 2*ne: (dy, -dx) of the edge along its L-cell: en = ed / elen, elen = |ed|
    std::vector<double> erl, err;            // 2*ne each: r_{L,e}, r_{R,e}
    std::vector<double> edlr;                // |x_R - x_L| between the centroids (0 on the boundary)
    std::vector<double> ernorm;              // 2*ne: |r_{L,e}|, |r_{R,e}| (multislope MUSCL face distances)
    std::vector<uint8_t> eside;              // ne: local side of the edge in its L cell | (in its R cell) << 2
    std::vector<int32_t> btag;               // ne-ne_int: user tag of the boundary edge (-1 = none)
};

struct ZoneLink {
    int src = -1;
    int32_t start = 0, count = 0;            // receive range, zone-local
    std::vector<int32_t> send;               // indices local to the source zone
};
struct ZoneDesc {
    int64_t nowned = 0;
    int64_t ncells = 0;                      // owned + ghost cells
    int64_t offset = 0;                      // first cell of the zone in the concatenated mesh
    std::vector<int32_t> cells;              // global DEVICE ids (un-zoned mesh): owned, then ghosts
    std::vector<int32_t> layer;
    std::vector<ZoneLink> links;
};
struct ZoneSet {
    int nz = 0, nlayers = 0;
    std::vector<int32_t> zone_of;            // per cell of the un-zoned mesh (device numbering)
    std::vector<ZoneDesc> z;
    MeshArrays mesh;                         // concatenated zoned mesh
    std::vector<int32_t> src_of_cell;        // per zoned cell: un-zoned device id it mirrors
    // flattened exchange lists over all links in (zone, link) order
    std::vector<int32_t> send_idx;           // concatenated-mesh index of every sent cell
    std::vector<int32_t> recv_idx;           // concatenated-mesh index of the ghost it lands in
    std::vector<int64_t> link_off;           // offsets into send_idx per link (+ total)
    std::vector<int32_t> link_src, link_dst; // zone ids per link
    // distribution over ranks (scope row f3): zones [zone_begin[r], zone_begin[r+1]) live on rank r.
    // Only this rank's zones are in `mesh`; links between two resident zones are in the lists
    // above; links that cross ranks are here, grouped by peer rank and, inside a peer, ordered by
    // (destination zone, source zone) -- the order both ends derive independently.
    int nranks = 1, rank = 0;
    std::vector<int32_t> zone_rank;          // owner rank per zone
    std::vector<int32_t> rsend_idx;          // resident cells packed for remote ghosts
    std::vector<int32_t> rsend_dst;          // where each of them lands: ghost index in the PEER's numbering
    std::vector<int32_t> rsend_peer;         // and the peer rank (for the one-kernel push over peer memory)
    std::vector<int32_t> rrecv_idx;          // resident ghost cells filled from remote owners
    std::vector<int64_t> rsend_off, rrecv_off;   // nranks + 1 each
    std::vector<int32_t> send_cells;         // distinct resident cells on any send list (remote or resident), ascending
};

struct HostMesh {
    int64_t nv = 0, nt = 0, nbe = 0;
    double min_rin = 0.0;
    std::vector<int32_t> user_cell;          // user id -> device id
    std::vector<double> cx, cy;              // centroids, device numbering (zone builder)
    MeshArrays m;                            // un-zoned mesh, device numbering
    std::vector<int32_t> tags;               // distinct user tags
    std::vector<double> tag_width;           // sum of edge lengths per tag
};

// Builds HostMesh; returns false and sets err on invalid input.
bool build_host_mesh(HostMesh& H, int64_t nv, const double* x, const double* y, const double* zb,
                     int64_t nt, const int32_t* tri, int64_t nb, const int32_t* bedge,
                     const int32_t* btag, int renumber, std::string& err);

// Builds the zone decomposition and the concatenated zoned mesh.  zone_of_cell_user may be null
// (recursive coordinate bisection).  Returns false and sets err on invalid arguments.
// ghost_finder (row f4, may be empty): returns the ghost entries of ALL zones as sorted 64-bit keys
//   ((z * nzones + src) * 4 + layer) << 32 | cell      (cell, src = zone_of[cell]: un-zoned device ids)
// i.e. in the order of A.12.3 (zone, source zone, layer, cell).  The library passes the device
// generator of swe_zone_kernels.cuh; without one the layers come from the host breadth-first
// search below (the host-inspection entry points, which must run without a GPU).
using GhostFinder = std::function<bool(const std::vector<int32_t>& zone_of, int nzones, int nlayers,
                                       std::vector<uint64_t>& keys, std::string& err)>;
// The library's device path (row f4, swe_zone_assembly.cuh) takes over what is O(cells) here: it
// hands in the zone of every cell, the number of owned cells per zone and, per ghost key, the
// position of that cell among its owner's cells (`ZoneDeviceLists`), gets the links and exchange
// lists back, and assembles the concatenated zoned mesh on the device itself (assemble = false:
// ZoneSet::mesh, src_of_cell and the owned part of ZoneDesc::cells / layer are then left empty;
// ZoneDesc::ncells always holds the count).
struct ZoneDeviceLists {
    std::vector<int32_t> zone_of;            // per cell of the un-zoned mesh, device numbering (may be left empty)
    std::vector<int64_t> nowned;             // per zone
    std::vector<int32_t> key_owned_pos;      // per ghost key: index of the cell among its owner zone's cells
};
bool build_zones(const HostMesh& H, ZoneSet& Z, int nzones, int nlayers,
                 const int32_t* zone_of_cell_user, std::string& err, int nranks = 1, int rank = 0,
                 const int32_t* zone_begin = nullptr, const GhostFinder& ghost_finder = GhostFinder(),
                 const ZoneDeviceLists* dev = nullptr, bool assemble = true);
// RCB of A.12.1 on the host (used by build_zones when no zone_of_cell is given and by the tests)
void rcb_zones(const HostMesh& H, int nzones, std::vector<int32_t>& zone_of);

}  // namespace swe
