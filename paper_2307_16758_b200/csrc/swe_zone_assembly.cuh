// swe_zone_assembly.cuh -- the zones' copies of the mesh, assembled on the device (SURVEY.md
// section 8(f) row f4, second half; PAPER.md:121-127 and section 3.3 "Renumbering the cells": every
// sub-domain gets its own numbering -- owned cells, then one contiguous block of ghost cells per
// neighbour -- and its own copy of the connectivity and geometry in that numbering).
//
// Round 1 grew the ghost layers on the device (swe_zone_kernels.cuh) but still built the zones'
// arrays in a single-core host loop (2.4 s at 13 M cells) and uploaded them (0.55 s).  Here the
// concatenated zoned mesh never exists on the host:
//   owned cells     stable radix pass of (zone << 32 | cell) on the zone bits: per zone its cells
//                   in ascending id, and for every cell its position among its zone's cells
//   ghost cells     the sorted ghost keys of swe_zone_kernels.cuh, still on the device
//   local index     of global cell g in zone z: offset + owned position if z owns g, else the rank
//                   of the key (z, zone_of[g], layer, g) among z's ghost keys (binary search, at
//                   most one search per possible layer; only cells at zone borders get that far)
//   edges           interior edges touching an owned cell and the boundary edges of cells whose
//                   gradient is evaluated, as keys (zone << 32 | edge), sorted: a zone's edges in
//                   ascending global id; local edge index = rank of the key (binary search)
//   arrays          gathered through those maps by two fill kernels (cells, edges)
// The results do not depend on the order of a zone's edges (a cell sums its three sides in side
// order), so zoned runs stay bit-identical to the un-zoned run; the host builder orders a zone's
// edges as its owned cells first meet them, this one by global edge id.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "swe_kernels.cuh"
#include "swe_zone_kernels.cuh"

namespace swe {

constexpr int ZA_OUTSIDE = INT32_MIN;      // = NB_OUTSIDE of host_mesh.hpp

// small per-zone tables (device arrays of nzr or nzr + 1 entries; r = index among the resident zones)
struct ZoneTabs {
    int nz, nzr, nlayers, gl;
    const int* zres;              // [nz]  zone id -> r, or -1 if the zone lives on another rank
    const int* zid;               // [nzr] r -> zone id
    const long long* coff;        // [nzr + 1] first cell of zone r in the concatenated mesh
    const long long* nown;        // [nzr] owned cells
    const long long* ownstart;    // [nzr] first entry of the zone in the sorted owned keys
    const long long* ghstart;     // [nzr + 1] range of the zone in the sorted ghost keys: [ghstart[r], ghend[r])
    const long long* ghend;
    const long long* ioff;        // [nzr + 1] interior edges of zone r in the concatenated edge list
    const long long* boff;        // [nzr + 1] boundary edges (after all interior edges)
};

__device__ __forceinline__ int za_find(const long long* __restrict__ off, int n, long long v) {   // largest r < n with off[r] <= v
    int lo = 0, hi = n - 1;
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (off[mid] <= v) lo = mid; else hi = mid - 1; }
    return lo;
}
__device__ __forceinline__ long long za_search(const unsigned long long* __restrict__ keys, long long lo, long long hi,
                                               unsigned long long key) {                        // index of key in [lo, hi), or -1
    const long long end = hi;
    while (lo < hi) { const long long mid = (lo + hi) >> 1; if (keys[mid] < key) lo = mid + 1; else hi = mid; }
    return (lo < end && keys[lo] == key) ? lo : -1;
}
// index of global cell g in the concatenated mesh as zone r sees it, or ZA_OUTSIDE
__device__ __forceinline__ int za_loc(const ZoneTabs& T, const int* __restrict__ zone_of, const int* __restrict__ owned_pos,
                                      const unsigned long long* __restrict__ gkeys, int r, int g) {
    const int z = T.zid[r], src = zone_of[g];
    if (src == z) return (int)(T.coff[r] + owned_pos[g]);
    for (int l = 1; l <= T.nlayers; ++l) {
        const unsigned long long key = ((((unsigned long long)z * T.nz + src) * 4ull + l) << 32) | (unsigned int)g;
        const long long p = za_search(gkeys, T.ghstart[r], T.ghend[r], key);
        if (p >= 0) return (int)(T.coff[r] + T.nown[r] + (p - T.ghstart[r]));
    }
    return ZA_OUTSIDE;
}

// ------------------------------------------------------------------------------------------
// A.12.1 recursive coordinate bisection on the device.  The host version sorts nothing: it takes,
// level by level, the lower floor(n/2) cells of every segment in the order (centroid coordinate
// along the longer side of the segment's bounding box, user id).  Here the cells are sorted ONCE
// by (x, user id) and ONCE by (y, user id) -- a stable radix sort of the order-preserving bit
// pattern of the coordinate, started from the cells listed by user id -- and both orders are kept
// segment-major: a level reads every segment's bounding box off the ends of its two ranges, marks
// the cells behind position floor(n/2) of the chosen order as the upper half, and re-partitions
// both orders with one stable radix pass on the new segment ids.  The segment sizes follow from
// the cell count alone (n -> floor(n/2), n - floor(n/2)), so the host knows every range.  Zone
// ids come out as in the host version (first split = most significant bit) and the partition is
// the same set for set (tests: the device lists against the host builder and the oracle).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long rcb_order_bits(double v) {
    unsigned long long b = (unsigned long long)__double_as_longlong(v);
    if (b == 0x8000000000000000ull) b = 0ull;                    // -0.0 compares equal to +0.0
    return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}
// cells in user order: key = order-preserving bits of the coordinate, value = device cell id
__global__ void __launch_bounds__(256) k_rcb_init(const int* __restrict__ user_cell, const double* __restrict__ coord,
                                                  unsigned long long* __restrict__ keys, unsigned int* __restrict__ vals, int nc) {
    for (int u = blockIdx.x * blockDim.x + threadIdx.x; u < nc; u += gridDim.x * blockDim.x) {
        const int cell = user_cell[u];
        keys[u] = rcb_order_bits(coord[cell]);
        vals[u] = (unsigned int)cell;
    }
}
__global__ void __launch_bounds__(256) k_rcb_order(const unsigned int* __restrict__ vals, unsigned long long* __restrict__ keys, int nc) {
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < nc; j += gridDim.x * blockDim.x) keys[j] = vals[j];   // segment 0
}
// one level: seg[] = nseg + 1 range starts (both orders share them); writes the new segment id of every cell
__global__ void __launch_bounds__(256) k_rcb_mark(const unsigned long long* __restrict__ kx, const unsigned long long* __restrict__ ky,
                                                  const double* __restrict__ cx, const double* __restrict__ cy,
                                                  const long long* __restrict__ seg, int nseg, int* __restrict__ newseg, int nc) {
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < nc; j += gridDim.x * blockDim.x) {
        const int s = za_find(seg, nseg, j);
        const long long beg = seg[s], end = seg[s + 1];
        const double xmin = cx[(unsigned int)kx[beg]], xmax = cx[(unsigned int)kx[end - 1]];
        const double ymin = cy[(unsigned int)ky[beg]], ymax = cy[(unsigned int)ky[end - 1]];
        const bool along_x = (xmax - xmin) >= (ymax - ymin);
        const long long nl = (end - beg) / 2;                        // the lower floor(n/2) go left
        const unsigned int cell = (unsigned int)(along_x ? kx[j] : ky[j]);
        newseg[cell] = 2 * s + ((j - beg) >= nl ? 1 : 0);
    }
}
__global__ void __launch_bounds__(256) k_rcb_rekey(unsigned long long* __restrict__ keys, const int* __restrict__ newseg, int nc) {
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < nc; j += gridDim.x * blockDim.x) {
        const unsigned int cell = (unsigned int)keys[j];
        keys[j] = ((unsigned long long)newseg[cell] << 32) | cell;
    }
}

// ---- owned cells ----
__global__ void __launch_bounds__(256) k_za_owned_keys(const int* __restrict__ zone_of, unsigned long long* __restrict__ keys, int nc) {
    for (int g = blockIdx.x * blockDim.x + threadIdx.x; g < nc; g += gridDim.x * blockDim.x)
        keys[g] = ((unsigned long long)zone_of[g] << 32) | (unsigned int)g;
}
// first index of every value of (key >> 32) in a sorted key array (start[] preset to -1)
__global__ void __launch_bounds__(256) k_za_starts(const unsigned long long* __restrict__ keys, long long n, long long* __restrict__ start) {
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < n; j += (long long)gridDim.x * blockDim.x) {
        const unsigned int a = (unsigned int)(keys[j] >> 32);
        if (j == 0 || (unsigned int)(keys[j - 1] >> 32) != a) start[a] = j;
    }
}
__global__ void __launch_bounds__(256) k_za_owned_pos(const unsigned long long* __restrict__ sorted, const long long* __restrict__ start,
                                                      int* __restrict__ owned_pos, int nc) {
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < nc; j += gridDim.x * blockDim.x) {
        const unsigned long long k = sorted[j];
        owned_pos[(unsigned int)k] = (int)(j - start[(unsigned int)(k >> 32)]);
    }
}
// per ghost key: where that cell sits among its owner's cells (the host turns these into send lists)
__global__ void __launch_bounds__(256) k_za_key_opos(const unsigned long long* __restrict__ gkeys, long long nk,
                                                     const int* __restrict__ owned_pos, int* __restrict__ out) {
    for (long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x; j < nk; j += (long long)gridDim.x * blockDim.x)
        out[j] = owned_pos[(unsigned int)gkeys[j]];
}

// ---- the cells of the concatenated mesh: source cell and ghost layer ----
__global__ void __launch_bounds__(256) k_za_cells(ZoneTabs T, const unsigned long long* __restrict__ own_sorted,
                                                  const unsigned long long* __restrict__ gkeys, int* __restrict__ src,
                                                  uint8_t* __restrict__ layer, int ncz) {
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < ncz; c += gridDim.x * blockDim.x) {
        const int r = za_find(T.coff, T.nzr, c);
        const long long j = c - T.coff[r];
        if (j < T.nown[r]) { src[c] = (int)(unsigned int)own_sorted[T.ownstart[r] + j]; layer[c] = 0; }
        else {
            const unsigned long long k = gkeys[T.ghstart[r] + (j - T.nown[r])];
            src[c] = (int)(unsigned int)k; layer[c] = (uint8_t)((k >> 32) & 3u);
        }
    }
}

// ---- edges: count, then emit one key (r << 32 | global edge) per (zone, edge) ----
// interior edge e belongs to every resident zone that owns one of its two cells
__global__ void __launch_bounds__(256) k_za_int_edges(ZoneTabs T, const int* __restrict__ zone_of, const int2* __restrict__ elr,
                                                      int ne_int, unsigned long long* __restrict__ keys, unsigned long long* cursor) {
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < ne_int; e += gridDim.x * blockDim.x) {
        const int2 lr = elr[e];
        const int zL = zone_of[lr.x], zR = zone_of[lr.y];
        const int rL = T.zres[zL], rR = (zR != zL) ? T.zres[zR] : -1;
        const unsigned int n = (rL >= 0) + (rR >= 0);
        if (!n) continue;
        if (keys == nullptr) { atomicAdd(cursor, (unsigned long long)n); continue; }
        unsigned long long at = atomicAdd(cursor, (unsigned long long)n);
        if (rL >= 0) keys[at++] = ((unsigned long long)rL << 32) | (unsigned int)e;
        if (rR >= 0) keys[at] = ((unsigned long long)rR << 32) | (unsigned int)e;
    }
}
// boundary edges of every cell of the concatenated mesh whose gradient is evaluated (layer <= gl)
__global__ void __launch_bounds__(256) k_za_bnd_edges(ZoneTabs T, const int* __restrict__ src, const uint8_t* __restrict__ layer,
                                                      const int4* __restrict__ c2c, int ncz, unsigned long long* __restrict__ keys,
                                                      unsigned long long* cursor) {
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < ncz; c += gridDim.x * blockDim.x) {
        if (layer[c] > T.gl) continue;
        const int4 nb = c2c[src[c]];
        const int nk[3] = {nb.x, nb.y, nb.z};
        const int r = za_find(T.coff, T.nzr, c);
        for (int k = 0; k < 3; ++k) {
            if (nk[k] >= 0) continue;
            const unsigned long long at = atomicAdd(cursor, 1ull);
            if (keys != nullptr) keys[at] = ((unsigned long long)r << 32) | (unsigned int)(-1 - nk[k]);
        }
    }
}

// ---- fill: per-cell arrays of the concatenated mesh ----
struct ZoneCellOut {
    int4* c2c; int4* c2e; int* cell_user; double* zc; double* area; double* rin; double4* dupw;
    double2* w[3]; double2* r[2]; float2* rres;
};
__global__ void __launch_bounds__(256) k_za_fill_cells(ZoneTabs T, DevMesh G, const int* __restrict__ g_cell_user,
                                                       const int* __restrict__ zone_of, const int* __restrict__ owned_pos,
                                                       const unsigned long long* __restrict__ gkeys,
                                                       const unsigned long long* __restrict__ ikeys,
                                                       const unsigned long long* __restrict__ bkeys,
                                                       const int* __restrict__ src, const uint8_t* __restrict__ layer,
                                                       ZoneCellOut O, int ncz, long long ne_int_z) {
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < ncz; c += gridDim.x * blockDim.x) {
        const int g = src[c], lay = layer[c];
        const int r = za_find(T.coff, T.nzr, c);
        O.cell_user[c] = g_cell_user[g];
        O.zc[c] = G.zc[g]; O.area[c] = G.area[g]; O.rin[c] = G.rin[g]; O.dupw[c] = G.dupw[g];
        #pragma unroll
        for (int k = 0; k < 3; ++k) O.w[k][c] = G.w[k][g];
        O.r[0][c] = G.r[0][g]; O.r[1][c] = G.r[1][g]; O.rres[c] = G.rres[g];
        const int4 nb = G.c2c[g], ce = G.c2e[g];
        const int nk[3] = {nb.x, nb.y, nb.z}, ek[3] = {ce.x, ce.y, ce.z};
        int on[3], oe[3];
        #pragma unroll
        for (int k = 0; k < 3; ++k) {
            if (nk[k] >= 0) on[k] = za_loc(T, zone_of, owned_pos, gkeys, r, nk[k]);
            else if (lay <= T.gl) {
                const long long p = za_search(bkeys, T.boff[r] - ne_int_z, T.boff[r + 1] - ne_int_z,
                                              ((unsigned long long)r << 32) | (unsigned int)(-1 - nk[k]));
                on[k] = (int)(-1 - (ne_int_z + p));
            } else on[k] = ZA_OUTSIDE;
            oe[k] = 0;
            if (lay == 0) {                                  // only owned cells are updated: they need their edges
                const int e = ek[k] >= 0 ? ek[k] : ~ek[k];
                long long d;
                if (e < G.ne_int) d = za_search(ikeys, T.ioff[r], T.ioff[r + 1], ((unsigned long long)r << 32) | (unsigned int)e);
                else d = ne_int_z + za_search(bkeys, T.boff[r] - ne_int_z, T.boff[r + 1] - ne_int_z, ((unsigned long long)r << 32) | (unsigned int)e);
                oe[k] = ek[k] >= 0 ? (int)d : ~(int)d;
            }
        }
        O.c2c[c] = make_int4(on[0], on[1], on[2], lay);
        O.c2e[c] = make_int4(oe[0], oe[1], oe[2], lay | (ce.w & 0xff00));      // the cell's Manning code travels along
    }
}
__global__ void __launch_bounds__(256) k_za_mark_send(int4* __restrict__ c2e, const int* __restrict__ cells, int n) {
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) c2e[cells[j]].w |= 0xff;   // flag -1, Manning code kept
}

// ---- fill: per-edge arrays (d < ne_int_z: interior edge ikeys[d]; else boundary edge bkeys[d - ne_int_z]) ----
struct ZoneEdgeOut {
    int2* elr; double2* en; double2* ed; double* elen; double* edx; double2* erl; double2* err; double* edlr; double2* ernorm;
    uint8_t* eside; int* gedge;      // gedge: global id of every boundary edge (for the tags), [ne_z - ne_int_z]
};
__global__ void __launch_bounds__(256) k_za_fill_edges(ZoneTabs T, DevMesh G, const int* __restrict__ zone_of,
                                                       const int* __restrict__ owned_pos,
                                                       const unsigned long long* __restrict__ gkeys,
                                                       const unsigned long long* __restrict__ ikeys,
                                                       const unsigned long long* __restrict__ bkeys, ZoneEdgeOut O,
                                                       long long ne_int_z, long long ne_z) {
    for (long long d = blockIdx.x * (long long)blockDim.x + threadIdx.x; d < ne_z; d += (long long)gridDim.x * blockDim.x) {
        const unsigned long long key = d < ne_int_z ? ikeys[d] : bkeys[d - ne_int_z];
        const int r = (int)(key >> 32), e = (int)(unsigned int)key;
        const int2 lr = G.elr[e];
        O.elr[d] = make_int2(za_loc(T, zone_of, owned_pos, gkeys, r, lr.x),
                             lr.y >= 0 ? za_loc(T, zone_of, owned_pos, gkeys, r, lr.y) : -1);
        O.en[d] = G.en[e]; O.ed[d] = G.ed[e]; O.elen[d] = G.elen[e]; O.edx[d] = G.edx[e]; O.erl[d] = G.erl[e]; O.err[d] = G.err[e];
        O.edlr[d] = G.edlr[e]; O.ernorm[d] = G.ernorm[e]; O.eside[d] = G.eside[e];
        if (d >= ne_int_z) O.gedge[d - ne_int_z] = e;
    }
}

}  // namespace swe
