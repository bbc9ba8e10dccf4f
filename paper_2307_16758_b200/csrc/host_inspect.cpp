// host_inspect.cpp -- host-only inspection entry points (no GPU needed): build the host mesh /
// zone set of host_mesh.cpp and copy named arrays out, so the set-up logic can be tested on a
// CPU-only machine.  Declared in include/swe_b200.h.
#include "../../include/swe_b200.h"
#include "host_mesh.hpp"

#include <cstring>
#include <new>
#include <string>

using namespace swe;

namespace {
struct HostHandle { HostMesh H; ZoneSet Z; bool zones = false; };
thread_local std::string h_err;

template <class T> int64_t copy_out(const std::vector<T>& v, void* out, int64_t cap_bytes) {
    const int64_t bytes = (int64_t)(v.size() * sizeof(T));
    if (out) {
        if (cap_bytes < bytes) return -1;
        if (bytes) std::memcpy(out, v.data(), (size_t)bytes);
    }
    return (int64_t)v.size();
}
int64_t mesh_get(const MeshArrays& M, const std::string& n, void* out, int64_t cap) {
    if (n == "cell_user") return copy_out(M.cell_user, out, cap);
    if (n == "c2c") return copy_out(M.c2c, out, cap);
    if (n == "c2e") return copy_out(M.c2e, out, cap);
    if (n == "zc") return copy_out(M.zc, out, cap);
    if (n == "area") return copy_out(M.area, out, cap);
    if (n == "rin") return copy_out(M.rin, out, cap);
    if (n == "w0") return copy_out(M.w[0], out, cap);
    if (n == "w1") return copy_out(M.w[1], out, cap);
    if (n == "w2") return copy_out(M.w[2], out, cap);
    if (n == "r0") return copy_out(M.r[0], out, cap);
    if (n == "r1") return copy_out(M.r[1], out, cap);
    if (n == "r2") return copy_out(M.r[2], out, cap);
    if (n == "rres") return copy_out(M.rres, out, cap);
    if (n == "elr") return copy_out(M.elr, out, cap);
    if (n == "en") return copy_out(M.en, out, cap);
    if (n == "elen") return copy_out(M.elen, out, cap);
    if (n == "ed") return copy_out(M.ed, out, cap);
    if (n == "edx") return copy_out(M.edx, out, cap);
    if (n == "erl") return copy_out(M.erl, out, cap);
    if (n == "err") return copy_out(M.err, out, cap);
    if (n == "btag") return copy_out(M.btag, out, cap);
    if (n == "dupw") return copy_out(M.dupw, out, cap);
    if (n == "edlr") return copy_out(M.edlr, out, cap);
    if (n == "eside") return copy_out(M.eside, out, cap);
    if (n == "ernorm") return copy_out(M.ernorm, out, cap);
    return -2;
}
}  // namespace

extern "C" {

const char* swe_host_last_error(void) { return h_err.c_str(); }

int swe_host_mesh_build(void** out, int64_t nv, const double* x, const double* y, const double* zb,
                        int64_t nt, const int32_t* tri, int64_t nb, const int32_t* bedge,
                        const int32_t* btag, int renumber) {
    if (!out || nv <= 0 || nt <= 0 || !x || !y || !zb || !tri) { h_err = "bad arguments"; return SWE_ERR_ARG; }
    HostHandle* h = new (std::nothrow) HostHandle();
    if (!h) { h_err = "out of memory"; return SWE_ERR_NOMEM; }
    std::string err;
    if (!build_host_mesh(h->H, nv, x, y, zb, nt, tri, nb, bedge, btag, renumber, err)) {
        delete h; h_err = err; return SWE_ERR_MESH;
    }
    *out = h;
    return SWE_OK;
}
int swe_host_zones_build(void* hh, int nzones, int nlayers, const int32_t* zone_of_cell) {
    HostHandle* h = (HostHandle*)hh;
    if (!h) { h_err = "null handle"; return SWE_ERR_ARG; }
    std::string err;
    h->zones = false;
    if (!build_zones(h->H, h->Z, nzones, nlayers, zone_of_cell, err)) { h_err = err; return SWE_ERR_ARG; }
    h->zones = true;
    return SWE_OK;
}
int swe_host_zones_build_dist(void* hh, int nzones, int nlayers, const int32_t* zone_of_cell, int nranks,
                              int rank, const int32_t* zone_begin) {
    HostHandle* h = (HostHandle*)hh;
    if (!h) { h_err = "null handle"; return SWE_ERR_ARG; }
    std::string err;
    h->zones = false;
    if (!build_zones(h->H, h->Z, nzones, nlayers, zone_of_cell, err, nranks, rank, zone_begin)) { h_err = err; return SWE_ERR_ARG; }
    h->zones = true;
    return SWE_OK;
}
void swe_host_mesh_free(void* hh) { delete (HostHandle*)hh; }

/* Copies the named array to `out` (capacity in bytes) and returns its element count; out == NULL
 * only returns the count.  Names: mesh arrays of host_mesh.hpp ("c2c", "elr", ...), with the prefix
 * "z:" for the concatenated zoned mesh; "user_cell", "cx", "cy"; zone lists "zone_of", "send_idx",
 * "recv_idx", "src_of_cell", "link_off", "link_src", "link_dst", "zone_offset", "zone_nowned";
 * scalars "ne_int", "z:ne_int" are returned as the count itself.  -1: capacity too small,
 * -2: unknown name. */
int64_t swe_host_get(void* hh, const char* name, void* out, int64_t cap_bytes) {
    HostHandle* h = (HostHandle*)hh;
    if (!h || !name) return -2;
    const std::string n(name);
    if (n == "ne_int") return h->H.m.ne_int;
    if (n == "user_cell") return copy_out(h->H.user_cell, out, cap_bytes);
    if (n == "cx") return copy_out(h->H.cx, out, cap_bytes);
    if (n == "cy") return copy_out(h->H.cy, out, cap_bytes);
    if (n == "tags") return copy_out(h->H.tags, out, cap_bytes);
    if (n == "tag_width") return copy_out(h->H.tag_width, out, cap_bytes);
    if (n.rfind("z:", 0) == 0) {
        if (!h->zones) return -2;
        if (n == "z:ne_int") return h->Z.mesh.ne_int;
        return mesh_get(h->Z.mesh, n.substr(2), out, cap_bytes);
    }
    if (h->zones) {
        if (n == "zone_of") return copy_out(h->Z.zone_of, out, cap_bytes);
        if (n == "send_idx") return copy_out(h->Z.send_idx, out, cap_bytes);
        if (n == "recv_idx") return copy_out(h->Z.recv_idx, out, cap_bytes);
        if (n == "src_of_cell") return copy_out(h->Z.src_of_cell, out, cap_bytes);
        if (n == "link_off") return copy_out(h->Z.link_off, out, cap_bytes);
        if (n == "link_src") return copy_out(h->Z.link_src, out, cap_bytes);
        if (n == "link_dst") return copy_out(h->Z.link_dst, out, cap_bytes);
        if (n == "zone_rank") return copy_out(h->Z.zone_rank, out, cap_bytes);
        if (n == "rsend_idx") return copy_out(h->Z.rsend_idx, out, cap_bytes);
        if (n == "rsend_dst") return copy_out(h->Z.rsend_dst, out, cap_bytes);
        if (n == "rsend_peer") return copy_out(h->Z.rsend_peer, out, cap_bytes);
        if (n == "rrecv_idx") return copy_out(h->Z.rrecv_idx, out, cap_bytes);
        if (n == "rsend_off") return copy_out(h->Z.rsend_off, out, cap_bytes);
        if (n == "rrecv_off") return copy_out(h->Z.rrecv_off, out, cap_bytes);
        if (n == "send_cells") return copy_out(h->Z.send_cells, out, cap_bytes);
        if (n == "zone_offset" || n == "zone_nowned" || n == "zone_ncells") {
            std::vector<int64_t> v;
            for (const ZoneDesc& zd : h->Z.z)
                v.push_back(n == "zone_offset" ? zd.offset : (n == "zone_nowned" ? zd.nowned : zd.ncells));
            return copy_out(v, out, cap_bytes);
        }
    }
    return mesh_get(h->H.m, n, out, cap_bytes);
}

}  // extern "C"
