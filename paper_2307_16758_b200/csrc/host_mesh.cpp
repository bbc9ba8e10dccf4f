// host_mesh.cpp -- host set-up: mesh topology / geometry (following the
// paper's "cell-to-cell adjacency from an edge map" PAPER.md:74), Hilbert renumbering for gather
// locality (BASELINE.json north_star), zone decomposition with ghost layers and send / receive
// lists (A.12).  Not on the timed path.
#include "host_mesh.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>
#include <chrono>
#include <cstdio>
#include <cstdlib>

namespace swe {
namespace {

// Hilbert curve index of integer point (px,py) on an n x n lattice, n = 2^order.
inline uint64_t hilbert_d(uint32_t order, uint32_t px, uint32_t py) {
    const uint32_t n = 1u << order;
    uint64_t d = 0;
    for (uint32_t s = n >> 1; s > 0; s >>= 1) {
        uint32_t rx = (px & s) ? 1u : 0u, ry = (py & s) ? 1u : 0u;
        d += (uint64_t)s * (uint64_t)s * (uint64_t)((3u * rx) ^ ry);
        if (ry == 0) {
            if (rx == 1) { px = n - 1 - px; py = n - 1 - py; }
            std::swap(px, py);
        }
    }
    return d;
}

struct HalfEdge { int32_t hi; int32_t slot; };

// ids sorted by (key, id): stable least-significant-digit radix sort, 16 bits per pass over the
// significant bits of the keys, started from the ids in ascending order (so equal keys stay in id
// order).  Replaces an indirect std::sort (1.1 s of the 4.3 s set-up of 3.3 M cells).
void sort_ids_by_key(const std::vector<uint64_t>& key, std::vector<int32_t>& ids) {
    const size_t n = key.size();
    uint64_t all = 0;
    for (size_t i = 0; i < n; ++i) all |= key[i];
    std::vector<uint64_t> ka(key), kb(n);
    std::vector<int32_t> ib(n);
    for (size_t i = 0; i < n; ++i) ids[i] = (int32_t)i;
    std::vector<size_t> cnt(65536);
    for (int shift = 0; shift < 64 && (all >> shift) != 0; shift += 16) {
        std::fill(cnt.begin(), cnt.end(), 0);
        for (size_t i = 0; i < n; ++i) cnt[(ka[i] >> shift) & 0xffff]++;
        size_t run = 0;
        for (size_t d = 0; d < 65536; ++d) { const size_t c = cnt[d]; cnt[d] = run; run += c; }
        for (size_t i = 0; i < n; ++i) {
            const size_t at = cnt[(ka[i] >> shift) & 0xffff]++;
            kb[at] = ka[i]; ib[at] = ids[i];
        }
        ka.swap(kb); ids.swap(ib);
    }
}

}  // namespace

bool build_host_mesh(HostMesh& H, int64_t nv, const double* x, const double* y, const double* zb,
                     int64_t nt, const int32_t* tri_in, int64_t nb, const int32_t* bedge,
                     const int32_t* btag, int renumber, std::string& err) {
    H = HostMesh();
    H.nv = nv; H.nt = nt;
    // SWE_SETUP_TRACE=1: cumulative seconds after every phase of the set-up, on stderr
    const bool trace = std::getenv("SWE_SETUP_TRACE") != nullptr;
    const auto t_begin = std::chrono::steady_clock::now();
    auto mark = [&](const char* what) {
        if (trace) std::fprintf(stderr, "[swe mesh] %-34s %7.3f s\n", what,
                                std::chrono::duration<double>(std::chrono::steady_clock::now() - t_begin).count());
    };
    if (nt > (int64_t)700000000) { err = "too many cells for int32 side indices"; return false; }
    std::vector<int32_t> tri(tri_in, tri_in + 3 * nt);
    for (int64_t i = 0; i < 3 * nt; ++i)
        if (tri[i] < 0 || tri[i] >= nv) { err = "triangle vertex id out of range"; return false; }

    // ---- A.1.1 / A.1.3 : orientation, area, centroid, cell bed (user numbering) ----
    // Vertex 0 is the pivot of the cross product; a clockwise triangle has its last two vertices
    // exchanged (which flips the sign of the product, re-evaluated so that the stored area is the
    // IEEE result of the counter-clockwise expression).  Means are summed in vertex order.
    std::vector<double> area(nt), ucx(nt), ucy(nt), uzc(nt);
    auto half_cross = [&](const int32_t* t) {
        const double px = x[t[0]], py = y[t[0]];
        return 0.5 * ((x[t[1]] - px) * (y[t[2]] - py) - (x[t[2]] - px) * (y[t[1]] - py));
    };
    auto vertex_mean = [](const double* f, const int32_t* t) { return (f[t[0]] + f[t[1]] + f[t[2]]) / 3.0; };
    // (the loops over cells / edges below that are marked `omp parallel for` touch only their own
    // entries: the threads change who computes an element, not how)
    int degenerate = 0;
    #pragma omp parallel for schedule(static) reduction(| : degenerate)
    for (int64_t c = 0; c < nt; ++c) {
        int32_t* t = tri.data() + 3 * c;
        double omega = half_cross(t);
        if (omega < 0.0) { std::swap(t[1], t[2]); omega = half_cross(t); }
        if (!(omega > 0.0)) degenerate |= 1;
        area[c] = omega;
        ucx[c] = vertex_mean(x, t); ucy[c] = vertex_mean(y, t); uzc[c] = vertex_mean(zb, t);
    }
    if (degenerate) { err = "degenerate (zero-area) triangle"; return false; }

    mark("areas, centroids");
    // ---- A.1.2 : global edges = distinct vertex pairs.  Counting sort of the 3*nt cell sides by
    // their lower vertex id, then pairing inside each bucket by the higher vertex id. ----
    const int64_t ns = 3 * nt;
    std::vector<int64_t> boff(nv + 1, 0);
    auto side_lo_hi = [&](int64_t s, int32_t& lo, int32_t& hi) {
        int64_t i = s / 3; int k = (int)(s % 3);
        int32_t a = tri[3 * i + k], b = tri[3 * i + (k + 1) % 3];
        lo = std::min(a, b); hi = std::max(a, b);
    };
    for (int64_t s = 0; s < ns; ++s) { int32_t lo, hi; side_lo_hi(s, lo, hi); boff[lo + 1]++; }
    for (int64_t v = 0; v < nv; ++v) boff[v + 1] += boff[v];
    std::vector<HalfEdge> he(ns);
    {
        std::vector<int64_t> fill(boff.begin(), boff.end() - 1);
        for (int64_t s = 0; s < ns; ++s) {  // ascending slot => ascending user cell id per bucket
            int32_t lo, hi; side_lo_hi(s, lo, hi);
            if (lo == hi) { err = "triangle repeats a vertex"; return false; }
            he[fill[lo]++] = HalfEdge{hi, (int32_t)s};
        }
    }
    // user-level edges: slot of the L side (smaller user cell id, A.1.4) and of the R side (-1)
    std::vector<int32_t> esL, esR;
    esL.reserve(ns / 2 + nt / 8 + 16); esR.reserve(ns / 2 + nt / 8 + 16);
    std::vector<int32_t> side_edge(ns, -1);
    for (int64_t v = 0; v < nv; ++v) {
        HalfEdge* b = he.data() + boff[v];
        int64_t n = boff[v + 1] - boff[v];
        std::sort(b, b + n, [](const HalfEdge& p, const HalfEdge& q) {
            return p.hi != q.hi ? p.hi < q.hi : p.slot < q.slot; });
        for (int64_t j = 0; j < n;) {
            int64_t j2 = j + 1;
            while (j2 < n && b[j2].hi == b[j].hi) ++j2;
            if (j2 - j > 2) { err = "non-manifold edge (more than two triangles)"; return false; }
            int32_t e = (int32_t)esL.size();
            esL.push_back(b[j].slot);
            esR.push_back(j2 - j == 2 ? b[j + 1].slot : -1);
            side_edge[b[j].slot] = e;
            if (j2 - j == 2) {
                if (b[j].slot / 3 == b[j + 1].slot / 3) { err = "triangle uses an edge twice"; return false; }
                side_edge[b[j + 1].slot] = e;
            }
            j = j2;
        }
    }
    const int64_t ne = (int64_t)esL.size();

    mark("edge pairing");
    // ---- A.1.4 / A.1.6 : edge geometry from the end points a->b as traversed by the L-cell ----
    std::vector<double> elen(ne), enx(ne), eny(ne), edx(ne), rlx(ne), rly(ne), rrx(ne), rry(ne), evx(ne), evy(ne);
    std::vector<int32_t> utag(ne, -1);
    int64_t nbe = 0;
    #pragma omp parallel for schedule(static) reduction(+ : nbe)
    for (int64_t e = 0; e < ne; ++e) {
        int64_t L = esL[e] / 3; int kL = esL[e] % 3;
        int32_t a = tri[3 * L + kL], b = tri[3 * L + (kL + 1) % 3];
        double dx = x[b] - x[a], dy = y[b] - y[a];
        double len = std::sqrt(dx * dx + dy * dy);
        double n1 = dy / len, n2 = -dx / len;
        double mx = 0.5 * (x[a] + x[b]), my = 0.5 * (y[a] + y[b]);
        elen[e] = len; enx[e] = n1; eny[e] = n2;
        evx[e] = dy; evy[e] = -dx;
        rlx[e] = mx - ucx[L]; rly[e] = my - ucy[L];
        if (esR[e] >= 0) {
            int64_t R = esR[e] / 3;
            rrx[e] = mx - ucx[R]; rry[e] = my - ucy[R];
            edx[e] = (rlx[e] * n1 + rly[e] * n2) - (rrx[e] * n1 + rry[e] * n2);
        } else {
            rrx[e] = 0.0; rry[e] = 0.0;
            edx[e] = 2.0 * (rlx[e] * n1 + rly[e] * n2);
            ++nbe;
        }
    }
    H.nbe = nbe;

    mark("edge geometry");
    // ---- boundary tags: look the pair up in its lower vertex's bucket ----
    for (int64_t j = 0; j < nb; ++j) {
        int32_t a = bedge[2 * j], b = bedge[2 * j + 1];
        if (a < 0 || b < 0 || a >= nv || b >= nv) { err = "boundary edge vertex id out of range"; return false; }
        if (btag[j] < 0) { err = "negative boundary tag"; return false; }
        int32_t lo = std::min(a, b), hi = std::max(a, b);
        int32_t e = -1;
        for (int64_t q = boff[lo]; q < boff[lo + 1]; ++q)
            if (he[q].hi == hi) { e = side_edge[he[q].slot]; break; }
        if (e < 0 || esR[e] >= 0) { err = "tagged edge is not a boundary edge"; return false; }
        utag[e] = btag[j];
    }
    he.clear(); he.shrink_to_fit();
    boff.clear(); boff.shrink_to_fit();

    mark("boundary tags");
    // ---- renumbering: Hilbert curve through the centroids (ties by user id) ----
    std::vector<int32_t> cell_user(nt);
    std::iota(cell_user.begin(), cell_user.end(), 0);
    if (renumber == 1 && nt > 1) {
        double xmin = ucx[0], xmax = ucx[0], ymin = ucy[0], ymax = ucy[0];
        for (int64_t i = 1; i < nt; ++i) {
            xmin = std::min(xmin, ucx[i]); xmax = std::max(xmax, ucx[i]);
            ymin = std::min(ymin, ucy[i]); ymax = std::max(ymax, ucy[i]);
        }
        const uint32_t order = 24;
        double ext = std::max(xmax - xmin, ymax - ymin);
        double sc = ext > 0.0 ? ((double)((1u << order) - 1)) / ext : 0.0;
        std::vector<uint64_t> key(nt);
        #pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < nt; ++i) {
            uint32_t px = (uint32_t)((ucx[i] - xmin) * sc), py = (uint32_t)((ucy[i] - ymin) * sc);
            uint64_t d = hilbert_d(order, px, py);
            key[i] = d;
        }
        sort_ids_by_key(key, cell_user);
    }
    // ---- or reverse Cuthill-McKee over the edge adjacency (north_star: "space-filling-curve or RCM
    // pass"): per connected component, root = a minimum-degree cell of the last level of a
    // breadth-first search from the component's lowest user id; neighbours by (degree, user id) ----
    if (renumber == 2 && nt > 1) {
        auto nbr = [&](int32_t u, int k) -> int32_t {
            const int32_t e = side_edge[3 * (int64_t)u + k];
            const int32_t L = esL[e] / 3, R = esR[e] >= 0 ? esR[e] / 3 : -1;
            return L == u ? R : L;
        };
        std::vector<uint8_t> deg(nt, 0), seen(nt, 0), done(nt, 0);
        for (int64_t u = 0; u < nt; ++u)
            for (int k = 0; k < 3; ++k) if (nbr((int32_t)u, k) >= 0) deg[u]++;
        std::vector<int32_t> order; order.reserve(nt);
        std::vector<int32_t> q;
        for (int64_t s0 = 0; s0 < nt; ++s0) {
            if (done[s0]) continue;
            // level structure from s0: the last level's minimum-degree cell becomes the root
            q.assign(1, (int32_t)s0); seen[s0] = 1;
            size_t lstart = 0, lend = 1;
            for (;;) {
                lend = q.size();
                for (size_t h2 = lstart; h2 < lend; ++h2)
                    for (int k = 0; k < 3; ++k) {
                        const int32_t v = nbr(q[h2], k);
                        if (v >= 0 && !seen[v]) { seen[v] = 1; q.push_back(v); }
                    }
                if (q.size() == lend) break;                  // [lstart, lend) is the last level
                lstart = lend;
            }
            int32_t root = q[lstart];
            for (size_t j = lstart; j < lend; ++j)
                if (deg[q[j]] < deg[root] || (deg[q[j]] == deg[root] && q[j] < root)) root = q[j];
            // Cuthill-McKee from the root
            const size_t first = order.size();
            order.push_back(root); done[root] = 1;
            for (size_t h2 = first; h2 < order.size(); ++h2) {
                const int32_t u = order[h2];
                int32_t cand[3]; int nc2 = 0;
                for (int k = 0; k < 3; ++k) {
                    const int32_t v = nbr(u, k);
                    if (v >= 0 && !done[v]) { done[v] = 1; cand[nc2++] = v; }
                }
                auto before = [&](int32_t a, int32_t b) { return deg[a] != deg[b] ? deg[a] < deg[b] : a < b; };
                for (int a = 1; a < nc2; ++a)                  // insertion sort of at most 3
                    for (int b = a; b > 0 && before(cand[b], cand[b - 1]); --b) std::swap(cand[b], cand[b - 1]);
                for (int j = 0; j < nc2; ++j) order.push_back(cand[j]);
            }
        }
        for (int64_t i = 0; i < nt; ++i) cell_user[i] = order[nt - 1 - i];      // reversed
    }
    H.user_cell.resize(nt);
    for (int64_t i = 0; i < nt; ++i) H.user_cell[cell_user[i]] = (int32_t)i;

    mark("renumbering");
    // ---- edge order: interior edges by their lower device cell id, boundary edges last ----
    std::vector<int32_t> eorder(ne);   // device edge id -> user-level edge id
    {
        std::vector<int64_t> cnt(nt + 1, 0);
        std::vector<int32_t> kmin(ne), kmax(ne);
        for (int64_t e = 0; e < ne; ++e) {
            int32_t dl = H.user_cell[esL[e] / 3];
            int32_t dr = esR[e] >= 0 ? H.user_cell[esR[e] / 3] : dl;
            kmin[e] = std::min(dl, dr); kmax[e] = std::max(dl, dr);
        }
        // pass 1: interior
        int64_t pos = 0;
        for (int pass = 0; pass < 2; ++pass) {
            std::fill(cnt.begin(), cnt.end(), 0);
            for (int64_t e = 0; e < ne; ++e)
                if ((esR[e] >= 0) == (pass == 0)) cnt[kmin[e] + 1]++;
            for (int64_t i = 0; i < nt; ++i) cnt[i + 1] += cnt[i];
            int64_t total = cnt[nt];
            std::vector<int64_t> fill(cnt.begin(), cnt.end() - 1);
            for (int64_t e = 0; e < ne; ++e)
                if ((esR[e] >= 0) == (pass == 0)) eorder[pos + fill[kmin[e]]++] = (int32_t)e;
            for (int64_t i = 0; i < nt; ++i) {   // at most 3 per bucket: order by the higher cell id
                int32_t* b = eorder.data() + pos + cnt[i];
                int64_t n = cnt[i + 1] - cnt[i];
                std::sort(b, b + n, [&](int32_t p, int32_t q) {
                    return kmax[p] != kmax[q] ? kmax[p] < kmax[q] : p < q; });
            }
            pos += total;
        }
    }
    std::vector<int32_t> edev(ne);     // user-level edge id -> device edge id
    for (int64_t e = 0; e < ne; ++e) edev[eorder[e]] = (int32_t)e;

    mark("edge order");
    // ---- fill the device-numbered arrays ----
    MeshArrays& M = H.m;
    M.nc = nt; M.ne = ne; M.ne_int = ne - nbe;
    M.cell_user = cell_user;
    M.c2c.assign(4 * nt, 0); M.c2e.assign(4 * nt, 0);
    M.zc.resize(nt); M.area.resize(nt); M.rin.resize(nt);
    for (int k = 0; k < 3; ++k) { M.w[k].resize(2 * nt); M.r[k].resize(2 * nt); }
    M.rres.resize(2 * nt);
    M.elr.resize(2 * ne); M.en.resize(2 * ne); M.elen.resize(ne); M.edx.resize(ne);
    M.erl.resize(2 * ne); M.err.resize(2 * ne); M.ed.resize(2 * ne);
    M.btag.assign(nbe, -1);
    H.cx.resize(nt); H.cy.resize(nt);
    #pragma omp parallel for schedule(static)
    for (int64_t d = 0; d < ne; ++d) {
        int32_t e = eorder[d];
        M.elr[2 * d] = H.user_cell[esL[e] / 3];
        M.elr[2 * d + 1] = esR[e] >= 0 ? H.user_cell[esR[e] / 3] : -1;
        M.en[2 * d] = enx[e]; M.en[2 * d + 1] = eny[e];
        M.elen[d] = elen[e]; M.edx[d] = edx[e];
        M.ed[2 * d] = evx[e]; M.ed[2 * d + 1] = evy[e];
        M.erl[2 * d] = rlx[e]; M.erl[2 * d + 1] = rly[e];
        M.err[2 * d] = rrx[e]; M.err[2 * d + 1] = rry[e];
        if (d >= M.ne_int) M.btag[d - M.ne_int] = utag[e];
    }
    double min_rin = 1e300;
    #pragma omp parallel for schedule(static) reduction(min : min_rin)
    for (int64_t i = 0; i < nt; ++i) {
        int64_t u = cell_user[i];
        M.zc[i] = uzc[u]; M.area[i] = area[u];
        H.cx[i] = ucx[u]; H.cy[i] = ucy[u];
        double rx[3], ry[3], nox[3], noy[3], dxk[3], dyk[3], lk[3];
        for (int k = 0; k < 3; ++k) {
            int32_t e = side_edge[3 * u + k];
            bool isL = (esL[e] == 3 * u + k);
            lk[k] = elen[e];
            if (isL) { rx[k] = rlx[e]; ry[k] = rly[e]; nox[k] = enx[e]; noy[k] = eny[e]; }
            else { rx[k] = rrx[e]; ry[k] = rry[e]; nox[k] = -enx[e]; noy[k] = -eny[e]; }
            int32_t other = isL ? esR[e] : esL[e];
            int32_t d = edev[e];
            M.c2e[4 * i + k] = isL ? d : ~d;
            if (other >= 0) {
                int64_t un = other / 3;
                M.c2c[4 * i + k] = H.user_cell[un];
                dxk[k] = ucx[un] - ucx[u];                    // A.1.7
                dyk[k] = ucy[un] - ucy[u];
            } else {
                M.c2c[4 * i + k] = -1 - d;
                double rn = rx[k] * nox[k] + ry[k] * noy[k];  // mirror point across the boundary edge
                dxk[k] = 2.0 * rn * nox[k];
                dyk[k] = 2.0 * rn * noy[k];
            }
            M.r[k][2 * i] = rx[k]; M.r[k][2 * i + 1] = ry[k];
        }
        for (int q = 0; q < 2; ++q)                           // residual of r_0 + r_1 + r_2 = 0 (exact in double: the sum cancels)
            M.rres[2 * i + q] = (float)(M.r[2][2 * i + q] + (M.r[0][2 * i + q] + M.r[1][2 * i + q]));
        M.rin[i] = 2.0 * area[u] / (lk[0] + lk[1] + lk[2]);   // A.1.5
        min_rin = std::min(min_rin, M.rin[i]);
        // A.1.7: w_k = N^-1 d_k with the normal matrix N = sum_k d_k d_k^T of the three stencil
        // offsets (symmetric 2 x 2, inverted by its adjugate; sums in side order)
        double nxx = 0.0, nxy = 0.0, nyy = 0.0;
        for (int k = 0; k < 3; ++k) {
            nxx += dxk[k] * dxk[k];
            nxy += dxk[k] * dyk[k];
            nyy += dyk[k] * dyk[k];
        }
        const double ndet = nxx * nyy - nxy * nxy;
        for (int k = 0; k < 3; ++k) {
            double* wk = &M.w[k][2 * i];
            wk[0] = (nyy * dxk[k] - nxy * dyk[k]) / ndet;
            wk[1] = (-nxy * dxk[k] + nxx * dyk[k]) / ndet;
        }
    }
    mark("cell arrays, LSQ weights");
    H.min_rin = nt > 0 ? min_rin : 0.0;
    // distances of the multislope MUSCL (eq. 22-25, reading R17): x_upw of side k = mean of the
    // centroids of the two other edge-neighbours (the cell's own centroid where one is missing)
    M.dupw.assign(4 * (size_t)nt, 0.0);
    M.edlr.assign(ne, 0.0);
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < nt; ++i)
        for (int k = 0; k < 3; ++k) {
            double sx = 0.0, sy = 0.0;
            for (int j = 0; j < 3; ++j) {
                if (j == k) continue;
                const int32_t nbq = M.c2c[4 * i + j];
                if (nbq >= 0) { sx += H.cx[nbq]; sy += H.cy[nbq]; }
                else { sx += H.cx[i]; sy += H.cy[i]; }
            }
            const double ux = H.cx[i] - 0.5 * sx, uy = H.cy[i] - 0.5 * sy;
            M.dupw[4 * i + k] = std::sqrt(ux * ux + uy * uy);
        }
    #pragma omp parallel for schedule(static)
    for (int64_t d = 0; d < M.ne_int; ++d) {
        const int32_t L = M.elr[2 * d], R = M.elr[2 * d + 1];
        const double ux = H.cx[R] - H.cx[L], uy = H.cy[R] - H.cy[L];
        M.edlr[d] = std::sqrt(ux * ux + uy * uy);
    }
    M.ernorm.assign(2 * (size_t)ne, 0.0);
    #pragma omp parallel for schedule(static)
    for (int64_t d = 0; d < ne; ++d) {
        M.ernorm[2 * d] = std::sqrt(M.erl[2 * d] * M.erl[2 * d] + M.erl[2 * d + 1] * M.erl[2 * d + 1]);
        M.ernorm[2 * d + 1] = std::sqrt(M.err[2 * d] * M.err[2 * d] + M.err[2 * d + 1] * M.err[2 * d + 1]);
    }
    // local side index of every edge in its two cells (the multislope slopes are stored per side)
    M.eside.assign(ne, 0);
    for (int64_t i = 0; i < nt; ++i)
        for (int k = 0; k < 3; ++k) {
            const int32_t ce = M.c2e[4 * i + k];
            if (ce >= 0) M.eside[ce] |= (uint8_t)k;
            else M.eside[~ce] |= (uint8_t)(k << 2);
        }

    // distinct tags and their widths (sum of edge lengths, reading R10)
    for (int64_t b = 0; b < nbe; ++b) {
        int32_t t = M.btag[b];
        if (t < 0) continue;
        size_t j = 0;
        for (; j < H.tags.size(); ++j) if (H.tags[j] == t) break;
        if (j == H.tags.size()) { H.tags.push_back(t); H.tag_width.push_back(0.0); }
    }
    // widths summed in USER-LEVEL edge order so they do not depend on the renumbering
    for (int64_t e = 0; e < ne; ++e) {
        if (esR[e] >= 0 || utag[e] < 0) continue;
        for (size_t j = 0; j < H.tags.size(); ++j)
            if (H.tags[j] == utag[e]) { H.tag_width[j] += elen[e]; break; }
    }
    mark("multislope distances, tags");
    return true;
}

// ---------------------------------------------------------------------------------------------
// zones (A.12)
// ---------------------------------------------------------------------------------------------
namespace {

void rcb_split(const HostMesh& H, std::vector<int32_t>& ids, int z0, int nz, std::vector<int32_t>& zone_of) {
    if (nz == 1) { for (int32_t i : ids) zone_of[i] = z0; return; }
    double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300;
    for (int32_t i : ids) {
        xmin = std::min(xmin, H.cx[i]); xmax = std::max(xmax, H.cx[i]);
        ymin = std::min(ymin, H.cy[i]); ymax = std::max(ymax, H.cy[i]);
    }
    const std::vector<double>& key = ((xmax - xmin) >= (ymax - ymin)) ? H.cx : H.cy;
    const std::vector<int32_t>& uid = H.m.cell_user;
    size_t nl = ids.size() / 2;
    auto cmp = [&](int32_t a, int32_t b) { return key[a] != key[b] ? key[a] < key[b] : uid[a] < uid[b]; };
    std::nth_element(ids.begin(), ids.begin() + nl, ids.end(), cmp);  // lower floor(n/2) go left
    std::vector<int32_t> left(ids.begin(), ids.begin() + nl), right(ids.begin() + nl, ids.end());
    ids.clear(); ids.shrink_to_fit();
    rcb_split(H, left, z0, nz / 2, zone_of);
    rcb_split(H, right, z0 + nz / 2, nz / 2, zone_of);
}

}  // namespace

void rcb_zones(const HostMesh& H, int nzones, std::vector<int32_t>& zone_of) {
    std::vector<int32_t> ids(H.m.nc);
    std::iota(ids.begin(), ids.end(), 0);
    zone_of.assign(H.m.nc, -1);
    rcb_split(H, ids, 0, nzones, zone_of);
}

bool build_zones(const HostMesh& H, ZoneSet& Z, int nz, int nlayers, const int32_t* zone_of_cell_user,
                 std::string& err, int nranks, int rank, const int32_t* zone_begin,
                 const GhostFinder& ghost_finder, const ZoneDeviceLists* dev, bool assemble) {
    const MeshArrays& G = H.m;
    const int64_t nc = G.nc;
    Z = ZoneSet();
    if (nz < 1) { err = "nzones must be >= 1"; return false; }
    if (nlayers < 1 || nlayers > 3) { err = "nlayers must be 1, 2 or 3"; return false; }
    Z.nz = nz; Z.nlayers = nlayers;
    if (nranks < 1 || rank < 0 || rank >= nranks) { err = "bad rank / nranks"; return false; }
    Z.nranks = nranks; Z.rank = rank;
    Z.zone_rank.assign(nz, 0);
    if (nranks > 1) {
        if (!zone_begin || zone_begin[0] != 0 || zone_begin[nranks] != nz) { err = "zone_begin must run from 0 to nzones"; return false; }
        for (int r = 0; r < nranks; ++r) {
            if (zone_begin[r + 1] < zone_begin[r]) { err = "zone_begin must be non-decreasing"; return false; }
            for (int zi = zone_begin[r]; zi < zone_begin[r + 1]; ++zi) Z.zone_rank[zi] = r;
        }
    }
    auto resident = [&](int zi) { return Z.zone_rank[zi] == rank; };
    Z.zone_of.assign(nc, -1);
    if (dev) {
        if ((!dev->zone_of.empty() && (int64_t)dev->zone_of.size() != nc) || (int64_t)dev->nowned.size() != nz) { err = "bad device zone lists"; return false; }
        Z.zone_of = dev->zone_of;            // may be empty: the zone ids then live on the device only
    } else if (zone_of_cell_user) {
        for (int64_t i = 0; i < nc; ++i) {
            int32_t zc = zone_of_cell_user[G.cell_user[i]];
            if (zc < 0 || zc >= nz) { err = "zone_of_cell value out of range"; return false; }
            Z.zone_of[i] = zc;
        }
    } else {
        if (nz & (nz - 1)) { err = "recursive coordinate bisection needs a power-of-two nzones"; return false; }
        rcb_zones(H, nz, Z.zone_of);
    }
    Z.z.assign(nz, ZoneDesc());
    std::vector<int32_t> owned_pos(dev ? 0 : nc);
    if (dev) {
        for (int zi = 0; zi < nz; ++zi) Z.z[zi].nowned = dev->nowned[zi];
    } else {
        for (int64_t i = 0; i < nc; ++i) {      // owned cells in ascending device id
            ZoneDesc& zd = Z.z[Z.zone_of[i]];
            owned_pos[i] = (int32_t)zd.cells.size();
            zd.cells.push_back((int32_t)i);
        }
        for (int zi = 0; zi < nz; ++zi) Z.z[zi].nowned = (int64_t)Z.z[zi].cells.size();
    }
    // A.12.2 ghost layers = breadth-first distance over the edge adjacency; A.12.3 numbering.
    // From the device generator (sorted keys of all zones) when the library runs, by the host
    // search below when the set-up is inspected without a GPU.
    std::vector<uint64_t> keys;
    if (ghost_finder) {
        if ((int64_t)nz * nz > (int64_t)1 << 29) { err = "too many zones"; return false; }
        if (!ghost_finder(Z.zone_of, nz, nlayers, keys, err)) return false;
    }
    if (dev && (!ghost_finder || dev->key_owned_pos.size() != keys.size())) { err = "bad device zone lists (keys)"; return false; }
    size_t kpos = 0;
    std::vector<int32_t> mark(ghost_finder ? 0 : nc, -1);
    struct Gh { int32_t cell, layer, src, opos; };
    for (int zi = 0; zi < nz; ++zi) {
        ZoneDesc& zd = Z.z[zi];
        zd.layer.assign(zd.cells.size(), 0);
        int64_t cur = zd.nowned;                 // next local index
        std::vector<Gh> ghosts;
        if (ghost_finder) {
            for (; kpos < keys.size(); ++kpos) {
                const uint64_t b = keys[kpos] >> 32;
                if ((int64_t)((b >> 2) / (uint64_t)nz) != zi) break;
                const int32_t cell = (int32_t)(keys[kpos] & 0xffffffffu);
                ghosts.push_back(Gh{cell, (int32_t)(b & 3), (int32_t)((b >> 2) % (uint64_t)nz),
                                    dev ? dev->key_owned_pos[kpos] : owned_pos[cell]});
            }
        } else {
            for (int32_t i : zd.cells) mark[i] = zi;
            std::vector<int32_t> frontier = zd.cells, next;
            for (int l = 1; l <= nlayers; ++l) {
                next.clear();
                for (int32_t i : frontier)
                    for (int k = 0; k < 3; ++k) {
                        int32_t nbq = G.c2c[4 * (int64_t)i + k];
                        if (nbq >= 0 && mark[nbq] != zi) {
                            mark[nbq] = zi; next.push_back(nbq);
                            ghosts.push_back(Gh{nbq, l, Z.zone_of[nbq], owned_pos[nbq]});
                        }
                    }
                frontier.swap(next);
            }
            std::sort(ghosts.begin(), ghosts.end(), [](const Gh& a, const Gh& b) {
                if (a.src != b.src) return a.src < b.src;
                if (a.layer != b.layer) return a.layer < b.layer;
                return a.cell < b.cell; });
        }
        for (const Gh& gq : ghosts) {
            if (zd.links.empty() || zd.links.back().src != gq.src) {
                ZoneLink lk; lk.src = gq.src; lk.start = (int32_t)cur; lk.count = 0;
                zd.links.push_back(lk);
            }
            ZoneLink& lk = zd.links.back();
            lk.count++;
            lk.send.push_back(gq.opos);
            if (!dev) { zd.cells.push_back(gq.cell); zd.layer.push_back(gq.layer); }
            ++cur;
        }
        zd.ncells = cur;
    }
    if (kpos != keys.size()) { err = "ghost keys are not sorted by zone"; return false; }
    // offset of every zone in the concatenated mesh of the rank that holds it
    std::vector<int64_t> owner_off(nz, 0), rank_cells(nranks, 0);
    for (int zi = 0; zi < nz; ++zi) {
        owner_off[zi] = rank_cells[Z.zone_rank[zi]];
        rank_cells[Z.zone_rank[zi]] += Z.z[zi].ncells;
        Z.z[zi].offset = resident(zi) ? owner_off[zi] : -1;
    }
    const int64_t ncz = rank_cells[rank];
    for (int r = 0; r < nranks; ++r)
        if (rank_cells[r] > (int64_t)INT32_MAX / 4) { err = "zoned mesh too large"; return false; }
    if (ncz > (int64_t)INT32_MAX / 4) { err = "zoned mesh too large"; return false; }

    MeshArrays& M = Z.mesh;
    if (assemble) {
    // ---- concatenated zoned mesh ----
    const int gl = (nlayers >= 2) ? 1 : 0;   // gradients are needed on layers <= gl (A.12.5)
    M.nc = ncz;
    M.cell_user.resize(ncz); M.c2c.assign(4 * ncz, 0); M.c2e.assign(4 * ncz, 0);
    M.zc.resize(ncz); M.area.resize(ncz); M.rin.resize(ncz);
    for (int k = 0; k < 3; ++k) { M.w[k].resize(2 * ncz); M.r[k].resize(2 * ncz); }
    M.rres.resize(2 * ncz);
    Z.src_of_cell.resize(ncz);
    std::vector<int32_t> loc(nc, -1);
    std::vector<int32_t> emark(G.ne, -1);
    std::vector<std::vector<int32_t>> zint(nz), zbnd(nz);   // global edge ids per zone
    for (int zi = 0; zi < nz; ++zi) {
        if (!resident(zi)) continue;
        ZoneDesc& zd = Z.z[zi];
        for (size_t j = 0; j < zd.cells.size(); ++j) loc[zd.cells[j]] = (int32_t)j;
        // interior edges touching an owned cell, in the order the owned cells meet them
        for (int64_t j = 0; j < zd.nowned; ++j) {
            int32_t g = zd.cells[j];
            for (int k = 0; k < 3; ++k) {
                int32_t ce = G.c2e[4 * (int64_t)g + k];
                int32_t e = ce >= 0 ? ce : ~ce;
                if (e < G.ne_int && emark[e] != zi) { emark[e] = zi; zint[zi].push_back(e); }
            }
        }
        // boundary edges of every cell whose gradient is evaluated
        for (size_t j = 0; j < zd.cells.size(); ++j) {
            if (zd.layer[j] > gl) continue;
            int32_t g = zd.cells[j];
            for (int k = 0; k < 3; ++k) {
                int32_t nbq = G.c2c[4 * (int64_t)g + k];
                if (nbq < 0) zbnd[zi].push_back(-1 - nbq);
            }
        }
        for (size_t j = 0; j < zd.cells.size(); ++j) loc[zd.cells[j]] = -1;
    }
    std::vector<int64_t> ioff(nz + 1, 0), boff(nz + 1, 0);
    for (int zi = 0; zi < nz; ++zi) { ioff[zi + 1] = ioff[zi] + (int64_t)zint[zi].size(); boff[zi + 1] = boff[zi] + (int64_t)zbnd[zi].size(); }
    M.ne_int = ioff[nz];
    M.ne = M.ne_int + boff[nz];
    if (M.ne > (int64_t)INT32_MAX / 2) { err = "zoned mesh too large"; return false; }
    M.elr.resize(2 * M.ne); M.en.resize(2 * M.ne); M.elen.resize(M.ne); M.edx.resize(M.ne);
    M.erl.resize(2 * M.ne); M.err.resize(2 * M.ne); M.edlr.resize(M.ne);
    M.eside.resize(M.ne); M.ernorm.resize(2 * M.ne); M.ed.resize(2 * M.ne);
    M.dupw.assign(4 * (size_t)ncz, 0.0);
    M.btag.assign(M.ne - M.ne_int, -1);
    std::vector<int32_t> eloc(G.ne, -1);
    for (int zi = 0; zi < nz; ++zi) {
        if (!resident(zi)) continue;
        ZoneDesc& zd = Z.z[zi];
        const int64_t o = zd.offset;
        for (size_t j = 0; j < zd.cells.size(); ++j) loc[zd.cells[j]] = (int32_t)j;
        auto put_edge = [&](int64_t d, int32_t e) {
            int32_t L = G.elr[2 * (int64_t)e], R = G.elr[2 * (int64_t)e + 1];
            M.elr[2 * d] = (int32_t)(o + loc[L]);
            M.elr[2 * d + 1] = R >= 0 ? (int32_t)(o + loc[R]) : -1;
            M.en[2 * d] = G.en[2 * (int64_t)e]; M.en[2 * d + 1] = G.en[2 * (int64_t)e + 1];
            M.ed[2 * d] = G.ed[2 * (int64_t)e]; M.ed[2 * d + 1] = G.ed[2 * (int64_t)e + 1];
            M.elen[d] = G.elen[e]; M.edx[d] = G.edx[e]; M.edlr[d] = G.edlr[e]; M.eside[d] = G.eside[e];
            M.ernorm[2 * d] = G.ernorm[2 * (int64_t)e]; M.ernorm[2 * d + 1] = G.ernorm[2 * (int64_t)e + 1];
            M.erl[2 * d] = G.erl[2 * (int64_t)e]; M.erl[2 * d + 1] = G.erl[2 * (int64_t)e + 1];
            M.err[2 * d] = G.err[2 * (int64_t)e]; M.err[2 * d + 1] = G.err[2 * (int64_t)e + 1];
            eloc[e] = (int32_t)d;
        };
        for (size_t q = 0; q < zint[zi].size(); ++q) put_edge(ioff[zi] + (int64_t)q, zint[zi][q]);
        for (size_t q = 0; q < zbnd[zi].size(); ++q) {
            int64_t d = M.ne_int + boff[zi] + (int64_t)q;
            put_edge(d, zbnd[zi][q]);
            M.btag[d - M.ne_int] = G.btag[zbnd[zi][q] - G.ne_int];
        }
        for (size_t j = 0; j < zd.cells.size(); ++j) {
            const int64_t g = zd.cells[j], c = o + (int64_t)j;
            const int lay = zd.layer[j];
            M.cell_user[c] = G.cell_user[g];
            Z.src_of_cell[c] = (int32_t)g;
            M.zc[c] = G.zc[g]; M.area[c] = G.area[g]; M.rin[c] = G.rin[g];
            for (int k = 0; k < 3; ++k) M.dupw[4 * c + k] = G.dupw[4 * g + k];
            M.rres[2 * c] = G.rres[2 * g]; M.rres[2 * c + 1] = G.rres[2 * g + 1];
            for (int k = 0; k < 3; ++k) {
                M.w[k][2 * c] = G.w[k][2 * g]; M.w[k][2 * c + 1] = G.w[k][2 * g + 1];
                M.r[k][2 * c] = G.r[k][2 * g]; M.r[k][2 * c + 1] = G.r[k][2 * g + 1];
                int32_t nbq = G.c2c[4 * g + k];
                int32_t v;
                if (nbq >= 0) v = loc[nbq] >= 0 ? (int32_t)(o + loc[nbq]) : NB_OUTSIDE;
                else v = (lay <= gl) ? (-1 - eloc[-1 - nbq]) : NB_OUTSIDE;
                M.c2c[4 * c + k] = v;
                if (lay == 0) {
                    int32_t ce = G.c2e[4 * g + k];
                    int32_t e = ce >= 0 ? ce : ~ce;
                    M.c2e[4 * c + k] = ce >= 0 ? eloc[e] : ~eloc[e];
                }
            }
            M.c2c[4 * c + 3] = lay;
            M.c2e[4 * c + 3] = lay;
        }
        for (size_t j = 0; j < zd.cells.size(); ++j) loc[zd.cells[j]] = -1;
    }
    }   // assemble
    // ---- flattened exchange lists: links between two resident zones ----
    Z.link_off.push_back(0);
    for (int zi = 0; zi < nz; ++zi) {
        if (!resident(zi)) continue;
        for (const ZoneLink& lk : Z.z[zi].links) {
            if (!resident(lk.src)) continue;
            for (int32_t j = 0; j < lk.count; ++j) {
                Z.send_idx.push_back((int32_t)(Z.z[lk.src].offset + lk.send[j]));
                Z.recv_idx.push_back((int32_t)(Z.z[zi].offset + lk.start + j));
            }
            Z.link_off.push_back((int64_t)Z.send_idx.size());
            Z.link_src.push_back(lk.src);
            Z.link_dst.push_back(zi);
        }
    }
    // ---- links that cross ranks, grouped by peer, ordered by (destination zone, source zone) ----
    Z.rsend_off.assign(nranks + 1, 0);
    Z.rrecv_off.assign(nranks + 1, 0);
    for (int p = 0; p < nranks; ++p) {
        if (p != rank)
            for (int zi = 0; zi < nz; ++zi)
                for (const ZoneLink& lk : Z.z[zi].links) {
                    if (Z.zone_rank[zi] == p && resident(lk.src))          // we own the source
                        for (int32_t j = 0; j < lk.count; ++j) {
                            Z.rsend_idx.push_back((int32_t)(Z.z[lk.src].offset + lk.send[j]));
                            Z.rsend_dst.push_back((int32_t)(owner_off[zi] + lk.start + j));
                            Z.rsend_peer.push_back(p);
                        }
                    if (resident(zi) && Z.zone_rank[lk.src] == p)          // we own the ghost
                        for (int32_t j = 0; j < lk.count; ++j)
                            Z.rrecv_idx.push_back((int32_t)(Z.z[zi].offset + lk.start + j));
                }
        Z.rsend_off[p + 1] = (int64_t)Z.rsend_idx.size();
        Z.rrecv_off[p + 1] = (int64_t)Z.rrecv_idx.size();
    }
    // ---- cells on any send list (remote or resident), ascending: the overlap schedule updates them
    // first; they carry -1 in c2e.w (owned cells otherwise carry 0).  Built for one rank too: the
    // links between resident zones are served by the same exchange ----
    {
        Z.send_cells = Z.rsend_idx;
        Z.send_cells.insert(Z.send_cells.end(), Z.send_idx.begin(), Z.send_idx.end());
        std::sort(Z.send_cells.begin(), Z.send_cells.end());
        Z.send_cells.erase(std::unique(Z.send_cells.begin(), Z.send_cells.end()), Z.send_cells.end());
        if (assemble) for (int32_t c : Z.send_cells) M.c2e[4 * (int64_t)c + 3] = -1;
    }
    return true;
}

}  // namespace swe
