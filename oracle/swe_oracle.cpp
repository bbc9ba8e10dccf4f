// swe_oracle.cpp -- CPU ORACLE for the shallow-water finite-volume time step.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
// header, table or helper with paper_2307_16758_b200/ (the CUDA library) and neither includes the
// other.  Plain C++17, double precision, compile with -O2 -ffp-contract=off.
//
// What it computes: the explicit time step of Delmas & Soulaimani (arxiv 2307.16758, PAPER.md)
// section 6.1-6.2 on an unstructured triangle mesh, cell by cell, in the paper's order and
// notation, with the readings of DESIGN.md ("Readings of the paper") where the paper is silent,
// garbled or at odds with itself:
//   eq. 1   state U=(h, hu, hv)
//   eq. 2   rotation T_n, T_n^-1
//   eq. 3   finite-volume update over the three sides
//   BCs     transmissive, imposed inflow Q, wall
//   eq. 5   CFL time step with d = in-circle radius
//   eq. 6-14  HLL / HLLC flux, wave speeds
//   eq. 15-21 WAF flux, TVD weights, SUPERBEE A(r,c)
//   eq. 24-25 limiter semantics (beta=1 MINBEE) for the cell limiter PAPER.md:410-420
//   eq. 22-25 the paper's own multislope MUSCL (scheme 3, scope row f1) PAPER.md:396-420
//   hydrostatic reconstruction, bed-slope and friction sources: named only;
//   formulas = DESIGN.md readings R12, R15.  LSQ gradients and Heun RK2: BASELINE.json north_star.
//   zones / ghost layers / send lists / contiguous receive ranges
//
// Structure: pass G (limited gradients of every cell into an array) then pass C (each cell loops
// over its three edges, evaluates the edge flux itself in the canonical L/R orientation, sums in
// the order k=0,1,2 and updates).  Both cells of an edge evaluate bit-identical fluxes, so mass is
// conserved to round-off without a flux buffer.  No blocking, fusion or reordering.
//
// Every rule of this file is pinned by tests/test_oracle_*.py against something the paper or the
// mathematics fixes (closed forms, invariants, exactness properties, the paper's printed tables;
// DESIGN.md section 2 lists what pins what), and the pins are checked by mutation
// (oracle/mutation_check.py: 74 single-rule mutants of this file, 73 killed).
// PARITY UNPINNED (only oracle<->GPU agreement and mass balance check these):
//   * edge_flux, inflow boundary: the momentum part of the flux on DRY faces (q^2/h dropped when
//     h* <= h_dry, reading R10); its mass part is pinned;
//   * ratio_r: r = 1 when |Delta_loc| is at round-off (reading R9; the three fluxes coincide there);
//   * cell_update: WHICH depth enters the Manning factor (the updated h', A.10); the depth before the
//     update is an equally consistent splitting and coincides with it at every steady state;
//   * the VALUES of h_dry and h_thin (parameters; that the two thresholds are distinct and which
//     rule uses which is pinned).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <limits>
#include <map>
#include <string>
#include <unordered_map>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum { SCH_HLLC = 0, SCH_MUSCL = 1, SCH_WAF = 2, SCH_MUSCL_MS = 3 };
enum { BC_WALL = 0, BC_INFLOW = 1, BC_LEVEL = 2, BC_TRANSMISSIVE = 3 };

struct Params {
    double g = 9.81, h_dry = 1e-6, h_thin = 1e-3, beta = 1.0;
};

struct BCInfo {
    int kind = BC_WALL;
    double value = 0.0;
    double width = 0.0;  // sum of the lengths of the tag's edges
};

struct Mesh {
    int64_t nv = 0, nt = 0, ne = 0, nbe = 0;
    std::vector<double> x, y, zb;
    std::vector<int32_t> tri;  // 3*nt, counter-clockwise
    // per cell
    std::vector<double> area, cx, cy, zc, rin;
    std::vector<int32_t> c2e, c2c;     // 3*nt; c2c = -1 on a boundary edge
    std::vector<double> rx, ry;        // 3*nt, r_{i,k} = m_e - c_i
    std::vector<double> nox, noy;      // 3*nt, unit normal of side k outward of cell i
    std::vector<double> wx, wy;        // 3*nt, least-squares weights
    std::vector<double> dupw;          // 3*nt, |x_i - x_upw| for side k (eq. 22-25): x_upw = mean of the
                                       // centroids of the two OTHER edge-neighbours (own centroid if missing)
    // per edge
    std::vector<int32_t> eL, eR, ekL, ekR, etag;  // eR=-1, etag=user tag (or -1 = untagged wall)
    std::vector<double> elen, enx, eny, edx;
    std::vector<double> edlr;          // |x_R - x_L| between the two centroids (0 on the boundary)
};

struct Ctx {
    Mesh m;
    Params p;
    std::map<int, BCInfo> bc;
    std::vector<double> nman;
    std::vector<double> h, hu, hv;
    double t = 0.0, last_dt = 0.0;
    int64_t steps = 0;
    // scratch
    std::vector<double> grad;               // 8*nt
    std::vector<double> a1, a2, a3, b1, b2, b3;
    std::string err;
};

int g_threads = 1;

// ---------------------------------------------------------------------------------------------
// A.1 geometry and topology (host, once)
// ---------------------------------------------------------------------------------------------
bool build_mesh(Mesh& m, int64_t nv, const double* x, const double* y, const double* zb, int64_t nt,
                const int32_t* tri, int64_t nb, const int32_t* bedge, const int32_t* btag,
                std::string& err) {
    m.nv = nv;
    m.nt = nt;
    m.x.assign(x, x + nv);
    m.y.assign(y, y + nv);
    m.zb.assign(zb, zb + nv);
    m.tri.assign(tri, tri + 3 * nt);
    for (int64_t i = 0; i < 3 * nt; ++i)
        if (m.tri[i] < 0 || m.tri[i] >= nv) { err = "triangle vertex id out of range"; return false; }
    m.area.resize(nt); m.cx.resize(nt); m.cy.resize(nt); m.zc.resize(nt); m.rin.resize(nt);
    // A.1.1 orientation and area; A.1.3 centroid and cell bed
    for (int64_t i = 0; i < nt; ++i) {
        int32_t* v = &m.tri[3 * i];
        double x0 = x[v[0]], y0 = y[v[0]];
        double a = 0.5 * ((x[v[1]] - x0) * (y[v[2]] - y0) - (x[v[2]] - x0) * (y[v[1]] - y0));
        if (a < 0.0) {
            std::swap(v[1], v[2]);
            a = 0.5 * ((x[v[1]] - x0) * (y[v[2]] - y0) - (x[v[2]] - x0) * (y[v[1]] - y0));
        }
        if (!(a > 0.0)) { err = "degenerate (zero-area) triangle"; return false; }
        m.area[i] = a;
        m.cx[i] = (x[v[0]] + x[v[1]] + x[v[2]]) / 3.0;
        m.cy[i] = (y[v[0]] + y[v[1]] + y[v[2]]) / 3.0;
        m.zc[i] = (zb[v[0]] + zb[v[1]] + zb[v[2]]) / 3.0;
    }
    // A.1.2 global edges = distinct vertex pairs (hash map keyed by the ordered pair)
    std::unordered_map<uint64_t, int32_t> emap;
    emap.reserve((size_t)(nt * 2));
    m.c2e.assign(3 * nt, -1);
    m.c2c.assign(3 * nt, -1);
    std::vector<int32_t> ecount;
    for (int64_t i = 0; i < nt; ++i) {
        for (int k = 0; k < 3; ++k) {
            int32_t a = m.tri[3 * i + k], b = m.tri[3 * i + (k + 1) % 3];
            uint64_t key = ((uint64_t)(uint32_t)std::min(a, b) << 32) | (uint32_t)std::max(a, b);
            auto it = emap.find(key);
            if (it == emap.end()) {
                int32_t e = (int32_t)m.eL.size();
                emap.emplace(key, e);
                // the cells are visited in increasing user id, so the first visitor is the L-cell
                // (A.1.4: L-cell = the adjacent cell with the smaller user id)
                m.eL.push_back((int32_t)i); m.ekL.push_back(k);
                m.eR.push_back(-1); m.ekR.push_back(-1);
                ecount.push_back(1);
                m.c2e[3 * i + k] = e;
            } else {
                int32_t e = it->second;
                if (ecount[e] >= 2) { err = "non-manifold edge (more than two triangles)"; return false; }
                ecount[e] = 2;
                m.eR[e] = (int32_t)i; m.ekR[e] = k;
                m.c2e[3 * i + k] = e;
            }
        }
    }
    m.ne = (int64_t)m.eL.size();
    m.etag.assign(m.ne, -1);
    m.elen.resize(m.ne); m.enx.resize(m.ne); m.eny.resize(m.ne); m.edx.resize(m.ne);
    m.rx.resize(3 * nt); m.ry.resize(3 * nt); m.nox.resize(3 * nt); m.noy.resize(3 * nt);
    m.wx.resize(3 * nt); m.wy.resize(3 * nt);
    m.nbe = 0;
    // A.1.4 edge geometry from the end points a->b as traversed by the L-cell; A.1.6 offsets
    for (int64_t e = 0; e < m.ne; ++e) {
        int32_t L = m.eL[e], kL = m.ekL[e], R = m.eR[e];
        int32_t a = m.tri[3 * L + kL], b = m.tri[3 * L + (kL + 1) % 3];
        double dx = x[b] - x[a], dy = y[b] - y[a];
        double len = std::sqrt(dx * dx + dy * dy);
        double n1 = dy / len, n2 = -dx / len;
        double mx = 0.5 * (x[a] + x[b]), my = 0.5 * (y[a] + y[b]);
        m.elen[e] = len; m.enx[e] = n1; m.eny[e] = n2;
        double rLx = mx - m.cx[L], rLy = my - m.cy[L];
        m.rx[3 * L + kL] = rLx; m.ry[3 * L + kL] = rLy;
        m.nox[3 * L + kL] = n1; m.noy[3 * L + kL] = n2;
        if (R >= 0) {
            int32_t kR = m.ekR[e];
            double rRx = mx - m.cx[R], rRy = my - m.cy[R];
            m.rx[3 * R + kR] = rRx; m.ry[3 * R + kR] = rRy;
            m.nox[3 * R + kR] = -n1; m.noy[3 * R + kR] = -n2;
            m.c2c[3 * L + kL] = R;
            m.c2c[3 * R + kR] = L;
            m.edx[e] = (rLx * n1 + rLy * n2) - (rRx * n1 + rRy * n2);
        } else {
            m.nbe++;
            m.edx[e] = 2.0 * (rLx * n1 + rLy * n2);
        }
    }
    // boundary tags
    for (int64_t j = 0; j < nb; ++j) {
        int32_t a = bedge[2 * j], b = bedge[2 * j + 1];
        if (a < 0 || b < 0 || a >= nv || b >= nv) { err = "boundary edge vertex id out of range"; return false; }
        uint64_t key = ((uint64_t)(uint32_t)std::min(a, b) << 32) | (uint32_t)std::max(a, b);
        auto it = emap.find(key);
        if (it == emap.end() || m.eR[it->second] >= 0) { err = "tagged edge is not a boundary edge"; return false; }
        if (btag[j] < 0) { err = "negative boundary tag"; return false; }
        m.etag[it->second] = btag[j];
    }
    // A.1.5 in-radius; A.1.7 least-squares weights
    for (int64_t i = 0; i < nt; ++i) {
        double l0 = m.elen[m.c2e[3 * i]], l1 = m.elen[m.c2e[3 * i + 1]], l2 = m.elen[m.c2e[3 * i + 2]];
        m.rin[i] = 2.0 * m.area[i] / (l0 + l1 + l2);
        double dxk[3], dyk[3];
        double a11 = 0.0, a12 = 0.0, a22 = 0.0;
        for (int k = 0; k < 3; ++k) {
            int32_t nb_ = m.c2c[3 * i + k];
            if (nb_ >= 0) {
                dxk[k] = m.cx[nb_] - m.cx[i];
                dyk[k] = m.cy[nb_] - m.cy[i];
            } else {  // mirror point across the boundary edge
                double rn = m.rx[3 * i + k] * m.nox[3 * i + k] + m.ry[3 * i + k] * m.noy[3 * i + k];
                dxk[k] = 2.0 * rn * m.nox[3 * i + k];
                dyk[k] = 2.0 * rn * m.noy[3 * i + k];
            }
            a11 += dxk[k] * dxk[k];
            a12 += dxk[k] * dyk[k];
            a22 += dyk[k] * dyk[k];
        }
        double det = a11 * a22 - a12 * a12;
        for (int k = 0; k < 3; ++k) {
            m.wx[3 * i + k] = (a22 * dxk[k] - a12 * dyk[k]) / det;
            m.wy[3 * i + k] = (-a12 * dxk[k] + a11 * dyk[k]) / det;
        }
    }
    // distances of the multislope MUSCL (eq. 22-25, reading R17)
    m.dupw.resize(3 * nt);
    m.edlr.assign(m.ne, 0.0);
    for (int64_t i = 0; i < nt; ++i)
        for (int k = 0; k < 3; ++k) {
            double sx = 0.0, sy = 0.0;
            for (int j = 0; j < 3; ++j) {
                if (j == k) continue;
                int32_t nb_ = m.c2c[3 * i + j];
                if (nb_ >= 0) { sx += m.cx[nb_]; sy += m.cy[nb_]; }
                else { sx += m.cx[i]; sy += m.cy[i]; }
            }
            double ux = m.cx[i] - 0.5 * sx, uy = m.cy[i] - 0.5 * sy;
            m.dupw[3 * i + k] = std::sqrt(ux * ux + uy * uy);
        }
    for (int64_t e = 0; e < m.ne; ++e)
        if (m.eR[e] >= 0) {
            double ux = m.cx[m.eR[e]] - m.cx[m.eL[e]], uy = m.cy[m.eR[e]] - m.cy[m.eL[e]];
            m.edlr[e] = std::sqrt(ux * ux + uy * uy);
        }
    return true;
}

// ---------------------------------------------------------------------------------------------
// eq. 21 SUPERBEE limiter function A(r,c), branch boundaries exactly as printed
// ---------------------------------------------------------------------------------------------
double limiter_A(double r, double c) {
    double ac = std::fabs(c);
    if (r <= 0.0) return 1.0;
    if (r <= 0.5) return 1.0 - 2.0 * (1.0 - ac) * r;
    if (r <= 1.0) return ac;
    if (r <= 2.0) return 1.0 - (1.0 - ac) * r;
    return 2.0 * ac - 1.0;
}

// ---------------------------------------------------------------------------------------------
// A.6 wave speeds (eq. 8-12, readings R1, R13) and HLLC flux (eq. 6, 7, 13, 14, reading R2)
// ---------------------------------------------------------------------------------------------
struct Waves {
    double SL, SR, Sstar, hstar, h0;
    double GL1, GL2, GR1, GR2;   // physical fluxes of the two states (first two components)
    double hL, uL, vL, hR, uR, vR;  // states actually used (a non-wet side contributes zeros)
    bool wetL, wetR;
};

void wave_speeds(double g, double h_dry, double hL, double uL, double vL, double hR, double uR,
                 double vR, Waves& w) {
    w.wetL = hL > h_dry;
    w.wetR = hR > h_dry;
    if (!w.wetL) { hL = 0.0; uL = 0.0; vL = 0.0; }
    if (!w.wetR) { hR = 0.0; uR = 0.0; vR = 0.0; }
    w.hL = hL; w.uL = uL; w.vL = vL; w.hR = hR; w.uR = uR; w.vR = vR;
    w.SL = w.SR = w.Sstar = w.hstar = w.h0 = 0.0;
    w.GL1 = hL * uL; w.GL2 = hL * uL * uL + 0.5 * g * hL * hL;
    w.GR1 = hR * uR; w.GR2 = hR * uR * uR + 0.5 * g * hR * hR;
    if (!w.wetL && !w.wetR) return;
    if (w.wetL && w.wetR) {
        double aL = std::sqrt(g * hL), aR = std::sqrt(g * hR);
        double h0 = (hL + hR) / 2.0 - (uR - uL) * (hL + hR) / (4.0 * (aL + aR));  // eq. 10
        double hs;
        if (h0 <= std::min(hL, hR)) {  // rarefaction, eq. 11 (bracket clamped at 0: vacuum)
            double s = std::max(0.0, (aL + aR) / 2.0 + (uL - uR) / 4.0);
            hs = s * s / g;
        } else {  // shock, eq. 12
            double gL = std::sqrt(g * (h0 + hL) / (2.0 * h0 * hL));
            double gR = std::sqrt(g * (h0 + hR) / (2.0 * h0 * hR));
            hs = (hL * gL + hR * gR + uL - uR) / (gL + gR);
        }
        double pL = (hs > hL) ? std::sqrt(0.5 * hs * (hs + hL)) / hL : 1.0;  // eq. 9, reading R1
        double pR = (hs > hR) ? std::sqrt(0.5 * hs * (hs + hR)) / hR : 1.0;
        w.SL = uL - aL * pL;  // eq. 8
        w.SR = uR + aR * pR;
        w.hstar = hs; w.h0 = h0;
    } else if (w.wetL) {  // right side dry (reading R13)
        double aL = std::sqrt(g * hL);
        w.SL = uL - aL;
        w.SR = uL + 2.0 * aL;
    } else {  // left side dry
        double aR = std::sqrt(g * hR);
        w.SL = uR - 2.0 * aR;
        w.SR = uR + aR;
    }
    double qR = hR * (uR - w.SR), qL = hL * (uL - w.SL);  // eq. 14
    double den = qR - qL;
    w.Sstar = (den == 0.0) ? 0.0 : (w.SL * qR - w.SR * qL) / den;
}

// star flux eq. 7 in the cancellation-free form G* = G_L + S_L [S_R (U_R-U_L) - (G_R-G_L)]/(S_R-S_L)
inline void star_flux(const Waves& w, double& Gs1, double& Gs2) {
    double d = w.SR - w.SL;
    Gs1 = w.GL1 + w.SL * (w.SR * (w.hR - w.hL) - (w.GR1 - w.GL1)) / d;
    Gs2 = w.GL2 + w.SL * (w.SR * (w.hR * w.uR - w.hL * w.uL) - (w.GR2 - w.GL2)) / d;
}

void hllc_flux(double g, double h_dry, double hL, double uL, double vL, double hR, double uR,
               double vR, double G[3], Waves* wout = nullptr) {
    Waves w;
    wave_speeds(g, h_dry, hL, uL, vL, hR, uR, vR, w);
    if (wout) *wout = w;
    if (!w.wetL && !w.wetR) { G[0] = G[1] = G[2] = 0.0; return; }
    if (w.SL >= 0.0) { G[0] = w.GL1; G[1] = w.GL2; }          // eq. 6
    else if (w.SR <= 0.0) { G[0] = w.GR1; G[1] = w.GR2; }
    else star_flux(w, G[0], G[1]);
    G[2] = G[0] * ((w.Sstar >= 0.0) ? w.vL : w.vR);           // eq. 13, reading R2
}

// ---------------------------------------------------------------------------------------------
// A.7 WAF flux (eq. 15-21; readings R3, R6-R9).  Both states wet.  q = eta for the outer waves,
// q = tangential velocity for the middle wave.
// ---------------------------------------------------------------------------------------------
inline double sgn(double c) { return (c > 0.0) ? 1.0 : ((c < 0.0) ? -1.0 : 0.0); }
inline double clamp1(double c) { return std::max(-1.0, std::min(1.0, c)); }

inline double ratio_r(double S, double qL, double qR, double qLupw, double qRupw) {
    double dloc = qR - qL;                                         // eq. 19
    double dupw = (S > 0.0) ? (qL - qLupw) : (qRupw - qR);         // eq. 20 (S=0 -> lower form)
    if (std::fabs(dloc) <= 1e-14 * std::max(1.0, std::fabs(qL))) return 1.0;
    return dupw / dloc;
}

void waf_flux(double g, double h_dry, double hL, double uL, double vL, double hR, double uR,
              double vR, double etaL, double etaR, double etaLupw, double etaRupw, double vLupw,
              double vRupw, double dt, double dx, int use_limiter, double G[3]) {
    Waves w;
    wave_speeds(g, h_dry, hL, uL, vL, hR, uR, vR, w);
    double Gs1, Gs2;
    star_flux(w, Gs1, Gs2);                                        // reading R3: always eq. 7
    double cL = clamp1(w.SL * dt / dx), cR = clamp1(w.SR * dt / dx), cS = clamp1(w.Sstar * dt / dx);
    double AL = 1.0, AR = 1.0, AS = 1.0;
    if (use_limiter) {
        double rL = ratio_r(w.SL, etaL, etaR, etaLupw, etaRupw);
        double rR = ratio_r(w.SR, etaL, etaR, etaLupw, etaRupw);
        double rS = ratio_r(w.Sstar, vL, vR, vLupw, vRupw);
        AL = limiter_A(rL, std::fabs(cL));
        AR = limiter_A(rR, std::fabs(cR));
        AS = limiter_A(rS, std::fabs(cS));
    }
    double sL = sgn(cL) * AL, sR = sgn(cR) * AR, sS = sgn(cS) * AS;  // eq. 18, reading R6
    // eq. 15 rewritten about the star flux so that equal states return the flux exactly
    G[0] = Gs1 + 0.5 * (1.0 + sL) * (w.GL1 - Gs1) + 0.5 * (1.0 - sR) * (w.GR1 - Gs1);
    G[1] = Gs2 + 0.5 * (1.0 + sL) * (w.GL2 - Gs2) + 0.5 * (1.0 - sR) * (w.GR2 - Gs2);
    G[2] = G[0] * (0.5 * (1.0 + sS) * vL + 0.5 * (1.0 - sS) * vR);   // eq. 16
}

// ---------------------------------------------------------------------------------------------
// A.2 time step (eq. 5, reading R5)
// ---------------------------------------------------------------------------------------------
double compute_dt(const Ctx& c, const double* h, const double* hu, const double* hv, double cfl) {
    const Mesh& m = c.m;
    double best = std::numeric_limits<double>::infinity();
#pragma omp parallel for reduction(min : best) num_threads(g_threads) schedule(static)
    for (int64_t i = 0; i < m.nt; ++i) {
        if (!(h[i] > c.p.h_dry)) continue;
        double u = hu[i] / h[i], v = hv[i] / h[i];
        double lam = std::sqrt(c.p.g * h[i]) + std::sqrt(u * u + v * v);
        double r = m.rin[i] / lam;
        if (r < best) best = r;
    }
    if (best == std::numeric_limits<double>::infinity()) return 0.0;
    return cfl * best;
}

// ---------------------------------------------------------------------------------------------
// A.1/A.3 primitives and limited least-squares gradients of (eta, h, u, v)
// ---------------------------------------------------------------------------------------------
struct Prim { double h, eta, u, v; bool wet; };

inline Prim prim_of(const Ctx& c, const double* h, const double* hu, const double* hv, int64_t i) {
    Prim p;
    p.h = h[i];
    p.eta = h[i] + c.m.zc[i];
    p.wet = h[i] > c.p.h_dry;
    if (p.wet) { p.u = hu[i] / h[i]; p.v = hv[i] / h[i]; }
    else { p.u = 0.0; p.v = 0.0; }
    return p;
}

void cell_gradient(const Ctx& c, const double* h, const double* hu, const double* hv, int64_t i,
                   double* out /*8: eta_x eta_y h_x h_y u_x u_y v_x v_y*/) {
    const Mesh& m = c.m;
    Prim pi = prim_of(c, h, hu, hv, i);
    double qi[4] = {pi.eta, pi.h, pi.u, pi.v};
    double qk[3][4];
    bool real[3];
    bool all_wet = pi.wet;
    for (int k = 0; k < 3; ++k) {
        int32_t nb = m.c2c[3 * i + k];
        real[k] = nb >= 0;
        if (nb >= 0) {
            Prim pk = prim_of(c, h, hu, hv, nb);
            qk[k][0] = pk.eta; qk[k][1] = pk.h; qk[k][2] = pk.u; qk[k][3] = pk.v;
            if (!pk.wet) all_wet = false;
        } else {
            qk[k][0] = pi.eta; qk[k][1] = pi.h; qk[k][2] = pi.u; qk[k][3] = pi.v;
            int32_t e = m.c2e[3 * i + k];
            int tag = m.etag[e];
            int kind = BC_WALL;
            if (tag >= 0) { auto it = c.bc.find(tag); if (it != c.bc.end()) kind = it->second.kind; }
            if (kind == BC_WALL) {  // mirror the velocity in the wall
                double n1 = m.nox[3 * i + k], n2 = m.noy[3 * i + k];
                double un = pi.u * n1 + pi.v * n2;
                qk[k][2] = pi.u - 2.0 * un * n1;
                qk[k][3] = pi.v - 2.0 * un * n2;
            }
        }
    }
    double kappa = c.p.beta / 2.0;
    for (int q = 0; q < 4; ++q) {
        double gx = 0.0, gy = 0.0;
        for (int k = 0; k < 3; ++k) {
            double dq = qk[k][q] - qi[q];
            gx += m.wx[3 * i + k] * dq;
            gy += m.wy[3 * i + k] * dq;
        }
        double phi = 1.0;
        if (!all_wet) phi = 0.0;
        else if (c.p.beta > 0.0) {
            double qmax = qi[q], qmin = qi[q];
            for (int k = 0; k < 3; ++k)
                if (real[k]) { qmax = std::max(qmax, qk[k][q]); qmin = std::min(qmin, qk[k][q]); }
            for (int k = 0; k < 3; ++k) {
                double d = gx * m.rx[3 * i + k] + gy * m.ry[3 * i + k];
                double pk = 1.0;
                if (d > 0.0) pk = std::min(1.0, kappa * (qmax - qi[q]) / d);
                else if (d < 0.0) pk = std::min(1.0, kappa * (qmin - qi[q]) / d);
                phi = std::min(phi, pk);
            }
        }
        out[2 * q] = phi * gx;
        out[2 * q + 1] = phi * gy;
    }
}

// ---------------------------------------------------------------------------------------------
// A.4-A.9 flux of one edge: face states, hydrostatic reconstruction, rotation, Riemann flux,
// bed-slope terms, rotation back, times the edge length.  PhiL / PhiR are the two sides' vectors.
// ---------------------------------------------------------------------------------------------
struct Face { double h, eta, u, v, z; };

inline Face face_state(const Ctx& c, const Prim& p, const double* grad, int64_t i, int k, int scheme) {
    Face f;
    if (scheme == SCH_MUSCL) {
        const double* gq = grad + 8 * i;
        double rx = c.m.rx[3 * i + k], ry = c.m.ry[3 * i + k];
        f.eta = p.eta + (gq[0] * rx + gq[1] * ry);
        f.h = p.h + (gq[2] * rx + gq[3] * ry);
        f.u = p.u + (gq[4] * rx + gq[5] * ry);
        f.v = p.v + (gq[6] * rx + gq[7] * ry);
    } else {
        f.eta = p.eta; f.h = p.h; f.u = p.u; f.v = p.v;
    }
    f.z = f.eta - f.h;
    return f;
}

bool waf_applicable(const Ctx& c, const double* h, int32_t L, int32_t R, double hsL, double hsR) {
    const Mesh& m = c.m;
    double ht = c.p.h_thin;
    if (!(h[L] > ht) || !(h[R] > ht)) return false;
    for (int k = 0; k < 3; ++k) {
        int32_t a = m.c2c[3 * L + k], b = m.c2c[3 * R + k];
        if (a >= 0 && !(h[a] > ht)) return false;
        if (b >= 0 && !(h[b] > ht)) return false;
    }
    return hsL > c.p.h_dry && hsR > c.p.h_dry;
}

// upwind average over the two other edge-neighbours of cell i; a missing one is
// replaced by the cell's own value
void upwind_mean(const Ctx& c, const double* h, const double* hu, const double* hv, int32_t i,
                 int kskip, const Prim& pi, double& eta, double& u, double& v, double* hmean = nullptr,
                 bool* all_wet = nullptr) {
    double se = 0.0, su = 0.0, sv = 0.0, sh = 0.0;
    for (int k = 0; k < 3; ++k) {
        if (k == kskip) continue;
        int32_t nb = c.m.c2c[3 * i + k];
        if (nb >= 0) {
            Prim pk = prim_of(c, h, hu, hv, nb);
            se += pk.eta; su += pk.u; sv += pk.v; sh += pk.h;
            if (all_wet && !pk.wet) *all_wet = false;
        } else {
            se += pi.eta; su += pi.u; sv += pi.v; sh += pi.h;
        }
    }
    eta = 0.5 * se; u = 0.5 * su; v = 0.5 * sv;
    if (hmean) *hmean = 0.5 * sh;
}

// eq. 24-25: limited slope from the slope x on one side and the slope y on the other; the case
// distinction of the paper is on the sign of y (the printed conditions U_R - U_L > 0 in eq. 24,
// U_Rupw - U_R > 0 in eq. 25).  beta = 1 MINBEE, beta = 2 SUPERBEE.
double ms_slope(double beta, double x, double y) {
    if (y > 0.0) return std::max(0.0, std::max(std::min(beta * x, y), std::min(x, beta * y)));
    if (y < 0.0) return std::min(0.0, std::min(std::max(beta * x, y), std::max(x, beta * y)));
    return 0.0;
}

// eq. 22: face values of the two sides of interior edge e by the multislope reconstruction of
// q = (eta, h, u, v); first order if a cell of the stencil is not wet (same rule as A.3.5)
void ms_face_states(const Ctx& c, const double* h, const double* hu, const double* hv, int32_t e,
                    const Prim& pL, const Prim& pR, Face& fL, Face& fR) {
    const Mesh& m = c.m;
    int32_t L = m.eL[e], R = m.eR[e], kL = m.ekL[e], kR = m.ekR[e];
    fL.eta = pL.eta; fL.h = pL.h; fL.u = pL.u; fL.v = pL.v;
    fR.eta = pR.eta; fR.h = pR.h; fR.u = pR.u; fR.v = pR.v;
    bool all_wet = pL.wet && pR.wet;
    double qLu[4], qRu[4];
    upwind_mean(c, h, hu, hv, L, kL, pL, qLu[0], qLu[2], qLu[3], &qLu[1], &all_wet);
    upwind_mean(c, h, hu, hv, R, kR, pR, qRu[0], qRu[2], qRu[3], &qRu[1], &all_wet);
    if (all_wet) {
        double beta = c.p.beta > 0.0 ? c.p.beta : 1.0;
        double dL = m.dupw[3 * L + kL], dR = m.dupw[3 * R + kR], dLR = m.edlr[e];
        double rL = std::sqrt(m.rx[3 * L + kL] * m.rx[3 * L + kL] + m.ry[3 * L + kL] * m.ry[3 * L + kL]);
        double rR = std::sqrt(m.rx[3 * R + kR] * m.rx[3 * R + kR] + m.ry[3 * R + kR] * m.ry[3 * R + kR]);
        double qL[4] = {pL.eta, pL.h, pL.u, pL.v}, qR[4] = {pR.eta, pR.h, pR.u, pR.v};
        double oL[4], oR[4];
        for (int q = 0; q < 4; ++q) {
            double a = (dL > 0.0) ? (qL[q] - qLu[q]) / dL : 0.0;      // upwind slope of L
            double b = (qR[q] - qL[q]) / dLR;                          // local slope
            double d = (dR > 0.0) ? (qRu[q] - qR[q]) / dR : 0.0;      // upwind slope of R
            oL[q] = qL[q] + rL * ms_slope(beta, a, b);                 // eq. 22 with eq. 24
            oR[q] = qR[q] - rR * ms_slope(beta, b, d);                 // eq. 22 with eq. 25
        }
        fL.eta = oL[0]; fL.h = oL[1]; fL.u = oL[2]; fL.v = oL[3];
        fR.eta = oR[0]; fR.h = oR[1]; fR.u = oR[2]; fR.v = oR[3];
    }
    fL.z = fL.eta - fL.h;
    fR.z = fR.eta - fR.h;
}

void edge_flux(const Ctx& c, const double* h, const double* hu, const double* hv, const double* grad,
               int32_t e, double dt, int scheme, double PhiL[3], double PhiR[3]) {
    const Mesh& m = c.m;
    const double g = c.p.g, h_dry = c.p.h_dry;
    int32_t L = m.eL[e], R = m.eR[e], kL = m.ekL[e];
    double n1 = m.enx[e], n2 = m.eny[e], len = m.elen[e];
    Prim pL = prim_of(c, h, hu, hv, L);
    Face fL = face_state(c, pL, grad, L, kL, scheme);
    double unL = fL.u * n1 + fL.v * n2, utL = -fL.u * n2 + fL.v * n1;   // eq. 2
    double G[3];
    if (R >= 0) {
        int32_t kR = m.ekR[e];
        Prim pR = prim_of(c, h, hu, hv, R);
        Face fR = face_state(c, pR, grad, R, kR, scheme);
        if (scheme == SCH_MUSCL_MS) {
            ms_face_states(c, h, hu, hv, e, pL, pR, fL, fR);
            unL = fL.u * n1 + fL.v * n2; utL = -fL.u * n2 + fL.v * n1;
        }
        double unR = fR.u * n1 + fR.v * n2, utR = -fR.u * n2 + fR.v * n1;
        double zs = std::max(fL.z, fR.z);                               // A.5
        double hsL = std::max(0.0, fL.eta - zs), hsR = std::max(0.0, fR.eta - zs);
        if (scheme == SCH_WAF && waf_applicable(c, h, L, R, hsL, hsR)) {
            double eLu, uLu, vLu, eRu, uRu, vRu;
            upwind_mean(c, h, hu, hv, L, kL, pL, eLu, uLu, vLu);
            upwind_mean(c, h, hu, hv, R, kR, pR, eRu, uRu, vRu);
            double utLu = -uLu * n2 + vLu * n1, utRu = -uRu * n2 + vRu * n1;
            waf_flux(g, h_dry, hsL, unL, utL, hsR, unR, utR, pL.eta, pR.eta, eLu, eRu, utLu, utRu,
                     dt, m.edx[e], 1, G);
        } else {
            hllc_flux(g, h_dry, hsL, unL, utL, hsR, unR, utR, G);
        }
        double PL = -0.5 * g * hsL * hsL + 0.5 * g * (fL.h + pL.h) * (fL.eta - pL.eta);  // A.9
        double PR = -0.5 * g * hsR * hsR + 0.5 * g * (fR.h + pR.h) * (fR.eta - pR.eta);
        double bL = G[1] + PL, bR = G[1] + PR;
        PhiL[0] = len * G[0];
        PhiL[1] = len * (bL * n1 - G[2] * n2);
        PhiL[2] = len * (bL * n2 + G[2] * n1);
        PhiR[0] = len * G[0];
        PhiR[1] = len * (bR * n1 - G[2] * n2);
        PhiR[2] = len * (bR * n2 + G[2] * n1);
        return;
    }
    // A.8 boundary edge: ghost bed = face bed, so h* = h_f (clamped at 0)
    double hs = std::max(0.0, fL.h);
    int kind = BC_WALL;
    double value = 0.0, width = 1.0;
    int tag = m.etag[e];
    if (tag >= 0) {
        auto it = c.bc.find(tag);
        if (it != c.bc.end()) { kind = it->second.kind; value = it->second.value; width = it->second.width; }
    }
    if (kind == BC_WALL) {                       // PAPER.md:286 with Q=0
        G[0] = 0.0; G[1] = 0.5 * g * hs * hs; G[2] = 0.0;
    } else if (kind == BC_INFLOW) {              // PAPER.md:286, outward-normal sign (reading R10)
        double qn = -value / width;
        G[0] = qn;
        G[1] = (hs > h_dry) ? (qn * qn / hs + 0.5 * g * hs * hs) : (0.5 * g * hs * hs);
        G[2] = 0.0;
    } else if (kind == BC_TRANSMISSIVE) {        // U_R = U_L
        if (hs > h_dry) {
            G[0] = hs * unL; G[1] = hs * unL * unL + 0.5 * g * hs * hs; G[2] = G[0] * utL;
        } else { G[0] = G[1] = G[2] = 0.0; }
    } else {                                     // fixed level (reading R11)
        double hb = std::max(0.0, value - fL.z);
        if (!(hs > h_dry) && !(hb > h_dry)) { G[0] = G[1] = G[2] = 0.0; }
        else {
            double ub = unL + 2.0 * (std::sqrt(g * hs) - std::sqrt(g * hb));
            hllc_flux(g, h_dry, hs, unL, utL, hb, ub, utL, G);
        }
    }
    double PL = -0.5 * g * hs * hs + 0.5 * g * (fL.h + pL.h) * (fL.eta - pL.eta);
    double bL = G[1] + PL;
    PhiL[0] = len * G[0];
    PhiL[1] = len * (bL * n1 - G[2] * n2);
    PhiL[2] = len * (bL * n2 + G[2] * n1);
    PhiR[0] = PhiR[1] = PhiR[2] = 0.0;
}

// ---------------------------------------------------------------------------------------------
// A.10 Euler stage of one cell from the state arrays (h,hu,hv) and gradient array
// ---------------------------------------------------------------------------------------------
inline void manning_step(double g, double n, double dt, double h, double& hu, double& hv) {
    double D = 1.0 + dt * g * n * n * std::sqrt(hu * hu + hv * hv) / h / (std::cbrt(h) * h);
    hu = hu / D;
    hv = hv / D;
}

void cell_update(const Ctx& c, const double* h, const double* hu, const double* hv,
                 const double* grad, int64_t i, double dt, int scheme, double& h1, double& hu1,
                 double& hv1) {
    const Mesh& m = c.m;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int k = 0; k < 3; ++k) {
        int32_t e = m.c2e[3 * i + k];
        double PL[3], PR[3];
        edge_flux(c, h, hu, hv, grad, e, dt, scheme, PL, PR);
        if (m.eL[e] == i) { s0 += PL[0]; s1 += PL[1]; s2 += PL[2]; }
        else { s0 -= PR[0]; s1 -= PR[1]; s2 -= PR[2]; }
    }
    double f = dt / m.area[i];
    double a = h[i] - f * s0, b = hu[i] - f * s1, d = hv[i] - f * s2;     // eq. 3
    a = std::max(a, 0.0);
    if (a > c.p.h_dry) {
        double n = c.nman.empty() ? 0.0 : c.nman[i];
        if (n > 0.0) manning_step(c.p.g, n, dt, a, b, d);
    } else { b = 0.0; d = 0.0; }
    h1 = a; hu1 = b; hv1 = d;
}

void compute_gradients(const Ctx& c, const double* h, const double* hu, const double* hv, double* grad) {
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int64_t i = 0; i < c.m.nt; ++i) cell_gradient(c, h, hu, hv, i, grad + 8 * i);
}

void euler_stage(Ctx& c, const double* h, const double* hu, const double* hv, double dt, int scheme,
                 double* h1, double* hu1, double* hv1) {
    const double* grad = nullptr;
    if (scheme == SCH_MUSCL) {
        c.grad.resize(8 * c.m.nt);
        compute_gradients(c, h, hu, hv, c.grad.data());   // pass G
        grad = c.grad.data();
    }
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int64_t i = 0; i < c.m.nt; ++i)                   // pass C
        cell_update(c, h, hu, hv, grad, i, dt, scheme, h1[i], hu1[i], hv1[i]);
}

// A.11 one full time step
double one_step(Ctx& c, double cfl, int scheme) {
    int64_t nt = c.m.nt;
    double dt = compute_dt(c, c.h.data(), c.hu.data(), c.hv.data(), cfl);
    c.a1.resize(nt); c.a2.resize(nt); c.a3.resize(nt);
    if (dt > 0.0) {
        if (scheme == SCH_MUSCL || scheme == SCH_MUSCL_MS) {
            c.b1.resize(nt); c.b2.resize(nt); c.b3.resize(nt);
            euler_stage(c, c.h.data(), c.hu.data(), c.hv.data(), dt, scheme, c.a1.data(), c.a2.data(), c.a3.data());
            euler_stage(c, c.a1.data(), c.a2.data(), c.a3.data(), dt, scheme, c.b1.data(), c.b2.data(), c.b3.data());
            for (int64_t i = 0; i < nt; ++i) {
                double hn = 0.5 * (c.h[i] + c.b1[i]);
                double hun = 0.5 * (c.hu[i] + c.b2[i]);
                double hvn = 0.5 * (c.hv[i] + c.b3[i]);
                if (!(hn > c.p.h_dry)) { hun = 0.0; hvn = 0.0; }
                c.h[i] = hn; c.hu[i] = hun; c.hv[i] = hvn;
            }
        } else {
            euler_stage(c, c.h.data(), c.hu.data(), c.hv.data(), dt, scheme, c.a1.data(), c.a2.data(), c.a3.data());
            c.h.swap(c.a1); c.hu.swap(c.a2); c.hv.swap(c.a3);
        }
    }
    c.t += dt;
    c.last_dt = dt;
    c.steps++;
    return dt;
}


// ---------------------------------------------------------------------------------------------
// A.12 zones, ghost layers, send lists / contiguous receive ranges, pack / unpack
// (PAPER.md:121-127 ghost layers and renumbering; 141 PointRange / PointList; 460 send buffer and
// in-place reception).  Every zone keeps its own state arrays (owned cells first, then one
// contiguous block of ghost cells per source zone).  A zone is evaluated with the SAME per-cell
// functions as the un-zoned run: its state is scattered into mesh-sized scratch arrays that hold
// NaN everywhere else, so any access outside the zone's owned+ghost cells poisons the result.
// ---------------------------------------------------------------------------------------------
struct Link {
    int src = -1;
    int32_t start = 0, count = 0;
    std::vector<int32_t> send;   // indices local to the SOURCE zone, same order as the block
};
struct Zone {
    int64_t nowned = 0;
    std::vector<int32_t> cells;  // global cell ids: owned (ascending), then ghost blocks
    std::vector<int32_t> layer;  // 0 = owned, l>=1 = ghost layer
    std::vector<Link> links;     // one per source zone, ascending source id
    std::vector<double> h, hu, hv, h0, hu0, hv0, grad;
    std::unordered_map<int32_t, int32_t> g2l;
};
struct Zones {
    int nz = 0, nlayers = 0;
    std::vector<int32_t> zone_of;
    std::vector<Zone> z;
    std::vector<double> sh, shu, shv, sgrad;   // mesh-sized scratch, NaN outside the active zone
    std::vector<std::vector<double>> sendbuf;  // one buffer per (zone, link), flattened
};

std::map<Ctx*, Zones> g_zones;

// recursive coordinate bisection (A.12.1)
void rcb(const Mesh& m, std::vector<int32_t>& ids, int z0, int nz, std::vector<int32_t>& zone_of) {
    if (nz == 1) { for (int32_t i : ids) zone_of[i] = z0; return; }
    double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300;
    for (int32_t i : ids) {
        xmin = std::min(xmin, m.cx[i]); xmax = std::max(xmax, m.cx[i]);
        ymin = std::min(ymin, m.cy[i]); ymax = std::max(ymax, m.cy[i]);
    }
    bool alongx = (xmax - xmin) >= (ymax - ymin);
    const std::vector<double>& key = alongx ? m.cx : m.cy;
    std::sort(ids.begin(), ids.end(), [&](int32_t a, int32_t b) {
        if (key[a] != key[b]) return key[a] < key[b];
        return a < b;
    });
    size_t nl = ids.size() / 2;
    std::vector<int32_t> left(ids.begin(), ids.begin() + nl), right(ids.begin() + nl, ids.end());
    rcb(m, left, z0, nz / 2, zone_of);
    rcb(m, right, z0 + nz / 2, nz / 2, zone_of);
}

int zones_build(Ctx& c, Zones& Z, int nz, int nlayers, const int32_t* zone_of_cell) {
    const Mesh& m = c.m;
    if (nz < 1 || nlayers < 1 || nlayers > 3) return -1;
    Z.nz = nz; Z.nlayers = nlayers;
    Z.zone_of.assign(m.nt, -1);
    if (zone_of_cell) {
        for (int64_t i = 0; i < m.nt; ++i) {
            if (zone_of_cell[i] < 0 || zone_of_cell[i] >= nz) return -1;
            Z.zone_of[i] = zone_of_cell[i];
        }
    } else {
        if (nz & (nz - 1)) return -1;   // RCB needs a power of two
        std::vector<int32_t> ids(m.nt);
        for (int64_t i = 0; i < m.nt; ++i) ids[i] = (int32_t)i;
        rcb(m, ids, 0, nz, Z.zone_of);
    }
    Z.z.assign(nz, Zone());
    for (int64_t i = 0; i < m.nt; ++i) Z.z[Z.zone_of[i]].cells.push_back((int32_t)i);
    std::vector<int32_t> mark(m.nt, -1);   // mark[i]==zone id  <=>  i already in that zone's set
    for (int zi = 0; zi < nz; ++zi) {
        Zone& zn = Z.z[zi];
        zn.nowned = (int64_t)zn.cells.size();
        zn.layer.assign(zn.cells.size(), 0);
        for (int32_t i : zn.cells) mark[i] = zi;
        // A.12.2 breadth-first ghost layers over edge adjacency
        std::vector<int32_t> frontier = zn.cells;
        std::vector<std::pair<int32_t, int32_t>> ghosts;   // (cell, layer)
        for (int l = 1; l <= nlayers; ++l) {
            std::vector<int32_t> next;
            for (int32_t i : frontier)
                for (int k = 0; k < 3; ++k) {
                    int32_t nb = m.c2c[3 * i + k];
                    if (nb >= 0 && mark[nb] != zi) { mark[nb] = zi; next.push_back(nb); ghosts.emplace_back(nb, l); }
                }
            frontier.swap(next);
        }
        // A.12.3 one contiguous block per source zone (ascending), ordered by layer then id
        std::sort(ghosts.begin(), ghosts.end(), [&](const std::pair<int32_t, int32_t>& a, const std::pair<int32_t, int32_t>& b) {
            int za = Z.zone_of[a.first], zb = Z.zone_of[b.first];
            if (za != zb) return za < zb;
            if (a.second != b.second) return a.second < b.second;
            return a.first < b.first;
        });
        for (size_t j = 0; j < ghosts.size(); ++j) {
            int src = Z.zone_of[ghosts[j].first];
            if (zn.links.empty() || zn.links.back().src != src) {
                Link lk; lk.src = src; lk.start = (int32_t)zn.cells.size(); lk.count = 0;
                zn.links.push_back(lk);
            }
            zn.links.back().count++;
            zn.cells.push_back(ghosts[j].first);
            zn.layer.push_back(ghosts[j].second);
        }
        for (size_t j = 0; j < zn.cells.size(); ++j) zn.g2l[zn.cells[j]] = (int32_t)j;
    }
    // send lists: local indices in the source zone (owned cells of the source)
    for (int zi = 0; zi < nz; ++zi)
        for (Link& lk : Z.z[zi].links) {
            lk.send.resize(lk.count);
            const Zone& s = Z.z[lk.src];
            for (int32_t j = 0; j < lk.count; ++j) {
                int32_t gl = Z.z[zi].cells[lk.start + j];
                int32_t loc = s.g2l.at(gl);
                if (loc >= s.nowned) return -2;
                lk.send[j] = loc;
            }
        }
    double nan = std::numeric_limits<double>::quiet_NaN();
    Z.sh.assign(m.nt, nan); Z.shu.assign(m.nt, nan); Z.shv.assign(m.nt, nan);
    Z.sgrad.assign(8 * m.nt, nan);
    for (Zone& zn : Z.z) {
        size_t n = zn.cells.size();
        zn.h.assign(n, nan); zn.hu.assign(n, nan); zn.hv.assign(n, nan);
        zn.h0.assign(n, nan); zn.hu0.assign(n, nan); zn.hv0.assign(n, nan);
        zn.grad.assign(8 * n, nan);
    }
    return 0;
}

// pack (index gather into the per-link send buffer) then unpack (contiguous copy into the ghost
// range): PAPER.md:460.  nf doubles per cell starting at arrays f[0..nf-1] (SoA) or one AoS array.
void exchange_state(Zones& Z) {
    size_t nb = 0;
    for (Zone& zn : Z.z) nb += zn.links.size();
    Z.sendbuf.resize(nb);
    size_t b = 0;
    for (Zone& zn : Z.z)
        for (Link& lk : zn.links) {   // pack, on the source zone's arrays
            const Zone& s = Z.z[lk.src];
            std::vector<double>& buf = Z.sendbuf[b++];
            buf.resize(3 * (size_t)lk.count);
            for (int32_t j = 0; j < lk.count; ++j) {
                buf[3 * j] = s.h[lk.send[j]]; buf[3 * j + 1] = s.hu[lk.send[j]]; buf[3 * j + 2] = s.hv[lk.send[j]];
            }
        }
    b = 0;
    for (Zone& zn : Z.z)
        for (Link& lk : zn.links) {   // unpack in place
            const std::vector<double>& buf = Z.sendbuf[b++];
            for (int32_t j = 0; j < lk.count; ++j) {
                zn.h[lk.start + j] = buf[3 * j]; zn.hu[lk.start + j] = buf[3 * j + 1]; zn.hv[lk.start + j] = buf[3 * j + 2];
            }
        }
}
void exchange_grad(Zones& Z) {
    size_t nb = 0;
    for (Zone& zn : Z.z) nb += zn.links.size();
    Z.sendbuf.resize(nb);
    size_t b = 0;
    for (Zone& zn : Z.z)
        for (Link& lk : zn.links) {
            const Zone& s = Z.z[lk.src];
            std::vector<double>& buf = Z.sendbuf[b++];
            buf.resize(8 * (size_t)lk.count);
            for (int32_t j = 0; j < lk.count; ++j)
                for (int q = 0; q < 8; ++q) buf[8 * j + q] = s.grad[8 * (size_t)lk.send[j] + q];
        }
    b = 0;
    for (Zone& zn : Z.z)
        for (Link& lk : zn.links) {
            const std::vector<double>& buf = Z.sendbuf[b++];
            for (int32_t j = 0; j < lk.count; ++j)
                for (int q = 0; q < 8; ++q) zn.grad[8 * (size_t)(lk.start + j) + q] = buf[8 * j + q];
        }
}

void zone_scatter(Zones& Z, const Zone& zn, bool with_grad) {
    for (size_t j = 0; j < zn.cells.size(); ++j) {
        int32_t gI = zn.cells[j];
        Z.sh[gI] = zn.h[j]; Z.shu[gI] = zn.hu[j]; Z.shv[gI] = zn.hv[j];
        if (with_grad) for (int q = 0; q < 8; ++q) Z.sgrad[8 * (size_t)gI + q] = zn.grad[8 * j + q];
    }
}
void zone_unscatter(Zones& Z, const Zone& zn) {
    double nan = std::numeric_limits<double>::quiet_NaN();
    for (size_t j = 0; j < zn.cells.size(); ++j) {
        int32_t gI = zn.cells[j];
        Z.sh[gI] = nan; Z.shu[gI] = nan; Z.shv[gI] = nan;
        for (int q = 0; q < 8; ++q) Z.sgrad[8 * (size_t)gI + q] = nan;
    }
}

// one Euler stage of every zone: zone state (h,hu,hv) -> new owned values written in place
int zones_stage(Ctx& c, Zones& Z, double dt, int scheme) {
    exchange_state(Z);                                        // A.12.5: exchange U
    if (scheme == SCH_MUSCL) {
        for (Zone& zn : Z.z) {                                // gradients, zone by zone
            zone_scatter(Z, zn, false);
            for (size_t j = 0; j < zn.cells.size(); ++j) {
                bool need = (Z.nlayers >= 2) ? (zn.layer[j] <= 1) : (zn.layer[j] == 0);
                if (need) cell_gradient(c, Z.sh.data(), Z.shu.data(), Z.shv.data(), zn.cells[j], &zn.grad[8 * j]);
            }
            zone_unscatter(Z, zn);
        }
        if (Z.nlayers == 1) exchange_grad(Z);                 // limited gradients of layer 1
    }
    for (Zone& zn : Z.z) {
        zone_scatter(Z, zn, scheme == SCH_MUSCL);
        std::vector<double> a(zn.nowned), b(zn.nowned), d(zn.nowned);
        for (int64_t j = 0; j < zn.nowned; ++j)
            cell_update(c, Z.sh.data(), Z.shu.data(), Z.shv.data(), scheme == SCH_MUSCL ? Z.sgrad.data() : nullptr,
                        zn.cells[j], dt, scheme, a[j], b[j], d[j]);
        zone_unscatter(Z, zn);
        for (int64_t j = 0; j < zn.nowned; ++j) {
            if (a[j] != a[j] || b[j] != b[j] || d[j] != d[j]) return -3;   // touched a cell outside the zone
            zn.h[j] = a[j]; zn.hu[j] = b[j]; zn.hv[j] = d[j];
        }
    }
    return 0;
}

int zones_step(Ctx& c, Zones& Z, double cfl, int scheme) {
    // A.12.6 dt = min over the owned cells of all zones
    double best = std::numeric_limits<double>::infinity();
    for (Zone& zn : Z.z)
        for (int64_t j = 0; j < zn.nowned; ++j) {
            if (!(zn.h[j] > c.p.h_dry)) continue;
            double u = zn.hu[j] / zn.h[j], v = zn.hv[j] / zn.h[j];
            double lam = std::sqrt(c.p.g * zn.h[j]) + std::sqrt(u * u + v * v);
            best = std::min(best, c.m.rin[zn.cells[j]] / lam);
        }
    double dt = (best == std::numeric_limits<double>::infinity()) ? 0.0 : cfl * best;
    if (dt > 0.0) {
        if (scheme == SCH_MUSCL || scheme == SCH_MUSCL_MS) {
            for (Zone& zn : Z.z)
                for (int64_t j = 0; j < zn.nowned; ++j) { zn.h0[j] = zn.h[j]; zn.hu0[j] = zn.hu[j]; zn.hv0[j] = zn.hv[j]; }
            int rc = zones_stage(c, Z, dt, scheme); if (rc) return rc;
            rc = zones_stage(c, Z, dt, scheme); if (rc) return rc;
            for (Zone& zn : Z.z)
                for (int64_t j = 0; j < zn.nowned; ++j) {
                    double hn = 0.5 * (zn.h0[j] + zn.h[j]);
                    double hun = 0.5 * (zn.hu0[j] + zn.hu[j]);
                    double hvn = 0.5 * (zn.hv0[j] + zn.hv[j]);
                    if (!(hn > c.p.h_dry)) { hun = 0.0; hvn = 0.0; }
                    zn.h[j] = hn; zn.hu[j] = hun; zn.hv[j] = hvn;
                }
        } else {
            int rc = zones_stage(c, Z, dt, scheme); if (rc) return rc;
        }
    }
    c.t += dt; c.last_dt = dt; c.steps++;
    return 0;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// C interface for tests (ctypes)
// ---------------------------------------------------------------------------------------------
extern "C" {

void orc_set_threads(int n) {
#ifdef _OPENMP
    g_threads = n > 0 ? n : omp_get_max_threads();
#else
    (void)n; g_threads = 1;
#endif
}
int orc_get_threads() { return g_threads; }

void* orc_create(int64_t nv, const double* x, const double* y, const double* zb, int64_t nt,
                 const int32_t* tri, int64_t nb, const int32_t* bedge, const int32_t* btag,
                 char* errbuf, int errlen) {
    Ctx* c = new Ctx();
    std::string err;
    if (!build_mesh(c->m, nv, x, y, zb, nt, tri, nb, bedge, btag, err)) {
        if (errbuf && errlen > 0) { std::strncpy(errbuf, err.c_str(), errlen - 1); errbuf[errlen - 1] = 0; }
        delete c;
        return nullptr;
    }
    // width of every tag
    for (int64_t e = 0; e < c->m.ne; ++e)
        if (c->m.eR[e] < 0 && c->m.etag[e] >= 0) c->bc[c->m.etag[e]].width += c->m.elen[e];
    c->h.assign(nt, 0.0); c->hu.assign(nt, 0.0); c->hv.assign(nt, 0.0);
    return c;
}
void orc_destroy(void* p);

int orc_info(void* p, int64_t* nt, int64_t* ne, int64_t* nbe, double* min_rin) {
    Ctx* c = (Ctx*)p;
    if (nt) *nt = c->m.nt;
    if (ne) *ne = c->m.ne;
    if (nbe) *nbe = c->m.nbe;
    if (min_rin) *min_rin = *std::min_element(c->m.rin.begin(), c->m.rin.end());
    return 0;
}
int orc_set_params(void* p, double g, double h_dry, double h_thin, double beta) {
    Ctx* c = (Ctx*)p;
    c->p.g = g; c->p.h_dry = h_dry; c->p.h_thin = h_thin; c->p.beta = beta;
    return 0;
}
int orc_set_manning(void* p, const double* n) {
    Ctx* c = (Ctx*)p;
    if (n) c->nman.assign(n, n + c->m.nt); else c->nman.clear();
    return 0;
}
int orc_set_bc(void* p, int tag, int kind, double value) {
    Ctx* c = (Ctx*)p;
    if (tag < 0 || kind < 0 || kind > 3) return -1;
    BCInfo& b = c->bc[tag];
    b.kind = kind; b.value = value;
    return 0;
}
int orc_set_state(void* p, const double* h, const double* hu, const double* hv) {
    Ctx* c = (Ctx*)p;
    int64_t nt = c->m.nt;
    for (int64_t i = 0; i < nt; ++i) if (!(h[i] >= 0.0)) return -4;
    c->h.assign(h, h + nt); c->hu.assign(hu, hu + nt); c->hv.assign(hv, hv + nt);
    return 0;
}
int orc_get_state(void* p, double* h, double* hu, double* hv) {
    Ctx* c = (Ctx*)p;
    std::copy(c->h.begin(), c->h.end(), h);
    std::copy(c->hu.begin(), c->hu.end(), hu);
    std::copy(c->hv.begin(), c->hv.end(), hv);
    return 0;
}
void orc_set_time(void* p, double t) { ((Ctx*)p)->t = t; }
int orc_step(void* p, int nsteps, double cfl, int scheme, double* t_out, double* dt_out) {
    Ctx* c = (Ctx*)p;
    if (scheme < 0 || scheme > 3 || nsteps < 0) return -1;
    for (int s = 0; s < nsteps; ++s) one_step(*c, cfl, scheme);
    if (t_out) *t_out = c->t;
    if (dt_out) *dt_out = c->last_dt;
    return 0;
}
double orc_compute_dt(void* p, double cfl) {
    Ctx* c = (Ctx*)p;
    return compute_dt(*c, c->h.data(), c->hu.data(), c->hv.data(), cfl);
}
int orc_gradients(void* p, double* out) {
    Ctx* c = (Ctx*)p;
    compute_gradients(*c, c->h.data(), c->hu.data(), c->hv.data(), out);
    return 0;
}
// one Euler stage from the current state with a given dt, result to caller arrays (state untouched)
int orc_euler_stage(void* p, double dt, int scheme, double* h1, double* hu1, double* hv1) {
    Ctx* c = (Ctx*)p;
    euler_stage(*c, c->h.data(), c->hu.data(), c->hv.data(), dt, scheme, h1, hu1, hv1);
    return 0;
}
int orc_cell_geometry(void* p, double* area, double* cx, double* cy, double* zc, double* rin) {
    Ctx* c = (Ctx*)p;
    const Mesh& m = c->m;
    if (area) std::copy(m.area.begin(), m.area.end(), area);
    if (cx) std::copy(m.cx.begin(), m.cx.end(), cx);
    if (cy) std::copy(m.cy.begin(), m.cy.end(), cy);
    if (zc) std::copy(m.zc.begin(), m.zc.end(), zc);
    if (rin) std::copy(m.rin.begin(), m.rin.end(), rin);
    return 0;
}
int orc_edge_geometry(void* p, int32_t* eL, int32_t* eR, double* len, double* nx, double* ny, double* dx) {
    Ctx* c = (Ctx*)p;
    const Mesh& m = c->m;
    if (eL) std::copy(m.eL.begin(), m.eL.end(), eL);
    if (eR) std::copy(m.eR.begin(), m.eR.end(), eR);
    if (len) std::copy(m.elen.begin(), m.elen.end(), len);
    if (nx) std::copy(m.enx.begin(), m.enx.end(), nx);
    if (ny) std::copy(m.eny.begin(), m.eny.end(), ny);
    if (dx) std::copy(m.edx.begin(), m.edx.end(), dx);
    return 0;
}
int orc_cell_topology(void* p, int32_t* c2c, int32_t* c2e) {
    Ctx* c = (Ctx*)p;
    if (c2c) std::copy(c->m.c2c.begin(), c->m.c2c.end(), c2c);
    if (c2e) std::copy(c->m.c2e.begin(), c->m.c2e.end(), c2e);
    return 0;
}
// flux of one edge from the current state: PhiL[3], PhiR[3] (already times the edge length)
int orc_edge_flux(void* p, int32_t e, double dt, int scheme, double* PhiL, double* PhiR) {
    Ctx* c = (Ctx*)p;
    if (e < 0 || e >= c->m.ne) return -1;
    const double* grad = nullptr;
    if (scheme == SCH_MUSCL) {
        c->grad.resize(8 * c->m.nt);
        compute_gradients(*c, c->h.data(), c->hu.data(), c->hv.data(), c->grad.data());
        grad = c->grad.data();
    }
    edge_flux(*c, c->h.data(), c->hu.data(), c->hv.data(), grad, e, dt, scheme, PhiL, PhiR);
    return 0;
}

// pure functions
// out = G1, G2, G3, SL, SR, Sstar, hstar, h0
void orc_hllc(double g, double h_dry, double hL, double uL, double vL, double hR, double uR, double vR,
              double* out) {
    Waves w;
    hllc_flux(g, h_dry, hL, uL, vL, hR, uR, vR, out, &w);
    out[3] = w.SL; out[4] = w.SR; out[5] = w.Sstar; out[6] = w.hstar; out[7] = w.h0;
}
void orc_waf(double g, double h_dry, double hL, double uL, double vL, double hR, double uR, double vR,
             double etaL, double etaR, double etaLupw, double etaRupw, double vLupw, double vRupw,
             double dt, double dx, int use_limiter, double* out) {
    waf_flux(g, h_dry, hL, uL, vL, hR, uR, vR, etaL, etaR, etaLupw, etaRupw, vLupw, vRupw, dt, dx,
             use_limiter, out);
}
double orc_limiter_A(double r, double c) { return limiter_A(r, c); }
double orc_ms_slope(double beta, double x, double y) { return ms_slope(beta, x, y); }
void orc_manning(double g, double n, double dt, double h, double* hu, double* hv) {
    manning_step(g, n, dt, h, *hu, *hv);
}


// ---- zones ----
void orc_destroy(void* p) { g_zones.erase((Ctx*)p); delete (Ctx*)p; }
int orc_zones_create(void* p, int nz, int nlayers, const int32_t* zone_of_cell) {
    Ctx* c = (Ctx*)p;
    Zones& Z = g_zones[c];
    Z = Zones();
    return zones_build(*c, Z, nz, nlayers, zone_of_cell);
}
// advances the zoned copy of the state; the context's global state is scattered to the zones'
// owned cells before and gathered back after, so orc_get_state returns the zoned result
int orc_zones_step(void* p, int nsteps, double cfl, int scheme, double* t_out, double* dt_out) {
    Ctx* c = (Ctx*)p;
    auto it = g_zones.find(c);
    if (it == g_zones.end()) return -4;
    Zones& Z = it->second;
    int need = (scheme == SCH_HLLC) ? 1 : ((scheme == SCH_WAF || scheme == SCH_MUSCL_MS) ? 2 : 1);
    if (Z.nlayers < need) return -4;
    for (Zone& zn : Z.z)
        for (int64_t j = 0; j < zn.nowned; ++j) {
            zn.h[j] = c->h[zn.cells[j]]; zn.hu[j] = c->hu[zn.cells[j]]; zn.hv[j] = c->hv[zn.cells[j]];
        }
    for (int s = 0; s < nsteps; ++s) { int rc = zones_step(*c, Z, cfl, scheme); if (rc) return rc; }
    for (Zone& zn : Z.z)
        for (int64_t j = 0; j < zn.nowned; ++j) {
            c->h[zn.cells[j]] = zn.h[j]; c->hu[zn.cells[j]] = zn.hu[j]; c->hv[zn.cells[j]] = zn.hv[j];
        }
    if (t_out) *t_out = c->t;
    if (dt_out) *dt_out = c->last_dt;
    return 0;
}
int orc_zones_counts(void* p, int64_t* send_cells, int64_t* bytes_per_exchange, int64_t* ghost_cells) {
    Ctx* c = (Ctx*)p;
    auto it = g_zones.find(c);
    if (it == g_zones.end()) return -4;
    int64_t s = 0, gh = 0;
    for (Zone& zn : it->second.z) {
        for (Link& lk : zn.links) s += lk.count;
        gh += (int64_t)zn.cells.size() - zn.nowned;
    }
    if (send_cells) *send_cells = s;
    if (bytes_per_exchange) *bytes_per_exchange = s * 24;
    if (ghost_cells) *ghost_cells = gh;
    return 0;
}
int orc_zones_zone_of_cell(void* p, int32_t* out) {
    Ctx* c = (Ctx*)p;
    auto it = g_zones.find(c);
    if (it == g_zones.end()) return -4;
    std::copy(it->second.zone_of.begin(), it->second.zone_of.end(), out);
    return 0;
}
int orc_zones_describe(void* p, int zone, int64_t* nowned, int64_t* nghost, int64_t* nlinks) {
    Ctx* c = (Ctx*)p;
    Zone& zn = g_zones.at(c).z.at(zone);
    *nowned = zn.nowned; *nghost = (int64_t)zn.cells.size() - zn.nowned; *nlinks = (int64_t)zn.links.size();
    return 0;
}
int orc_zones_cells(void* p, int zone, int32_t* cells, int32_t* layer) {
    Ctx* c = (Ctx*)p;
    Zone& zn = g_zones.at(c).z.at(zone);
    std::copy(zn.cells.begin(), zn.cells.end(), cells);
    std::copy(zn.layer.begin(), zn.layer.end(), layer);
    return 0;
}
int orc_zones_links(void* p, int zone, int32_t* src, int32_t* start, int32_t* count) {
    Ctx* c = (Ctx*)p;
    Zone& zn = g_zones.at(c).z.at(zone);
    for (size_t j = 0; j < zn.links.size(); ++j) { src[j] = zn.links[j].src; start[j] = zn.links[j].start; count[j] = zn.links[j].count; }
    return 0;
}
int orc_zones_sendlist(void* p, int zone, int link, int32_t* out) {
    Ctx* c = (Ctx*)p;
    Link& lk = g_zones.at(c).z.at(zone).links.at(link);
    std::copy(lk.send.begin(), lk.send.end(), out);
    return 0;
}

}  // extern "C"
