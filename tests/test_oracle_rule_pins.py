"""Pins for the oracle rules that the round-1 mutation run found unpinned (VERDICT.md, row c):

  A.3.1  the velocity of a boundary neighbour is mirrored in a WALL (gradient stencil)
  A.3.3  the limiter's extrema run over REAL neighbours only (mirror values excluded)
  R14    WAF falls back to HLLC within one cell of a cell with h <= h_thin
  R8     the outer WAF waves are limited on q = eta, not q = h
  R7     |c_k| is clamped to 1
  BC     the transmissive boundary carries the tangential momentum G3 = G1 u_t
  R17    the multislope reconstruction is first order if a cell of its stencil is not wet

Each test states a property that the mathematics (or the reading as DESIGN.md words it) fixes and
that a broken rule violates; none re-types the oracle's arithmetic.  The mutants of VERDICT.md
"What's weak" 1 each fail at least one test of this file (oracle/mutation_check.py runs them).
"""
import numpy as np
import pytest

import swe_inputs as si
from oracle import pyoracle as po

G = 9.81


def _rot(x, y, ang):
    c, s = np.cos(ang), np.sin(ang)
    return c * x - s * y, s * x + c * y


# ---------------------------------------------------------------------------------------------
# A.3.1: wall mirror of the velocity
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ang", [0.0, 0.6, -2.1])
def test_wall_mirror_makes_lsq_exact_for_velocity_linear_in_wall_distance(ang):
    """Flow normal to a straight wall and proportional to the distance s from it, U = a s m
    (m = unit normal into the domain).  Reflecting a cell's velocity in the wall, U - 2(U.n)n,
    gives -a s m: exactly the value the linear field takes at the cell's mirror point (s -> -s).
    The least-squares gradient over {two real neighbours, mirror point} is exact for linear data,
    so the unlimited gradient of a wall cell must be a m m^T to round-off.  Copying the cell's own
    velocity into the mirror point instead (no reflection) cannot give that."""
    nx, ny, lx, ly, a = 12, 8, 12.0, 8.0, 0.37
    x0, y0, tri = si.grid_mesh(nx, ny, lx, ly, 0.2, 5)
    x, y = _rot(x0, y0, ang)
    mx, my = _rot(0.0, 1.0, ang)                                   # inward normal of the wall y0 = 0
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    o.set_params(beta=0.0)                                         # unlimited (A.3.4)
    s = y0[tri].mean(axis=1)                                       # distance of the centroid from the wall
    h = np.full(o.nt, 2.0)
    o.set_state(h, h * a * s * mx, h * a * s * my)
    gr = o.gradients()
    c2c, _ = o.cell_topology()
    on_wall = (y0[tri] == 0.0).sum(axis=1) == 2                    # an edge on the wall y0 = 0
    one_bnd = (c2c < 0).sum(axis=1) == 1                           # ... and no other boundary edge
    cells = np.nonzero(on_wall & one_bnd)[0]
    assert cells.size >= nx - 2
    want = a * np.array([mx * mx, mx * my, my * mx, my * my])      # u_x u_y v_x v_y
    np.testing.assert_allclose(gr[cells, 4:8], np.tile(want, (cells.size, 1)), rtol=0, atol=1e-13)
    np.testing.assert_allclose(gr[cells, 0:4], 0.0, rtol=0, atol=1e-13)


def test_wall_mirror_leaves_tangential_velocity_unreflected():
    """A uniform stream along a straight wall: the reflection changes nothing (U.n = 0), every
    neighbour value equals the cell's, the gradient is zero and the stream is steady along the
    wall.  A mirror that flipped the whole velocity would see a jump of 2|U| at the wall."""
    x, y, tri = si.grid_mesh(10, 6, 10.0, 6.0, 0.2, 3)
    x, y = _rot(x, y, 0.4)
    ux, uy = _rot(1.3, 0.0, 0.4)
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    h = np.full(o.nt, 1.5)
    o.set_state(h, h * ux, h * uy)
    c2c, _ = o.cell_topology()
    x0, y0 = _rot(x, y, -0.4)
    long_wall = ((np.abs(y0[tri]) < 1e-9).sum(axis=1) == 2) | ((np.abs(y0[tri] - 6.0) < 1e-9).sum(axis=1) == 2)
    cells = np.nonzero(long_wall & ((c2c < 0).sum(axis=1) == 1))[0]
    for beta in (0.0, 1.0):
        o.set_params(beta=beta)
        np.testing.assert_allclose(o.gradients()[cells], 0.0, rtol=0, atol=1e-14)


# ---------------------------------------------------------------------------------------------
# A.3.3: extrema over real neighbours only
# ---------------------------------------------------------------------------------------------
def test_limiter_extrema_exclude_the_mirror_value():
    """A wall cell whose normal velocity v_i = -1 is a strict maximum among its REAL neighbours
    (v = -3) while its mirror value is +1.  With the extrema over real neighbours only, q_max = q_i,
    so any face increment > 0 is limited to zero (A.3.4: phi_k = kappa (q_max - q_i)/Delta_k = 0)
    and the limited gradient of v is exactly zero -- the cell is a local extremum of the data.
    Counting the mirror value (+1) among the extrema would leave a non-zero slope."""
    x, y, tri = si.grid_mesh(10, 6, 10.0, 6.0, 0.2, 9)
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    c2c, _ = o.cell_topology()
    on_wall = (y[tri] == 0.0).sum(axis=1) == 2
    cells = np.nonzero(on_wall & ((c2c < 0).sum(axis=1) == 1))[0]
    assert cells.size >= 6
    for i in cells[1:-1:2]:
        h = np.full(o.nt, 1.0)
        v = np.full(o.nt, -3.0)
        v[i] = -1.0
        o.set_state(h, 0.5 * h, h * v)
        o.set_params(beta=0.0)
        g0 = o.gradients()[i]
        assert np.abs(g0[6:8]).max() > 0.1                         # the unlimited slope is not zero
        for beta in (1.0, 2.0):
            o.set_params(beta=beta)
            g1 = o.gradients()[i]
            assert g1[6] == 0.0 and g1[7] == 0.0, (i, beta, g1)
    # and the other way round: a cell strictly inside the range of its real neighbours keeps a slope
    i = cells[2]
    nb = [n for n in c2c[i] if n >= 0]
    h = np.full(o.nt, 1.0)
    v = np.full(o.nt, -3.0)
    v[i] = -1.0
    v[nb[0]] = 0.5
    o.set_state(h, 0.5 * h, h * v)
    o.set_params(beta=1.0)
    assert np.abs(o.gradients()[i][6:8]).max() > 1e-3


# ---------------------------------------------------------------------------------------------
# R14: WAF -> HLLC within one cell of a thin cell;  R17: multislope first order next to dry cells
# ---------------------------------------------------------------------------------------------
def _smooth_monotone_case(nx=16, ny=10, seed=13):
    x, y, tri = si.grid_mesh(nx, ny, 16.0, 10.0, 0.15, seed)
    cx = x[tri].mean(axis=1)
    cy = y[tri].mean(axis=1)
    h = 1.5 + 0.02 * cx + 0.013 * cy
    u = 0.30 + 0.004 * cx + 0.002 * cy
    v = 0.10 + 0.003 * cx + 0.005 * cy
    return x, y, tri, h, u, v


def _graph_distance(c2c, seeds, nmax=4):
    d = np.full(c2c.shape[0], 99, np.int64)
    d[seeds] = 0
    for l in range(1, nmax + 1):
        for i in np.nonzero(d == l - 1)[0]:
            for n in c2c[i]:
                if n >= 0 and d[n] > l:
                    d[n] = l
    return d


def _edge_fluxes(o, dt, scheme, edges):
    return np.array([np.concatenate(o.edge_flux(int(e), dt, scheme)) for e in edges])


@pytest.mark.parametrize("film", [5e-4, 0.0])
def test_waf_is_hllc_exactly_within_one_cell_of_a_thin_cell_and_only_there(film):
    """Reading R14 as DESIGN.md states it: WAF is used on an edge iff both cells and all their real
    edge-neighbours are deeper than h_thin = 1e-3 m.  A film of 5e-4 m is wet (> h_dry = 1e-6 m) but
    thin, which separates h_thin from h_dry.  On a smooth monotone flow every limiter ratio is
    positive, A < 1, and the WAF flux differs from the HLLC flux -- except where the rule says
    HLLC."""
    x, y, tri, h, u, v = _smooth_monotone_case()
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    c2c, _ = o.cell_topology()
    inner_cells = np.nonzero((c2c >= 0).all(axis=1))[0]
    thin = inner_cells[[7, len(inner_cells) // 2, -9]]
    h = h.copy()
    h[thin] = film
    o.set_state(h, h * u, h * v)
    dt = o.compute_dt(0.45)
    e = o.edge_geometry()
    inner = np.nonzero(e["eR"] >= 0)[0]
    d = _graph_distance(c2c, thin)
    dmin = np.minimum(d[e["eL"][inner]], d[e["eR"][inner]])
    near, far = inner[dmin <= 1], inner[dmin >= 2]
    assert near.size >= 15 and far.size > 200
    fw, fh = _edge_fluxes(o, dt, "waf", near), _edge_fluxes(o, dt, "hllc", near)
    assert np.array_equal(fw, fh)                                  # bit for bit
    fw, fh = _edge_fluxes(o, dt, "waf", far), _edge_fluxes(o, dt, "hllc", far)
    differ = np.any(fw != fh, axis=1)
    assert differ.all(), "WAF fell back to HLLC on %d edges away from thin cells" % (~differ).sum()


def test_multislope_is_first_order_exactly_where_the_stencil_holds_a_dry_cell_and_only_there():
    """Reading R17: the multislope face values are the cell values if any cell of the stencil
    (the two cells and their other edge-neighbours) is not wet -- the flux is then the first-order
    HLLC flux bit for bit.  Away from dry cells a smooth monotone flow has non-zero limited slopes
    and the two fluxes differ."""
    x, y, tri, h, u, v = _smooth_monotone_case(seed=14)
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    c2c, _ = o.cell_topology()
    inner_cells = np.nonzero((c2c >= 0).all(axis=1))[0]
    dry = inner_cells[[5, len(inner_cells) // 2 + 3, -12]]
    h = h.copy()
    h[dry] = [0.0, 5e-7, 0.0]                                       # 5e-7 <= h_dry: not wet either
    o.set_state(h, h * u, h * v)
    dt = o.compute_dt(0.45)
    e = o.edge_geometry()
    inner = np.nonzero(e["eR"] >= 0)[0]
    d = _graph_distance(c2c, dry)
    dmin = np.minimum(d[e["eL"][inner]], d[e["eR"][inner]])
    near, far = inner[dmin <= 1], inner[dmin >= 2]
    fm, fh = _edge_fluxes(o, dt, "muscl_ms", near), _edge_fluxes(o, dt, "hllc", near)
    assert np.array_equal(fm, fh)
    fm, fh = _edge_fluxes(o, dt, "muscl_ms", far), _edge_fluxes(o, dt, "hllc", far)
    assert np.any(fm != fh, axis=1).all()


@pytest.mark.parametrize("scheme,cfl", [("waf", 0.45), ("muscl_ms", 0.45)])
def test_mass_and_positivity_through_wet_dry_front_waf_and_multislope(scheme, cfl, oracle_threads):
    """without the WAF -> HLLC fallback a dry-bed run loses positivity (the clamp
    h = max(h, 0) then creates mass, drift 1e-7); with it mass is exact.  Same for the multislope
    reconstruction without its dry-stencil rule."""
    cfg = si.config0(nx=100, ny=5, h_left=4.0, h_right=0.0)
    o = po.Oracle.from_config(cfg)
    area = o.cell_geometry()["area"]
    m0 = float((cfg["h"] * area).sum())
    for _ in range(10):
        o.step(20, cfl, scheme)
        h, hu, hv = o.get_state()
        assert h.min() >= 0.0
        assert abs(float((h * area).sum()) - m0) <= 1e-13 * m0
        dry = h <= 1e-6
        assert np.all(hu[dry] == 0.0) and np.all(hv[dry] == 0.0)


# ---------------------------------------------------------------------------------------------
# R8: q = eta for the outer WAF waves
# ---------------------------------------------------------------------------------------------
def test_waf_outer_wave_limiter_sees_the_free_surface_not_the_depth():
    """Three states on one mesh that differ only in the UPWIND cells of an edge (the two other
    edge-neighbours of its L- and R-cell):
      A: reference, a smooth monotone free surface over an uneven bed: the upwind jumps have the
         sign of the local jump, r > 0, A(r, c) < 1 on both outer waves;
      B: the bed under the upwind cells moved by +-0.1 m, their free surface kept (depth changes);
      C: the same bed as B, their depth kept (free surface changes by +-0.1 m, signs chosen so that
         both upwind jumps change sign: r < 0, A = 1, fully upwind).
    The two cells of the edge, and therefore the Riemann problem, are the same in all three.  With
    the limiter ratios of the outer waves formed on eta (R8: bathymetry jumps must not masquerade
    as waves), the edge flux of B equals that of A and the flux of C does not; formed on h it
    would be the other way round."""
    x, y, tri = si.grid_mesh(12, 9, 12.0, 9.0, 0.15, 21)
    rng = np.random.default_rng(3)
    zb = 0.3 * np.sin(0.7 * x) + 0.2 * np.cos(0.9 * y)
    oA = po.Oracle(x, y, zb, tri)
    c2c, _ = oA.cell_topology()
    e = oA.edge_geometry()
    cx = x[tri].mean(axis=1)
    cy = y[tri].mean(axis=1)
    eta = 2.5 + 0.02 * cx + 0.015 * cy
    u = 0.4 + 0.01 * cx
    v = 0.1 + 0.01 * cy
    zcA = oA.cell_geometry()["zc"]
    hA = eta - zcA
    oA.set_state(hA, hA * u, hA * v)
    dt = oA.compute_dt(0.45)
    inner = np.nonzero(e["eR"] >= 0)[0]
    checked = 0
    for ed in rng.permutation(inner):
        L, R = int(e["eL"][ed]), int(e["eR"][ed])
        upL = [int(n) for n in c2c[L] if n != R]
        upR = [int(n) for n in c2c[R] if n != L]
        upw = upL + upR
        if min(upw) < 0 or len(set(upw)) != 4:
            continue
        own = set(tri[L]) | set(tri[R])
        far = [sorted(set(tri[n]) - own) for n in upw]             # each upwind cell's vertex off L, R
        if any(len(f) != 1 for f in far) or len({f[0] for f in far}) != 4:
            continue
        far = [int(f[0]) for f in far]
        dloc = eta[R] - eta[L]
        dL = eta[L] - 0.5 * (eta[upL[0]] + eta[upL[1]])
        dR = 0.5 * (eta[upR[0]] + eta[upR[1]]) - eta[R]
        if not (dL * dloc > 0.0 and dR * dloc > 0.0 and abs(dloc) > 1e-3):
            continue
        zb2 = zb.copy()
        zb2[far[0:2]] += 0.3 * np.sign(dL)                          # cell bed = vertex mean: +-0.1 m
        zb2[far[2:4]] -= 0.3 * np.sign(dR)
        oB = po.Oracle(x, y, zb2, tri)
        zc2 = oB.cell_geometry()["zc"]
        assert zc2[L] == zcA[L] and zc2[R] == zcA[R]
        assert min(abs(zc2[n] - zcA[n]) for n in upw) > 0.09
        hB = eta - zc2                                             # same free surface, other depth
        oB.set_state(hB, hB * u, hB * v)
        oC = po.Oracle(x, y, zb2, tri)
        oC.set_state(hA, hA * u, hA * v)                           # same depth, other free surface
        fA = np.concatenate(oA.edge_flux(ed, dt, "waf"))
        fB = np.concatenate(oB.edge_flux(ed, dt, "waf"))
        fC = np.concatenate(oC.edge_flux(ed, dt, "waf"))
        scale = np.abs(fA).max()
        assert np.abs(fB - fA).max() <= 1e-13 * scale, (ed, fA, fB)
        assert np.abs(fC - fA).max() >= 1e-4 * scale, (ed, fA, fC)
        checked += 1
        if checked == 8:
            break
    assert checked == 8


# ---------------------------------------------------------------------------------------------
# R7: |c| <= 1
# ---------------------------------------------------------------------------------------------
def test_waf_courant_numbers_are_clamped_to_one():
    """eq. 21 at |c| = 1 gives A = 1 for every r, i.e. the fully upwind flux of eq. 6.  With the
    clamp |c_k| <= 1 (R7) a time step far beyond the CFL limit therefore returns the HLLC flux; an
    unclamped c > 1 would extrapolate (A = 2|c| - 1 > 1 for r > 2)."""
    args = (2.0, 0.3, 0.2, 1.2, -0.1, 0.5)
    hl = po.hllc(G, 1e-6, *args)
    for etaLupw, etaRupw in ((2.6, 0.9), (1.9, 1.25), (2.0, 1.2)):
        w = po.waf(G, 1e-6, *args, 2.0, 1.2, etaLupw, etaRupw, 0.1, 0.6, dt=50.0, dx=1.0)
        np.testing.assert_allclose(w, [hl["G1"], hl["G2"], hl["G3"]], rtol=1e-14)
    w = po.waf(G, 1e-6, *args, 2.0, 1.2, 2.6, 0.9, 0.1, 0.6, dt=0.05, dx=1.0)
    assert abs(w[0] - hl["G1"]) > 1e-3                             # inside the CFL limit WAF is not upwind


# ---------------------------------------------------------------------------------------------
# transmissive boundary: tangential momentum
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme,cfl", [("hllc", 0.9), ("muscl", 0.45), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_oblique_uniform_stream_through_an_open_box_stays_uniform(scheme, cfl):
    """U_R = U_L on every side: a uniform stream crossing the box obliquely is an
    exact steady state, because the physical flux of a constant state sums to zero over a closed
    cell.  That needs all three components of the boundary flux, including the tangential
    momentum G3 = G1 u_t that a stream normal to the boundary never exercises."""
    x, y, tri = si.grid_mesh(14, 9, 14.0, 9.0, 0.2, 17)
    be = si.boundary_edges(tri)
    o = po.Oracle(x, y, np.zeros_like(x), tri, be, np.full(len(be), 3, np.int32))
    o.set_bc(3, "transmissive")
    h0 = np.full(o.nt, 2.0)
    o.set_state(h0, h0 * 1.5, h0 * 0.5)
    o.step(40, cfl, scheme)
    h, hu, hv = o.get_state()
    np.testing.assert_allclose(h, 2.0, rtol=0, atol=1e-12)
    np.testing.assert_allclose(hu, 3.0, rtol=0, atol=1e-12)
    np.testing.assert_allclose(hv, 1.0, rtol=0, atol=1e-12)


# ---------------------------------------------------------------------------------------------
# fixed-level boundary: tangential velocity of the ghost state (R11)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme,cfl", [("hllc", 0.9), ("muscl", 0.45), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_oblique_uniform_stream_through_level_boundaries_stays_uniform(scheme, cfl):
    """A box whose four sides all hold the free surface at the level of the water inside, crossed
    obliquely by a uniform stream.  The ghost state of reading R11 (depth from the level, normal
    velocity from the outgoing invariant, the interior's tangential velocity) then equals the
    interior state on every side, the boundary flux is the physical flux of a constant state, and
    the stream is steady.  On the two sides where the water ENTERS the contact wave upwinds the
    tangential momentum from the ghost: a ghost without the interior's tangential velocity breaks
    the steady state there."""
    x, y, tri = si.grid_mesh(14, 9, 14.0, 9.0, 0.2, 23)
    be = si.boundary_edges(tri)
    o = po.Oracle(x, y, np.zeros_like(x), tri, be, np.full(len(be), 2, np.int32))
    o.set_bc(2, "level", 2.0)
    h0 = np.full(o.nt, 2.0)
    o.set_state(h0, h0 * 1.5, h0 * 0.5)
    o.step(40, cfl, scheme)
    h, hu, hv = o.get_state()
    np.testing.assert_allclose(h, 2.0, rtol=0, atol=1e-12)
    np.testing.assert_allclose(hu, 3.0, rtol=0, atol=1e-12)
    np.testing.assert_allclose(hv, 1.0, rtol=0, atol=1e-12)


# ---------------------------------------------------------------------------------------------
# eq. 22 / 24 / 25 worked on a skewed pair of cells: which distances divide which jumps
# ---------------------------------------------------------------------------------------------
def test_multislope_face_values_on_a_skewed_stencil_worked_from_eq_22_24():
    """Still water of varying depth over a flat bed, beta = 1 (MINBEE).  The upwind cells of an
    interior edge are set so far beyond the local jump that both limited slopes of eq. 24-25 are the
    LOCAL slope (h_R - h_L) / |x_R - x_L| (the smaller of two slopes of equal sign), so eq. 22 gives
    the face depths  h_L + |r_L| s  and  h_R - |r_R| s  with |r| the distance from the centroid to
    the edge midpoint (reading R17).  With zero velocity and a flat bed the mass component of the
    edge flux is then the HLLC mass flux between those two face depths (a routine pinned on its own
    in test_oracle_flux.py) times the edge length.  On a strongly jittered mesh the midpoint is off
    the line between the centroids, |r_L| + |r_R| > |x_R - x_L|, so mixing up the distances shows."""
    x, y, tri = si.grid_mesh(10, 8, 10.0, 8.0, 0.3, 31)
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    o.set_params(beta=1.0)
    c2c, _ = o.cell_topology()
    e = o.edge_geometry()
    cx = x[tri].mean(axis=1)
    cy = y[tri].mean(axis=1)
    rng = np.random.default_rng(5)
    inner = np.nonzero(e["eR"] >= 0)[0]
    checked, skew = 0, 0.0
    for ed in rng.permutation(inner):
        L, R = int(e["eL"][ed]), int(e["eR"][ed])
        upL = [int(n) for n in c2c[L] if n != R]
        upR = [int(n) for n in c2c[R] if n != L]
        if min(upL + upR) < 0 or len(set(upL + upR)) != 4:
            continue
        shared = sorted(set(tri[L]) & set(tri[R]))
        mx, my = x[shared].mean(), y[shared].mean()                # edge midpoint
        rL = np.hypot(mx - cx[L], my - cy[L])
        rR = np.hypot(mx - cx[R], my - cy[R])
        dLR = np.hypot(cx[R] - cx[L], cy[R] - cy[L])
        hL, hR = 2.0, 2.3
        h = np.full(o.nt, 2.0)
        h[L], h[R] = hL, hR
        h[upL] = hL - 5.0 * (hR - hL) * 0.3                        # upwind slopes: same sign, much steeper
        h[upR] = hR + 5.0 * (hR - hL) * 0.3
        o.set_state(h, np.zeros(o.nt), np.zeros(o.nt))
        s = (hR - hL) / dLR
        want = po.hllc(G, 1e-6, hL + rL * s, 0.0, 0.0, hR - rR * s, 0.0, 0.0)["G1"] * e["len"][ed]
        got = o.edge_flux(ed, 0.01, "muscl_ms")[0][0]
        assert got == pytest.approx(want, rel=1e-12), (ed, got, want)
        first = o.edge_flux(ed, 0.01, "hllc")[0][0]
        assert abs(got - first) > 1e-3 * abs(first)                # the reconstruction is active
        skew = max(skew, (rL + rR) / dLR - 1.0)
        checked += 1
        if checked == 12:
            break
    assert checked == 12 and skew > 0.01                           # the two distances really differ


def test_mutation_list_still_applies_to_the_oracle_source():
    """oracle/mutation_check.py breaks one rule at a time by exact text replacement: every pattern
    must occur exactly once in oracle/swe_oracle.cpp, or the mutant silently tests nothing (the
    script reports such a mutant as STALE).  The mutation run itself takes ~10 minutes and is not
    part of the suite."""
    import os
    from oracle import mutation_check as mc
    src = open(os.path.join(os.path.dirname(mc.__file__), "swe_oracle.cpp")).read()
    names = [m[0] for m in mc.MUTANTS]
    assert len(names) == len(set(names)) and len(names) >= 56
    for name, rule, find, repl in mc.MUTANTS:
        assert src.count(find) == 1, name
        assert find != repl and rule


# ---------------------------------------------------------------------------------------------
# A.10: h' = max(h', 0), whatever the time step
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", ["hllc", "muscl", "waf", "muscl_ms"])
def test_a_stage_never_returns_a_negative_depth_whatever_the_time_step(scheme):
    """A.10 clamps the updated depth at zero and zeroes the momentum of a cell that ends up not wet.
    At the CFL numbers the schemes are run with, the hydrostatic reconstruction keeps depths positive
    by itself and the clamp never acts; a stage with forty times the stable time step drains cells
    below zero, and the rule must still hold: no negative depth, no momentum without water."""
    cfg = si.config0(nx=60, ny=4, h_left=2.0, h_right=0.02)
    o = po.Oracle.from_config(cfg)
    o.step(5, 0.45, "hllc")                                        # a moving front
    dt = 40.0 * o.compute_dt(0.9)
    h, hu, hv = o.euler_stage(dt, scheme)
    assert np.all(np.isfinite(h)) and np.all(np.isfinite(hu)) and np.all(np.isfinite(hv))
    assert h.min() >= 0.0
    assert (h == 0.0).any()                                        # the clamp was needed somewhere
    dry = h <= 1e-6
    assert np.all(hu[dry] == 0.0) and np.all(hv[dry] == 0.0)


# ---------------------------------------------------------------------------------------------
# R11: the level boundary's ghost depth stands over the FACE bed
# ---------------------------------------------------------------------------------------------
def test_lake_at_rest_against_a_level_boundary_with_unlimited_gradients():
    """C-property at the open boundary.  With z_ghost = z_f (A.8) a lake at rest at the imposed
    level sees its own face state in the ghost -- h_b = level - z_f = h_f -- and nothing moves,
    however the depth is reconstructed.  The cell limiter hides this at boundary cells (they are
    local extrema among their two real neighbours, so their limited gradient is zero and
    z_f = z_cell); with unlimited gradients (beta <= 0) over an uneven bed the face bed differs from
    the cell bed by centimetres, and a ghost standing over the CELL bed would drive a flow."""
    x, y, tri = si.grid_mesh(20, 4, 20.0, 4.0, 0.15, 11)
    be = si.boundary_edges(tri)
    xm = 0.5 * (x[be[:, 0]] + x[be[:, 1]])
    east = be[xm > 20.0 - 1e-9]
    zb = 0.2 * np.sin(x) + 0.1 * y + 0.03 * x
    o = po.Oracle(x, y, zb, tri, east, np.full(len(east), 2, np.int32))
    o.set_bc(2, "level", 3.0)
    o.set_params(beta=0.0)
    zc = o.cell_geometry()["zc"]
    h0 = 3.0 - zc
    o.set_state(h0, np.zeros(o.nt), np.zeros(o.nt))
    gr = o.gradients()
    c2c, _ = o.cell_topology()
    cx = x[tri].mean(axis=1)
    at_outlet = (cx > 19.0) & ((c2c < 0).sum(axis=1) >= 1)
    assert np.abs(gr[at_outlet, 2:4]).max() > 0.02                 # the depth gradient is alive there
    o.step(40, 0.45, "muscl")
    h, hu, hv = o.get_state()
    assert np.abs(hu / h).max() <= 1e-12 and np.abs(hv / h).max() <= 1e-12
    assert np.abs(h - h0).max() <= 1e-12


# ---------------------------------------------------------------------------------------------
# eq. 15-17: the Courant numbers c_k = S_k dt / dx inside the edge flux
# ---------------------------------------------------------------------------------------------
def test_waf_edge_flux_with_unit_ratios_is_eq17_with_c_from_dt_over_dx():
    """Upwind cells set so that every limiter ratio is exactly 1 (q_L - q_Lupw = q_R - q_L =
    q_Rupw - q_R for eta and for the velocity vector): SUPERBEE then gives A = |c| (eq. 21, middle
    branch) and the WAF flux is the paper's eq. 16-17 with weights (1 +- c_k)/2,
        G = G* + (1 + c_L)/2 (G_L - G*) + (1 - c_R)/2 (G_R - G*),   G_3 = G_1 [(1 + c_*)/2 v_L + (1 - c_*)/2 v_R],
    c_k = S_k dt / dx.  The wave speeds and G* come from the HLLC routine (pinned on its own), dx and
    the normal from the edge geometry (pinned on its own): what is checked is that the edge flux puts
    them together with THIS dt and THIS dx -- half the time step or another length fails."""
    x, y, tri = si.grid_mesh(10, 8, 10.0, 8.0, 0.2, 41)
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    c2c, _ = o.cell_topology()
    e = o.edge_geometry()
    rng = np.random.default_rng(9)
    inner = np.nonzero(e["eR"] >= 0)[0]
    checked = 0
    for ed in rng.permutation(inner):
        L, R = int(e["eL"][ed]), int(e["eR"][ed])
        upL = [int(n) for n in c2c[L] if n != R]
        upR = [int(n) for n in c2c[R] if n != L]
        if min(upL + upR) < 0 or len(set(upL + upR)) != 4:
            continue
        n1, n2, length, dx = e["nx"][ed], e["ny"][ed], e["len"][ed], e["dx"][ed]
        h = np.full(o.nt, 2.0); u = np.zeros(o.nt); v = np.zeros(o.nt)
        qL = np.array([2.0, 0.30, -0.10]); qR = np.array([1.7, 0.45, 0.05])        # (h, u, v), subcritical
        for cells, q in ((([L]), qL), ([R], qR), (upL, qL - (qR - qL)), (upR, qR + (qR - qL))):
            h[cells], u[cells], v[cells] = q
        o.set_state(h, h * u, h * v)
        unL, utL = qL[1] * n1 + qL[2] * n2, -qL[1] * n2 + qL[2] * n1                # eq. 2
        unR, utR = qR[1] * n1 + qR[2] * n2, -qR[1] * n2 + qR[2] * n1
        w = po.hllc(G, 1e-6, qL[0], unL, utL, qR[0], unR, utR)
        assert w["SL"] < 0.0 < w["SR"] and abs(w["Sstar"]) > 1e-3                   # G = G* for HLLC here
        dt = 0.4 * dx / max(abs(w["SL"]), abs(w["SR"]))
        cL, cR, cS = w["SL"] * dt / dx, w["SR"] * dt / dx, w["Sstar"] * dt / dx
        GL = np.array([qL[0] * unL, qL[0] * unL ** 2 + 0.5 * G * qL[0] ** 2])       # eq. 1, normal frame
        GR = np.array([qR[0] * unR, qR[0] * unR ** 2 + 0.5 * G * qR[0] ** 2])
        Gs = np.array([w["G1"], w["G2"]])
        Gw = Gs + 0.5 * (1.0 + cL) * (GL - Gs) + 0.5 * (1.0 - cR) * (GR - Gs)
        G3 = Gw[0] * (0.5 * (1.0 + cS) * utL + 0.5 * (1.0 - cS) * utR)
        bL = Gw[1] - 0.5 * G * qL[0] ** 2                                           # A.9, first-order faces, flat bed
        want = length * np.array([Gw[0], bL * n1 - G3 * n2, bL * n2 + G3 * n1])
        got = o.edge_flux(ed, dt, "waf")[0]
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-12 * np.abs(want).max())
        half = o.edge_flux(ed, 0.5 * dt, "waf")[0]
        assert np.abs(half - want).max() > 1e-3 * np.abs(want).max()
        checked += 1
        if checked == 10:
            break
    assert checked == 10
