"""Pins of the oracle's mesh geometry, least-squares gradient, cell limiter and CFL time step
 against textbook geometry, exactness properties and brute force."""
import numpy as np
import pytest

import swe_inputs as si
from oracle import pyoracle as po


def _mesh(nx=12, ny=9, jitter=0.25, seed=5, permute=True):
    x, y, tri = si.grid_mesh(nx, ny, 6.0, 4.5, jitter, seed, permute)
    return x, y, tri


def test_areas_centroids_inradius_textbook():
    x, y, tri = _mesh()
    # flip the winding of every other triangle: the library must orient them itself
    tri = tri.copy()
    tri[::2] = tri[::2][:, [0, 2, 1]]
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    g = o.cell_geometry()
    assert g["area"].sum() == pytest.approx(6.0 * 4.5, rel=1e-13)
    assert np.all(g["area"] > 0)
    # Heron's formula and r = Area / semi-perimeter (inscribed circle)
    p = np.stack([x[tri], y[tri]], axis=-1)
    a = np.linalg.norm(p[:, 1] - p[:, 2], axis=1)
    b = np.linalg.norm(p[:, 2] - p[:, 0], axis=1)
    c = np.linalg.norm(p[:, 0] - p[:, 1], axis=1)
    s = 0.5 * (a + b + c)
    heron = np.sqrt(s * (s - a) * (s - b) * (s - c))
    np.testing.assert_allclose(g["area"], heron, rtol=1e-11)
    np.testing.assert_allclose(g["rin"], heron / s, rtol=1e-11)
    np.testing.assert_allclose(g["cx"], p[:, :, 0].mean(axis=1), rtol=1e-14)
    assert o.min_inradius == g["rin"].min()


def test_right_triangle_inradius_closed_form():
    # legs 3,4, hypotenuse 5: r = (3+4-5)/2 = 1
    x = np.array([0.0, 3.0, 0.0, 3.0])
    y = np.array([0.0, 0.0, 4.0, 4.0])
    tri = np.array([[0, 1, 2], [1, 3, 2]], np.int32)
    o = po.Oracle(x, y, np.zeros(4), tri)
    np.testing.assert_allclose(o.cell_geometry()["rin"], [1.0, 1.0], rtol=1e-15)


def test_edge_normals_unit_outward_and_closed():
    x, y, tri = _mesh()
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    g, e = o.cell_geometry(), o.edge_geometry()
    np.testing.assert_allclose(e["nx"] ** 2 + e["ny"] ** 2, 1.0, rtol=1e-14)
    inner = e["eR"] >= 0
    L, R = e["eL"][inner], e["eR"][inner]
    assert np.all(L < R)                      # A.1.4: L-cell = smaller user id
    d = (g["cx"][R] - g["cx"][L]) * e["nx"][inner] + (g["cy"][R] - g["cy"][L]) * e["ny"][inner]
    assert np.all(d > 0)                      # normal points from L to R
    np.testing.assert_allclose(e["dx"][inner], d, rtol=1e-12)   # A.1.6 projected centroid distance
    # Euler: V - E + F = 1 for a disc
    assert x.size - o.ne + o.nt == 1
    # closed cells: sum_k L_k n_out,k = 0  (needed by the regrouped bed-slope term, reading R12)
    c2c, c2e = o.cell_topology()
    sx = np.zeros(o.nt)
    sy = np.zeros(o.nt)
    for k in range(3):
        ed = c2e[:, k]
        sgn = np.where(e["eL"][ed] == np.arange(o.nt), 1.0, -1.0)
        sx += sgn * e["len"][ed] * e["nx"][ed]
        sy += sgn * e["len"][ed] * e["ny"][ed]
    assert np.abs(sx).max() < 1e-13 and np.abs(sy).max() < 1e-13


def test_mesh_errors():
    x = np.array([0.0, 1.0, 2.0, 0.0])
    y = np.array([0.0, 0.0, 0.0, 1.0])
    with pytest.raises(ValueError):
        po.Oracle(x, y, np.zeros(4), np.array([[0, 1, 2]], np.int32))          # zero area
    with pytest.raises(ValueError):
        po.Oracle(x, y, np.zeros(4), np.array([[0, 1, 7]], np.int32))          # bad index
    with pytest.raises(ValueError):                                            # non-manifold edge
        po.Oracle(np.array([0.0, 1.0, 0.0, 1.0, 0.5]), np.array([0.0, 0.0, 1.0, 1.0, -1.0]), np.zeros(5),
                  np.array([[0, 1, 2], [0, 1, 3], [0, 1, 4]], np.int32))


def test_lsq_gradient_exact_for_linear_fields():
    # A.1.7 / A.3: the unlimited (beta<=0) LSQ gradient reproduces a linear field exactly on any
    # mesh (interior cells; boundary cells use a mirror value and are excluded)
    x, y, tri = _mesh(jitter=0.3)
    zb = 0.3 * x - 0.2 * y                       # linear bed
    o = po.Oracle(x, y, zb, tri)
    o.set_params(beta=0.0)
    g = o.cell_geometry()
    cx, cy = g["cx"], g["cy"]
    eta = 5.0 + 0.11 * cx + 0.07 * cy
    h = eta - g["zc"]
    u = 0.4 - 0.05 * cx + 0.02 * cy
    v = -0.1 + 0.03 * cx + 0.06 * cy
    o.set_state(h, h * u, h * v)
    gr = o.gradients()
    c2c, _ = o.cell_topology()
    interior = np.all(c2c >= 0, axis=1)
    assert interior.sum() > 50
    expect = np.array([0.11, 0.07, 0.11 - 0.3, 0.07 + 0.2, -0.05, 0.02, 0.03, 0.06])
    np.testing.assert_allclose(gr[interior], np.broadcast_to(expect, gr[interior].shape), atol=2e-12)


def _four_triangle_stencil(F, B, beta):
    """Central triangle whose neighbour centroids sit at (+1,0), (-1,0), (0,-delta) from its own,
    data varying in x only: a uniform 1-D stencil of cell width 1 (faces at +-1/2)."""
    hgt = 1.2
    P0, P1, P2 = (-1.0, 0.0), (1.0, 0.0), (0.0, hgt)
    Q0 = (0.0, hgt - 3.0 * 0.9)       # neighbour across the base
    Q1 = (2.0, 0.0)
    Q2 = (-2.0, 0.0)
    x = np.array([P0[0], P1[0], P2[0], Q0[0], Q1[0], Q2[0]])
    y = np.array([P0[1], P1[1], P2[1], Q0[1], Q1[1], Q2[1]])
    tri = np.array([[0, 1, 2], [0, 1, 3], [1, 2, 4], [2, 0, 5]], np.int32)
    o = po.Oracle(x, y, np.zeros(6), tri)
    o.set_params(beta=beta)
    q = 3.0
    h = np.array([q, q, q + F, q - B])      # centre, below (same x), right, left
    o.set_state(h, np.zeros(4), np.zeros(4))
    g = o.cell_geometry()
    assert g["cx"][2] - g["cx"][0] == pytest.approx(1.0) and g["cx"][3] - g["cx"][0] == pytest.approx(-1.0)
    assert g["cx"][1] == pytest.approx(g["cx"][0])
    return o.gradients()[0]


def _minmod(a, b):
    return 0.0 if a * b <= 0 else (min(a, b) if a > 0 else max(a, b))


def test_cell_limiter_reduces_to_minmod_on_1d_stencil():
    # beta=1 (MINBEE): limited slope = minmod(forward, backward) difference
    for F, B in [(0.4, 0.1), (0.1, 0.4), (0.3, 0.3), (-0.2, -0.5), (0.3, -0.2), (-0.1, 0.2), (0.0, 0.3)]:
        gr = _four_triangle_stencil(F, B, 1.0)
        assert gr[2] == pytest.approx(_minmod(F, B), abs=1e-14), (F, B)   # dh/dx
        assert gr[3] == pytest.approx(0.0, abs=1e-14)
        assert gr[0] == pytest.approx(gr[2], abs=1e-14)                   # eta = h on a flat bed
    # beta<=0: unlimited central slope
    gr = _four_triangle_stencil(0.4, 0.1, 0.0)
    assert gr[2] == pytest.approx(0.25, abs=1e-14)
    # beta=2 (Barth-Jespersen bound): min(central, 2F, 2B)
    gr = _four_triangle_stencil(0.4, 0.05, 2.0)
    assert gr[2] == pytest.approx(0.1, abs=1e-14)


def test_cell_limiter_bound_property_and_dry_fallback():
    x, y, tri = _mesh(20, 15, 0.2, 9)
    rng = np.random.default_rng(3)
    o = po.Oracle(x, y, np.zeros_like(x), tri)
    h = rng.uniform(0.5, 2.0, o.nt)
    u = rng.uniform(-1, 1, o.nt)
    v = rng.uniform(-1, 1, o.nt)
    dry = rng.random(o.nt) < 0.03
    h[dry] = 0.0
    o.set_state(h, h * u, h * v)
    c2c, c2e = o.cell_topology()
    g = o.cell_geometry()
    e = o.edge_geometry()
    for beta in (1.0, 2.0):
        o.set_params(beta=beta)
        gr = o.gradients()
        wet = h > 1e-6
        nb_ok = np.ones(o.nt, bool)
        for k in range(3):
            nb = c2c[:, k]
            nb_ok &= np.where(nb >= 0, wet[np.maximum(nb, 0)], True)
        front = ~(wet & nb_ok)
        assert np.all(gr[front] == 0.0)              # A.3.5 first order at wet/dry fronts
        # face increments stay within kappa x (distance to the neighbourhood extremum), q = h
        qmax = h.copy()
        qmin = h.copy()
        for k in range(3):
            nb = c2c[:, k]
            val = np.where(nb >= 0, h[np.maximum(nb, 0)], h)
            qmax = np.maximum(qmax, val)
            qmin = np.minimum(qmin, val)
        # edge midpoints from the mesh
        t = o.tri
        for k in range(3):
            mx = 0.5 * (x[t[:, k]] + x[t[:, (k + 1) % 3]])
            my = 0.5 * (y[t[:, k]] + y[t[:, (k + 1) % 3]])
            # the oracle may have re-oriented a triangle: the set of three midpoints is the same
            inc = gr[:, 2] * (mx - g["cx"]) + gr[:, 3] * (my - g["cy"])
            assert np.all(inc <= 0.5 * beta * (qmax - h) + 1e-13)
            assert np.all(inc >= 0.5 * beta * (qmin - h) - 1e-13)


def test_cfl_time_step_is_brute_force_minimum():
    # eq. 5 with d = in-circle radius (reading R5)
    cfg = si.lake_case(n=30)
    o = po.Oracle.from_config(cfg)
    rng = np.random.default_rng(4)
    h = cfg["h"].copy()
    u = rng.uniform(-2, 2, o.nt)
    v = rng.uniform(-2, 2, o.nt)
    o.set_state(h, h * u, h * v)
    x, y, tri = cfg["x"], cfg["y"], cfg["tri"]
    p = np.stack([x[tri], y[tri]], axis=-1)
    per = sum(np.linalg.norm(p[:, k] - p[:, (k + 1) % 3], axis=1) for k in range(3))
    a_, b_ = p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]
    area = 0.5 * np.abs(a_[:, 0] * b_[:, 1] - a_[:, 1] * b_[:, 0])
    rin = 2.0 * area / per
    wet = h > 1e-6
    assert 0 < wet.sum() < o.nt
    lam = np.sqrt(9.81 * h[wet]) + np.sqrt(u[wet] ** 2 + v[wet] ** 2)
    assert o.compute_dt(0.9) == pytest.approx(0.9 * np.min(rin[wet] / lam), rel=1e-13)
    o.set_state(np.zeros(o.nt), np.zeros(o.nt), np.zeros(o.nt))
    assert o.compute_dt(0.9) == 0.0
    t, dt = o.step(3, 0.9, "hllc")      # all dry: no-op
    assert (t, dt) == (0.0, 0.0)
