"""Pins of the oracle's multislope MUSCL (the paper's own MUSCL, eq. 22-25, PAPER.md:396-420;
scope row f1, reading R17): textbook limiter values, closed forms (Stoker, Ritter, exact
simple wave), invariants (C-property, mass, positivity, zoned == un-zoned)."""
import os

import numpy as np
import pytest

import closed_forms as cf
import swe_inputs as si
from oracle import pyoracle as po

HERE = os.path.dirname(os.path.abspath(__file__))


def l1(cfg, a, b):
    A = cf.tri_areas(cfg["x"], cfg["y"], cfg["tri"])
    return float(np.sum(A * np.abs(a - b)) / np.sum(A))


def run_to(o, T, cfl, scheme):
    t = 0.0
    while True:
        dt = o.compute_dt(cfl)
        if t + dt >= T or dt == 0.0:
            return t
        t, _ = o.step(1, cfl, scheme)


def test_limited_slope_reproduces_minbee_and_superbee():
    rows = [ln.split() for ln in open(os.path.join(HERE, "golden", "minbee_superbee_slope.txt"))
            if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 9
    for r, mb, sb in rows:
        r, mb, sb = float(r), float(mb), float(sb)
        for scale in (1.0, 0.37, 12.5):                      # homogeneous of degree one
            assert po.ms_slope(1.0, r * scale, scale) == pytest.approx(mb * scale, abs=1e-15)
            assert po.ms_slope(2.0, r * scale, scale) == pytest.approx(sb * scale, abs=1e-15)
            # negative local slope: mirror image (eq. 24, second case)
            assert po.ms_slope(1.0, -r * scale, -scale) == pytest.approx(-mb * scale, abs=1e-15)
            assert po.ms_slope(2.0, -r * scale, -scale) == pytest.approx(-sb * scale, abs=1e-15)
    assert po.ms_slope(2.0, 3.0, 0.0) == 0.0                 # flat local slope: no reconstruction
    rng = np.random.default_rng(0)
    for x, y in rng.normal(size=(200, 2)):                   # symmetric in its two slopes
        for beta in (1.0, 1.5, 2.0):
            assert po.ms_slope(beta, x, y) == po.ms_slope(beta, y, x)
            if x * y <= 0:
                assert po.ms_slope(beta, x, y) == 0.0
            else:                                            # between minmod and the larger slope
                lo, hi = min(abs(x), abs(y)), max(abs(x), abs(y))
                assert lo - 1e-15 <= abs(po.ms_slope(beta, x, y)) <= hi + 1e-15


@pytest.mark.parametrize("beta,jitter", [(2.0, 0.0), (2.0, 0.1), (1.0, 0.1)])
def test_observed_order_on_exact_simple_wave(beta, jitter, oracle_threads):
    errs = []
    for nx in (100, 200, 400):
        cfg = si.simple_wave_case(nx, jitter=jitter)
        o = po.Oracle.from_config(cfg)
        o.set_params(beta=beta)
        t = run_to(o, 3.0, 0.45, "muscl_ms")
        he, _ = cf.cell_average(lambda xm: cf.simple_wave(xm, t), cfg["x"], cfg["y"], cfg["tri"])
        errs.append(l1(cfg, o.get_state()[0], he))
        o.close()
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(1.4 < v < 2.2 for v in orders), (errs, orders)     # limited second order
    cfg = si.simple_wave_case(200, jitter=jitter)
    o = po.Oracle.from_config(cfg)
    t = run_to(o, 3.0, 0.9, "hllc")
    he, _ = cf.cell_average(lambda xm: cf.simple_wave(xm, t), cfg["x"], cfg["y"], cfg["tri"])
    assert errs[1] < 0.4 * l1(cfg, o.get_state()[0], he)         # far more accurate than HLLC


def test_stoker_and_ritter(oracle_threads):
    # "WAF and MUSCL more accurate than HLLC" on the paper's validation case
    e = {}
    for scheme, cfl, beta in (("hllc", 0.9, 1.0), ("muscl_ms", 0.45, 2.0), ("muscl_ms", 0.45, 1.0)):
        cfg = si.config0()
        o = po.Oracle.from_config(cfg)
        o.set_params(beta=beta)
        A = o.cell_geometry()["area"]
        t = run_to(o, 1.5, cfl, scheme)
        h = o.get_state()[0]
        he, _ = cf.cell_average(lambda xm: cf.stoker(xm, t, 50.0, 10.0, 1.0), cfg["x"], cfg["y"], cfg["tri"])
        e[(scheme, beta)] = l1(cfg, h, he)
        assert abs(np.sum(h * A) - np.sum(cfg["h"] * A)) <= 1e-13 * np.sum(cfg["h"] * A)
        if beta == 1.0:
            assert h.min() >= 1.0 - 1e-9 and h.max() <= 10.0 + 1e-9      # MINBEE is monotone here
        o.close()
    assert e[("muscl_ms", 2.0)] < 0.4 * e[("hllc", 1.0)] and e[("muscl_ms", 1.0)] < 0.6 * e[("hllc", 1.0)]
    cfg = si.config0(nx=200, ny=10, h_right=0.0, h_left=4.0)
    o = po.Oracle.from_config(cfg)
    o.set_params(beta=2.0)
    A = o.cell_geometry()["area"]
    t = run_to(o, 2.0, 0.45, "muscl_ms")
    h = o.get_state()[0]
    he, _ = cf.cell_average(lambda xm: cf.ritter(xm, t, 50.0, 4.0), cfg["x"], cfg["y"], cfg["tri"])
    assert h.min() >= 0.0 and l1(cfg, h, he) < 0.008
    assert abs(np.sum(h * A) - np.sum(cfg["h"] * A)) <= 1e-13 * np.sum(cfg["h"] * A)


@pytest.mark.parametrize("level", [5.0, np.pi + 1.7])
def test_c_property_and_mass(level, oracle_threads):
    cfg = si.lake_case(n=40, level=level)
    o = po.Oracle.from_config(cfg)
    A = o.cell_geometry()["area"]
    m0 = np.sum(cfg["h"] * A)
    o.step(300, 0.45, "muscl_ms")
    h, hu, hv = o.get_state()
    w = h > 1e-6
    assert np.array_equal(w, cfg["h"] > 1e-6)
    assert (np.sqrt(hu[w] ** 2 + hv[w] ** 2) / h[w]).max() <= 1e-12
    assert abs(np.sum(h * A) - m0) <= 1e-14 * m0


def test_uniform_state_is_first_order_exact_and_zones_are_invisible(oracle_threads):
    # a uniform flow between walls parallel to it: every slope is zero, so the scheme returns the
    # first-order HLLC update bit for bit
    cfg = si.config0(nx=40, ny=4)
    a = po.Oracle.from_config(cfg)
    b = po.Oracle.from_config(cfg)
    for o in (a, b):
        o.set_state(np.full(a.nt, 2.0), np.zeros(a.nt), np.zeros(a.nt))
    a.step(5, 0.45, "hllc")
    b.step(5, 0.45, "muscl_ms")
    assert np.array_equal(a.get_state()[0], b.get_state()[0])
    # zoned run with two ghost layers == un-zoned run, bit for bit
    cfg = si.config3(length=1600.0, half_width=400.0, w2=20.0, n4=3, n8=2)
    u = po.Oracle.from_config(cfg)
    z = po.Oracle.from_config(cfg)
    z.zones_create(4, 2)
    u.step(20, 0.45, "muscl_ms")
    z.zones_step(20, 0.45, "muscl_ms")
    for x, y in zip(u.get_state(), z.get_state()):
        assert np.array_equal(x, y)
    z1 = po.Oracle.from_config(cfg)
    z1.zones_create(4, 1)
    with pytest.raises(ValueError):
        z1.zones_step(1, 0.45, "muscl_ms")               # needs two layers
