"""The oracle's whole time-step path against closed-form solutions: Stoker wet-bed dam break (the
case the paper validates on), Ritter dry-bed dam break, and observed order of
accuracy on a smooth simple wave (north_star: ~1 for HLLC, ~2 for MUSCL/WAF)."""
import os

import numpy as np
import pytest

import closed_forms as cf
import swe_inputs as si
from oracle import pyoracle as po

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def run_to(o, T, cfl, scheme):
    t = 0.0
    while True:
        dt = o.compute_dt(cfl)
        if dt <= 0 or t + dt >= T:
            return t
        t, _ = o.step(1, cfl, scheme)


def l1(cfg, h, he):
    A = cf.tri_areas(cfg["x"], cfg["y"], cfg["tri"])
    return float((np.abs(h - he) * A).sum() / A.sum())


def test_stoker_constants_match_golden():
    with open(os.path.join(GOLD, "stoker_constants.txt")) as f:
        rows = [[float(v) for v in ln.split()] for ln in f if ln.strip() and not ln.startswith("#")]
    for hL, hR, hm, um, shock, head, tail in rows:
        k = cf.stoker_constants(hL, hR)
        np.testing.assert_allclose([k["hm"], k["um"], k["shock"], k["head"], k["tail"]],
                                   [hm, um, shock, head, tail], rtol=1e-11)


def _stoker_errors(scheme, cfl, hL, hR, T, sizes=(100, 200, 400), lx=100.0):
    errs = []
    for nx in sizes:
        cfg = si.config0(nx=nx, ny=nx // 20, h_left=hL, h_right=hR)
        o = po.Oracle.from_config(cfg)
        t = run_to(o, T, cfl, scheme)
        h, hu, hv = o.get_state()
        if hR > 0:
            he, _ = cf.cell_average(lambda xm: cf.stoker(xm, t, 0.5 * lx, hL, hR), cfg["x"], cfg["y"], cfg["tri"])
        else:
            he, _ = cf.cell_average(lambda xm: cf.ritter(xm, t, 0.5 * lx, hL), cfg["x"], cfg["y"], cfg["tri"])
        errs.append(l1(cfg, h, he))
        assert h.min() >= 0.0
    return errs


def test_config0_hllc_200_steps_vs_stoker(oracle_threads):
    # configs[0] exactly: 4 000 cells, HLLC, CFL 0.9, 200 steps (L1(h) ~ 0.048 m)
    cfg = si.config0()
    o = po.Oracle.from_config(cfg)
    t, _ = o.step(200, 0.9, "hllc")
    h, hu, hv = o.get_state()
    he, hue = cf.cell_average(lambda xm: cf.stoker(xm, t, 50.0, 10.0, 1.0), cfg["x"], cfg["y"], cfg["tri"])
    assert 1.5 < t < 1.8
    assert l1(cfg, h, he) < 0.06
    assert l1(cfg, hu, hue) < 0.6
    # plateau between the rarefaction tail and the shock sits at (h_m, u_m)
    k = cf.stoker_constants(10.0, 1.0)
    cx = cfg["x"][cfg["tri"]].mean(axis=1)
    mid = (cx > 50 + (k["tail"] + 1.5) * t) & (cx < 50 + (k["shock"] - 2.0) * t)
    assert mid.sum() > 100
    assert np.abs(h[mid] - k["hm"]).max() < 0.05 * k["hm"]
    assert np.abs(hu[mid] / h[mid] - k["um"]).max() < 0.05 * k["um"]


@pytest.mark.parametrize("scheme,cfl", [("hllc", 0.9), ("muscl", 0.45), ("waf", 0.45)])
def test_stoker_convergence(scheme, cfl, oracle_threads):
    e = _stoker_errors(scheme, cfl, 10.0, 1.0, 1.5)
    orders = [np.log2(e[i] / e[i + 1]) for i in range(2)]
    assert all(0.6 < o < 1.3 for o in orders), (e, orders)   # discontinuous solution: order <= 1
    if scheme != "hllc":
        # second-order schemes are more accurate than HLLC on the same mesh
        eh = _stoker_errors("hllc", 0.9, 10.0, 1.0, 1.5, sizes=(200,))
        assert e[1] < 0.6 * eh[0]


def test_paper_own_dam_break_case(oracle_threads):
    # h = 1 | 0.5 on [0,10]x[0,1], t = 1 s
    errs = {}
    for scheme, cfl in [("hllc", 0.9), ("muscl", 0.45), ("waf", 0.45)]:
        x, y, tri = si.grid_mesh(100, 10, 10.0, 1.0, 0.1, 0)
        cx = x[tri].mean(axis=1)
        o = po.Oracle(x, y, np.zeros_like(x), tri)
        o.set_state(np.where(cx < 5.0, 1.0, 0.5), np.zeros(len(tri)), np.zeros(len(tri)))
        t = run_to(o, 1.0, cfl, scheme)
        h = o.get_state()[0]
        he, _ = cf.cell_average(lambda xm: cf.stoker(xm, t, 5.0, 1.0, 0.5), x, y, tri)
        errs[scheme] = l1({"x": x, "y": y, "tri": tri}, h, he)
    assert errs["hllc"] < 0.012
    assert errs["muscl"] < 0.6 * errs["hllc"] and errs["waf"] < 0.7 * errs["hllc"]


@pytest.mark.parametrize("scheme,cfl", [("hllc", 0.9), ("muscl", 0.45)])
def test_ritter_dry_bed(scheme, cfl, oracle_threads):
    e = _stoker_errors(scheme, cfl, 4.0, 0.0, 2.0)
    orders = [np.log2(e[i] / e[i + 1]) for i in range(2)]
    assert e[-1] < 0.03 and all(o > 0.55 for o in orders), (e, orders)


def _wave_errors(scheme, cfl, beta, jitter, sizes=(100, 200, 400)):
    errs = []
    for nx in sizes:
        cfg = si.simple_wave_case(nx, jitter=jitter)
        o = po.Oracle.from_config(cfg)
        o.set_params(beta=beta)
        t = run_to(o, 3.0, cfl, scheme)
        h = o.get_state()[0]
        he, _ = cf.cell_average(lambda xm: cf.simple_wave(xm, t), cfg["x"], cfg["y"], cfg["tri"])
        errs.append(l1(cfg, h, he))
    return errs, [np.log2(errs[i] / errs[i + 1]) for i in range(len(errs) - 1)]


@pytest.mark.parametrize("jitter", [0.0, 0.1])
def test_observed_order_hllc_is_one(jitter, oracle_threads):
    e, o = _wave_errors("hllc", 0.9, 1.0, jitter)
    assert all(0.8 < v < 1.15 for v in o), (e, o)


@pytest.mark.parametrize("beta", [0.0, 2.0])
def test_observed_order_muscl_is_two(beta, oracle_threads):
    e, o = _wave_errors("muscl", 0.45, beta, 0.1)
    assert all(1.85 < v < 2.4 for v in o), (e, o)


def test_observed_order_muscl_minmod_and_waf(oracle_threads):
    # beta=1 clips smooth extrema (order between 1 and 2); the per-edge WAF on triangles is
    # formally second order only for edge-normal flow: report as observed, > 1
    e, o = _wave_errors("muscl", 0.45, 1.0, 0.1)
    assert all(1.2 < v < 2.0 for v in o), (e, o)
    eh, _ = _wave_errors("hllc", 0.9, 1.0, 0.1, sizes=(200,))
    assert e[1] < 0.35 * eh[0]
    ew, ow = _wave_errors("waf", 0.45, 1.0, 0.1)
    assert all(v > 1.0 for v in ow), (ew, ow)
    assert ew[1] < 0.5 * eh[0]
