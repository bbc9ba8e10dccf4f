"""The oracle's invariants on a genuinely unstructured mesh (Delaunay triangulation of random points:
vertex valence 2..11, every third triangle clockwise, no grid structure anywhere) over a bumpy bed
with dry bump tops -- the paper's meshes are of this kind, the five configs
are triangulated lattices.  C-property, mass conservation, positivity, zoned == un-zoned, rotation."""
import numpy as np
import pytest

import closed_forms as cf
import swe_inputs as si
from oracle import pyoracle as po

SCHEMES = [("hllc", 0.9), ("muscl", 0.45), ("waf", 0.45), ("muscl_ms", 0.45)]


def test_the_mesh_is_unstructured():
    c = si.delaunay_case()
    tri = c["tri"]
    val = np.bincount(tri.ravel())
    assert val.min() <= 3 and val.max() >= 9 and len(np.unique(val)) >= 6
    a = cf.tri_areas(c["x"], c["y"], tri)
    assert abs(a.sum() - 200.0 * 120.0) < 1e-9 * 24000.0           # covers the rectangle exactly once
    x, y = c["x"], c["y"]
    signed = 0.5 * ((x[tri[:, 1]] - x[tri[:, 0]]) * (y[tri[:, 2]] - y[tri[:, 0]])
                    - (y[tri[:, 1]] - y[tri[:, 0]]) * (x[tri[:, 2]] - x[tri[:, 0]]))
    assert (signed < 0).sum() > 0.3 * tri.shape[0] and (signed > 0).sum() > 0.6 * tri.shape[0]
    assert 0.1 < (c["h"] == 0.0).mean() < 0.3


@pytest.mark.parametrize("scheme,cfl", SCHEMES)
def test_lake_at_rest_stays_at_rest(scheme, cfl, oracle_threads):
    c = si.delaunay_case(dam=False)
    o = po.Oracle.from_config(c)
    o.step(300, cfl, scheme)
    h, hu, hv = o.get_state()
    wet = h > 1e-6
    vel = np.sqrt(hu[wet] ** 2 + hv[wet] ** 2) / h[wet]
    assert vel.max() < 1e-12
    assert np.array_equal(wet, c["h"] > 1e-6)                        # the shoreline does not move
    zc = c["zb"][c["tri"]].mean(axis=1)
    assert np.abs((h + zc)[wet] - 3.0).max() < 1e-12


@pytest.mark.parametrize("scheme,cfl", SCHEMES)
def test_dam_break_over_bumps_conserves_mass_and_stays_positive(scheme, cfl, oracle_threads):
    c = si.delaunay_case(dam=True)
    area = cf.tri_areas(c["x"], c["y"], c["tri"])
    o = po.Oracle.from_config(c)
    m0 = float((c["h"] * area).sum())
    for _ in range(3):
        o.step(100, cfl, scheme)
        h, hu, hv = o.get_state()
        assert h.min() >= 0.0
        assert abs(float((h * area).sum()) - m0) < 2e-13 * m0
    assert np.abs(h - c["h"]).max() > 0.5   # the wave has run over the bumps
    assert np.sqrt(hu ** 2 + hv ** 2).max() > 1.0


@pytest.mark.parametrize("scheme,cfl,layers", [("hllc", 0.9, 1), ("muscl", 0.45, 1), ("muscl", 0.45, 2), ("waf", 0.45, 2),
                                               ("muscl_ms", 0.45, 2), ("muscl", 0.45, 3)])
def test_zoned_equals_unzoned(scheme, cfl, layers, oracle_threads):
    c = si.delaunay_case(n=1500, dam=True)
    a = po.Oracle.from_config(c)
    b = po.Oracle.from_config(c)
    ta = a.step(40, cfl, scheme)
    b.zones_create(8, layers)
    tb = b.zones_step(40, cfl, scheme)
    assert ta == tb
    for u, v in zip(a.get_state(), b.get_state()):
        assert np.array_equal(u, v)


@pytest.mark.parametrize("scheme,cfl", [("muscl", 0.45), ("hllc", 0.9)])
def test_rotating_the_problem_rotates_the_solution(scheme, cfl, oracle_threads):
    # (MUSCL with the limiter off: the cell limiter bounds u and v component by component, which
    # depends on the frame by construction -- tests/test_oracle_invariants.py)
    c = si.delaunay_case(n=1500, dam=True)
    c["params"] = dict(c["params"], beta=0.0 if scheme == "muscl" else c["params"]["beta"])
    th = 0.7
    cs, sn = np.cos(th), np.sin(th)
    r = dict(c)
    r["x"] = np.ascontiguousarray(cs * c["x"] - sn * c["y"])
    r["y"] = np.ascontiguousarray(sn * c["x"] + cs * c["y"])
    a = po.Oracle.from_config(c)
    b = po.Oracle.from_config(r)
    a.step(40, cfl, scheme)
    b.step(40, cfl, scheme)
    ha, hua, hva = a.get_state()
    hb, hub, hvb = b.get_state()
    assert np.abs(ha - hb).max() < 1e-11 * ha.max()
    q = max(np.abs(hua).max(), np.abs(hva).max())
    assert np.abs(cs * hua - sn * hva - hub).max() < 1e-11 * q
    assert np.abs(sn * hua + cs * hva - hvb).max() < 1e-11 * q
