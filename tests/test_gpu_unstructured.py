"""GPU parity on a genuinely unstructured mesh (Delaunay triangulation, mixed windings, valence
2..11, bumpy bed with dry tops; tests/test_oracle_unstructured.py pins the oracle on it): single
passes, every step from the oracle's state, free runs, zones and ranks bit-identical, numbering
invisible."""
import numpy as np
import pytest

import paper_2307_16758_b200 as sw
from paper_2307_16758_b200 import dist as swdist
from oracle import pyoracle as po
from swe_inputs import delaunay_case
from parity import assert_parity

pytestmark = pytest.mark.gpu
SCHEMES = [("hllc", 0.9), ("muscl", 0.45), ("waf", 0.45), ("muscl_ms", 0.45)]


@pytest.fixture(autouse=True)
def _threads():
    po.set_threads(0)


@pytest.mark.parametrize("scheme,cfl", SCHEMES)
def test_per_step_and_free_run(scheme, cfl):
    cfg = delaunay_case(dam=True)
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    f = sw.create_from_config(cfg, sw.SWE_RENUM_RCM)
    try:
        assert abs(sw.swe_compute_dt(c, cfl) - o.compute_dt(cfl)) <= 4e-16 * o.compute_dt(cfl)
        for s in range(60):
            sw.swe_set_state(c, *o.get_state())
            o.step(1, cfl, scheme)
            sw.swe_step(c, 1, cfl, scheme)
            got = sw.swe_get_state(c)
            assert_parity(o.get_state(), got, 1e-11, what="delaunay %s step %d" % (scheme, s))
            assert np.array_equal(o.get_state()[0] > 1e-6, got[0] > 1e-6)
        sw.swe_step(f, 60, cfl, scheme)                   # free run from the start, other numbering
        assert_parity(o.get_state(), sw.swe_get_state(f), 1e-8, what="delaunay free run " + scheme)
    finally:
        sw.swe_mesh_destroy(c)
        sw.swe_mesh_destroy(f)
        o.close()


def test_single_passes():
    cfg = delaunay_case(dam=True)
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    try:
        o.step(20, 0.45, "muscl")
        sw.swe_set_state(c, *o.get_state())
        go, gg = o.gradients(), sw.swe_gradients(c)
        assert np.abs(gg - go).max() <= 1e-11 * max(np.abs(go).max(), 1e-3)
        dt = o.compute_dt(0.45)
        for scheme in ("hllc", "muscl", "waf", "muscl_ms"):
            ho = o.euler_stage(dt, scheme)
            hg = sw.swe_euler_stage(c, dt, scheme)
            assert_parity(ho, hg, 1e-11, what="euler stage " + scheme)
    finally:
        sw.swe_mesh_destroy(c)
        o.close()


@pytest.mark.parametrize("scheme,cfl", SCHEMES)
def test_lake_at_rest_on_the_gpu(scheme, cfl):
    cfg = delaunay_case(dam=False)
    c = sw.create_from_config(cfg)
    try:
        sw.swe_step(c, 300, cfl, scheme)
        h, hu, hv = sw.swe_get_state(c)
        wet = h > 1e-6
        assert np.array_equal(wet, cfg["h"] > 1e-6)
        assert (np.sqrt(hu[wet] ** 2 + hv[wet] ** 2) / h[wet]).max() < 1e-12
    finally:
        sw.swe_mesh_destroy(c)


@pytest.mark.parametrize("scheme,cfl,nl", [("muscl", 0.45, 2), ("hllc", 0.9, 1), ("waf", 0.45, 2), ("muscl_ms", 0.45, 3),
                                           ("muscl", 0.45, 1)])
def test_zones_and_ranks_bit_identical(scheme, cfl, nl):
    cfg = delaunay_case(dam=True)
    a = sw.create_from_config(cfg)
    b = sw.create_from_config(cfg)
    ranks = [sw.create_from_config(cfg) for _ in range(3)] if not (scheme == "muscl" and nl == 1) else []
    try:
        ta = sw.swe_step(a, 40, cfl, scheme)
        sw.swe_zones_create(b, 8, nl)
        assert sw.swe_step(b, 40, cfl, scheme) == ta
        ref = sw.swe_get_state(a)
        for x, y in zip(ref, sw.swe_get_state(b)):
            assert np.array_equal(x, y)
        if ranks:                                              # 3 ranks, 8 zones, peer-memory push
            blocks = swdist.zone_blocks(8, 3)
            for r, c in enumerate(ranks):
                sw.swe_zones_create_dist(c, 8, nl, None, 3, r, blocks)
            raw = [sw.swe_peer_raw(c) for c in ranks]
            for r, c in enumerate(ranks):
                for p in range(3):
                    if p != r:
                        sw.swe_peer_set_raw(c, p, *raw[p])
            import torch
            mins = torch.zeros(3, dtype=torch.float64, device="cuda")
            heun = scheme in ("muscl", "muscl_ms")
            for _ in range(40):
                for c in ranks:
                    sw.swe_halo_push(c, 0)
                for r, c in enumerate(ranks):
                    sw.swe_dist_local_min(c, mins[r:r + 1])
                m = mins.min().reshape(1)
                for c in ranks:
                    sw.swe_dist_begin_step(c, m, cfl)
                    sw.swe_dist_stage(c, scheme, 0)
                if heun:
                    for c in ranks:
                        sw.swe_halo_push(c, 1)
                    for c in ranks:
                        sw.swe_dist_stage(c, scheme, 1)
            out = [np.full(ref[0].size, np.nan) for _ in range(3)]
            for c in ranks:
                sw.swe_get_state(c, *out)
            for x, y in zip(ref, out):
                assert np.array_equal(x, y)
    finally:
        for c in [a, b] + ranks:
            sw.swe_mesh_destroy(c)


def test_large_delaunay_mesh_against_the_oracle():
    """The same comparison at a size that spans many thousands of tiles: a Delaunay triangulation of
    400 000 jittered points (~0.8 M triangles, valence 3-10, every third triangle clockwise, listed in
    the triangulator's order), a dam break over bumps with dry tops: per-step bar after step 1, run
    bar after 60 steps for the two Heun schemes, identical masks; then 8 zones, bit-identical."""
    cfg = delaunay_case(n=400_000, lx=4000.0, ly=2400.0, seed=5, dam=True)
    assert cfg["tri"].shape[0] > 700_000
    po.set_threads(0)
    for scheme, cfl in (("muscl", 0.45), ("muscl_ms", 0.45), ("hllc", 0.9)):
        o = po.Oracle.from_config(cfg)
        c = sw.create_from_config(cfg)
        try:
            for chunk, tol in ((1, 1e-11), (59, 1e-8)):
                o.step(chunk, cfl, scheme)
                sw.swe_step(c, chunk, cfl, scheme)
                e = assert_parity(o.get_state(), sw.swe_get_state(c), tol, what="delaunay 0.8M %s +%d" % (scheme, chunk))
                print("delaunay 0.8M %s +%d steps: %s" % (scheme, chunk, e))
            ref = sw.swe_get_state(c)
            if scheme == "muscl":
                z = sw.create_from_config(cfg)
                try:
                    sw.swe_zones_create(z, 8, 2)
                    sw.swe_step(z, 60, cfl, scheme)
                    for a, b in zip(ref, sw.swe_get_state(z)):
                        assert np.array_equal(a, b)
                finally:
                    sw.swe_mesh_destroy(z)
        finally:
            sw.swe_mesh_destroy(c)
            o.close()
