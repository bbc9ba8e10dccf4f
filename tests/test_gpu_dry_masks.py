"""Dry-record bit masks (swe_set_dry_masks, include/swe_b200.h): on the un-zoned mesh swe_step keeps
one bit per cell / edge for "this record holds nothing" and neither rewrites nor rereads such
records.  That is an implementation device, not a change of the scheme (SURVEY.md A.3.5, A.5-A.9:
those records are exactly zero): the run must be BIT-identical to the step that works on every
cell, through wetting and drying fronts, scheme changes, state changes between calls and graph
replay, and it must still agree with the oracle."""
import numpy as np
import pytest

import paper_2307_16758_b200 as sw
from oracle import pyoracle as po
from swe_inputs import config3, delaunay_case, lake_case
from parity import assert_parity

pytestmark = pytest.mark.gpu

SCHEMES = [("muscl", 0.45), ("hllc", 0.9), ("waf", 0.45), ("muscl_ms", 0.45)]


def _river():
    return config3(length=3200.0, half_width=600.0, w2=30.0, n4=4, n8=3)


def _bits(ctx):
    return [a.view(np.int64).copy() for a in sw.swe_get_state(ctx)]


def _same_bits(a, b, what):
    for name, u, v in zip(("h", "hu", "hv"), _bits(a), _bits(b)):
        bad = np.nonzero(u != v)[0]
        assert bad.size == 0, "%s: %s differs in %d cells (first %d)" % (what, name, bad.size, bad[0])
    assert sw.swe_get_time(a) == sw.swe_get_time(b), what


def _pair(cfg):
    a = sw.create_from_config(cfg)
    b = sw.create_from_config(cfg)
    sw.swe_set_dry_masks(a, True)                     # b: the default, every cell worked on
    return a, b


@pytest.mark.parametrize("scheme,cfl", SCHEMES)
@pytest.mark.parametrize("case", ["river", "dam_over_bumps"])
def test_masked_step_is_bit_identical(case, scheme, cfl):
    """Flood wave advancing over a dry flood plain (cells wetting) / dam break over bumps with dry
    tops (cells wetting and drying): several calls in a row, so that the masks stay live and the
    captured graph is replayed."""
    cfg = _river() if case == "river" else delaunay_case(n=4000)
    a, b = _pair(cfg)
    try:
        dry0 = int((sw.swe_get_state(a)[0] == 0.0).sum())
        assert dry0 > 200
        for n in (1, 7, 60, 2, 130):
            sw.swe_step(a, n, cfl, scheme)
            sw.swe_step(b, n, cfl, scheme)
            _same_bits(a, b, "%s %s after a call of %d steps" % (case, scheme, n))
        if case == "river":
            h = sw.swe_get_state(a)[0]
            assert int((h == 0.0).sum()) != dry0        # the flood front has moved over dry cells
    finally:
        sw.swe_mesh_destroy(a)
        sw.swe_mesh_destroy(b)


def test_masks_survive_everything_between_calls():
    """Scheme changes (the gradient buffer holds other records for the multislope pass), parameter
    and boundary changes, a state written by the user (water poured onto dry cells, water removed,
    momentum and negative zeros left in dry cells), zones built and removed, the single passes of
    the test interface, graph replay switched off and on: after each the next steps equal those of
    the context without masks."""
    cfg = _river()
    a, b = _pair(cfg)
    rng = np.random.default_rng(11)
    try:
        def both(f):
            f(a); f(b)

        def steps(scheme, cfl, n):
            both(lambda c: sw.swe_step(c, n, cfl, scheme))
            _same_bits(a, b, "%s x %d" % (scheme, n))

        steps("muscl", 0.45, 9)
        steps("muscl_ms", 0.45, 5)
        steps("muscl", 0.45, 6)
        steps("waf", 0.45, 4)
        steps("hllc", 0.9, 8)
        steps("muscl", 0.45, 3)
        both(lambda c: sw.swe_set_params(c, beta=2.0))
        steps("muscl", 0.45, 5)
        h, hu, hv = [x.copy() for x in sw.swe_get_state(a)]
        dry = np.nonzero(h == 0.0)[0]
        wet = np.nonzero(h > 0.1)[0]
        assert dry.size > 200 and wet.size > 200
        h[rng.choice(dry, 50, replace=False)] = 0.3                 # water poured onto dry cells
        gone = rng.choice(wet, 50, replace=False)
        h[gone] = 0.0                                                # water removed, momentum left behind
        left = rng.choice(dry, 80, replace=False)
        hu[left[:40]] = rng.normal(size=40)                          # momentum in cells without water
        hv[left[40:]] = -0.0                                         # negative zeros
        both(lambda c: sw.swe_set_state(c, h, hu, hv))
        steps("muscl", 0.45, 4)
        steps("muscl", 0.45, 30)
        both(lambda c: sw.swe_set_bc(c, 1, "inflow", 300.0))
        steps("muscl", 0.45, 10)
        both(lambda c: sw.swe_gradients(c))
        both(lambda c: sw.swe_euler_stage(c, 1e-3, "muscl"))
        steps("muscl", 0.45, 10)
        both(lambda c: sw.swe_zones_create(c, 4, 2))
        steps("muscl", 0.45, 5)
        both(lambda c: sw.swe_zones_create(c, 0, 1))
        steps("muscl", 0.45, 10)
        both(lambda c: sw.swe_set_graphs(c, False))
        steps("muscl", 0.45, 10)
        both(lambda c: sw.swe_set_graphs(c, True))
        steps("hllc", 0.9, 10)
        sw.swe_set_dry_masks(a, False)                               # and the switch itself
        steps("muscl", 0.45, 5)
        sw.swe_set_dry_masks(a, True)
        steps("muscl", 0.45, 12)
    finally:
        sw.swe_mesh_destroy(a)
        sw.swe_mesh_destroy(b)


@pytest.mark.parametrize("scheme,cfl", SCHEMES)
def test_masked_free_run_against_the_oracle(scheme, cfl):
    """The masked step over a wetting / drying front against the oracle's free run (1e-8), with the
    masks live from the second step on."""
    cfg = delaunay_case(n=2500)
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    sw.swe_set_dry_masks(c, True)
    try:
        o.step(60, cfl, scheme)
        sw.swe_step(c, 60, cfl, scheme)
        assert_parity(o.get_state(), sw.swe_get_state(c), 1e-8, what="masked %s" % scheme)
        # one more step from the oracle's own state: the per-step bound with a fresh set of masks
        sw.swe_set_state(c, *o.get_state())
        o.step(1, cfl, scheme)
        sw.swe_step(c, 1, cfl, scheme)
        assert_parity(o.get_state(), sw.swe_get_state(c), 1e-11, what="masked %s, one step" % scheme)
    finally:
        sw.swe_mesh_destroy(c)
        o.close()


def test_lake_at_rest_all_quiet_cells_are_left_alone():
    """configs[2]-like lake: the dry bump tops are never touched, the wet part stays at rest; the
    launch count is that of the unmasked step (same kernels, only less work inside)."""
    cfg = lake_case(n=60)
    a, b = _pair(cfg)
    try:
        for scheme, cfl in SCHEMES:
            sw.swe_step(a, 40, cfl, scheme)
            sw.swe_step(b, 40, cfl, scheme)
            _same_bits(a, b, "lake %s" % scheme)
        assert sw.swe_get_stats(a) == sw.swe_get_stats(b)
        h, hu, hv = sw.swe_get_state(a)
        assert np.abs(hu[h > 1e-6] / h[h > 1e-6]).max() <= 1e-12
    finally:
        sw.swe_mesh_destroy(a)
        sw.swe_mesh_destroy(b)
