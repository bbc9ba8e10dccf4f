"""The fused flux + update pass of the Heun schemes (k_cell_flux_update, swe_set_fused) against
the three-kernel pipeline: bit-identical states, clocks and time steps, un-zoned and zoned, and
against the oracle within the parity bars."""
import numpy as np
import pytest

import paper_2307_16758_b200 as sw
from oracle import pyoracle as po
from swe_inputs import config0, config1, config3, lake_case, delaunay_case, channel_flow_case
from parity import assert_parity

pytestmark = pytest.mark.gpu


def _cases():
    return {"river": config3(length=3200.0, half_width=600.0, w2=30.0, n4=4, n8=3),
            "ritter": config0(nx=100, ny=6, h_right=0.0),
            "c1": config1(n=48), "lake": lake_case(n=40), "delaunay": delaunay_case(n=1500),
            "channel": channel_flow_case(discharge=10.0, level=2.0, manning=0.03)}


@pytest.mark.parametrize("name", ["river", "ritter", "c1", "lake", "delaunay", "channel"])
@pytest.mark.parametrize("scheme", ["muscl", "muscl_ms"])
def test_fused_pass_is_bit_identical_to_the_three_kernel_pipeline(name, scheme):
    cfg = _cases()[name]
    a = sw.create_from_config(cfg)
    b = sw.create_from_config(cfg)
    try:
        sw.swe_set_fused(a, True)
        sw.swe_set_fused(b, False)
        for chunk in (1, 2, 40):                                   # kernel by kernel, then graph replay
            ta = sw.swe_step(a, chunk, 0.45, scheme)
            tb = sw.swe_step(b, chunk, 0.45, scheme)
            assert ta == tb
            for x, y in zip(sw.swe_get_state(a), sw.swe_get_state(b)):
                assert np.array_equal(x, y)
        # fewer launches: no separate update kernel
        la, lb = sw.swe_get_stats(a)["kernel_launches"], sw.swe_get_stats(b)["kernel_launches"]
        assert la < lb
        # beta = 2, unlimited, and a scheme change in between
        for beta in (2.0, 0.0):
            sw.swe_set_params(a, beta=beta)
            sw.swe_set_params(b, beta=beta)
            sw.swe_step(a, 5, 0.45, scheme); sw.swe_step(b, 5, 0.45, scheme)
            sw.swe_step(a, 3, 0.9, "hllc"); sw.swe_step(b, 3, 0.9, "hllc")
            for x, y in zip(sw.swe_get_state(a), sw.swe_get_state(b)):
                assert np.array_equal(x, y)
    finally:
        sw.swe_mesh_destroy(a)
        sw.swe_mesh_destroy(b)


@pytest.mark.parametrize("nlayers", [1, 2, 3])
def test_fused_pass_on_zones_is_bit_identical_to_the_unzoned_run(nlayers):
    cfg = _cases()["river"]
    a = sw.create_from_config(cfg)
    b = sw.create_from_config(cfg)
    try:
        sw.swe_zones_create(b, 8, nlayers)
        schemes = ["muscl"] + (["muscl_ms"] if nlayers >= 2 else [])
        for scheme in schemes:
            sw.swe_step(a, 25, 0.45, scheme)
            sw.swe_step(b, 25, 0.45, scheme)
            for x, y in zip(sw.swe_get_state(a), sw.swe_get_state(b)):
                assert np.array_equal(x, y)
    finally:
        sw.swe_mesh_destroy(a)
        sw.swe_mesh_destroy(b)


@pytest.mark.parametrize("scheme", ["muscl", "muscl_ms"])
def test_fused_pass_against_the_oracle(scheme):
    cfg = _cases()["river"]
    po.set_threads(0)
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    try:
        sw.swe_set_fused(c, True)
        for s in range(30):
            sw.swe_set_state(c, *o.get_state())
            o.step(1, 0.45, scheme)
            sw.swe_step(c, 1, 0.45, scheme)
            assert_parity(o.get_state(), sw.swe_get_state(c), 1e-11, what="fused %s step %d" % (scheme, s))
    finally:
        sw.swe_mesh_destroy(c)
        o.close()
