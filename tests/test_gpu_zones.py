"""configs[4]: zone decomposition resident on one GPU with ghost layers and device-side
pack / unpack.  The zoned run must be BIT-identical to the un-zoned run (with two
ghost layers the decomposed MUSCL solution is exactly the undecomposed one), and both agree with
the oracle's own zoned run."""
import numpy as np
import pytest

import paper_2307_16758_b200 as sw
from oracle import pyoracle as po
from swe_inputs import config1, config3, lake_case
from parity import assert_parity

pytestmark = pytest.mark.gpu


def _river():
    return config3(length=3200.0, half_width=600.0, w2=30.0, n4=4, n8=3)


@pytest.mark.parametrize("nz,nl", [(4, 1), (8, 2), (32, 2), (4, 3)])
@pytest.mark.parametrize("scheme,cfl", [("muscl", 0.45), ("hllc", 0.9), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_zoned_run_is_bit_identical(nz, nl, scheme, cfl):
    cfg = _river()
    a = sw.create_from_config(cfg)
    b = sw.create_from_config(cfg)
    try:
        sw.swe_zones_create(b, nz, nl)
        if scheme in ("waf", "muscl_ms") and nl < 2:
            with pytest.raises(sw.SweError) as e:
                sw.swe_step(b, 1, cfl, scheme)
            assert e.value.code == sw.SWE_ERR_STATE
            return
        ta = sw.swe_step(a, 40, cfl, scheme)
        tb = sw.swe_step(b, 40, cfl, scheme)
        assert ta == tb
        for x, y in zip(sw.swe_get_state(a), sw.swe_get_state(b)):
            assert np.array_equal(x, y)
        # removing the zones keeps the state
        sw.swe_zones_create(b, 0, 1)
        for x, y in zip(sw.swe_get_state(a), sw.swe_get_state(b)):
            assert np.array_equal(x, y)
    finally:
        sw.swe_mesh_destroy(a)
        sw.swe_mesh_destroy(b)


def test_zoned_run_matches_zoned_oracle():
    cfg = config1(n=48)
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    try:
        o.zones_create(8, 2)
        sw.swe_zones_create(c, 8, 2)
        o.zones_step(30, 0.45, "muscl")
        sw.swe_step(c, 30, 0.45, "muscl")
        assert_parity(o.get_state(), sw.swe_get_state(c), 1e-8, what="zoned c1")
        st, so = sw.swe_zone_stats(c), o.zones_counts()
        assert st == so
    finally:
        sw.swe_mesh_destroy(c)
        o.close()


def test_pack_unpack_move_the_right_cells():
    """After set_state the ghosts are filled; corrupt nothing, but check pack -> unpack is the
    identity on a consistent state and that per-zone calls equal the all-zones call."""
    cfg = lake_case(n=40)
    c = sw.create_from_config(cfg)
    try:
        sw.swe_zones_create(c, 4, 2)
        d = [sw.swe_zone_describe(c, z) for z in range(4)]
        # structure: send lists index owned cells of the source, receive ranges are ghost blocks
        for z in range(4):
            pos = d[z]["nowned"]
            for src, start, cnt, sl in d[z]["links"]:
                assert start == pos and src != z
                pos += cnt
                assert np.all(sl < d[src]["nowned"])
                assert np.array_equal(d[src]["cells"][sl], d[z]["cells"][start:start + cnt])
            assert pos == len(d[z]["cells"])
        s0 = sw.swe_get_stats(c)["halo_bytes"]
        sw.swe_pack_ghosts(c, -1)
        sw.swe_unpack_ghosts(c, -1)
        for z in range(4):
            sw.swe_pack_ghosts(c, z)
        for z in range(4):
            sw.swe_unpack_ghosts(c, z)
        assert sw.swe_get_stats(c)["halo_bytes"] == s0 + 2 * sw.swe_zone_stats(c)["send_cells_total"] * 128
        ref = sw.create_from_config(cfg)
        sw.swe_step(ref, 5, 0.45, "muscl")
        sw.swe_step(c, 5, 0.45, "muscl")
        for x, y in zip(sw.swe_get_state(ref), sw.swe_get_state(c)):
            assert np.array_equal(x, y)
        sw.swe_mesh_destroy(ref)
    finally:
        sw.swe_mesh_destroy(c)


def test_config4_full_bit_identity():
    """configs[4] at full size: ~13 M cells, 32 zones by recursive coordinate bisection,
    1, 2 and 3 ghost layers; 3 MUSCL-RK2 steps bit-identical to the un-zoned run."""
    cfg = config3()
    a = sw.create_from_config(cfg)
    try:
        sw.swe_step(a, 3, 0.45, "muscl")
        ref = sw.swe_get_state(a)
        sw.swe_set_state(a, cfg["h"], cfg["hu"], cfg["hv"])
        prev = None
        for nl in (1, 2, 3):
            sw.swe_zones_create(a, 32, nl)
            sw.swe_set_state(a, cfg["h"], cfg["hu"], cfg["hv"])
            sw.swe_step(a, 3, 0.45, "muscl")
            for x, y in zip(ref, sw.swe_get_state(a)):
                assert np.array_equal(x, y)
            st = sw.swe_zone_stats(a)
            assert st["bytes_per_exchange"] == 24 * st["send_cells_total"]
            if prev is not None:
                assert st["send_cells_total"] > prev
            prev = st["send_cells_total"]
    finally:
        sw.swe_mesh_destroy(a)


# ---- row f4: ghost layers and their numbering generated on the device ----
def _zone_assignments(nt, cx):
    rng = np.random.default_rng(7)
    return {
        "rcb4": (4, None), "rcb32": (32, None), "one": (1, None),
        # every cell in a random zone of 70: masks of two 64-bit words, nearly every cell is a
        # ghost of several zones, several radix-sort tiles
        "random70": (70, rng.integers(0, 70, nt).astype(np.int32)),
        # thin stripes along x: with 3 layers ghosts come from non-adjacent zones too
        "stripes130": (130, np.minimum(129, (130 * (cx - cx.min()) / (np.ptp(cx) + 1e-9)).astype(np.int32))),
        "two": (2, (rng.random(nt) < 0.5).astype(np.int32)),
    }


@pytest.mark.parametrize("name", ["rcb4", "rcb32", "one", "random70", "stripes130", "two"])
@pytest.mark.parametrize("nl", [1, 2, 3])
def test_device_ghost_layers_match_host_search_and_oracle(name, nl):
    """swe_zones_create builds the ghost layers on the device (mask wavefronts + radix sort).
    They must equal, array for array, the host breadth-first search of the set-up inspection
    entry points (same numbering, so the order of A.12.3 is checked exactly), and, as sets per
    zone / layer / source zone, the oracle's independent zone builder."""
    from swe_inputs import delaunay_case
    cfg = delaunay_case(n=6000) if name in ("random70", "two") else _river()
    tri = cfg["tri"].reshape(-1, 3)
    cx = cfg["x"][tri].mean(axis=1)
    nz, zone_of = _zone_assignments(tri.shape[0], cx)[name]
    c = sw.create_from_config(cfg)
    h = sw.swe_host_mesh_build(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], cfg["bedge"], cfg["btag"], sw.SWE_RENUM_HILBERT)
    o = po.Oracle.from_config(cfg)
    try:
        l0 = sw.swe_get_stats(c)["kernel_launches"]
        sw.swe_zones_create(c, nz, nl, zone_of)
        assert sw.swe_get_stats(c)["kernel_launches"] > l0 + nl          # the device generator ran
        assert sw.swe_zone_setup_ms(c)["ghost_layers_ms"] > 0.0
        sw.swe_host_zones_build(h, nz, nl, zone_of)
        o.zones_create(nz, nl, zone_of)
        off = sw.swe_host_get(h, "zone_offset")
        ncell = sw.swe_host_get(h, "zone_ncells")
        zcu = sw.swe_host_get(h, "z:cell_user")
        zlay = sw.swe_host_get(h, "z:c2c").reshape(-1, 4)[:, 3]
        hs, hr = sw.swe_host_get(h, "send_idx"), sw.swe_host_get(h, "recv_idx")
        sends, recvs = [], []
        for z in range(nz):
            d = sw.swe_zone_describe(c, z)
            assert np.array_equal(d["cells"], zcu[off[z]:off[z] + ncell[z]])
            assert np.array_equal(d["layer"], zlay[off[z]:off[z] + ncell[z]])
            od = o.zones_describe(z)
            assert d["nowned"] == od["nowned"] and len(d["cells"]) == len(od["cells"])
            for l in range(0, nl + 1):
                assert set(d["cells"][d["layer"] == l].tolist()) == set(od["cells"][od["layer"] == l].tolist())
            assert [(s, st, n) for s, st, n, _ in d["links"]] == [(s, st, n) for s, st, n, _ in od["links"]]
            for (s, st, n, sl), (_, _, _, _osl) in zip(d["links"], od["links"]):
                assert set(d["cells"][st:st + n].tolist()) == set(od["cells"][st:st + n].tolist())
                sends.append(off[s] + sl)
                recvs.append(off[z] + st + np.arange(n))
        if sends:
            assert np.array_equal(np.concatenate(sends), hs) and np.array_equal(np.concatenate(recvs), hr)
        else:
            assert len(hs) == 0
        assert sw.swe_zone_stats(c)["send_cells_total"] == len(hs) == o.zones_counts()["send_cells_total"]
    finally:
        sw.swe_mesh_destroy(c)
        sw.swe_host_mesh_free(h)
        o.close()


def test_zoned_run_on_device_built_random_zones_is_bit_identical():
    """A decomposition no partitioner would make (random zone per cell, 70 zones, 2 layers): the
    zoned MUSCL run on the device-built ghost lists still equals the un-zoned run bit for bit."""
    from swe_inputs import delaunay_case
    cfg = delaunay_case(n=6000)
    nt = cfg["tri"].size // 3
    zone_of = np.random.default_rng(11).integers(0, 70, nt).astype(np.int32)
    a = sw.create_from_config(cfg)
    b = sw.create_from_config(cfg)
    try:
        sw.swe_zones_create(b, 70, 2, zone_of)
        sw.swe_step(a, 20, 0.45, "muscl")
        sw.swe_step(b, 20, 0.45, "muscl")
        for x, y in zip(sw.swe_get_state(a), sw.swe_get_state(b)):
            assert np.array_equal(x, y)
    finally:
        sw.swe_mesh_destroy(a)
        sw.swe_mesh_destroy(b)
