"""The input variants bench.py measures besides the five configs: same mesh in a random triangle
order (`permuted`), same mesh flooded (`flooded`), the open channel (`channel_flow_case`)."""
import numpy as np

import swe_inputs as si


def _small():
    return si.config3(length=1600.0, half_width=400.0, w2=20.0, n4=3, n8=2)


def test_permuted_is_the_same_case_in_another_order():
    c = _small()
    p = si.permuted(c, seed=7)
    assert p["tri"].shape == c["tri"].shape and not np.array_equal(p["tri"], c["tri"])
    key = lambda t: np.sort(np.sort(t, axis=1).view([("a", t.dtype), ("b", t.dtype), ("c", t.dtype)]).ravel())
    assert np.array_equal(key(np.ascontiguousarray(p["tri"])), key(np.ascontiguousarray(c["tri"])))
    # the fields travel with their triangles
    order = np.lexsort(np.sort(c["tri"], axis=1).T[::-1])
    order_p = np.lexsort(np.sort(p["tri"], axis=1).T[::-1])
    for k in ("h", "manning"):
        assert np.array_equal(c[k][order], p[k][order_p])
    assert np.array_equal(p["x"], c["x"]) and p["bc"] == c["bc"] and np.array_equal(p["bedge"], c["bedge"])
    assert np.array_equal(si.permuted(c, seed=7)["tri"], p["tri"])            # seeded


def test_flooded_has_no_dry_cell_and_a_flat_surface():
    c = _small()
    assert (c["h"] == 0.0).mean() > 0.2
    f = si.flooded(c, 18.0)
    zc = c["zb"][c["tri"]].mean(axis=1)
    assert f["h"].min() > 1.0 and np.allclose(f["h"] + zc, 18.0, rtol=0, atol=1e-12)
    assert not f["hu"].any() and not f["hv"].any() and f["tri"] is c["tri"]


def test_channel_flow_case_tags_the_two_ends():
    c = si.channel_flow_case(nx=20, ny=4, lx=50.0, ly=8.0, discharge=6.0, level=1.5, u_init=0.5, manning=0.02)
    assert c["tri"].shape[0] == 160 and c["bedge"].shape == (8, 2) and list(c["btag"]) == [1] * 4 + [2] * 4
    assert np.all(c["x"][c["bedge"][:4]] == 0.0) and np.all(c["x"][c["bedge"][4:]] == 50.0)
    assert c["bc"] == {1: ("inflow", 6.0), 2: ("level", 1.5)}
    assert np.all(c["h"] == 1.5) and np.all(c["hu"] == 0.75) and np.all(c["manning"] == 0.02)
