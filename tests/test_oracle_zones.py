"""Pins of the oracle's zone decomposition, ghost layers, send lists / receive ranges and
pack/unpack."""
import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import dijkstra

import swe_inputs as si
from oracle import pyoracle as po


@pytest.mark.parametrize("scheme,cfl,layers", [("hllc", 0.9, 1), ("hllc", 0.9, 2), ("muscl", 0.45, 1),
                                               ("muscl", 0.45, 2), ("muscl", 0.45, 3), ("waf", 0.45, 2)])
def test_zoned_run_is_bit_identical_to_unzoned(scheme, cfl, layers):
    # "the solution generated when using two layers of ghost cells is exactly the same as the
    # solution generated on the original mesh before the decomposition"
    cfg = si.lake_case(n=28, level=6.0)      # wet/dry fronts, rough bed, Manning
    rng = np.random.default_rng(0)
    cfg["hu"] = np.where(cfg["h"] > 0, rng.uniform(-0.5, 0.5, cfg["h"].size), 0.0)
    a = po.Oracle.from_config(cfg)
    b = po.Oracle.from_config(cfg)
    ta = a.step(25, cfl, scheme)
    b.zones_create(8, layers)
    tb = b.zones_step(25, cfl, scheme)
    assert ta == tb
    for u, v in zip(a.get_state(), b.get_state()):
        assert np.array_equal(u, v)


def test_insufficient_ghost_layers_are_refused():
    # WAF needs the upwind cells of R (Fig. 18): one layer is not enough
    cfg = si.config1(n=16)
    b = po.Oracle.from_config(cfg)
    b.zones_create(4, 1)
    with pytest.raises(ValueError):
        b.zones_step(1, 0.45, "waf")


def _adjacency(o):
    c2c, _ = o.cell_topology()
    i = np.repeat(np.arange(o.nt), 3)
    j = c2c.ravel()
    ok = j >= 0
    return coo_matrix((np.ones(ok.sum()), (i[ok], j[ok])), shape=(o.nt, o.nt)).tocsr()


@pytest.mark.parametrize("layers", [1, 2, 3])
def test_zone_structure(layers):
    cfg = si.config3(length=320.0, half_width=360.0)
    o = po.Oracle.from_config(cfg)
    nz = 8
    o.zones_create(nz, layers)
    zone_of = o.zones_zone_of_cell()
    # RCB: sizes differ by at most one per bisection level (lower floor(n/2) go left)
    sizes = np.bincount(zone_of, minlength=nz)
    assert sizes.sum() == o.nt and sizes.max() - sizes.min() <= 3
    adj = _adjacency(o)
    total_send = 0
    total_ghost = 0
    descr = [o.zones_describe(z) for z in range(nz)]
    for z, d in enumerate(descr):
        no = d["nowned"]
        owned = d["cells"][:no]
        assert np.array_equal(owned, np.flatnonzero(zone_of == z))      # ascending ids
        ghosts = d["cells"][no:]
        glayer = d["layer"][no:]
        assert np.all(d["layer"][:no] == 0)
        # ghost layer l = graph distance l from the zone over edge adjacency (library BFS)
        dist = dijkstra(adj, unweighted=True, indices=owned, min_only=True)
        expect = np.flatnonzero((dist >= 1) & (dist <= layers))
        assert np.array_equal(np.sort(ghosts), expect)
        assert np.array_equal(glayer, dist[ghosts].astype(int))
        # receive ranges: contiguous per source, ascending source, tile the ghost range exactly
        pos = no
        prev_src = -1
        for src, start, count, send in d["links"]:
            assert src > prev_src and src != z and start == pos and count > 0
            blk = d["cells"][start:start + count]
            assert np.all(zone_of[blk] == src)
            # ordered by layer then id
            key = d["layer"][start:start + count].astype(np.int64) * o.nt + blk
            assert np.all(np.diff(key) > 0)
            # the send list holds the source-local indices of exactly these cells (PointList)
            sd = descr[src]
            assert np.all(send < sd["nowned"])
            assert np.array_equal(sd["cells"][send], blk)
            pos += count
            prev_src = src
            total_send += count
        assert pos == len(d["cells"])
        total_ghost += len(ghosts)
    cnt = o.zones_counts()
    assert cnt["send_cells_total"] == total_send == total_ghost == cnt["ghost_cells_total"]
    assert cnt["bytes_per_exchange"] == 24 * total_send


def test_user_supplied_partition_and_single_zone():
    cfg = si.config1(n=12)
    a = po.Oracle.from_config(cfg)
    b = po.Oracle.from_config(cfg)
    rng = np.random.default_rng(1)
    zoc = rng.integers(0, 3, a.nt).astype(np.int32)      # scattered, non-contiguous zones
    a.step(10, 0.45, "muscl")
    b.zones_create(3, 2, zoc)
    b.zones_step(10, 0.45, "muscl")
    for u, v in zip(a.get_state(), b.get_state()):
        assert np.array_equal(u, v)
    c = po.Oracle.from_config(cfg)
    c.zones_create(1, 2)
    assert c.zones_counts()["ghost_cells_total"] == 0
    c.zones_step(10, 0.45, "muscl")
    assert np.array_equal(c.get_state()[0], a.get_state()[0])
