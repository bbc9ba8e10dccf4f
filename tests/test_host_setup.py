"""CPU tests of the CUDA library's HOST logic (no GPU): the C-ABI library loads and exports every
symbol include/swe_b200.h declares; the host mesh set-up (topology, geometry of SURVEY.md A.1,
Hilbert renumbering) and the zone builder (A.12) agree with the oracle's independent set-up."""
import os
import re

import numpy as np
import pytest

import paper_2307_16758_b200 as sw
from oracle import pyoracle as po
from swe_inputs import config0, config1, config3, lake_case, delaunay_case

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "swe_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(swe_[a-z_0-9]+)\s*\(", hdr))
    assert len(declared) >= 30
    L = sw.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(sw.SIGNATURES), declared ^ set(sw.SIGNATURES)


def test_no_device_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    cfg = config0(nx=4, ny=2)
    with pytest.raises(sw.SweError) as e:
        sw.create_from_config(cfg)
    assert e.value.code == sw.SWE_ERR_CUDA


def _cases():
    return {
        "c0": config0(nx=40, ny=4),
        "c1": config1(n=24),
        "lake": lake_case(n=20),
        "river": config3(length=1600.0, half_width=400.0, w2=20.0, n4=3, n8=2),
        "delaunay": delaunay_case(n=1500),          # genuinely unstructured, mixed windings
    }


@pytest.mark.parametrize("name", ["c0", "c1", "lake", "river", "delaunay"])
@pytest.mark.parametrize("renum", [sw.SWE_RENUM_NONE, sw.SWE_RENUM_HILBERT, sw.SWE_RENUM_RCM])
def test_host_mesh_matches_oracle_geometry(name, renum):
    cfg = _cases()[name]
    o = po.Oracle.from_config(cfg)
    h = sw.swe_host_mesh_build(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], cfg["bedge"], cfg["btag"], renum)
    try:
        cu = sw.swe_host_get(h, "cell_user")
        nt = o.nt
        assert sorted(cu.tolist()) == list(range(nt))            # a permutation
        uc = sw.swe_host_get(h, "user_cell")
        assert np.array_equal(uc[cu], np.arange(nt))
        if renum == sw.SWE_RENUM_NONE:
            assert np.array_equal(cu, np.arange(nt))
        og = o.cell_geometry()
        for k_mine, k_or in (("area", "area"), ("zc", "zc"), ("rin", "rin"), ("cx", "cx"), ("cy", "cy")):
            assert np.array_equal(sw.swe_host_get(h, k_mine), og[k_or][cu]), k_mine   # bit-exact
        # edges, matched by their (L user id, R user id) pair
        oe = o.edge_geometry()
        elr = sw.swe_host_get(h, "elr").reshape(-1, 2)
        ne_int = sw.swe_host_get(h, "ne_int")
        assert elr.shape[0] == o.ne and o.ne - ne_int == o.nbe
        assert np.all(elr[:ne_int, 1] >= 0) and np.all(elr[ne_int:, 1] == -1)
        Lu = cu[elr[:, 0]]
        Ru = np.where(elr[:, 1] >= 0, cu[np.maximum(elr[:, 1], 0)], -1)
        assert np.all((Ru < 0) | (Lu < Ru))                      # L-cell = smaller user id (A.1.4)
        c2c_o, c2e_o = o.cell_topology()
        # oracle edge id of my edge: the side of Lu whose neighbour is Ru (boundary: match geometry)
        en = sw.swe_host_get(h, "en").reshape(-1, 2)
        elen = sw.swe_host_get(h, "elen")
        edx = sw.swe_host_get(h, "edx")
        my_to_or = np.empty(o.ne, np.int64)
        for e in range(o.ne):
            cand = [c2e_o[Lu[e], k] for k in range(3) if c2c_o[Lu[e], k] == Ru[e]]
            if Ru[e] >= 0:
                assert len(cand) == 1
                my_to_or[e] = cand[0]
            else:
                hit = [q for q in cand if oe["len"][q] == elen[e] and oe["nx"][q] == en[e, 0] and oe["ny"][q] == en[e, 1]]
                assert len(hit) >= 1
                my_to_or[e] = hit[0]
        assert len(set(my_to_or.tolist())) == o.ne
        assert np.array_equal(elen, oe["len"][my_to_or])
        assert np.array_equal(en[:, 0], oe["nx"][my_to_or]) and np.array_equal(en[:, 1], oe["ny"][my_to_or])
        assert np.array_equal(edx, oe["dx"][my_to_or])
        # interior edges are sorted by their lower device cell id; c2e / c2c are consistent
        lo = np.minimum(elr[:ne_int, 0], elr[:ne_int, 1])
        assert np.all(np.diff(lo) >= 0)
        c2c = sw.swe_host_get(h, "c2c").reshape(-1, 4)
        c2e = sw.swe_host_get(h, "c2e").reshape(-1, 4)
        for i in range(nt):
            for k in range(3):
                ce = c2e[i, k]
                e = ce if ce >= 0 else ~ce
                assert elr[e, 0 if ce >= 0 else 1] == i
                nb = c2c[i, k]
                if nb >= 0:
                    assert nb == elr[e, 1 if ce >= 0 else 0]
                    assert cu[nb] == c2c_o[cu[i], k]            # same local side order as the oracle
                else:
                    assert -1 - nb == e and e >= ne_int and c2c_o[cu[i], k] == -1
        # least-squares weights reproduce the gradient of a linear field exactly (A.1.7)
        cx, cy = sw.swe_host_get(h, "cx"), sw.swe_host_get(h, "cy")
        q = 0.3 + 1.7 * cx - 0.9 * cy
        gx = np.zeros(nt)
        gy = np.zeros(nt)
        for k in range(3):
            w = sw.swe_host_get(h, "w%d" % k).reshape(-1, 2)
            r = sw.swe_host_get(h, "r%d" % k).reshape(-1, 2)
            nb = c2c[:, k]
            # mirror point of a boundary side: 2 (r.n) n, with n along r's normal component
            e = np.where(nb < 0, -1 - nb, 0)
            n = en[e] * np.where((c2e[:, k] >= 0)[:, None], 1.0, -1.0)
            rn = (r * n).sum(1)
            px = np.where(nb >= 0, cx[np.maximum(nb, 0)], cx + 2 * rn * n[:, 0])
            py = np.where(nb >= 0, cy[np.maximum(nb, 0)], cy + 2 * rn * n[:, 1])
            dq = (0.3 + 1.7 * px - 0.9 * py) - q
            gx += w[:, 0] * dq
            gy += w[:, 1] * dq
        assert np.allclose(gx, 1.7, atol=1e-9) and np.allclose(gy, -0.9, atol=1e-9)
    finally:
        sw.swe_host_mesh_free(h)
        o.close()


def test_hilbert_order_is_local():
    """Consecutive device cells are spatial neighbours: mean index distance to the edge-neighbours
    is small compared with a random order (configs[1] permutes the triangles on purpose)."""
    cfg = config1(n=64)
    h = sw.swe_host_mesh_build(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], None, None, sw.SWE_RENUM_HILBERT)
    h0 = sw.swe_host_mesh_build(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], None, None, sw.SWE_RENUM_NONE)
    try:
        def spread(hh):
            c2c = sw.swe_host_get(hh, "c2c").reshape(-1, 4)[:, :3]
            i = np.arange(c2c.shape[0])[:, None]
            m = c2c >= 0
            return np.abs(c2c - i)[m].mean()
        assert spread(h) < 0.02 * spread(h0)
    finally:
        sw.swe_host_mesh_free(h)
        sw.swe_host_mesh_free(h0)


@pytest.mark.parametrize("name,nz,nl", [("c1", 4, 2), ("c1", 8, 1), ("river", 4, 3), ("lake", 2, 2),
                                        ("delaunay", 8, 2), ("delaunay", 4, 3)])
def test_zone_builder_matches_oracle(name, nz, nl):
    cfg = _cases()[name]
    o = po.Oracle.from_config(cfg)
    o.zones_create(nz, nl)
    h = sw.swe_host_mesh_build(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], cfg["bedge"], cfg["btag"], sw.SWE_RENUM_HILBERT)
    try:
        sw.swe_host_zones_build(h, nz, nl)
        cu = sw.swe_host_get(h, "cell_user")
        zone_of = sw.swe_host_get(h, "zone_of")
        zo = o.zones_zone_of_cell()
        assert np.array_equal(zone_of, zo[cu])                   # same RCB partition
        off = sw.swe_host_get(h, "zone_offset")
        nown = sw.swe_host_get(h, "zone_nowned")
        ncell = sw.swe_host_get(h, "zone_ncells")
        zcu = sw.swe_host_get(h, "z:cell_user")
        zc2c = sw.swe_host_get(h, "z:c2c").reshape(-1, 4)
        src = sw.swe_host_get(h, "src_of_cell")
        for z in range(nz):
            d = o.zones_describe(z)
            mine = zcu[off[z]:off[z] + ncell[z]]
            lay = zc2c[off[z]:off[z] + ncell[z], 3]
            assert nown[z] == d["nowned"] and ncell[z] == len(d["cells"])
            assert set(mine[:nown[z]].tolist()) == set(d["cells"][:d["nowned"]].tolist())
            assert np.all(lay[:nown[z]] == 0)
            for l in range(1, nl + 1):
                assert set(mine[lay == l].tolist()) == set(d["cells"][d["layer"] == l].tolist())
        # exchange lists: every ghost mirrors the owned cell it receives from
        s, r = sw.swe_host_get(h, "send_idx"), sw.swe_host_get(h, "recv_idx")
        assert np.array_equal(src[s], src[r])
        assert np.all(zc2c[s, 3] == 0) and np.all(zc2c[r, 3] >= 1)
        assert len(set(r.tolist())) == len(r) == int((zc2c[:, 3] >= 1).sum())
        assert o.zones_counts()["send_cells_total"] == len(s)
        # zoned geometry is a bit-copy of the un-zoned one
        for nm in ("zc", "area", "rin"):
            assert np.array_equal(sw.swe_host_get(h, "z:" + nm), sw.swe_host_get(h, nm)[src])
        # zoned edges: both cells inside the same zone, orientation kept
        zelr = sw.swe_host_get(h, "z:elr").reshape(-1, 2)
        zne_int = sw.swe_host_get(h, "z:ne_int")
        zid = np.searchsorted(off, np.arange(len(zcu)), side="right") - 1
        assert np.all(zid[zelr[:zne_int, 0]] == zid[zelr[:zne_int, 1]])
        assert np.all(zcu[zelr[:zne_int, 0]] < zcu[zelr[:zne_int, 1]])
        assert np.all((zc2c[zelr[:zne_int, 0], 3] == 0) | (zc2c[zelr[:zne_int, 1], 3] == 0))
    finally:
        sw.swe_host_mesh_free(h)
        o.close()


def test_mesh_errors():
    x = np.array([0.0, 1.0, 0.0, 1.0])
    y = np.array([0.0, 0.0, 1.0, 1.0])
    z = np.zeros(4)
    with pytest.raises(sw.SweError):   # vertex id out of range
        sw.swe_host_mesh_build(x, y, z, np.array([[0, 1, 7]], np.int32))
    with pytest.raises(sw.SweError):   # zero area
        sw.swe_host_mesh_build(np.array([0.0, 1.0, 2.0]), np.zeros(3), np.zeros(3), np.array([[0, 1, 2]], np.int32))
    with pytest.raises(sw.SweError):   # non-manifold: three triangles on edge (0,1)
        sw.swe_host_mesh_build(np.array([0.0, 1.0, 0.0, 1.0, 0.5]), np.array([0.0, 0.0, 1.0, 1.0, -1.0]), np.zeros(5),
                               np.array([[0, 1, 2], [0, 1, 3], [0, 1, 4]], np.int32))
    with pytest.raises(sw.SweError):   # tagged edge is interior
        sw.swe_host_mesh_build(x, y, z, np.array([[0, 1, 2], [1, 3, 2]], np.int32),
                               np.array([[1, 2]], np.int32), np.array([1], np.int32))
    h = sw.swe_host_mesh_build(x, y, z, np.array([[0, 2, 1], [1, 3, 2]], np.int32))   # clockwise input is fixed
    assert np.all(sw.swe_host_get(h, "area") > 0)
    with pytest.raises(sw.SweError):
        sw.swe_host_zones_build(h, 3, 1)      # RCB needs a power of two
    with pytest.raises(sw.SweError):
        sw.swe_host_zones_build(h, 2, 4)      # nlayers in 1..3
    sw.swe_host_mesh_free(h)


def test_rcm_order_has_a_small_bandwidth():
    """Reverse Cuthill-McKee: neighbours get close numbers.  On the permuted configs[1] mesh the
    identity numbering has a bandwidth of the order of the cell count; RCM brings it down to the
    order of the number of cells across the domain."""
    from swe_inputs import config1
    cfg = config1(n=60)
    nt = cfg["tri"].shape[0]
    bw = {}
    for renum in (sw.SWE_RENUM_NONE, sw.SWE_RENUM_RCM, sw.SWE_RENUM_HILBERT):
        h = sw.swe_host_mesh_build(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], cfg["bedge"], cfg["btag"], renum)
        c2c = sw.swe_host_get(h, "c2c").reshape(-1, 4)[:, :3]
        i = np.repeat(np.arange(nt), 3).reshape(-1, 3)
        d = np.abs(c2c - i)[c2c >= 0]
        bw[renum] = (int(d.max()), float(d.mean()))
        sw.swe_host_mesh_free(h)
    assert bw[sw.SWE_RENUM_NONE][0] > nt // 2
    assert bw[sw.SWE_RENUM_RCM][0] < 6 * 60                  # a few rows of the 60 x 60 x 2 mesh
    assert bw[sw.SWE_RENUM_RCM][1] < 0.05 * bw[sw.SWE_RENUM_NONE][1]


def test_third_offset_travels_as_a_single_precision_residual():
    """The device stores r_0, r_1 and rres = float(r_2 + (r_0 + r_1)) instead of r_2 (8 bytes less
    per cell and stage in the gradient kernel; swe_kernels.cuh stencil_r2): the reconstruction
    rres - (r_0 + r_1) must give back the stored r_2 -- bit for bit except where a component of r_2
    is tiny against |r| (there within an ulp of |r|) -- on meshes with coordinates up to 6e4 m."""
    for cfg in (config3(length=3200.0, half_width=600.0, w2=30.0, n4=4, n8=3), config1(n=60),
                delaunay_case(n=1500)):
        shift = dict(cfg)
        shift["x"] = cfg["x"] + 56000.0                     # the far end of the 60 km reach
        for c in (cfg, shift):
            h = sw.swe_host_mesh_build(c["x"], c["y"], c["zb"], c["tri"], c["bedge"], c["btag"])
            try:
                r0, r1, r2 = [sw.swe_host_get(h, k).reshape(-1, 2) for k in ("r0", "r1", "r2")]
                res = sw.swe_host_get(h, "rres").reshape(-1, 2)
                assert res.dtype == np.float32
                exact = r2 + (r0 + r1)                          # the sum cancels: exact in double
                assert np.array_equal(res, exact.astype(np.float32))
                back = res.astype(np.float64) - (r0 + r1)
                scale = np.sqrt((r2 ** 2).sum(axis=1, keepdims=True))
                assert np.abs(back - r2).max() <= 1.2e-16 * scale.max()
                big = np.abs(r2) > 1e-2 * scale
                assert np.array_equal(back[big], r2[big])
                assert (back == r2).mean() > 0.999
            finally:
                sw.swe_host_mesh_free(h)


def test_build_check_fails_loudly_when_a_source_is_missing(monkeypatch):
    """A library next to an incomplete source tree must not be picked up silently
    (paper_2307_16758_b200/build.py needs_build)."""
    from paper_2307_16758_b200 import build as b
    assert b.needs_build() is False                       # the suite runs on a freshly built library
    monkeypatch.setattr(b, "DEPS", list(b.DEPS) + ["no_such_file.cuh"])
    with pytest.raises(FileNotFoundError) as e:
        b.needs_build()
    assert "no_such_file.cuh" in str(e.value)
