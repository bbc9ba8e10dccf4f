"""The five BASELINE.json configs (and scaled-down variants of each) as plain input dictionaries.

Every builder returns a dict with
  x, y, zb      per-vertex coordinates and bed elevation (float64)
  tri           (nt,3) int32 vertex ids
  bedge, btag   (nb,2) int32 vertex pairs of tagged boundary edges and their tag ids
                (untagged boundary edges are walls)
  bc            {tag: (kind, value)} with kind in {"wall","inflow","level","transmissive"}
  h, hu, hv     initial cell state in the order of `tri`
  manning       per-cell Manning n, or None
  params        g, h_dry, h_thin, beta
  runs          list of (scheme, cfl, steps)
Cell-centred inputs (initial depth, Manning zone) are evaluated at the vertex-average point of
each triangle; the cell bed used for `h = max(0, level - z)` is (zb[v0]+zb[v1]+zb[v2])/3 in that
order, the same expression both libraries use.
"""
import numpy as np

from .meshes import grid_mesh, river_mesh
from .noise import value_noise, gaussian_bumps

PARAMS = {"g": 9.81, "h_dry": 1e-6, "h_thin": 1e-3, "beta": 1.0}


def _centroids(x, y, tri):
    cx = (x[tri[:, 0]] + x[tri[:, 1]] + x[tri[:, 2]]) / 3.0
    cy = (y[tri[:, 0]] + y[tri[:, 1]] + y[tri[:, 2]]) / 3.0
    return cx, cy


def _cell_bed(zb, tri):
    return (zb[tri[:, 0]] + zb[tri[:, 1]] + zb[tri[:, 2]]) / 3.0


def _base(name, x, y, zb, tri, h, runs, manning=None, bedge=None, btag=None, bc=None, params=None):
    nt = tri.shape[0]
    return {
        "name": name, "x": np.ascontiguousarray(x), "y": np.ascontiguousarray(y),
        "zb": np.ascontiguousarray(zb), "tri": np.ascontiguousarray(tri, dtype=np.int32),
        "bedge": np.zeros((0, 2), np.int32) if bedge is None else np.ascontiguousarray(bedge, dtype=np.int32),
        "btag": np.zeros((0,), np.int32) if btag is None else np.ascontiguousarray(btag, dtype=np.int32),
        "bc": {} if bc is None else dict(bc),
        "h": np.ascontiguousarray(h, dtype=np.float64), "hu": np.zeros(nt), "hv": np.zeros(nt),
        "manning": manning, "params": dict(PARAMS if params is None else params), "runs": list(runs),
    }


def config0(nx=200, ny=10, lx=100.0, ly=5.0, jitter=0.1, seed=0, h_left=10.0, h_right=1.0,
            steps=200):
    """configs[0]: wet-bed dam break on a 100 m x 5 m channel, 200x10 quads -> 4 000 triangles,
    jitter +-10 %, flat bed, h=10 | 1 about x=lx/2, walls, HLLC CFL 0.9, 200 steps.
    h_right=0 gives the Ritter dry-bed case on the same channel."""
    x, y, tri = grid_mesh(nx, ny, lx, ly, jitter, seed)
    cx, _ = _centroids(x, y, tri)
    h = np.where(cx < 0.5 * lx, h_left, h_right)
    return _base("c0", x, y, np.zeros_like(x), tri, h, [("hllc", 0.9, steps)])


def config1(n=350, l=100.0, jitter=0.2, seed=1, steps=500, radius=11.0):
    """configs[1]: circular dam break, 350x350 quads -> 245 000 triangles, jitter +-20 %,
    triangle order randomly permuted, h=10 inside r<11 m else 1, MUSCL(beta=1) RK2 CFL 0.45."""
    x, y, tri = grid_mesh(n, n, l, l, jitter, seed, permute=True)
    cx, cy = _centroids(x, y, tri)
    r = np.sqrt((cx - 0.5 * l) ** 2 + (cy - 0.5 * l) ** 2)
    h = np.where(r < radius * (l / 100.0), 10.0, 1.0)
    return _base("c1", x, y, np.zeros_like(x), tri, h, [("muscl", 0.45, steps)])


def lake_bed(x, y, seed, extent=2000.0):
    """configs[2] bathymetry: 40 Gaussian bumps (H~U[1,8] m, W~U[20,200] m scaled with the extent)
    + 4-octave value noise, amplitude 0.5 m, lambda0 = extent/10."""
    sc = extent / 2000.0
    z = gaussian_bumps(x, y, seed, 40, extent, 1.0, 8.0, 20.0 * sc, 200.0 * sc)
    z += value_noise(x, y, seed, 4, 0.5, 200.0 * sc)
    return z


def config2(n=707, extent=2000.0, jitter=0.1, seed=2, level=5.0, steps=1000, manning=0.03):
    """configs[2]: lake at rest over rough bathymetry with dry bump tops, ~1.0 M triangles."""
    x, y, tri = grid_mesh(n, n, extent, extent, jitter, seed)
    zb = lake_bed(x, y, seed, extent)
    zc = _cell_bed(zb, tri)
    h = np.maximum(0.0, level - zc)
    nman = np.full(tri.shape[0], manning)
    return _base("c2", x, y, zb, tri, h, [("waf", 0.45, steps), ("muscl", 0.45, steps)],
                 manning=nman)


def lake_case(n=60, extent=200.0, seed=2, level=5.0, jitter=0.1, manning=0.03):
    """Scaled-down configs[2] (same recipe, smaller extent and cell count) for CPU pins."""
    return config2(n=n, extent=extent, jitter=jitter, seed=seed, level=level, steps=1000,
                   manning=manning)


def river_bed(m, seed):
    """configs[3] bed: thalweg 4.5*(1-x/L) m, banks +6 m outside the 300 m channel (cosine ramp
    between d=0.8*w2 and d=w2), valley sides +4.5 m over 0.75*half_width, + 5-octave value noise
    (amplitude 0.5 m, lambda0 400 m): range about 0-15 m."""
    x, d = m["x"], m["d"]
    length, hw, w2 = m["length"], m["half_width"], m["w2"]
    thal = 4.5 * (1.0 - x / length)
    d0 = 0.8 * w2
    chi = np.where(d < d0, 1.0, np.where(d >= w2, 0.0,
                                         0.5 * (1.0 + np.cos(np.pi * (d - d0) / (w2 - d0)))))
    side = 4.5 * np.minimum(1.0, np.maximum(0.0, d - w2) / (0.75 * hw))
    z = thal + 6.0 * (1.0 - chi) + side
    z += value_noise(x, m["y"], seed, 5, 0.5, 400.0)
    return z, thal


def config3(length=60000.0, half_width=4000.0, seed=3, jitter=0.1, discharge=8000.0,
            steps=200, **mesh_kw):
    """configs[3]: river-scale mesh (~13 M triangles at the default size), partly dry, inflow Q
    on the upstream channel edges (tag 1), fixed level downstream (tag 2), walls elsewhere,
    Manning 0.025/0.03/0.035/0.04 by band.  Smaller `length`/`half_width` give the same
    structure at test size."""
    m = river_mesh(length, half_width, seed, jitter, **mesh_kw)
    x, y, tri = m["x"], m["y"], m["tri"]
    zb, thal = river_bed(m, seed)
    zc = _cell_bed(zb, tri)
    thal_c = _cell_bed(thal, tri)
    h = np.maximum(0.0, (thal_c + 4.0) - zc)
    nman = np.array([0.025, 0.03, 0.035, 0.04])[m["band"]]
    west, east = m["west_edges"], m["east_edges"]
    dW = np.maximum(m["d"][west[:, 0]], m["d"][west[:, 1]])
    inflow = west[dW <= m["w2"] + 1e-9]
    bedge = np.concatenate([inflow, east], axis=0)
    btag = np.concatenate([np.full(inflow.shape[0], 1), np.full(east.shape[0], 2)]).astype(np.int32)
    bc = {1: ("inflow", float(discharge)), 2: ("level", 4.0)}
    cfg = _base("c3", x, y, zb, tri, h, [("muscl", 0.45, steps), ("hllc", 0.9, steps)],
                manning=nman, bedge=bedge, btag=btag, bc=bc)
    return cfg


def simple_wave_case(nx, ny=None, lx=100.0, ly=None, jitter=0.0, seed=0, h0=1.0, a=0.2, w=5.0,
                     x0=30.0, g=9.81):
    """Smooth right-running simple wave into still water on the configs[0] channel
    (SURVEY.md Appendix C.3): h(x,0)=h0+a exp(-((x-x0)/w)^2), u=2(sqrt(g h)-sqrt(g h0)), v=0.
    Cell values are edge-midpoint-quadrature averages of the conserved variables."""
    if ny is None:
        ny = max(1, nx // 20)
    if ly is None:
        ly = lx * ny / nx
    x, y, tri = grid_mesh(nx, ny, lx, ly, jitter, seed)

    def prof(xx):
        hh = h0 + a * np.exp(-((xx - x0) / w) ** 2)
        uu = 2.0 * (np.sqrt(g * hh) - np.sqrt(g * h0))
        return hh, hh * uu

    xm = [0.5 * (x[tri[:, k]] + x[tri[:, (k + 1) % 3]]) for k in range(3)]
    hs = [prof(v) for v in xm]
    h = (hs[0][0] + hs[1][0] + hs[2][0]) / 3.0
    hu = (hs[0][1] + hs[1][1] + hs[2][1]) / 3.0
    cfg = _base("simple_wave", x, y, np.zeros_like(x), tri, h, [("hllc", 0.9, 0)])
    cfg["hu"] = np.ascontiguousarray(hu)
    cfg["profile"] = {"h0": h0, "a": a, "w": w, "x0": x0, "g": g}
    return cfg


def permuted(cfg, seed=7):
    """The same case with its triangles listed in a random order (as a mesh generator or a
    partitioner may hand them over): tri and every per-cell field are permuted together."""
    rng = np.random.default_rng(seed)
    p = rng.permutation(cfg["tri"].shape[0])
    out = dict(cfg)
    out["tri"] = np.ascontiguousarray(cfg["tri"][p])
    for k in ("h", "hu", "hv", "manning"):
        if cfg.get(k) is not None:
            out[k] = np.ascontiguousarray(cfg[k][p])
    out["name"] = cfg["name"] + "_permuted"
    return out


def flooded(cfg, level):
    """The same case with a flat free surface at `level` (above every cell's bed where level is
    high enough): no dry cells, velocity zero.  depth = max(0, level - cell bed)."""
    out = dict(cfg)
    zc = _cell_bed(cfg["zb"], cfg["tri"])
    out["h"] = np.ascontiguousarray(np.maximum(0.0, level - zc))
    out["hu"] = np.zeros_like(out["h"])
    out["hv"] = np.zeros_like(out["h"])
    out["name"] = cfg["name"] + "_flooded"
    return out


def delaunay_case(n=3000, lx=200.0, ly=120.0, seed=5, level=3.0, dam=True):
    """An unstructured (Delaunay) mesh over a bumpy bed with dry bump tops: lake at rest at `level`
    (dam=False) or the same with the left third raised by 2 m (a dam break running over the bumps
    and around the dry tops).  Walls all round, Manning 0.03."""
    from .meshes import delaunay_mesh
    x, y, tri = delaunay_mesh(n, lx, ly, seed)
    sc = lx / 200.0                                   # bump widths and noise wavelength follow the domain
    zb = gaussian_bumps(x, y, seed, 10, max(lx, ly), 2.0, 6.0, 8.0 * sc, 25.0 * sc) + value_noise(x, y, seed, 3, 0.3, 40.0 * sc)
    zc = _cell_bed(zb, tri)
    cx, _ = _centroids(x, y, tri)
    eta = np.where((cx < lx / 3.0) & dam, level + 2.0, level)
    h = np.maximum(0.0, eta - zc)
    return _base("delaunay", x, y, zb, tri, h, [("muscl", 0.45, 100)], manning=np.full(tri.shape[0], 0.03))


def channel_flow_case(nx=100, ny=5, lx=100.0, ly=5.0, jitter=0.1, seed=4, discharge=10.0, level=2.0,
                      manning=0.0, h_init=None, u_init=0.0):
    """Straight flat channel with the two open boundaries of configs[3]: imposed discharge Q on the
    upstream side x = 0 (tag 1), fixed water level on the downstream side x = lx (tag 2), walls on
    the long sides.  Initial state: depth h_init (default: the level) and velocity u_init along x,
    uniform.  Used to pin the oracle's open boundaries (uniform flow, backwater curve)."""
    x, y, tri = grid_mesh(nx, ny, lx, ly, jitter, seed)
    j = np.arange(ny)
    west = np.stack([j * (nx + 1), (j + 1) * (nx + 1)], axis=1)
    east = west + nx
    bedge = np.concatenate([west, east], axis=0)
    btag = np.concatenate([np.full(ny, 1), np.full(ny, 2)]).astype(np.int32)
    nt = tri.shape[0]
    h0 = float(level if h_init is None else h_init)
    cfg = _base("channel_flow", x, y, np.zeros_like(x), tri, np.full(nt, h0), [("hllc", 0.9, 0)],
                manning=np.full(nt, float(manning)) if manning else None, bedge=bedge, btag=btag,
                bc={1: ("inflow", float(discharge)), 2: ("level", float(level))})
    cfg["hu"] = np.full(nt, h0 * float(u_init))
    return cfg


CONFIG_BUILDERS = {"c0": config0, "c1": config1, "c2": config2, "c3": config3}
