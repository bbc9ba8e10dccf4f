"""Synthetic triangle meshes (input recipe; BASELINE.json configs[0..3]).

* grid_mesh   -- jittered grid of quads, each split into two triangles (configs 0-2)
* river_mesh  -- banded 2->4->8->16(-20) m triangulation of a meandering valley (configs 3-4)

Meshes are returned as plain arrays: vertex coordinates x, y (float64) and tri (int32, shape
(nt,3), any winding).  No mesh *geometry* used by the numerical method (areas, normals, ...) is
computed here; both the oracle and the CUDA library derive it themselves.
"""
import numpy as np


def grid_mesh(nx, ny, lx, ly, jitter=0.0, seed=0, permute=False):
    """(nx x ny) quads on [0,lx]x[0,ly]; interior vertices displaced by jitter*spacing*U[-1,1];
    quad (i,j) -> triangles (a,b,c),(a,c,d), a=(i,j), b=(i+1,j), c=(i+1,j+1), d=(i,j+1).
    `permute` applies a random permutation to the triangle list (configs[1])."""
    rng = np.random.default_rng(seed)
    dx = lx / nx
    dy = ly / ny
    ii, jj = np.meshgrid(np.arange(nx + 1), np.arange(ny + 1), indexing="xy")
    x = ii.astype(np.float64) * dx
    y = jj.astype(np.float64) * dy
    if jitter > 0.0:
        jx = rng.uniform(-1.0, 1.0, x.shape) * (jitter * dx)
        jy = rng.uniform(-1.0, 1.0, y.shape) * (jitter * dy)
        interior = (ii > 0) & (ii < nx) & (jj > 0) & (jj < ny)
        x = np.where(interior, x + jx, x)
        y = np.where(interior, y + jy, y)
    x = x.ravel()
    y = y.ravel()
    qi, qj = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    a = (qj * (nx + 1) + qi).ravel()
    b = a + 1
    c = a + (nx + 1) + 1
    d = a + (nx + 1)
    tri = np.empty((2 * nx * ny, 3), dtype=np.int32)
    tri[0::2, 0] = a
    tri[0::2, 1] = b
    tri[0::2, 2] = c
    tri[1::2, 0] = a
    tri[1::2, 1] = c
    tri[1::2, 2] = d
    if permute:
        tri = tri[rng.permutation(tri.shape[0])]
    return x, y, np.ascontiguousarray(tri)


def delaunay_mesh(n, lx, ly, seed=0):
    """A genuinely unstructured triangulation of [0,lx]x[0,ly]: n seeded random interior points
    (rejected if closer than 0.45 of the mean spacing to an earlier one) plus equispaced boundary
    points, Delaunay-triangulated (scipy).  Vertex valence, triangle shape, winding and order are
    whatever the triangulator returns (every third triangle is then turned clockwise); needle
    triangles along the boundary are dropped."""
    from scipy.spatial import Delaunay, cKDTree
    rng = np.random.default_rng(seed)
    spacing = np.sqrt(lx * ly / n)
    nbx, nby = max(2, int(round(lx / spacing))), max(2, int(round(ly / spacing)))
    bx = np.linspace(0.0, lx, nbx + 1)
    by = np.linspace(0.0, ly, nby + 1)
    border = np.concatenate([np.stack([bx, np.zeros_like(bx)], 1), np.stack([bx, np.full_like(bx, ly)], 1),
                             np.stack([np.zeros_like(by[1:-1]), by[1:-1]], 1),
                             np.stack([np.full_like(by[1:-1], lx), by[1:-1]], 1)])
    if n > 50000:
        # large meshes: one point per lattice site, displaced by up to 0.45 of the spacing (the
        # Poisson-disc thinning below is a Python loop); the connectivity is still the triangulator's
        gx, gy = np.meshgrid(bx[1:-1], by[1:-1], indexing="xy")
        inner = np.stack([gx.ravel(), gy.ravel()], 1)
        inner += rng.uniform(-0.45, 0.45, inner.shape) * [lx / nbx, ly / nby]
        p = np.concatenate([border, inner])
        tri = Delaunay(p).simplices.astype(np.int32)
        a = p[tri[:, 1]] - p[tri[:, 0]]
        b = p[tri[:, 2]] - p[tri[:, 0]]
        area = 0.5 * np.abs(a[:, 0] * b[:, 1] - a[:, 1] * b[:, 0])
        tri = tri[area > 1e-3 * spacing * spacing]
        tri[::3] = tri[::3, ::-1]
        return np.ascontiguousarray(p[:, 0]), np.ascontiguousarray(p[:, 1]), np.ascontiguousarray(tri)
    cand = rng.uniform([0.3 * spacing, 0.3 * spacing], [lx - 0.3 * spacing, ly - 0.3 * spacing], (3 * n, 2))
    pts = list(border)
    tree_pts = np.array(pts)
    keep = []
    for start in range(0, cand.shape[0], 256):                     # thinning in blocks
        block = cand[start:start + 256]
        tree = cKDTree(np.concatenate([tree_pts, np.array(keep).reshape(-1, 2)]))
        d, _ = tree.query(block)
        ok = block[d > 0.45 * spacing]
        if ok.shape[0]:
            sub = cKDTree(ok)
            pairs = sub.query_pairs(0.45 * spacing)
            drop = {j for _, j in pairs}
            keep.extend(ok[[i for i in range(ok.shape[0]) if i not in drop]])
        if len(keep) >= n:
            break
    p = np.concatenate([border, np.array(keep[:n]).reshape(-1, 2)])
    tri = Delaunay(p).simplices.astype(np.int32)
    a = p[tri[:, 1]] - p[tri[:, 0]]
    b = p[tri[:, 2]] - p[tri[:, 0]]
    area = 0.5 * np.abs(a[:, 0] * b[:, 1] - a[:, 1] * b[:, 0])
    tri = tri[area > 1e-3 * spacing * spacing]                      # collinear boundary points give slivers
    tri[::3] = tri[::3, ::-1]                                       # every third triangle clockwise
    return np.ascontiguousarray(p[:, 0]), np.ascontiguousarray(p[:, 1]), np.ascontiguousarray(tri)


def boundary_edges(tri):
    """Vertex pairs (nb,2) of edges that belong to exactly one triangle (used only to attach
    boundary tags; the libraries find boundary edges themselves)."""
    tri = np.asarray(tri, dtype=np.int64)
    e = np.concatenate([tri[:, [0, 1]], tri[:, [1, 2]], tri[:, [2, 0]]], axis=0)
    lo = np.minimum(e[:, 0], e[:, 1])
    hi = np.maximum(e[:, 0], e[:, 1])
    nv = int(tri.max()) + 1
    key = lo * nv + hi
    uk, cnt = np.unique(key, return_counts=True)
    bk = uk[cnt == 1]
    return np.stack([bk // nv, bk % nv], axis=1).astype(np.int32)


def _river_rows(half_width, w2, n4, n8, target16):
    """Row layout of one side of the valley, from the band edge outward:
    list of (offset from centre line, spacing in s).  Transition strips have height 1.5x the
    finer spacing."""
    rows = []
    t = w2
    # transition 2 -> 4
    t += 3.0
    rows.append((t, 4.0))
    for _ in range(n4):
        t += 4.0
        rows.append((t, 4.0))
    t += 6.0
    rows.append((t, 8.0))
    for _ in range(n8):
        t += 8.0
        rows.append((t, 8.0))
    t += 12.0
    rows.append((t, 16.0))
    rest = half_width - t
    n16 = max(1, int(round(rest / target16)))
    h16 = rest / n16
    for k in range(n16):
        rows.append((t + (k + 1) * h16 if k + 1 < n16 else half_width, 16.0))
    return rows


def river_mesh(length=60000.0, half_width=4000.0, seed=3, jitter=0.1, w2=150.0, n4=15, n8=10,
               target16=20.0, amp=None, wavelength=None):
    """Banded triangulation of [0,length] x [0,2*half_width] in logical coordinates (s,t), mapped to
    a meandering valley (BASELINE.json configs[3]).

    Bands, symmetric about the centre line t=half_width: 2 m squares for |t-centre|<=w2, then n4
    rows of 4 m, n8 rows of 8 m and 16 m x ~target16 m rows out to the valley edge, joined by
    conforming 2:1 transition strips (per coarse segment, fine nodes b0,b1,b2 and coarse nodes
    t0,t2 give triangles (b0,b1,t0),(b1,t2,t0),(b1,b2,t2)).
    Physical map: x=s, y=t+amp*sin(2 pi s/wavelength)*psi(t); psi=1 near the channel with a cosine
    taper to 0 at 0.75*half_width.

    Returns dict with x, y, tri, and per-vertex logical coords s, t, d=|t-centre|, per-cell band
    id (0..3 for the 2/4/8/16 m bands; transition strips take the coarser band).
    `length` must be a multiple of 16.
    """
    if abs(length / 16.0 - round(length / 16.0)) > 1e-9:
        raise ValueError("length must be a multiple of 16 m")
    if amp is None:
        amp = min(0.02 * length, 0.3 * half_width)
    if wavelength is None:
        wavelength = length / 4.0
    rng = np.random.default_rng(seed)
    side = _river_rows(half_width, w2, n4, n8, target16)
    n2 = int(round(w2 / 2.0))
    # rows ordered by increasing t: (t', spacing)
    rows = [(-off, sp) for off, sp in reversed(side)]
    rows += [(2.0 * k, 2.0) for k in range(-n2, n2 + 1)]
    rows += list(side)
    nrow = len(rows)
    counts = [int(round(length / sp)) + 1 for _, sp in rows]
    offs = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    nv = int(offs[-1])
    s = np.empty(nv)
    t = np.empty(nv)
    hloc = np.empty(nv)       # local spacing used to scale the jitter
    fixed = np.zeros(nv, dtype=bool)
    for r, (tp, sp) in enumerate(rows):
        o, n = offs[r], counts[r]
        s[o:o + n] = np.arange(n) * sp
        s[o + n - 1] = length
        t[o:o + n] = half_width + tp
        hloc[o:o + n] = sp
        fixed[o] = True
        fixed[o + n - 1] = True
        if r == 0 or r == nrow - 1:
            fixed[o:o + n] = True
    # finer spacing governs the jitter of rows that border a transition strip
    for r in range(nrow - 1):
        if rows[r][1] != rows[r + 1][1]:
            fine = min(rows[r][1], rows[r + 1][1])
            for q in (r, r + 1):
                hloc[offs[q]:offs[q] + counts[q]] = np.minimum(hloc[offs[q]:offs[q] + counts[q]], fine)
    if jitter > 0.0:
        js = rng.uniform(-1.0, 1.0, nv) * jitter * hloc
        jt = rng.uniform(-1.0, 1.0, nv) * jitter * hloc
        s = np.where(fixed, s, s + js)
        t = np.where(fixed, t, t + jt)
    tris = []
    bands = []
    band_of = {2.0: 0, 4.0: 1, 8.0: 2, 16.0: 3}
    for r in range(nrow - 1):
        lo, hi = offs[r], offs[r + 1]
        nlo, nhi = counts[r], counts[r + 1]
        band = band_of[max(rows[r][1], rows[r + 1][1])]
        if nlo == nhi:
            i = np.arange(nlo - 1, dtype=np.int64)
            a = lo + i
            b = lo + i + 1
            c = hi + i + 1
            d = hi + i
            tt = np.empty((2 * (nlo - 1), 3), dtype=np.int64)
            tt[0::2] = np.stack([a, b, c], axis=1)
            tt[1::2] = np.stack([a, c, d], axis=1)
        elif nlo == 2 * nhi - 1:      # fine below, coarse above
            j = np.arange(nhi - 1, dtype=np.int64)
            b0 = lo + 2 * j
            b1 = b0 + 1
            b2 = b0 + 2
            t0 = hi + j
            t2 = hi + j + 1
            tt = np.empty((3 * (nhi - 1), 3), dtype=np.int64)
            tt[0::3] = np.stack([b0, b1, t0], axis=1)
            tt[1::3] = np.stack([b1, t2, t0], axis=1)
            tt[2::3] = np.stack([b1, b2, t2], axis=1)
        elif nhi == 2 * nlo - 1:      # coarse below, fine above
            j = np.arange(nlo - 1, dtype=np.int64)
            b0 = hi + 2 * j
            b1 = b0 + 1
            b2 = b0 + 2
            t0 = lo + j
            t2 = lo + j + 1
            tt = np.empty((3 * (nlo - 1), 3), dtype=np.int64)
            tt[0::3] = np.stack([t0, b1, b0], axis=1)
            tt[1::3] = np.stack([t0, t2, b1], axis=1)
            tt[2::3] = np.stack([t2, b2, b1], axis=1)
        else:
            raise AssertionError("row counts are not 1:1 or 2:1")
        tris.append(tt)
        bands.append(np.full(tt.shape[0], band, dtype=np.int8))
    tri = np.concatenate(tris, axis=0).astype(np.int32)
    band = np.concatenate(bands)
    d = np.abs(t - half_width)
    a0 = 0.15 * half_width
    a1 = 0.75 * half_width
    psi = np.where(d <= a0, 1.0,
                   np.where(d >= a1, 0.0, 0.5 * (1.0 + np.cos(np.pi * (d - a0) / (a1 - a0)))))
    x = s.copy()
    y = t + amp * np.sin(2.0 * np.pi * s / wavelength) * psi
    # boundary edge sets on x=0 (first node of consecutive rows) and x=length (last nodes)
    first = offs[:-1]
    last = offs[:-1] + np.asarray(counts, dtype=np.int64) - 1
    west = np.stack([first[:-1], first[1:]], axis=1).astype(np.int32)
    east = np.stack([last[:-1], last[1:]], axis=1).astype(np.int32)
    return {"x": x, "y": y, "tri": np.ascontiguousarray(tri), "s": s, "t": t, "d": d,
            "band": band, "length": length, "half_width": half_width, "w2": w2,
            "west_edges": west, "east_edges": east}
