"""Counter-based lattice value noise and Gaussian-bump bathymetry (input recipe).

The lattice values come from an integer hash of (ix, iy, octave, seed), so the same field can be
regenerated anywhere without carrying generator state.
"""
import numpy as np

_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_G = np.uint64(0x9E3779B97F4A7C15)


def _mix64(z):
    """splitmix64 finaliser on a uint64 array (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def lattice_hash(ix, iy, octave, seed):
    """U[-1,1) value attached to lattice point (ix, iy) of a given octave and seed."""
    ix = np.asarray(ix, dtype=np.int64).astype(np.uint64)
    iy = np.asarray(iy, dtype=np.int64).astype(np.uint64)
    with np.errstate(over="ignore"):
        k = _mix64(ix * _G + np.uint64(octave + 1))
        k = _mix64(k ^ (iy * _M2 + np.uint64(seed) * _M1))
    # top 53 bits -> [0,1)
    u = (k >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    return 2.0 * u - 1.0


def value_noise(x, y, seed, octaves, amplitude, lambda0):
    """Sum of `octaves` octaves of bilinear (smoothstep) lattice noise.

    Octave o has lattice spacing lambda0 / 2**o and amplitude `amplitude` / 2**o.
    """
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    out = np.zeros_like(x)
    for o in range(octaves):
        lam = lambda0 / (2 ** o)
        amp = amplitude / (2 ** o)
        fx = x / lam
        fy = y / lam
        ix = np.floor(fx)
        iy = np.floor(fy)
        tx = fx - ix
        ty = fy - iy
        sx = tx * tx * (3.0 - 2.0 * tx)
        sy = ty * ty * (3.0 - 2.0 * ty)
        ix = ix.astype(np.int64)
        iy = iy.astype(np.int64)
        v00 = lattice_hash(ix, iy, o, seed)
        v10 = lattice_hash(ix + 1, iy, o, seed)
        v01 = lattice_hash(ix, iy + 1, o, seed)
        v11 = lattice_hash(ix + 1, iy + 1, o, seed)
        a = v00 + sx * (v10 - v00)
        b = v01 + sx * (v11 - v01)
        out += amp * (a + sy * (b - a))
    return out


def gaussian_bumps(x, y, seed, n, extent, hmin, hmax, wmin, wmax):
    """Sum of n Gaussian bumps H_k exp(-r^2 / (2 W_k^2)); H~U[hmin,hmax], W~U[wmin,wmax],
    centres U[0,extent]^2 (BASELINE.json configs[2])."""
    rng = np.random.default_rng(seed)
    H = rng.uniform(hmin, hmax, n)
    W = rng.uniform(wmin, wmax, n)
    cx = rng.uniform(0.0, extent, n)
    cy = rng.uniform(0.0, extent, n)
    z = np.zeros_like(np.asarray(x, dtype=np.float64))
    for k in range(n):
        r2 = (x - cx[k]) ** 2 + (y - cy[k]) ** 2
        z += H[k] * np.exp(-r2 / (2.0 * W[k] * W[k]))
    return z
