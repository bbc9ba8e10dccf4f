"""Closed-form shallow-water solutions used to pin the oracle (never derived from the oracle or
from the CUDA library).

* Stoker wet-bed dam break  -- the paper's validation case ("analytical
  solution that can be found in Toro (2001)")
* Ritter dry-bed dam break
* right-running simple wave into still water (exact by characteristics until breaking)
"""
import numpy as np
from scipy.optimize import brentq


def stoker_constants(hL, hR, g=9.81):
    """Middle state (h_m, u_m), shock speed, rarefaction head and tail speeds."""
    aL = np.sqrt(g * hL)

    def f(hm):
        um_rar = 2.0 * (aL - np.sqrt(g * hm))                      # left rarefaction invariant
        um_shock = (hm - hR) * np.sqrt(0.5 * g * (hm + hR) / (hm * hR))  # right shock
        return um_rar - um_shock

    hm = brentq(f, hR * (1 + 1e-12), hL, xtol=1e-15, rtol=1e-15)
    um = 2.0 * (aL - np.sqrt(g * hm))
    S = hm * um / (hm - hR)
    return {"hm": hm, "um": um, "shock": S, "head": -aL, "tail": um - np.sqrt(g * hm)}


def stoker(x, t, x0, hL, hR, g=9.81):
    """h, u at positions x and time t>0 for a dam at x0."""
    k = stoker_constants(hL, hR, g)
    aL = np.sqrt(g * hL)
    xi = (np.asarray(x, dtype=np.float64) - x0) / t
    h = np.where(xi < k["head"], hL,
                 np.where(xi < k["tail"], (2.0 * aL - xi) ** 2 / (9.0 * g),
                          np.where(xi < k["shock"], k["hm"], hR)))
    u = np.where(xi < k["head"], 0.0,
                 np.where(xi < k["tail"], 2.0 / 3.0 * (aL + xi),
                          np.where(xi < k["shock"], k["um"], 0.0)))
    return h, u


def ritter(x, t, x0, h0, g=9.81):
    a0 = np.sqrt(g * h0)
    xi = (np.asarray(x, dtype=np.float64) - x0) / t
    h = np.where(xi < -a0, h0, np.where(xi < 2.0 * a0, (2.0 * a0 - xi) ** 2 / (9.0 * g), 0.0))
    u = np.where(xi < -a0, 0.0, np.where(xi < 2.0 * a0, 2.0 / 3.0 * (a0 + xi), 0.0))
    return h, u


def simple_wave(x, t, h0=1.0, a=0.2, w=5.0, x0=30.0, g=9.81):
    """Exact h, u at time t of the right-running simple wave that starts from
    h(x,0)=h0+a exp(-((x-x0)/w)^2), u=2(sqrt(g h)-sqrt(g h0)): solve
    x = xi + (3 sqrt(g h(xi,0)) - 2 sqrt(g h0)) t for xi by bisection (monotone before breaking)."""
    x = np.asarray(x, dtype=np.float64)

    def hinit(xi):
        return h0 + a * np.exp(-((xi - x0) / w) ** 2)

    def speed(xi):
        return 3.0 * np.sqrt(g * hinit(xi)) - 2.0 * np.sqrt(g * h0)

    smax = 3.0 * np.sqrt(g * (h0 + a)) - 2.0 * np.sqrt(g * h0)
    smin = np.sqrt(g * h0)
    lo = x - smax * t - 1e-9
    hi = x - smin * t + 1e-9
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        f = mid + speed(mid) * t - x
        hi = np.where(f > 0, mid, hi)
        lo = np.where(f > 0, lo, mid)
    xi = 0.5 * (lo + hi)
    h = hinit(xi)
    u = 2.0 * (np.sqrt(g * h) - np.sqrt(g * h0))
    return h, u


def cell_average(fun, x, y, tri):
    """Edge-midpoint quadrature (exact for quadratics) of fun(x)->(h,u) on each triangle."""
    acc_h = 0.0
    acc_hu = 0.0
    for k in range(3):
        xm = 0.5 * (x[tri[:, k]] + x[tri[:, (k + 1) % 3]])
        h, u = fun(xm)
        acc_h = acc_h + h
        acc_hu = acc_hu + h * u
    return acc_h / 3.0, acc_hu / 3.0


def tri_areas(x, y, tri):
    return 0.5 * np.abs((x[tri[:, 1]] - x[tri[:, 0]]) * (y[tri[:, 2]] - y[tri[:, 0]])
                        - (x[tri[:, 2]] - x[tri[:, 0]]) * (y[tri[:, 1]] - y[tri[:, 0]]))
