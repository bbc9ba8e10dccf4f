"""Pins for the oracle's open boundaries ("incoming flow Q", and the fixed water level
the paper uses at PAPER.md:518, 548 without defining it; readings R10, R11) against what
the mathematics fixes, on a straight flat channel with inflow Q upstream and a level downstream:

 * uniform subcritical flow h = level, u = Q/(W h) is an exact steady solution of the equations
   and of both boundary formulas: it must be preserved to round-off by every scheme (a wrong sign,
   magnitude or per-width distribution of Q, or a wrong ghost depth, breaks it at once);
 * with Manning friction the steady state is the gradually-varied-flow (backwater) profile
       dh/dx = -S_f / (1 - Fr^2),  S_f = n^2 q^2 / h^(10/3),  Fr^2 = q^2 / (g h^3),  h(L) = level,
   a textbook ODE integrated here with scipy, independently of the oracle: the oracle started from
   still water must relax to it (first-order accurate: the error halves with the mesh size), with
   the discharge per unit width equal to Q / W along the whole channel.
"""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import swe_inputs as si
from oracle import pyoracle as po

G = 9.81


@pytest.mark.parametrize("scheme,cfl", [("hllc", 0.9), ("muscl", 0.45), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_uniform_flow_is_an_exact_steady_state(scheme, cfl, oracle_threads):
    Q, level, W = 10.0, 2.0, 5.0
    u0 = Q / (W * level)                       # Fr = 0.23: subcritical
    cfg = si.channel_flow_case(discharge=Q, level=level, u_init=u0)
    o = po.Oracle.from_config(cfg)
    o.step(200, cfl, scheme)
    h, hu, hv = o.get_state()
    assert np.abs(h - level).max() < 1e-13
    assert np.abs(hu - level * u0).max() < 1e-13
    assert np.abs(hv).max() < 1e-13


def test_wrong_discharge_does_not_keep_the_uniform_flow(oracle_threads):
    # the same state with half the discharge imposed is NOT steady: the pin above can fail
    cfg = si.channel_flow_case(discharge=5.0, level=2.0, u_init=1.0)
    o = po.Oracle.from_config(cfg)
    o.step(50, 0.9, "hllc")
    h, hu, hv = o.get_state()
    assert np.abs(hu - 2.0).max() > 0.1


def _backwater(x, q, n, level, length):
    f = lambda s, h: -(n * n * q * q / h ** (10.0 / 3.0)) / (1.0 - q * q / (G * h ** 3))
    sol = solve_ivp(f, [length, 0.0], [level], dense_output=True, rtol=1e-10, atol=1e-12)
    return sol.sol(x)[0]


def _relax(scheme, cfl, nx, steps):
    n, Q, level, lx, ly = 0.03, 20.0, 1.0, 200.0, 10.0
    cfg = si.channel_flow_case(nx=nx, ny=nx // 20, lx=lx, ly=ly, discharge=Q, level=level, manning=n)
    o = po.Oracle.from_config(cfg)
    o.step(steps, cfl, scheme)
    h, hu, hv = o.get_state()
    cx = cfg["x"][cfg["tri"]].mean(axis=1)
    he = _backwater(cx, Q / ly, n, level, lx)
    return h, hu, hv, cx, he, Q / ly


def test_backwater_curve_hllc_first_order(oracle_threads):
    errs = []
    for nx, steps in ((100, 8000), (200, 16000)):
        h, hu, hv, cx, he, q = _relax("hllc", 0.9, nx, steps)
        errs.append(np.abs(h - he).mean() / he.mean())
        assert np.abs(hu - q).max() < 0.01 * q            # discharge per unit width = Q / W everywhere
        assert np.abs(hv).max() < 0.01 * q
        # inlet depth of the M-type curve (1.447 m for these numbers) and the imposed outlet level
        assert abs(h[cx < 4.0].mean() - he[cx < 4.0].mean()) < 5e-3
        assert abs(h[cx > 196.0].mean() - he[cx > 196.0].mean()) < 5e-3
    assert errs[0] < 1.0e-3 and errs[1] < 0.6 * errs[0], errs
    assert 1.40 < h[cx < 4.0].mean() < 1.46           # the M-type curve rises 0.44 m above the level


@pytest.mark.parametrize("scheme,cfl", [("muscl", 0.45), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_backwater_curve_second_order_schemes(scheme, cfl, oracle_threads):
    h, hu, hv, cx, he, q = _relax(scheme, cfl, 100, 12000)
    assert np.abs(h - he).mean() / he.mean() < 1.0e-3
    assert np.abs(h - he).max() < 0.01
    assert np.abs(hu - q).max() < 0.025 * q


def test_backwater_reference_is_the_textbook_curve():
    # the ODE solution used above against its own closed-form check: x(h) by quadrature of
    # dx/dh = -(1 - Fr^2)/S_f from the outlet depth (independent of solve_ivp)
    q, n, level, L = 2.0, 0.03, 1.0, 200.0
    hs = np.linspace(level, 1.4, 4001)
    dxdh = -(1.0 - q * q / (G * hs ** 3)) / (n * n * q * q / hs ** (10.0 / 3.0))
    x_of_h = L + np.concatenate([[0.0], np.cumsum(0.5 * (dxdh[1:] + dxdh[:-1]) * np.diff(hs))])
    for k in (500, 2000, 4000):
        assert abs(_backwater(np.array([x_of_h[k]]), q, n, level, L)[0] - hs[k]) < 1e-6


@pytest.mark.parametrize("scheme,cfl,keep", [("muscl", 0.45, 0.9), ("hllc", 0.9, 0.8), ("waf", 0.45, 0.85),
                                             ("muscl_ms", 0.45, 0.85)])
def test_fixed_level_boundary_reflects_with_coefficient_minus_one(scheme, cfl, keep, oracle_threads):
    """Transient behaviour of the fixed-level boundary (the outgoing Riemann invariant of R11):
    linear theory -- a boundary that holds the free surface reflects a small long wave with
    coefficient -1 in elevation and +1 in velocity.  A right-running simple-wave pulse of amplitude
    a = 1 cm on h0 = 1 m, centred at x0 = 60 m, comes back inverted: after t = (100 - x0)/c +
    50/c its trough sits at x = 50 m with eta = -a and u = +a c / h0 (less the scheme's damping).
    A wall-like treatment, or the invariant with the wrong sign, returns a crest instead."""
    h0, a, x0, w = 1.0, 0.01, 60.0, 6.0
    cfg = si.channel_flow_case(nx=400, ny=4, lx=100.0, ly=1.0, jitter=0.1, discharge=0.0, level=h0)
    cx = cfg["x"][cfg["tri"]].mean(axis=1)
    h = h0 + a * np.exp(-((cx - x0) / w) ** 2)
    cfg["h"] = h
    cfg["hu"] = h * 2.0 * (np.sqrt(G * h) - np.sqrt(G * h0))       # right-running simple wave
    o = po.Oracle.from_config(cfg)
    c = np.sqrt(G * h0)
    T = (100.0 - x0) / c + 50.0 / c
    t, _ = o.step(int(0.98 * T / o.compute_dt(cfl)), cfl, scheme)   # dt is almost constant (a << h0)
    while t < T:
        t, _ = o.step(1, cfl, scheme)
    hh, hu, hv = o.get_state()
    eta = hh - h0
    i = int(np.argmin(eta))
    assert -1.02 * a < eta[i] < -keep * a                  # inverted, amplitude kept up to the damping
    assert abs(cx[i] - 50.0) < 3.0                         # where linear theory puts it
    assert eta.max() < 0.05 * a                            # no crest comes back
    u = hu[i] / hh[i]
    assert keep * a * c / h0 < u < 1.05 * a * c / h0       # velocity perturbation keeps its sign


@pytest.mark.parametrize("scheme,cfl", [("hllc", 0.9), ("muscl", 0.45), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_inflow_onto_a_dry_bed_fills_the_channel_with_Q_t(scheme, cfl, oracle_threads):
    """Imposed discharge onto a dry bed (reading R10): whatever the momentum part of the boundary flux
    on a dry face, the mass part is q_n = -Q / W on every tagged edge, so a closed channel holds
    exactly Q t of water after time t (to round-off), depths never go negative, and the water has
    got as far as a front moving at a few m/s can -- not further, not nowhere.  (The pool is 0.5 m
    deep: with a 5 cm film the inflow is a Froude-17 jet, the second Heun stage -- which uses the
    dt of U^n, A.2 -- overshoots, and the clamp h' = max(h', 0) of A.10 creates mass in the first
    steps of MUSCL / MUSCL_MS, 0.24 m3 here; HLLC and WAF stay exact.  DESIGN.md, tolerances.)"""
    Q, lx, ly = 3.0, 100.0, 5.0
    cfg = si.channel_flow_case(nx=200, ny=10, lx=lx, ly=ly, discharge=Q, level=0.0, h_init=0.0)
    cfg["bc"] = {1: ("inflow", Q), 2: ("wall", 0.0)}
    o = po.Oracle.from_config(cfg)
    assert o.compute_dt(cfl) == 0.0                        # nothing is wet yet: dt = 0, the step is a no-op
    # a pool next to the inlet gets the clock going (its volume is accounted for)
    import closed_forms as cf
    cx = cfg["x"][cfg["tri"]].mean(axis=1)
    area = cf.tri_areas(cfg["x"], cfg["y"], cfg["tri"])
    h0 = np.where(cx < 4.0, 0.5, 0.0)
    o.set_state(h0, np.zeros_like(h0), np.zeros_like(h0))
    v0 = float((h0 * area).sum())
    t, _ = o.step(600, cfl, scheme)
    h, hu, hv = o.get_state()
    assert h.min() >= 0.0
    vol = float((h * area).sum())
    assert abs(vol - (v0 + Q * t)) < 1e-11 * (v0 + Q * t)
    front = cx[h > 1e-3].max()
    assert 5.0 < front and (front < lx - 1.0 or t > 10.0)
    assert t > 1.0
