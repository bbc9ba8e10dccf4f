"""Pins of the oracle's flux functions against what the paper and the mathematics fix
(no GPU, no CUDA library).  Citations: PAPER.md line numbers; readings R# = DESIGN.md."""
import os

import numpy as np
import pytest

from oracle import pyoracle as po

G = 9.81
HD = 1e-6
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.split("#")[0].replace("|", " ").strip()
            if line:
                out.append([float(v) for v in line.split()])
    return out


def phys_flux(h, u, v):
    """G(U) of eq. 1."""
    return np.array([h * u, h * u * u + 0.5 * G * h * h, h * u * v])


def test_superbee_table_eq21():
    for r, c, A in _rows("superbee_eq21.txt"):
        assert po.limiter_A(r, c) == pytest.approx(A, abs=1e-15), (r, c)


def test_superbee_properties():
    # A(r,c) = 1 - (1-|c|) phi(r) with the SUPERBEE flux limiter phi: phi(1)=1,
    # phi in [0,2], A(r,1) = 1 for every r (a wave that crosses the whole cell is fully upwinded)
    for r in np.linspace(-2, 5, 57):
        assert po.limiter_A(r, 1.0) == pytest.approx(1.0, abs=1e-15)
        assert po.limiter_A(r, -1.0) == pytest.approx(1.0, abs=1e-15)
        for c in (0.0, 0.2, 0.7):
            phi = (1.0 - po.limiter_A(r, c)) / (1.0 - c)
            sb = max(0.0, min(2.0 * r, 1.0), min(r, 2.0))  # textbook SUPERBEE
            assert phi == pytest.approx(sb, abs=1e-14), (r, c)


def test_hllc_consistency_equal_states():
    # G~(U,U) = G(U) exactly (invariant of eq. 6-7, 13)
    rng = np.random.default_rng(0)
    for _ in range(200):
        h = rng.uniform(0.01, 20)
        u = rng.uniform(-15, 15)
        v = rng.uniform(-5, 5)
        r = po.hllc(G, HD, h, u, v, h, u, v)
        np.testing.assert_allclose([r["G1"], r["G2"], r["G3"]], phys_flux(h, u, v), rtol=1e-15, atol=1e-15)


def test_hllc_mirror_symmetry():
    # flux(L,R;n) = -flux(R,L;-n): in the frame of -n the states swap and both velocity
    # components change sign; mass flux changes sign, momentum-flux components keep theirs,
    # and T_{-n}^{-1} flips them (eq. 2)
    rng = np.random.default_rng(1)
    for _ in range(300):
        hL, hR = rng.uniform(0.01, 10, 2)
        uL, uR = rng.uniform(-6, 6, 2)
        vL, vR = rng.uniform(-3, 3, 2)
        a = po.hllc(G, HD, hL, uL, vL, hR, uR, vR)
        b = po.hllc(G, HD, hR, -uR, -vR, hL, -uL, -vL)
        assert b["G1"] == pytest.approx(-a["G1"], rel=1e-12, abs=1e-12)
        assert b["G2"] == pytest.approx(a["G2"], rel=1e-12, abs=1e-12)
        assert b["G3"] == pytest.approx(a["G3"], rel=1e-12, abs=1e-12)
        assert b["SL"] == pytest.approx(-a["SR"], rel=1e-12, abs=1e-12)


def test_hllc_supercritical_is_upwind():
    # eq. 6: S_L >= 0 -> G(U_L); S_R <= 0 -> G(U_R)
    r = po.hllc(G, HD, 1.0, 10.0, 0.5, 1.1, 10.0, -0.5)
    assert r["SL"] > 0
    np.testing.assert_allclose([r["G1"], r["G2"], r["G3"]], phys_flux(1.0, 10.0, 0.5), rtol=1e-15)
    r = po.hllc(G, HD, 1.0, -10.0, 0.5, 1.1, -10.0, -0.5)
    assert r["SR"] < 0
    np.testing.assert_allclose([r["G1"], r["G2"], r["G3"]], phys_flux(1.1, -10.0, -0.5), rtol=1e-15)


def test_hllc_star_flux_is_eq7():
    # the cancellation-free form must equal eq. 7 as printed, here written with the
    # returned speeds for a subcritical case
    hL, uL, vL, hR, uR, vR = 2.0, 1.0, 0.5, 1.0, -0.5, -0.25
    r = po.hllc(G, HD, hL, uL, vL, hR, uR, vR)
    SL, SR = r["SL"], r["SR"]
    GL, GR = phys_flux(hL, uL, vL), phys_flux(hR, uR, vR)
    UL, UR = np.array([hL, hL * uL]), np.array([hR, hR * uR])
    star = (SR * GL[:2] - SL * GR[:2] + SR * SL * (UR - UL)) / (SR - SL)
    np.testing.assert_allclose([r["G1"], r["G2"]], star, rtol=1e-13)
    # eq. 14 as printed
    Ss = (SL * hR * (uR - SR) - SR * hL * (uL - SL)) / (hR * (uR - SR) - hL * (uL - SL))
    assert r["Sstar"] == pytest.approx(Ss, rel=1e-13)
    # eq. 13 (reading R2): contact moving right carries the left tangential velocity
    assert Ss > 0 and r["G3"] == pytest.approx(r["G1"] * vL, rel=1e-15)


def test_hllc_wave_speed_estimates_bracket_exact_stoker():
    # two-rarefaction / two-shock depth estimate (eq. 10-12) against the exact Riemann solution
    # of the Stoker problems (closed form): h* within 1 %, S_L = exact rarefaction head, S_R
    # within 0.5 % of the exact shock speed (reading R1: p_R = sqrt(h*(h*+h_R)/2)/h_R is the exact
    # shock relation evaluated at the estimated h*)
    for hL, hR, hm, um, shock, head, tail in _rows("stoker_constants.txt"):
        r = po.hllc(G, HD, hL, 0.0, 0.0, hR, 0.0, 0.0)
        assert r["SL"] == pytest.approx(head, rel=1e-11)
        assert r["hstar"] == pytest.approx(hm, rel=1e-2)
        assert r["SR"] == pytest.approx(shock, rel=5e-3)
        # exact shock relation: with the exact h_m the printed reading returns the exact speed
        exact = np.sqrt(G * hR) * np.sqrt(0.5 * hm * (hm + hR)) / hR
        assert exact == pytest.approx(shock, rel=1e-11)


def test_hllc_dry_bed_speeds_match_ritter_front():
    # reading R13: right side dry -> S_L = u_L - a_L (rarefaction head), S_R = u_L + 2 a_L
    # (the Ritter front speed 2 sqrt(g h0))
    r = po.hllc(G, HD, 4.0, 0.0, 0.0, 0.0, 0.0, 0.0)
    a = np.sqrt(G * 4.0)
    assert r["SL"] == pytest.approx(-a, rel=1e-15)
    assert r["SR"] == pytest.approx(2 * a, rel=1e-15)
    assert r["G1"] > 0
    m = po.hllc(G, HD, 0.0, 0.0, 0.0, 4.0, 0.0, 0.0)
    assert m["G1"] == pytest.approx(-r["G1"], rel=1e-14)
    z = po.hllc(G, HD, 0.0, 0.0, 0.0, 0.5e-6, 3.0, 0.0)
    assert (z["G1"], z["G2"], z["G3"]) == (0.0, 0.0, 0.0)


def test_hllc_cross_check_survey_table():
    for row in _rows("hllc_survey_c2.txt"):
        hL, uL, vL, hR, uR, vR, h0, hs, SL, SR, Ss, G1, G2, G3 = row
        r = po.hllc(G, HD, hL, uL, vL, hR, uR, vR)
        got = [r["h0"], r["hstar"], r["SL"], r["SR"], r["Sstar"], r["G1"], r["G2"], r["G3"]]
        np.testing.assert_allclose(got, [h0, hs, SL, SR, Ss, G1, G2, G3], rtol=2e-11, atol=1e-11)


# ------------------------------------------------------------------------------------------ WAF
def _waf(hL, uL, vL, hR, uR, vR, dt, dx, lim, up=None):
    etaL, etaR = hL, hR
    if up is None:
        up = (etaL, etaR, vL, vR)
    return po.waf(G, HD, hL, uL, vL, hR, uR, vR, etaL, etaR, up[0], up[1], up[2], up[3], dt, dx, lim)


def test_waf_with_A_equal_one_is_hll_flux():
    # eq. 18 with A=1 gives weights that select the upwind HLL flux of eq. 6 (reading R6)
    rng = np.random.default_rng(2)
    n = {"sub": 0, "supL": 0, "supR": 0}
    for _ in range(400):
        hL, hR = rng.uniform(0.05, 5, 2)
        uL, uR = rng.uniform(-8, 8, 2)
        vL, vR = rng.uniform(-2, 2, 2)
        r = po.hllc(G, HD, hL, uL, vL, hR, uR, vR)
        if r["SL"] == 0.0 or r["SR"] == 0.0 or r["SR"] <= r["SL"]:
            continue
        n["supL" if r["SL"] > 0 else ("supR" if r["SR"] < 0 else "sub")] += 1
        w = _waf(hL, uL, vL, hR, uR, vR, 0.01, 1.0, False)
        sc = max(1.0, abs(r["G1"]), abs(r["G2"]))
        assert abs(w[0] - r["G1"]) <= 1e-12 * sc
        assert abs(w[1] - r["G2"]) <= 1e-12 * sc
        # third component: A=1 upwinds on S* exactly like eq. 13 (reading R2)
        if r["Sstar"] != 0.0:
            assert abs(w[2] - r["G3"]) <= 1e-12 * max(1.0, abs(r["G3"]))
    assert min(n.values()) > 5


def test_waf_equal_states_returns_physical_flux_exactly():
    w = _waf(2.0, 0.7, -0.3, 2.0, 0.7, -0.3, 0.02, 1.0, True)
    np.testing.assert_array_equal(w, phys_flux(2.0, 0.7, -0.3))


def test_waf_unlimited_weights_are_eq17():
    # with r in (1/2, 1] the limiter returns A=|c| and eq. 18 must reduce to eq. 17
    hL, uL, vL, hR, uR, vR = 1.2, 0.3, 0.2, 1.0, 0.1, -0.1
    dt, dx = 0.05, 1.0
    r = po.hllc(G, HD, hL, uL, vL, hR, uR, vR)
    # choose upwind values so that every ratio r_k = 0.75
    dl = hR - hL
    dv = vR - vL
    up = (hL - 0.75 * dl, hR + 0.75 * dl, vL - 0.75 * dv, vR + 0.75 * dv)
    w = _waf(hL, uL, vL, hR, uR, vR, dt, dx, True, up)
    cL, cR, cS = r["SL"] * dt / dx, r["SR"] * dt / dx, r["Sstar"] * dt / dx
    GL, GR = phys_flux(hL, uL, vL), phys_flux(hR, uR, vR)
    SL, SR = r["SL"], r["SR"]
    UL, UR = np.array([hL, hL * uL]), np.array([hR, hR * uR])
    star = (SR * GL[:2] - SL * GR[:2] + SR * SL * (UR - UL)) / (SR - SL)
    wL, wR, wLR = (1 + cL) / 2, (1 - cR) / 2, (cR - cL) / 2             # eq. 17
    expect = wL * GL[:2] + wLR * star + wR * GR[:2]                      # eq. 15 (reading R3)
    np.testing.assert_allclose(w[:2], expect, rtol=1e-13)
    exp3 = ((1 + cS) / 2 * vL + (1 - cS) / 2 * vR) * expect[0]           # eq. 16
    assert w[2] == pytest.approx(exp3, rel=1e-13)


def _waf_1d_error(n, T=3.0, cfl=0.9):
    """1-D finite-volume driver (test code) around the oracle's WAF flux function: uniform grid on
    [0,100], simple wave of SURVEY Appendix C.3, transmissive ends."""
    from closed_forms import simple_wave
    dx = 100.0 / n
    xe = np.linspace(0.0, 100.0, n + 1)
    # Simpson cell averages
    def avg(f):
        a, m, b = f(xe[:-1]), f(0.5 * (xe[:-1] + xe[1:])), f(xe[1:])
        return (a + 4 * m + b) / 6.0
    h = avg(lambda x: simple_wave(x, 0.0)[0])
    hu = avg(lambda x: simple_wave(x, 0.0)[0] * simple_wave(x, 0.0)[1])
    t = 0.0
    while t < T:
        u = hu / h
        dt = cfl * dx / np.max(np.abs(u) + np.sqrt(G * h))
        dt = min(dt, T - t)
        hp = np.concatenate([[h[0], h[0]], h, [h[-1], h[-1]]])
        up = np.concatenate([[u[0], u[0]], u, [u[-1], u[-1]]])
        F = np.zeros((n + 1, 2))
        for i in range(n + 1):
            L, R = i + 1, i + 2
            w = po.waf(G, HD, hp[L], up[L], 0.0, hp[R], up[R], 0.0, hp[L], hp[R], hp[L - 1], hp[R + 1],
                       0.0, 0.0, dt, dx, True)
            F[i] = w[:2]
        h = h - dt / dx * (F[1:, 0] - F[:-1, 0])
        hu = hu - dt / dx * (F[1:, 1] - F[:-1, 1])
        t += dt
    he = avg(lambda x: simple_wave(x, T)[0])
    return np.abs(h - he).sum() * dx / 100.0


def test_waf_flux_is_second_order_in_1d():
    # Toro's WAF is second order in space and time for smooth flow
    e = [_waf_1d_error(n) for n in (200, 400, 800)]
    o1, o2 = np.log2(e[0] / e[1]), np.log2(e[1] / e[2])
    assert o1 > 1.7 and o2 > 1.85, (e, o1, o2)


def test_manning_is_exact_solution_of_friction_ode():
    # du/dt = -(g n^2 / h^(4/3)) u |u| at constant h, integrated numerically by an ODE library
    from scipy.integrate import solve_ivp
    g, n, dt, h = 9.81, 0.03, 0.7, 0.4
    hu0, hv0 = 0.9, -0.5
    k = g * n * n / h ** (4.0 / 3.0)

    def rhs(t, y):
        s = np.hypot(y[0], y[1])
        return [-k * s * y[0], -k * s * y[1]]

    sol = solve_ivp(rhs, [0, dt], [hu0 / h, hv0 / h], rtol=1e-12, atol=1e-14)
    a, b = po.manning(g, n, dt, h, hu0, hv0)
    assert a / h == pytest.approx(sol.y[0, -1], rel=1e-9)
    assert b / h == pytest.approx(sol.y[1, -1], rel=1e-9)
