"""Parity norm shared by the GPU-vs-oracle tests.

Per field, max_i |a_i - b_i| / scale: scale = max|h_ref| for the depth; for the two momentum
components the common scale max(max|hu_ref|, max|hv_ref|, 1e-3 * h_max * sqrt(g h_max)) -- the
floor keeps the norm meaningful on a lake at rest, where the momenta are round-off noise (their
size is checked separately against the 1e-12 velocity bound)."""
import numpy as np


def rel_errors(ref, got, g=9.81):
    h, hu, hv = [np.asarray(a) for a in ref]
    H, HU, HV = [np.asarray(a) for a in got]
    hmax = max(float(np.max(np.abs(h))), 1e-300)
    qs = max(float(np.max(np.abs(hu))), float(np.max(np.abs(hv))), 1e-3 * hmax * np.sqrt(g * hmax))
    return {"h": float(np.max(np.abs(H - h))) / hmax,
            "hu": float(np.max(np.abs(HU - hu))) / qs,
            "hv": float(np.max(np.abs(HV - hv))) / qs}


def assert_parity(ref, got, tol, h_dry=1e-6, what=""):
    for a in got:
        assert np.all(np.isfinite(a)), what + " non-finite values"
    e = rel_errors(ref, got)
    assert max(e.values()) <= tol, "%s parity %s > %g" % (what, e, tol)
    m_ref = np.asarray(ref[0]) > h_dry
    m_got = np.asarray(got[0]) > h_dry
    nflip = int(np.count_nonzero(m_ref != m_got))
    assert nflip == 0, "%s wet/dry masks differ in %d cells" % (what, nflip)
    return e
