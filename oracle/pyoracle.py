"""ctypes wrapper of the CPU oracle (oracle/swe_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the cpu_baseline /
--impl reference legs of bench.py.  The CUDA library never imports this module.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

SCHEMES = {"hllc": 0, "muscl": 1, "waf": 2, "muscl_ms": 3}
BC_KINDS = {"wall": 0, "inflow": 1, "level": 2, "transmissive": 3}

_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_int64, _ip, C.c_int64, _ip, _ip,
                                 C.c_char_p, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_info.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64),
                               C.POINTER(C.c_int64), _dp]
        L.orc_set_params.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double]
        L.orc_set_manning.argtypes = [C.c_void_p, _dp]
        L.orc_set_bc.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double]
        L.orc_set_state.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.orc_get_state.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.orc_set_time.argtypes = [C.c_void_p, C.c_double]
        L.orc_step.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_int, _dp, _dp]
        L.orc_compute_dt.restype = C.c_double
        L.orc_compute_dt.argtypes = [C.c_void_p, C.c_double]
        L.orc_gradients.argtypes = [C.c_void_p, _dp]
        L.orc_euler_stage.argtypes = [C.c_void_p, C.c_double, C.c_int, _dp, _dp, _dp]
        L.orc_cell_geometry.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
        L.orc_edge_geometry.argtypes = [C.c_void_p, _ip, _ip, _dp, _dp, _dp, _dp]
        L.orc_cell_topology.argtypes = [C.c_void_p, _ip, _ip]
        L.orc_edge_flux.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_int, _dp, _dp]
        L.orc_hllc.argtypes = [C.c_double] * 8 + [_dp]
        L.orc_waf.argtypes = [C.c_double] * 16 + [C.c_int, _dp]
        L.orc_limiter_A.restype = C.c_double
        L.orc_limiter_A.argtypes = [C.c_double, C.c_double]
        L.orc_ms_slope.restype = C.c_double
        L.orc_ms_slope.argtypes = [C.c_double, C.c_double, C.c_double]
        L.orc_manning.argtypes = [C.c_double] * 4 + [_dp, _dp]
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_get_threads.restype = C.c_int
        if hasattr(L, "orc_zones_create"):
            L.orc_zones_create.argtypes = [C.c_void_p, C.c_int, C.c_int, _ip]
            L.orc_zones_step.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_int, _dp, _dp]
            L.orc_zones_counts.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64),
                                           C.POINTER(C.c_int64)]
            L.orc_zones_zone_of_cell.argtypes = [C.c_void_p, _ip]
            L.orc_zones_describe.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int64),
                                             C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
            L.orc_zones_cells.argtypes = [C.c_void_p, C.c_int, _ip, _ip]
            L.orc_zones_links.argtypes = [C.c_void_p, C.c_int, _ip, _ip, _ip]
            L.orc_zones_sendlist.argtypes = [C.c_void_p, C.c_int, C.c_int, _ip]
        _lib = L
    return _lib


def set_threads(n):
    """n<=0: every core OpenMP grants."""
    lib().orc_set_threads(int(n))
    return lib().orc_get_threads()


def hllc(g, h_dry, hL, uL, vL, hR, uR, vR):
    """Returns dict G1,G2,G3,SL,SR,Sstar,hstar,h0 of one HLLC evaluation (A.6)."""
    out = np.zeros(8)
    lib().orc_hllc(g, h_dry, hL, uL, vL, hR, uR, vR, _d(out))
    return dict(zip(["G1", "G2", "G3", "SL", "SR", "Sstar", "hstar", "h0"], out.tolist()))


def waf(g, h_dry, hL, uL, vL, hR, uR, vR, etaL, etaR, etaLupw, etaRupw, vLupw, vRupw, dt, dx,
        use_limiter=True):
    out = np.zeros(3)
    lib().orc_waf(g, h_dry, hL, uL, vL, hR, uR, vR, etaL, etaR, etaLupw, etaRupw, vLupw, vRupw,
                  dt, dx, 1 if use_limiter else 0, _d(out))
    return out


def limiter_A(r, c):
    return lib().orc_limiter_A(float(r), float(c))


def ms_slope(beta, x, y):
    """Limited slope of the multislope MUSCL, eq. 24-25."""
    return lib().orc_ms_slope(float(beta), float(x), float(y))


def manning(g, n, dt, h, hu, hv):
    a = C.c_double(hu)
    b = C.c_double(hv)
    lib().orc_manning(g, n, dt, h, C.byref(a), C.byref(b))
    return a.value, b.value


class Oracle:
    """One mesh + state in the oracle.  Construct from an input dict of swe_inputs.configs."""

    def __init__(self, x, y, zb, tri, bedge=None, btag=None):
        L = lib()
        self.x = np.ascontiguousarray(x, dtype=np.float64)
        self.y = np.ascontiguousarray(y, dtype=np.float64)
        self.zb = np.ascontiguousarray(zb, dtype=np.float64)
        self.tri = np.ascontiguousarray(tri, dtype=np.int32).reshape(-1, 3)
        bedge = np.zeros((0, 2), np.int32) if bedge is None else np.ascontiguousarray(bedge, dtype=np.int32)
        btag = np.zeros((0,), np.int32) if btag is None else np.ascontiguousarray(btag, dtype=np.int32)
        err = C.create_string_buffer(256)
        self._h = L.orc_create(self.x.size, _d(self.x), _d(self.y), _d(self.zb), self.tri.shape[0],
                               _i(self.tri), btag.size, _i(bedge), _i(btag), err, 256)
        if not self._h:
            raise ValueError("oracle mesh error: " + err.value.decode())
        nt, ne, nbe = C.c_int64(), C.c_int64(), C.c_int64()
        mr = C.c_double()
        L.orc_info(self._h, C.byref(nt), C.byref(ne), C.byref(nbe), C.byref(mr))
        self.nt, self.ne, self.nbe, self.min_inradius = nt.value, ne.value, nbe.value, mr.value

    @classmethod
    def from_config(cls, cfg):
        o = cls(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], cfg["bedge"], cfg["btag"])
        p = cfg["params"]
        o.set_params(p["g"], p["h_dry"], p["h_thin"], p["beta"])
        for tag, (kind, value) in cfg["bc"].items():
            o.set_bc(tag, kind, value)
        if cfg.get("manning") is not None:
            o.set_manning(cfg["manning"])
        o.set_state(cfg["h"], cfg["hu"], cfg["hv"])
        return o

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_params(self, g=9.81, h_dry=1e-6, h_thin=1e-3, beta=1.0):
        lib().orc_set_params(self._h, g, h_dry, h_thin, beta)

    def set_manning(self, n):
        if n is None:
            lib().orc_set_manning(self._h, None)
        else:
            n = np.ascontiguousarray(n, dtype=np.float64)
            assert n.size == self.nt
            lib().orc_set_manning(self._h, _d(n))

    def set_bc(self, tag, kind, value=0.0):
        k = BC_KINDS[kind] if isinstance(kind, str) else int(kind)
        if lib().orc_set_bc(self._h, int(tag), k, float(value)) != 0:
            raise ValueError("bad bc")

    def set_state(self, h, hu, hv):
        h = np.ascontiguousarray(h, dtype=np.float64)
        hu = np.ascontiguousarray(hu, dtype=np.float64)
        hv = np.ascontiguousarray(hv, dtype=np.float64)
        assert h.size == hu.size == hv.size == self.nt
        if lib().orc_set_state(self._h, _d(h), _d(hu), _d(hv)) != 0:
            raise ValueError("bad state (NaN or negative depth)")

    def get_state(self):
        h = np.empty(self.nt)
        hu = np.empty(self.nt)
        hv = np.empty(self.nt)
        lib().orc_get_state(self._h, _d(h), _d(hu), _d(hv))
        return h, hu, hv

    def step(self, nsteps, cfl, scheme):
        s = SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
        t = C.c_double()
        dt = C.c_double()
        if lib().orc_step(self._h, int(nsteps), float(cfl), s, C.byref(t), C.byref(dt)) != 0:
            raise ValueError("bad step arguments")
        return t.value, dt.value

    def compute_dt(self, cfl):
        return lib().orc_compute_dt(self._h, float(cfl))

    def gradients(self):
        out = np.empty((self.nt, 8))
        lib().orc_gradients(self._h, _d(out))
        return out

    def euler_stage(self, dt, scheme):
        s = SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
        h = np.empty(self.nt)
        hu = np.empty(self.nt)
        hv = np.empty(self.nt)
        lib().orc_euler_stage(self._h, float(dt), s, _d(h), _d(hu), _d(hv))
        return h, hu, hv

    def cell_geometry(self):
        a = {k: np.empty(self.nt) for k in ("area", "cx", "cy", "zc", "rin")}
        lib().orc_cell_geometry(self._h, _d(a["area"]), _d(a["cx"]), _d(a["cy"]), _d(a["zc"]), _d(a["rin"]))
        return a

    def edge_geometry(self):
        eL = np.empty(self.ne, np.int32)
        eR = np.empty(self.ne, np.int32)
        a = {k: np.empty(self.ne) for k in ("len", "nx", "ny", "dx")}
        lib().orc_edge_geometry(self._h, _i(eL), _i(eR), _d(a["len"]), _d(a["nx"]), _d(a["ny"]), _d(a["dx"]))
        a["eL"], a["eR"] = eL, eR
        return a

    def cell_topology(self):
        c2c = np.empty((self.nt, 3), np.int32)
        c2e = np.empty((self.nt, 3), np.int32)
        lib().orc_cell_topology(self._h, _i(c2c), _i(c2e))
        return c2c, c2e

    def edge_flux(self, e, dt, scheme):
        s = SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
        a = np.zeros(3)
        b = np.zeros(3)
        if lib().orc_edge_flux(self._h, int(e), float(dt), s, _d(a), _d(b)) != 0:
            raise ValueError("bad edge")
        return a, b

    # ---- zones (A.12) ----
    def zones_create(self, nzones, nlayers, zone_of_cell=None):
        z = None if zone_of_cell is None else np.ascontiguousarray(zone_of_cell, dtype=np.int32)
        rc = lib().orc_zones_create(self._h, int(nzones), int(nlayers), None if z is None else _i(z))
        if rc != 0:
            raise ValueError("zones_create failed (%d)" % rc)

    def zones_step(self, nsteps, cfl, scheme):
        s = SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
        t = C.c_double()
        dt = C.c_double()
        rc = lib().orc_zones_step(self._h, int(nsteps), float(cfl), s, C.byref(t), C.byref(dt))
        if rc != 0:
            raise ValueError("zones_step failed (%d)" % rc)
        return t.value, dt.value

    def zones_counts(self):
        a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
        lib().orc_zones_counts(self._h, C.byref(a), C.byref(b), C.byref(c))
        return {"send_cells_total": a.value, "bytes_per_exchange": b.value, "ghost_cells_total": c.value}

    def zones_zone_of_cell(self):
        z = np.empty(self.nt, np.int32)
        lib().orc_zones_zone_of_cell(self._h, _i(z))
        return z

    def zones_describe(self, zone):
        """Returns owned cell ids, ghost cell ids (global), ghost layers, and the links:
        list of (source zone, recv_start, count, send list as source-local indices)."""
        no, ng, nl = C.c_int64(), C.c_int64(), C.c_int64()
        lib().orc_zones_describe(self._h, int(zone), C.byref(no), C.byref(ng), C.byref(nl))
        cells = np.empty(no.value + ng.value, np.int32)
        layer = np.empty(no.value + ng.value, np.int32)
        lib().orc_zones_cells(self._h, int(zone), _i(cells), _i(layer))
        src = np.empty(nl.value, np.int32)
        start = np.empty(nl.value, np.int32)
        cnt = np.empty(nl.value, np.int32)
        lib().orc_zones_links(self._h, int(zone), _i(src), _i(start), _i(cnt))
        links = []
        for j in range(nl.value):
            sl = np.empty(cnt[j], np.int32)
            lib().orc_zones_sendlist(self._h, int(zone), j, _i(sl))
            links.append((int(src[j]), int(start[j]), int(cnt[j]), sl))
        return {"nowned": no.value, "cells": cells, "layer": layer, "links": links}
