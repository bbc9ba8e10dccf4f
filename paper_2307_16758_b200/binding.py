"""Thin ctypes binding of include/swe_b200.h: same names, argument marshalling only.

Every array argument may be a numpy array (host pointer) or a torch tensor (host or CUDA: its
data_ptr() is passed straight through).  Nothing here computes: every step of the path runs in the
CUDA kernels of libswe_b200.so.  There is no CPU fallback: if the library is missing it is built
with nvcc, and if that fails the import raises.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

SWE_OK = 0
SWE_ERR_ARG, SWE_ERR_MESH, SWE_ERR_CUDA, SWE_ERR_STATE, SWE_ERR_NOMEM = -1, -2, -3, -4, -5
SWE_HLLC, SWE_MUSCL, SWE_WAF, SWE_MUSCL_MS = 0, 1, 2, 3
SWE_BC_WALL, SWE_BC_INFLOW_Q, SWE_BC_LEVEL, SWE_BC_TRANSMISSIVE = 0, 1, 2, 3
SWE_RENUM_NONE, SWE_RENUM_HILBERT, SWE_RENUM_RCM = 0, 1, 2
SWE_STATIC_MAX_CELLS = 262144      # include/swe_b200.h: the most cells swe_get_state_static serves
SCHEMES = {"hllc": SWE_HLLC, "muscl": SWE_MUSCL, "waf": SWE_WAF, "muscl_ms": SWE_MUSCL_MS}
BC_KINDS = {"wall": SWE_BC_WALL, "inflow": SWE_BC_INFLOW_Q, "level": SWE_BC_LEVEL,
            "transmissive": SWE_BC_TRANSMISSIVE}
KERNEL_KINDS = ("dt_reduce", "grad_limit", "edge_flux", "cell_update", "pack", "unpack", "dt_finalize")

_lib = None
_vp, _i64p, _dp = C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_double)

# name -> (restype, argtypes); also the list of symbols the header declares
SIGNATURES = {
    "swe_mesh_create": (C.c_int, [C.POINTER(_vp), C.c_int64, _vp, _vp, _vp, C.c_int64, _vp, C.c_int64, _vp, _vp, C.c_int, _vp]),
    "swe_mesh_destroy": (C.c_int, [_vp]),
    "swe_mesh_info": (C.c_int, [_vp, _i64p, _i64p, _i64p, _dp]),
    "swe_set_params": (C.c_int, [_vp, C.c_double, C.c_double, C.c_double, C.c_double]),
    "swe_set_manning": (C.c_int, [_vp, _vp]),
    "swe_set_bc": (C.c_int, [_vp, C.c_int, C.c_int, C.c_double]),
    "swe_set_state": (C.c_int, [_vp, _vp, _vp, _vp]),
    "swe_get_state": (C.c_int, [_vp, _vp, _vp, _vp]),
    "swe_get_state_static": (C.c_int, [_vp, _vp, _vp, _vp]),
    "swe_set_time": (C.c_int, [_vp, C.c_double]),
    "swe_step": (C.c_int, [_vp, C.c_int, C.c_double, C.c_int, _dp, _dp]),
    "swe_set_graphs": (C.c_int, [_vp, C.c_int]),
    "swe_set_dry_masks": (C.c_int, [_vp, C.c_int]),
    "swe_fp64_peak": (C.c_int, [_vp, _dp]),
    "swe_dry_counts": (C.c_int, [_vp, _i64p]),
    "swe_fastmath_check": (C.c_int, [_vp, C.c_int64, _vp, _vp, _i64p, _dp]),
    "swe_zones_create": (C.c_int, [_vp, C.c_int, C.c_int, _vp]),
    "swe_pack_ghosts": (C.c_int, [_vp, C.c_int]),
    "swe_unpack_ghosts": (C.c_int, [_vp, C.c_int]),
    "swe_zone_stats": (C.c_int, [_vp, _i64p, _i64p, _i64p]),
    "swe_zone_setup_ms": (C.c_int, [_vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "swe_zone_setup_detail": (C.c_int, [_vp, _dp]),
    "swe_zone_describe": (C.c_int, [_vp, C.c_int, _i64p, _i64p, _i64p]),
    "swe_zone_cells": (C.c_int, [_vp, C.c_int, _vp, _vp]),
    "swe_zone_links": (C.c_int, [_vp, C.c_int, _vp, _vp, _vp]),
    "swe_zone_sendlist": (C.c_int, [_vp, C.c_int, C.c_int, _vp]),
    "swe_zones_create_dist": (C.c_int, [_vp, C.c_int, C.c_int, _vp, C.c_int, C.c_int, _vp]),
    "swe_halo_counts": (C.c_int, [_vp, _vp, _vp]),
    "swe_halo_pack": (C.c_int, [_vp, C.c_int, _vp]),
    "swe_halo_unpack": (C.c_int, [_vp, C.c_int, _vp]),
    "swe_peer_export": (C.c_int, [_vp, _vp]),
    "swe_peer_import": (C.c_int, [_vp, C.c_int, _vp]),
    "swe_peer_raw": (C.c_int, [_vp, C.POINTER(_vp), C.POINTER(_vp)]),
    "swe_peer_set_raw": (C.c_int, [_vp, C.c_int, _vp, _vp]),
    "swe_halo_push": (C.c_int, [_vp, C.c_int]),
    "swe_dist_local_min": (C.c_int, [_vp, _vp]),
    "swe_dist_begin_step": (C.c_int, [_vp, _vp, C.c_double]),
    "swe_dist_stage": (C.c_int, [_vp, C.c_int, C.c_int]),
    "swe_dist_flux": (C.c_int, [_vp, C.c_int, C.c_int]),
    "swe_dist_update": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int]),
    "swe_get_time": (C.c_int, [_vp, _dp, _dp]),
    "swe_compute_dt": (C.c_int, [_vp, C.c_double, _dp]),
    "swe_gradients": (C.c_int, [_vp, _vp]),
    "swe_side_fluxes": (C.c_int, [_vp, C.c_double, C.c_int, _vp]),
    "swe_euler_stage": (C.c_int, [_vp, C.c_double, C.c_int, _vp, _vp, _vp]),
    "swe_get_stats": (C.c_int, [_vp, _i64p, _i64p, _i64p]),
    "swe_account_replays": (C.c_int, [_vp, C.c_int64, C.c_int64, C.c_int64]),
    "swe_step_timed": (C.c_int, [_vp, C.c_int, C.c_double, C.c_int, C.POINTER(C.c_float)]),
    "swe_kernel_timed": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float)]),
    "swe_set_profile": (C.c_int, [_vp, C.c_int]),
    "swe_get_profile": (C.c_int, [_vp, _dp, _i64p]),
    "swe_last_error": (C.c_char_p, []),
    "swe_host_mesh_build": (C.c_int, [C.POINTER(_vp), C.c_int64, _vp, _vp, _vp, C.c_int64, _vp, C.c_int64, _vp, _vp, C.c_int]),
    "swe_host_zones_build": (C.c_int, [_vp, C.c_int, C.c_int, _vp]),
    "swe_host_zones_build_dist": (C.c_int, [_vp, C.c_int, C.c_int, _vp, C.c_int, C.c_int, _vp]),
    "swe_host_mesh_free": (None, [_vp]),
    "swe_host_get": (C.c_int64, [_vp, C.c_char_p, _vp, C.c_int64]),
    "swe_host_last_error": (C.c_char_p, []),
}


class SweError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("swe error %d: %s" % (code, msg))
        self.code = code


def lib():
    """Loads (building if needed) libswe_b200.so.  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            f = getattr(L, name)
            f.restype = res
            f.argtypes = args
        _lib = L
    return _lib


def _check(rc):
    if rc != SWE_OK:
        raise SweError(rc, lib().swe_last_error().decode())


def _ptr(a):
    """Raw pointer of a numpy array or torch tensor (None -> NULL)."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        assert a.is_contiguous()
        return a.data_ptr()
    raise TypeError("expected numpy array or torch tensor")


def _f64(a):
    if a is None or hasattr(a, "data_ptr"):
        return a
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    if a is None or hasattr(a, "data_ptr"):
        return a
    return np.ascontiguousarray(a, dtype=np.int32)


def _scheme(s):
    return SCHEMES[s] if isinstance(s, str) else int(s)


# ---- functions with the names of the C ABI -------------------------------------------------
def swe_mesh_create(x, y, zb, tri, bedge=None, btag=None, renumber=SWE_RENUM_HILBERT, cuda_stream=None):
    x, y, zb, tri = _f64(x), _f64(y), _f64(zb), _i32(tri)
    bedge, btag = _i32(bedge), _i32(btag)
    nv = int(x.shape[0])
    nt = int(np.prod(tri.shape)) // 3
    nb = 0 if btag is None else int(btag.shape[0])
    h = _vp()
    _check(lib().swe_mesh_create(C.byref(h), nv, _ptr(x), _ptr(y), _ptr(zb), nt, _ptr(tri), nb,
                                 _ptr(bedge) if nb else None, _ptr(btag) if nb else None,
                                 int(renumber), cuda_stream))
    return h


def swe_mesh_destroy(ctx):
    _check(lib().swe_mesh_destroy(ctx))


def swe_mesh_info(ctx):
    a, b, c, d = C.c_int64(), C.c_int64(), C.c_int64(), C.c_double()
    _check(lib().swe_mesh_info(ctx, C.byref(a), C.byref(b), C.byref(c), C.byref(d)))
    return {"ncell": a.value, "nedge": b.value, "nbedge": c.value, "min_inradius": d.value}


def swe_set_params(ctx, g=9.81, h_dry=1e-6, h_thin=1e-3, beta=1.0):
    _check(lib().swe_set_params(ctx, g, h_dry, h_thin, beta))


def swe_set_manning(ctx, n_cell):
    n_cell = _f64(n_cell)
    _check(lib().swe_set_manning(ctx, _ptr(n_cell)))


def swe_set_bc(ctx, tag, kind, value=0.0):
    k = BC_KINDS[kind] if isinstance(kind, str) else int(kind)
    _check(lib().swe_set_bc(ctx, int(tag), k, float(value)))


def swe_set_state(ctx, h, hu, hv):
    h, hu, hv = _f64(h), _f64(hu), _f64(hv)
    _check(lib().swe_set_state(ctx, _ptr(h), _ptr(hu), _ptr(hv)))


def swe_get_state(ctx, h=None, hu=None, hv=None):
    """Fills the given arrays / tensors, or returns three new numpy arrays."""
    if h is None:
        n = swe_mesh_info(ctx)["ncell"]
        h, hu, hv = np.empty(n), np.empty(n), np.empty(n)
    _check(lib().swe_get_state(ctx, _ptr(h), _ptr(hu), _ptr(hv)))
    return h, hu, hv


def swe_get_state_static(ctx, h=None, hu=None, hv=None):
    """swe_get_state without any allocation in the library: host arrays are staged through a static
    device array (meshes of up to SWE_STATIC_MAX_CELLS cells; see include/swe_b200.h)."""
    if h is None:
        n = swe_mesh_info(ctx)["ncell"]
        h, hu, hv = np.empty(n), np.empty(n), np.empty(n)
    _check(lib().swe_get_state_static(ctx, _ptr(h), _ptr(hu), _ptr(hv)))
    return h, hu, hv


def swe_set_time(ctx, t):
    _check(lib().swe_set_time(ctx, float(t)))


def swe_step(ctx, nsteps, cfl, scheme, sync=True):
    """Returns (t, last_dt) when sync, else None (asynchronous on the context's stream)."""
    if not sync:
        _check(lib().swe_step(ctx, int(nsteps), float(cfl), _scheme(scheme), None, None))
        return None
    t, dt = C.c_double(), C.c_double()
    _check(lib().swe_step(ctx, int(nsteps), float(cfl), _scheme(scheme), C.byref(t), C.byref(dt)))
    return t.value, dt.value


def swe_fastmath_check(ctx, a, x):
    a, x = _f64(a), _f64(x)
    nd = (C.c_int64 * 2)()
    mr = (C.c_double * 2)()
    _check(lib().swe_fastmath_check(ctx, a.size, _ptr(a), _ptr(x), nd, mr))
    return {"div_differs": nd[0], "sqrt_differs": nd[1], "div_maxrel": mr[0], "sqrt_maxrel": mr[1]}


def swe_dry_counts(ctx):
    v = (C.c_int64 * 5)()
    _check(lib().swe_dry_counts(ctx, v))
    return {"cells_not_wet": v[0], "cells_empty": v[1], "edges_between_empty_cells": v[2], "cells": v[3],
            "interior_edges": v[4]}


def swe_fp64_peak(ctx):
    v = C.c_double()
    _check(lib().swe_fp64_peak(ctx, C.byref(v)))
    return v.value


def swe_set_dry_masks(ctx, on):
    _check(lib().swe_set_dry_masks(ctx, 1 if on else 0))


def swe_set_graphs(ctx, on):
    _check(lib().swe_set_graphs(ctx, 1 if on else 0))


def swe_zones_create(ctx, nzones, nlayers, zone_of_cell=None):
    z = _i32(zone_of_cell)
    _check(lib().swe_zones_create(ctx, int(nzones), int(nlayers), _ptr(z)))


def swe_pack_ghosts(ctx, zone=-1):
    _check(lib().swe_pack_ghosts(ctx, int(zone)))


def swe_unpack_ghosts(ctx, zone=-1):
    _check(lib().swe_unpack_ghosts(ctx, int(zone)))


def swe_zone_stats(ctx):
    a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
    _check(lib().swe_zone_stats(ctx, C.byref(a), C.byref(b), C.byref(c)))
    return {"send_cells_total": a.value, "bytes_per_exchange": b.value, "ghost_cells_total": c.value}


def swe_zone_setup_detail(ctx):
    v = (C.c_double * 5)()
    _check(lib().swe_zone_setup_detail(ctx, v))
    return dict(zip(["zone_of_ms", "ghost_layers_ms", "lists_ms", "assembly_ms", "total_ms"], list(v)))


def swe_zone_setup_ms(ctx):
    """wall-clock ms of the last swe_zones_create: device ghost layers, zone build, whole call."""
    a, b, c = C.c_double(), C.c_double(), C.c_double()
    _check(lib().swe_zone_setup_ms(ctx, C.byref(a), C.byref(b), C.byref(c)))
    return {"ghost_layers_ms": a.value, "build_ms": b.value, "total_ms": c.value}


def swe_zone_describe_counts(ctx, zone):
    """(owned cells, ghost cells, links) of one zone."""
    no, ng, nl = C.c_int64(), C.c_int64(), C.c_int64()
    _check(lib().swe_zone_describe(ctx, int(zone), C.byref(no), C.byref(ng), C.byref(nl)))
    return no.value, ng.value, nl.value


def swe_zone_describe(ctx, zone):
    """counts + arrays of one zone (swe_zone_describe / _cells / _links / _sendlist)."""
    no, ng, nl = C.c_int64(), C.c_int64(), C.c_int64()
    _check(lib().swe_zone_describe(ctx, int(zone), C.byref(no), C.byref(ng), C.byref(nl)))
    cells = np.empty(no.value + ng.value, np.int32)
    layer = np.empty(no.value + ng.value, np.int32)
    _check(lib().swe_zone_cells(ctx, int(zone), _ptr(cells), _ptr(layer)))
    src = np.empty(nl.value, np.int32)
    start = np.empty(nl.value, np.int32)
    cnt = np.empty(nl.value, np.int32)
    _check(lib().swe_zone_links(ctx, int(zone), _ptr(src), _ptr(start), _ptr(cnt)))
    links = []
    for j in range(nl.value):
        sl = np.empty(int(cnt[j]), np.int32)
        _check(lib().swe_zone_sendlist(ctx, int(zone), j, _ptr(sl)))
        links.append((int(src[j]), int(start[j]), int(cnt[j]), sl))
    return {"nowned": no.value, "cells": cells, "layer": layer, "links": links}


# ---- zones distributed over ranks (the caller moves / synchronises; see dist.py) ----
def swe_zones_create_dist(ctx, nzones, nlayers, zone_of_cell, nranks, rank, zone_begin):
    z = _i32(zone_of_cell)
    zb = None if zone_begin is None else np.ascontiguousarray(zone_begin, dtype=np.int32)
    _check(lib().swe_zones_create_dist(ctx, int(nzones), int(nlayers), _ptr(z), int(nranks), int(rank), _ptr(zb)))


def swe_halo_counts(ctx, nranks):
    s, r = np.zeros(nranks, np.int64), np.zeros(nranks, np.int64)
    _check(lib().swe_halo_counts(ctx, _ptr(s), _ptr(r)))
    return s, r


def swe_halo_pack(ctx, buffer, sendbuf):
    _check(lib().swe_halo_pack(ctx, int(buffer), _ptr(sendbuf)))


def swe_halo_unpack(ctx, buffer, recvbuf):
    _check(lib().swe_halo_unpack(ctx, int(buffer), _ptr(recvbuf)))


def swe_peer_export(ctx):
    h = np.zeros(128, np.uint8)
    _check(lib().swe_peer_export(ctx, _ptr(h)))
    return h


def swe_peer_import(ctx, peer, handles):
    h = np.ascontiguousarray(handles, dtype=np.uint8)
    assert h.size == 128
    _check(lib().swe_peer_import(ctx, int(peer), _ptr(h)))


def swe_peer_raw(ctx):
    a, b = _vp(), _vp()
    _check(lib().swe_peer_raw(ctx, C.byref(a), C.byref(b)))
    return a.value, b.value


def swe_peer_set_raw(ctx, peer, buf0, buf1):
    _check(lib().swe_peer_set_raw(ctx, int(peer), buf0, buf1))


def swe_halo_push(ctx, buffer):
    _check(lib().swe_halo_push(ctx, int(buffer)))


def swe_dist_local_min(ctx, min_out):
    _check(lib().swe_dist_local_min(ctx, _ptr(min_out)))


def swe_dist_begin_step(ctx, min_in, cfl):
    _check(lib().swe_dist_begin_step(ctx, _ptr(min_in), float(cfl)))


def swe_dist_stage(ctx, scheme, stage):
    _check(lib().swe_dist_stage(ctx, _scheme(scheme), int(stage)))


def swe_dist_flux(ctx, scheme, stage):
    _check(lib().swe_dist_flux(ctx, _scheme(scheme), int(stage)))


def swe_dist_update(ctx, scheme, stage, part=0):
    _check(lib().swe_dist_update(ctx, _scheme(scheme), int(stage), int(part)))


def swe_get_time(ctx):
    t, dt = C.c_double(), C.c_double()
    _check(lib().swe_get_time(ctx, C.byref(t), C.byref(dt)))
    return t.value, dt.value


def swe_compute_dt(ctx, cfl):
    dt = C.c_double()
    _check(lib().swe_compute_dt(ctx, float(cfl), C.byref(dt)))
    return dt.value


def swe_gradients(ctx, out=None):
    if out is None:
        out = np.empty((swe_mesh_info(ctx)["ncell"], 8))
    _check(lib().swe_gradients(ctx, _ptr(out)))
    return out


def swe_side_fluxes(ctx, dt, scheme, out=None):
    if out is None:
        out = np.empty((swe_mesh_info(ctx)["ncell"], 3, 3))
    _check(lib().swe_side_fluxes(ctx, float(dt), _scheme(scheme), _ptr(out)))
    return out


def swe_euler_stage(ctx, dt, scheme):
    n = swe_mesh_info(ctx)["ncell"]
    h, hu, hv = np.empty(n), np.empty(n), np.empty(n)
    _check(lib().swe_euler_stage(ctx, float(dt), _scheme(scheme), _ptr(h), _ptr(hu), _ptr(hv)))
    return h, hu, hv


def swe_account_replays(ctx, steps, kernel_launches, halo_bytes):
    _check(lib().swe_account_replays(ctx, int(steps), int(kernel_launches), int(halo_bytes)))


def swe_get_stats(ctx):
    a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
    _check(lib().swe_get_stats(ctx, C.byref(a), C.byref(b), C.byref(c)))
    return {"steps": a.value, "kernel_launches": b.value, "halo_bytes": c.value}


def swe_step_timed(ctx, nsteps, cfl, scheme):
    ms = C.c_float()
    _check(lib().swe_step_timed(ctx, int(nsteps), float(cfl), _scheme(scheme), C.byref(ms)))
    return ms.value


def swe_kernel_timed(ctx, which, scheme, reps):
    ms = C.c_float()
    _check(lib().swe_kernel_timed(ctx, int(which), _scheme(scheme), int(reps), C.byref(ms)))
    return ms.value


def swe_set_profile(ctx, on):
    _check(lib().swe_set_profile(ctx, 1 if on else 0))


def swe_get_profile(ctx):
    ms = (C.c_double * 7)()
    n = (C.c_int64 * 7)()
    _check(lib().swe_get_profile(ctx, ms, n))
    return {k: (ms[i], n[i]) for i, k in enumerate(KERNEL_KINDS)}


def swe_last_error():
    return lib().swe_last_error().decode()


def create_from_config(cfg, renumber=SWE_RENUM_HILBERT, cuda_stream=None):
    """Marshals one input dictionary of swe_inputs.configs through the calls above."""
    ctx = swe_mesh_create(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], cfg["bedge"], cfg["btag"],
                          renumber, cuda_stream)
    p = cfg["params"]
    swe_set_params(ctx, p["g"], p["h_dry"], p["h_thin"], p["beta"])
    for tag, (kind, value) in cfg["bc"].items():
        swe_set_bc(ctx, tag, kind, value)
    if cfg.get("manning") is not None:
        swe_set_manning(ctx, cfg["manning"])
    swe_set_state(ctx, cfg["h"], cfg["hu"], cfg["hv"])
    return ctx


# ---- host-only inspection (no GPU) ----------------------------------------------------------
_HOST_DTYPES = {"eside": np.uint8, "rres": np.float32, "cell_user": np.int32, "c2c": np.int32, "c2e": np.int32, "elr": np.int32, "btag": np.int32,
                "user_cell": np.int32, "zone_of": np.int32, "send_idx": np.int32, "recv_idx": np.int32,
                "src_of_cell": np.int32, "link_src": np.int32, "link_dst": np.int32, "tags": np.int32,
                "zone_rank": np.int32, "rsend_idx": np.int32, "rsend_dst": np.int32, "rsend_peer": np.int32,
                "rrecv_idx": np.int32, "send_cells": np.int32, "rsend_off": np.int64, "rrecv_off": np.int64,
                "link_off": np.int64, "zone_offset": np.int64, "zone_nowned": np.int64, "zone_ncells": np.int64}


def swe_host_mesh_build(x, y, zb, tri, bedge=None, btag=None, renumber=SWE_RENUM_HILBERT):
    x, y, zb, tri = _f64(x), _f64(y), _f64(zb), _i32(tri)
    bedge, btag = _i32(bedge), _i32(btag)
    nb = 0 if btag is None else int(btag.shape[0])
    h = _vp()
    rc = lib().swe_host_mesh_build(C.byref(h), int(x.shape[0]), _ptr(x), _ptr(y), _ptr(zb),
                                   int(np.prod(tri.shape)) // 3, _ptr(tri), nb,
                                   _ptr(bedge) if nb else None, _ptr(btag) if nb else None, int(renumber))
    if rc != SWE_OK:
        raise SweError(rc, lib().swe_host_last_error().decode())
    return h


def swe_host_zones_build(handle, nzones, nlayers, zone_of_cell=None):
    z = _i32(zone_of_cell)
    rc = lib().swe_host_zones_build(handle, int(nzones), int(nlayers), _ptr(z))
    if rc != SWE_OK:
        raise SweError(rc, lib().swe_host_last_error().decode())


def swe_host_zones_build_dist(handle, nzones, nlayers, zone_of_cell, nranks, rank, zone_begin):
    z = _i32(zone_of_cell)
    zb = None if zone_begin is None else np.ascontiguousarray(zone_begin, dtype=np.int32)
    rc = lib().swe_host_zones_build_dist(handle, int(nzones), int(nlayers), _ptr(z), int(nranks), int(rank), _ptr(zb))
    if rc != SWE_OK:
        raise SweError(rc, lib().swe_host_last_error().decode())


def swe_host_mesh_free(handle):
    lib().swe_host_mesh_free(handle)


def swe_host_get(handle, name):
    """Named array of the host set-up as numpy (scalars "ne_int", "z:ne_int" as int)."""
    key = name.encode()
    n = lib().swe_host_get(handle, key, None, 0)
    if n == -2:
        raise KeyError(name)
    if name.endswith("ne_int"):
        return int(n)
    base = name[2:] if name.startswith("z:") else name
    out = np.empty(int(n), dtype=_HOST_DTYPES.get(base, np.float64))
    got = lib().swe_host_get(handle, key, _ptr(out), out.nbytes)
    assert got == n
    return out
