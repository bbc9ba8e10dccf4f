"""More GPU parity and API cases: limiter parameter, every boundary kind, parameters changed after
the mesh / zones exist, launch accounting, per-kernel timing and profiling entry points."""
import numpy as np
import pytest

import paper_2307_16758_b200 as sw
from oracle import pyoracle as po
from swe_inputs import config0, config3, simple_wave_case, lake_case, channel_flow_case
from parity import assert_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _threads():
    po.set_threads(0)


def _river():
    return config3(length=3200.0, half_width=600.0, w2=30.0, n4=4, n8=3)


@pytest.mark.parametrize("beta", [2.0, 0.0, 1.5])
def test_limiter_parameter(beta):
    """beta = 2 (Barth-Jespersen bound), beta <= 0 (unlimited), and a value in between."""
    cfg = simple_wave_case(120, jitter=0.1)
    cfg["params"] = dict(cfg["params"], beta=beta)
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    try:
        o.step(5, 0.45, "muscl")
        sw.swe_set_state(c, *o.get_state())
        go, gg = o.gradients(), sw.swe_gradients(c)
        assert np.abs(gg - go).max() <= 1e-11 * max(np.abs(go).max(), 1e-3)
        for s in range(30):
            sw.swe_set_state(c, *o.get_state())
            o.step(1, 0.45, "muscl")
            sw.swe_step(c, 1, 0.45, "muscl")
            assert_parity(o.get_state(), sw.swe_get_state(c), 1e-11, what="beta %g step %d" % (beta, s))
    finally:
        sw.swe_mesh_destroy(c)
        o.close()


@pytest.mark.parametrize("kinds", [("transmissive", "transmissive"), ("inflow", "transmissive"),
                                   ("level", "level"), ("wall", "level")])
@pytest.mark.parametrize("scheme,cfl", [("muscl", 0.45), ("hllc", 0.9), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_boundary_kinds(kinds, scheme, cfl):
    """Every boundary kind (PAPER.md:286 + fixed level) on both tagged boundaries of the river case."""
    cfg = _river()
    val = {"transmissive": 0.0, "inflow": 300.0, "level": 3.5, "wall": 0.0}
    cfg["bc"] = {1: (kinds[0], val[kinds[0]]), 2: (kinds[1], val[kinds[1]])}
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    try:
        for s in range(25):
            sw.swe_set_state(c, *o.get_state())
            o.step(1, cfl, scheme)
            sw.swe_step(c, 1, cfl, scheme)
            assert_parity(o.get_state(), sw.swe_get_state(c), 1e-11, what="%s %s step %d" % (kinds, scheme, s))
    finally:
        sw.swe_mesh_destroy(c)
        o.close()


@pytest.mark.parametrize("scheme,cfl", [("muscl", 0.45), ("hllc", 0.9), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_open_channel_flow_free_run(scheme, cfl):
    """The case that pins the oracle's open boundaries (tests/test_oracle_boundaries.py): inflow Q,
    fixed level, Manning friction, relaxing from still water towards the backwater curve -- a free
    run of 400 steps on the GPU stays within 1e-8 of the oracle, and the GPU keeps the uniform flow
    exactly as the oracle does.  WAF: 100 steps -- on this case the per-edge WAF with SUPERBEE
    amplifies round-off tenfold every 25 steps (both sides agree to 3e-16 when restarted every step;
    free trajectories are 2e-12 apart after 100 steps, 5e-8 after 200, 1e-2 after 400: DESIGN.md 3)."""
    cfg = channel_flow_case(nx=100, ny=5, lx=200.0, ly=10.0, discharge=20.0, level=1.0, manning=0.03)
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    try:
        if scheme == "waf":                              # every step from the oracle's state: 1e-11
            for s in range(150):
                sw.swe_set_state(c, *o.get_state())
                o.step(1, cfl, scheme)
                sw.swe_step(c, 1, cfl, scheme)
                assert_parity(o.get_state(), sw.swe_get_state(c), 1e-11, what="channel waf step %d" % s)
            o.close()
            o = po.Oracle.from_config(cfg)               # and a free run from the start
            sw.swe_set_state(c, cfg["h"], cfg["hu"], cfg["hv"])
            sw.swe_set_time(c, 0.0)
        n = 100 if scheme == "waf" else 400
        to = o.step(n, cfl, scheme)
        tg = sw.swe_step(c, n, cfl, scheme)
        assert abs(to[0] - tg[0]) <= 1e-10 * to[0]
        assert_parity(o.get_state(), sw.swe_get_state(c), 1e-8, what="channel " + scheme)
    finally:
        sw.swe_mesh_destroy(c)
        o.close()
    cfg = channel_flow_case(discharge=10.0, level=2.0, u_init=1.0)
    c = sw.create_from_config(cfg)
    try:
        sw.swe_step(c, 200, cfl, scheme)
        h, hu, hv = sw.swe_get_state(c)
        assert np.abs(h - 2.0).max() < 1e-13 and np.abs(hu - 2.0).max() < 1e-13 and np.abs(hv).max() < 1e-13
    finally:
        sw.swe_mesh_destroy(c)


@pytest.mark.parametrize("beta", [2.0, 1.0])
def test_multislope_muscl_limiter_parameter(beta):
    """The paper's MUSCL (eq. 22-25) with SUPERBEE (beta = 2, the paper's choice) and MINBEE."""
    cfg = config0()
    cfg["params"] = dict(cfg["params"], beta=beta)
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    try:
        for s in range(60):
            sw.swe_set_state(c, *o.get_state())
            o.step(1, 0.45, "muscl_ms")
            sw.swe_step(c, 1, 0.45, "muscl_ms")
            assert_parity(o.get_state(), sw.swe_get_state(c), 1e-11, what="ms beta %g step %d" % (beta, s))
    finally:
        sw.swe_mesh_destroy(c)
        o.close()


def test_parameters_changed_after_zones_exist():
    """swe_set_bc / swe_set_manning / swe_set_params reach the zoned copy as well."""
    cfg = _river()
    a = sw.create_from_config(cfg)
    b = sw.create_from_config(cfg)
    try:
        sw.swe_zones_create(b, 8, 2)
        n2 = np.where(cfg["manning"] > 0.03, 0.05, 0.02)
        for ctx in (a, b):
            sw.swe_set_bc(ctx, 1, "inflow", 500.0)
            sw.swe_set_bc(ctx, 2, "transmissive", 0.0)
            sw.swe_set_manning(ctx, n2)
            sw.swe_set_params(ctx, 9.81, 1e-6, 1e-3, 2.0)
            sw.swe_step(ctx, 20, 0.45, "muscl")
        for x, y in zip(sw.swe_get_state(a), sw.swe_get_state(b)):
            assert np.array_equal(x, y)
        for ctx in (a, b):
            sw.swe_set_manning(ctx, None)
            sw.swe_step(ctx, 5, 0.45, "waf")
        for x, y in zip(sw.swe_get_state(a), sw.swe_get_state(b)):
            assert np.array_equal(x, y)
        o = po.Oracle.from_config(cfg)          # and the un-zoned one still matches the oracle
        o.set_bc(1, "inflow", 500.0); o.set_bc(2, "transmissive", 0.0); o.set_manning(n2)
        o.set_params(9.81, 1e-6, 1e-3, 2.0)
        o.step(20, 0.45, "muscl")
        o.set_manning(None)
        o.step(5, 0.45, "waf")
        assert_parity(o.get_state(), sw.swe_get_state(a), 1e-8, what="changed parameters")
        o.close()
    finally:
        sw.swe_mesh_destroy(a)
        sw.swe_mesh_destroy(b)


def test_launch_accounting_and_timing_entry_points():
    cfg = lake_case(n=40)
    c = sw.create_from_config(cfg)
    try:
        sw.swe_step(c, 1, 0.45, "muscl")                   # includes the stand-alone dt_reduce
        l0 = sw.swe_get_stats(c)["kernel_launches"]
        sw.swe_step(c, 10, 0.45, "muscl")
        l1 = sw.swe_get_stats(c)["kernel_launches"]
        assert l1 - l0 == 10 * 7                           # finalize + 2 x (grad, flux, update)
        sw.swe_step(c, 10, 0.9, "hllc")
        assert sw.swe_get_stats(c)["kernel_launches"] - l1 == 10 * 3
        assert sw.swe_get_stats(c)["steps"] == 21
        ms = sw.swe_step_timed(c, 5, 0.45, "muscl")
        assert ms > 0.0
        for which in range(5):
            assert sw.swe_kernel_timed(c, which, "muscl", 3) > 0.0
        ref = sw.swe_get_state(c)
        sw.swe_set_profile(c, True)
        sw.swe_step(c, 4, 0.45, "muscl")
        p = sw.swe_get_profile(c)
        sw.swe_set_profile(c, False)
        assert p["grad_limit"][1] == 8 and p["edge_flux"][1] == 8 and p["cell_update"][1] == 8
        assert p["dt_finalize"][1] == 4 and p["dt_reduce"][1] == 0
        assert all(v[0] > 0.0 for k, v in p.items() if v[1])
        # the timing entry points of single kernels leave the state alone
        c2 = sw.create_from_config(cfg)
        sw.swe_step(c2, 1 + 10, 0.45, "muscl"); sw.swe_step(c2, 10, 0.9, "hllc"); sw.swe_step(c2, 5, 0.45, "muscl")
        for x, y in zip(ref, sw.swe_get_state(c2)):
            assert np.array_equal(x, y)
        sw.swe_mesh_destroy(c2)
    finally:
        sw.swe_mesh_destroy(c)


def test_time_accumulates_and_can_be_set():
    cfg = config0(nx=60, ny=4)
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    try:
        t1, dt1 = sw.swe_step(c, 7, 0.9, "hllc")
        to, dto = o.step(7, 0.9, "hllc")
        assert abs(t1 - to) <= 1e-13 * to and abs(dt1 - dto) <= 4e-16 * dto
        sw.swe_set_time(c, 100.0)
        t2, dt2 = sw.swe_step(c, 1, 0.9, "hllc")
        assert abs(t2 - (100.0 + dt2)) <= 1e-12
    finally:
        sw.swe_mesh_destroy(c)
        o.close()


@pytest.mark.parametrize("scheme,cfl", [("muscl", 0.45), ("hllc", 0.9), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_dry_cells_with_leftover_momentum(scheme, cfl):
    """Cells without water are skipped by the gradient and flux kernels (their records are exactly
    zero by A.3.5 / A.5-A.9).  A user state may still carry momentum in such cells, and depths
    between 0 and h_dry are NOT skipped: both must behave as in the oracle."""
    cfg = lake_case(n=40)
    rng = np.random.default_rng(5)
    h = cfg["h"].copy()
    dry = h == 0.0
    assert dry.sum() > 100
    hu = np.where(dry, rng.normal(size=h.size), 0.0)          # leftover momentum in dry cells
    hv = np.where(dry, rng.normal(size=h.size), 0.0)
    thin = rng.random(h.size) < 0.3
    h = np.where(dry & thin, 5e-7, h)                          # below h_dry but not zero
    o = po.Oracle.from_config(cfg)
    c = sw.create_from_config(cfg)
    try:
        o.set_state(h, hu, hv)
        for s in range(10):
            sw.swe_set_state(c, *o.get_state())
            o.step(1, cfl, scheme)
            sw.swe_step(c, 1, cfl, scheme)
            assert_parity(o.get_state(), sw.swe_get_state(c), 1e-11, what="dry %s step %d" % (scheme, s))
        go, gg = o.gradients(), sw.swe_gradients(c)
        assert np.abs(gg - go).max() <= 1e-11 * max(np.abs(go).max(), 1e-3)
    finally:
        sw.swe_mesh_destroy(c)
        o.close()


def test_error_paths_leave_the_context_usable():
    cfg = lake_case(n=20)
    c = sw.create_from_config(cfg)
    try:
        ref = sw.swe_get_state(c)
        for call, code in [
            (lambda: sw.swe_set_bc(c, -1, "wall", 0.0), sw.SWE_ERR_ARG),
            (lambda: sw.swe_set_bc(c, 1, 9, 0.0), sw.SWE_ERR_ARG),
            (lambda: sw.swe_set_params(c, -9.81, 1e-6, 1e-3, 1.0), sw.SWE_ERR_ARG),
            (lambda: sw.swe_zones_create(c, 3, 2), sw.SWE_ERR_ARG),          # RCB needs a power of two
            (lambda: sw.swe_zones_create(c, 4, 0), sw.SWE_ERR_ARG),
            (lambda: sw.swe_zones_create(c, 2, 2, np.full(cfg["h"].size, 5, np.int32)), sw.SWE_ERR_ARG),
            (lambda: sw.swe_pack_ghosts(c, -1), sw.SWE_ERR_STATE),           # no zones yet
            (lambda: sw.swe_zone_stats(c), sw.SWE_ERR_STATE),
            (lambda: sw.swe_kernel_timed(c, 99, "muscl", 1), sw.SWE_ERR_ARG),
            (lambda: sw.swe_step(c, -1, 0.5, "hllc"), sw.SWE_ERR_ARG),
            (lambda: sw.swe_compute_dt(c, 0.0), sw.SWE_ERR_ARG),
        ]:
            with pytest.raises(sw.SweError) as e:
                call()
            assert e.value.code == code and str(e.value)
        for x, y in zip(ref, sw.swe_get_state(c)):
            assert np.array_equal(x, y)
        # explicit zone map (not RCB), then single-pass calls are refused while zones exist
        zmap = (np.arange(cfg["h"].size) % 3).astype(np.int32)
        sw.swe_zones_create(c, 3, 2, zmap)
        with pytest.raises(sw.SweError) as e:
            sw.swe_gradients(c)
        assert e.value.code == sw.SWE_ERR_STATE
        with pytest.raises(sw.SweError):
            sw.swe_pack_ghosts(c, 7)
        a = sw.create_from_config(cfg)
        sw.swe_step(a, 15, 0.45, "muscl")
        sw.swe_step(c, 15, 0.45, "muscl")                   # scattered zones: still bit-identical
        for x, y in zip(sw.swe_get_state(a), sw.swe_get_state(c)):
            assert np.array_equal(x, y)
        sw.swe_mesh_destroy(a)
    finally:
        sw.swe_mesh_destroy(c)


def test_mesh_errors_through_the_gpu_entry_point():
    x = np.array([0.0, 1.0, 0.0, 1.0]); y = np.array([0.0, 0.0, 1.0, 1.0]); z = np.zeros(4)
    with pytest.raises(sw.SweError) as e:
        sw.swe_mesh_create(x, y, z, np.array([[0, 1, 9]], np.int32))
    assert e.value.code == sw.SWE_ERR_MESH
    with pytest.raises(sw.SweError) as e:
        sw.swe_mesh_create(x, y, z, np.array([[0, 1, 2], [1, 3, 2]], np.int32),
                           np.array([[1, 2]], np.int32), np.array([1], np.int32))
    assert e.value.code == sw.SWE_ERR_MESH and "boundary" in str(e.value)
    with pytest.raises(sw.SweError) as e:
        sw.swe_mesh_create(x, y, z, np.array([[0, 1, 2]], np.int32), renumber=5)
    assert e.value.code == sw.SWE_ERR_ARG


def test_graph_replay_equals_kernel_by_kernel_launches():
    """swe_step replays one captured CUDA graph per step (nsteps >= 2): same kernels, same order --
    the state, the clock and the launch count must be those of the plain launches, through scheme
    changes, parameter changes and zones (each invalidates the captured graph)."""
    cfg = _river()
    a = sw.create_from_config(cfg)
    b = sw.create_from_config(cfg)
    try:
        sw.swe_set_graphs(b, False)
        seq = [("muscl", 0.45, 12), ("hllc", 0.9, 7), ("muscl", 0.45, 1), ("waf", 0.45, 5), ("muscl", 0.3, 6),
               ("muscl_ms", 0.45, 4)]
        for x in (a, b):
            for scheme, cfl, n in seq:
                t = sw.swe_step(x, n, cfl, scheme)
            sw.swe_set_params(x, beta=2.0)
            sw.swe_step(x, 5, 0.45, "muscl")
            sw.swe_zones_create(x, 8, 2)
            sw.swe_step(x, 6, 0.45, "muscl")
            sw.swe_step(x, 3, 0.9, "hllc")
            sw.swe_zones_create(x, 0, 1)
            sw.swe_step(x, 4, 0.45, "muscl")
        for u, v in zip(sw.swe_get_state(a), sw.swe_get_state(b)):
            assert np.array_equal(u, v)
        assert sw.swe_get_time(a) == sw.swe_get_time(b)
        sa, sb = sw.swe_get_stats(a), sw.swe_get_stats(b)
        assert sa == sb
    finally:
        sw.swe_mesh_destroy(a)
        sw.swe_mesh_destroy(b)


def test_fp64_peak_microbenchmark():
    """The DFMA micro-benchmark BASELINE.md asks for: a plausible B200 figure (tens of TFLOP/s)."""
    c = sw.create_from_config(config0())
    try:
        v = sw.swe_fp64_peak(c)
        assert 10.0 < v < 100.0, v
        assert abs(sw.swe_fp64_peak(c) - v) < 0.2 * v
    finally:
        sw.swe_mesh_destroy(c)


def test_division_and_square_root_sequences_equal_ieee():
    """The kernels do not use the compiler's fp64 division / sqrt but a MUFU seed, one Newton step and
    a residual correction (swe_kernels.cuh).  On 4 M seeded samples over 24 decades (numerators of
    either sign over 10 decades) every quotient and every root is the IEEE-rounded one, so the
    per-step agreement with the oracle does not depend on them."""
    rng = np.random.default_rng(3)
    n = 1 << 22
    x = 10.0 ** rng.uniform(-12, 12, n) * (1.0 + rng.random(n))
    a = rng.choice([-1.0, 1.0], n) * 10.0 ** rng.uniform(-5, 5, n) * (1.0 + rng.random(n))
    # the arguments the kernels see most: depths from h_dry up, g h, sums of squares, near powers of two
    x[: n // 8] = rng.uniform(1e-6, 30.0, n // 8)
    x[n // 8: n // 4] = 2.0 ** rng.integers(-20, 20, n // 8) * (1.0 + rng.choice([-1, 1], n // 8) * 2.0 ** -rng.integers(30, 53, n // 8))
    cfg = lake_case(n=10)
    c = sw.create_from_config(cfg)
    try:
        r = sw.swe_fastmath_check(c, a, x)
        assert r["div_differs"] == 0 and r["sqrt_differs"] == 0, r
    finally:
        sw.swe_mesh_destroy(c)


@pytest.mark.parametrize("ndistinct", [1, 4, 255, 256, 0])
def test_manning_table_and_per_cell_fallback(ndistinct):
    """Manning n travels as a one-byte code per cell + a table of the distinct values (at most 255);
    with more distinct values every cell carries code 255 and the update kernel reads the per-cell
    array.  Both routes against the oracle (<= 1e-11 per step), un-zoned and with zones created
    before and after swe_set_manning, device and host pointers.  ndistinct = 0: one value per cell."""
    import torch
    cfg = config3(length=1600.0, half_width=400.0, w2=20.0, n4=3, n8=2)
    nt = cfg["tri"].shape[0]
    rng = np.random.default_rng(11)
    if ndistinct == 0:
        nman = rng.uniform(0.01, 0.06, nt)
        assert np.unique(nman).size > 255
    else:
        vals = np.concatenate([[0.0], rng.uniform(0.01, 0.06, ndistinct - 1)]) if ndistinct > 1 else np.array([0.033])
        nman = vals[rng.integers(0, ndistinct, nt)]
        nman[:ndistinct] = vals                                    # every value occurs
    po.set_threads(0)
    o = po.Oracle.from_config(cfg)
    o.set_manning(nman)
    a = sw.create_from_config(cfg)                                 # un-zoned, host pointer
    b = sw.create_from_config(cfg)                                 # zones first, then Manning from a device pointer
    c = sw.create_from_config(cfg)                                 # Manning first, then zones
    try:
        sw.swe_set_manning(a, nman)
        sw.swe_zones_create(b, 4, 2)
        sw.swe_set_manning(b, torch.tensor(nman, device="cuda"))
        sw.swe_set_manning(c, nman)
        sw.swe_zones_create(c, 8, 2)
        o.step(15, 0.45, "muscl")                                  # water starts to move: friction matters
        for x in (a, b, c):
            sw.swe_step(x, 15, 0.45, "muscl")
        ref = sw.swe_get_state(a)
        assert_parity(o.get_state(), ref, 1e-9, what="manning %d run" % ndistinct)
        for x in (b, c):
            for p, q in zip(ref, sw.swe_get_state(x)):
                assert np.array_equal(p, q)
        for s in range(5):
            sw.swe_set_state(a, *o.get_state())
            o.step(1, 0.45, "muscl")
            sw.swe_step(a, 1, 0.45, "muscl")
            assert_parity(o.get_state(), sw.swe_get_state(a), 1e-11, what="manning %d step %d" % (ndistinct, s))
        # back to no friction at all, and to a table again: the codes are rewritten every time
        sw.swe_set_manning(a, None); o.set_manning(None)
        o.step(3, 0.9, "hllc"); sw.swe_set_state(a, *o.get_state())
        sw.swe_set_manning(a, np.full(nt, 0.02)); o.set_manning(np.full(nt, 0.02))
        o.step(1, 0.9, "hllc"); sw.swe_step(a, 1, 0.9, "hllc")
        assert_parity(o.get_state(), sw.swe_get_state(a), 1e-11, what="manning reset")
    finally:
        for x in (a, b, c):
            sw.swe_mesh_destroy(x)
        o.close()


def test_dry_counts_and_zone_setup_detail():
    """swe_dry_counts against numpy on the state the library holds (un-zoned and zoned; bench.py
    prints these fractions beside the roofline), swe_zone_setup_detail adds up, swe_account_replays
    moves the counters."""
    cfg = config3(length=3200.0, half_width=600.0, w2=30.0, n4=4, n8=3)
    c = sw.create_from_config(cfg)
    o = po.Oracle.from_config(cfg)
    try:
        sw.swe_step(c, 7, 0.45, "muscl")
        h, hu, hv = sw.swe_get_state(c)
        eg = o.edge_geometry()
        inner = eg["eR"] >= 0
        want_edges = int(np.count_nonzero((h[eg["eL"][inner]] == 0.0) & (h[eg["eR"][inner]] == 0.0)))
        d = sw.swe_dry_counts(c)
        assert d["cells"] == h.size and d["interior_edges"] == int(inner.sum())
        assert d["cells_not_wet"] == int(np.count_nonzero(~(h > 1e-6)))
        assert d["cells_empty"] == int(np.count_nonzero(h == 0.0)) > 0
        assert d["edges_between_empty_cells"] == want_edges > 0
        sw.swe_zones_create(c, 4, 2)
        dz = sw.swe_dry_counts(c)                                    # owned cells of the zoned copy
        assert dz["cells_not_wet"] == d["cells_not_wet"] and dz["cells_empty"] == d["cells_empty"]
        t = sw.swe_zone_setup_detail(c)
        parts = t["zone_of_ms"] + t["ghost_layers_ms"] + t["lists_ms"] + t["assembly_ms"]
        assert all(v >= 0.0 for v in t.values()) and parts <= t["total_ms"] * 1.001 and t["assembly_ms"] > 0.0
        s0 = sw.swe_get_stats(c)
        sw.swe_account_replays(c, 3, 39, 1000)
        s1 = sw.swe_get_stats(c)
        assert (s1["steps"] - s0["steps"], s1["kernel_launches"] - s0["kernel_launches"],
                s1["halo_bytes"] - s0["halo_bytes"]) == (3, 39, 1000)
        sw.swe_account_replays(c, -3, -39, -1000)
        assert sw.swe_get_stats(c) == s0
    finally:
        sw.swe_mesh_destroy(c)
        o.close()
