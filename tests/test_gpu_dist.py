"""Multi-GPU driver (scope row f3) on ONE GPU: the ranks' kernels never wait on one
another, so the path can be run rank after rank.

 * in-process: `world` contexts in one process stand for the ranks; every phase of dist.DistSolver's
   step (push / pack-transfer-unpack, min-reduce, stages) is run for all ranks in turn, the
   "transfer" being a device copy between the ranks' halo buffers.  The result must be BIT-identical
   to the un-zoned run for every scheme, both transports, 1..3 zones per rank.
 * two processes sharing cuda:0 over gloo (host-staged collectives, CUDA IPC between the
   processes): dist.DistSolver itself, the code bench.py runs at N > 1.
"""
import os
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

import paper_2307_16758_b200 as sw
from paper_2307_16758_b200 import dist as swdist
from swe_inputs import config3

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _river():
    return config3(length=3200.0, half_width=600.0, w2=30.0, n4=4, n8=3)


class _Ranks:
    """`world` ranks as contexts of one process."""

    def __init__(self, cfg, world, nz, nl, transport):
        self.world, self.transport = world, transport
        self.ctx = [sw.create_from_config(cfg) for _ in range(world)]
        blocks = swdist.zone_blocks(nz, world)
        for r, c in enumerate(self.ctx):
            sw.swe_zones_create_dist(c, nz, nl, None, world, r, blocks)
        self.counts = [sw.swe_halo_counts(c, world) for c in self.ctx]
        dev = torch.device("cuda")
        self.mins = torch.zeros(world, dtype=torch.float64, device=dev)
        if transport == "p2p":
            raw = [sw.swe_peer_raw(c) for c in self.ctx]
            for r, c in enumerate(self.ctx):
                for p in range(world):
                    if p != r:
                        sw.swe_peer_set_raw(c, p, *raw[p])
        else:
            self.sendbuf = [torch.zeros(max(1, 3 * int(s.sum())), dtype=torch.float64, device=dev) for s, _ in self.counts]
            self.recvbuf = [torch.full((max(1, 3 * int(r.sum())),), np.nan, dtype=torch.float64, device=dev) for _, r in self.counts]

    def exchange(self, buffer):
        if self.transport == "p2p":
            for c in self.ctx:
                sw.swe_halo_push(c, buffer)
            return
        for r, c in enumerate(self.ctx):
            sw.swe_halo_pack(c, buffer, self.sendbuf[r])
        soff = [np.concatenate([[0], 3 * np.cumsum(s)]) for s, _ in self.counts]
        roff = [np.concatenate([[0], 3 * np.cumsum(r)]) for _, r in self.counts]
        for a in range(self.world):            # the all-to-all
            for b in range(self.world):
                n = int(soff[a][b + 1] - soff[a][b])
                assert n == int(roff[b][a + 1] - roff[b][a])
                if n:
                    self.recvbuf[b][int(roff[b][a]):int(roff[b][a]) + n] = self.sendbuf[a][int(soff[a][b]):int(soff[a][b]) + n]
        for r, c in enumerate(self.ctx):
            sw.swe_halo_unpack(c, buffer, self.recvbuf[r])

    def step(self, nsteps, cfl, scheme, overlap=False):
        if overlap:
            return self.step_overlap(nsteps, cfl, scheme)
        heun = scheme in ("muscl", "muscl_ms")
        for _ in range(nsteps):
            self.exchange(0)
            for r, c in enumerate(self.ctx):
                sw.swe_dist_local_min(c, self.mins[r:r + 1])
            m = self.mins.min().reshape(1)                      # the all-reduce(min)
            for c in self.ctx:
                sw.swe_dist_begin_step(c, m, cfl)
                sw.swe_dist_stage(c, scheme, 0)
            if heun:
                self.exchange(1)
                for c in self.ctx:
                    sw.swe_dist_stage(c, scheme, 1)

    def step_overlap(self, nsteps, cfl, scheme):
        """The phases of DistSolver._step_overlap: send cells first, exchange, then the rest."""
        heun = scheme in ("muscl", "muscl_ms")
        self.exchange(0)
        for _ in range(nsteps):
            for r, c in enumerate(self.ctx):
                sw.swe_dist_local_min(c, self.mins[r:r + 1])
            m = self.mins.min().reshape(1)
            for c in self.ctx:
                if scheme == "waf":
                    sw.swe_dist_begin_step(c, m, cfl)
                sw.swe_dist_flux(c, scheme, 0)
                if scheme != "waf":
                    sw.swe_dist_begin_step(c, m, cfl)
                sw.swe_dist_update(c, scheme, 0, 1)
            if heun:
                self.exchange(1)
                for c in self.ctx:
                    sw.swe_dist_update(c, scheme, 0, 2)
                    sw.swe_dist_flux(c, scheme, 1)
                    sw.swe_dist_update(c, scheme, 1, 1)
            self.exchange(0)
            for c in self.ctx:
                sw.swe_dist_update(c, scheme, 1 if heun else 0, 2)

    def state(self, n):
        out = [np.full(n, np.nan) for _ in range(3)]
        for c in self.ctx:
            sw.swe_get_state(c, *out)          # each rank fills the cells it owns
        return out

    def close(self):
        torch.cuda.synchronize()
        for c in self.ctx:
            sw.swe_mesh_destroy(c)


@pytest.mark.parametrize("transport,overlap", [("p2p", False), ("staged", False), ("p2p", True)])
@pytest.mark.parametrize("world,nz,nl", [(2, 2, 2), (4, 4, 2), (2, 8, 3), (3, 8, 2)])
@pytest.mark.parametrize("scheme,cfl", [("muscl", 0.45), ("hllc", 0.9), ("waf", 0.45), ("muscl_ms", 0.45)])
def test_ranks_in_one_process_bit_identical(transport, overlap, world, nz, nl, scheme, cfl):
    cfg = _river()
    a = sw.create_from_config(cfg)
    R = _Ranks(cfg, world, nz, nl, transport)
    try:
        n = sw.swe_mesh_info(a)["ncell"]
        ta = sw.swe_step(a, 30, cfl, scheme)
        R.step(30, cfl, scheme, overlap)
        ref = sw.swe_get_state(a)
        got = R.state(n)
        for x, y in zip(ref, got):
            assert np.array_equal(x, y)
        for c in R.ctx:
            assert sw.swe_get_time(c) == ta
        # a rank refuses the single-GPU step while its zones are distributed
        with pytest.raises(sw.SweError) as e:
            sw.swe_step(R.ctx[0], 1, cfl, scheme)
        assert e.value.code == sw.SWE_ERR_STATE
    finally:
        sw.swe_mesh_destroy(a)
        R.close()


def test_config3_full_size_two_ranks_overlap_schedule():
    """The workload bench.py runs at N = 2 (configs[3], 13.1 M cells, 2 zones over 2 ranks, 2 ghost
    layers, peer-memory push, overlap schedule), ranks in one process: 3 MUSCL-RK2 steps
    bit-identical to the single-GPU run."""
    from swe_inputs import config3 as full
    cfg = full()
    a = sw.create_from_config(cfg)
    try:
        ta = sw.swe_step(a, 3, 0.45, "muscl")
        ref = sw.swe_get_state(a)
    finally:
        sw.swe_mesh_destroy(a)
    R = _Ranks(cfg, 2, 2, 2, "p2p")
    try:
        R.step(3, 0.45, "muscl", overlap=True)
        got = R.state(ref[0].size)
        for x, y in zip(ref, got):
            assert np.array_equal(x, y)
        assert sw.swe_get_time(R.ctx[1]) == ta
        s, r = R.counts[0]
        assert s[1] == r[1] and 500 < s[1] < 100000          # two layers of the cells along the cut
    finally:
        R.close()


def test_one_layer_hllc_and_errors():
    cfg = _river()
    a = sw.create_from_config(cfg)
    R = _Ranks(cfg, 2, 4, 1, "p2p")
    try:
        n = sw.swe_mesh_info(a)["ncell"]
        sw.swe_step(a, 20, 0.9, "hllc")
        R.step(20, 0.9, "hllc")
        for x, y in zip(sw.swe_get_state(a), R.state(n)):
            assert np.array_equal(x, y)
        c = R.ctx[0]
        for bad in (lambda: sw.swe_dist_stage(c, "muscl", 0),        # one ghost layer: HLLC only
                    lambda: sw.swe_dist_stage(c, "hllc", 1),         # Euler schemes have one stage
                    lambda: sw.swe_halo_push(c, 2),
                    lambda: sw.swe_peer_set_raw(c, 0, *sw.swe_peer_raw(c)),     # own rank is not a peer
                    lambda: sw.swe_halo_pack(c, 0, np.zeros(8)),     # host pointer
                    lambda: sw.swe_dist_local_min(c, np.zeros(1))):
            with pytest.raises(sw.SweError):
                bad()
        # a rank whose peers were never connected cannot push
        d = sw.create_from_config(cfg)
        try:
            sw.swe_zones_create_dist(d, 4, 1, None, 2, 0, [0, 2, 4])
            with pytest.raises(sw.SweError) as e:
                sw.swe_halo_push(d, 0)
            assert e.value.code == sw.SWE_ERR_STATE
        finally:
            sw.swe_mesh_destroy(d)
    finally:
        sw.swe_mesh_destroy(a)
        R.close()


def _worker(rank, world, port, transport, scheme, cfl, schedule, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK="0", WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port), SWE_DIST_GLOO="1")
    try:
        from paper_2307_16758_b200 import dist as d
        d.init_from_env()
        cfg = _river()
        S = d.DistSolver(cfg, nzones=4, nlayers=2, transport=transport, schedule=schedule)
        S.step(10, cfl, scheme)
        S.step(15, cfl, scheme)            # the overlap schedule carries collectives across calls
        t = S.time()
        st = S.get_state()
        S.close()
        out = None
        if rank == 0:
            a = sw.create_from_config(cfg)
            ta = sw.swe_step(a, 25, cfl, scheme)
            ref = sw.swe_get_state(a)
            sw.swe_mesh_destroy(a)
            out = bool(ta == t and all(np.array_equal(x, y) for x, y in zip(ref, st)))
        d.finalize()
        q.put((rank, out, ""))
    except Exception as e:       # report instead of hanging the parent
        import traceback
        q.put((rank, False, traceback.format_exc() + str(e)))


@pytest.mark.parametrize("transport,scheme,cfl,schedule", [
    ("p2p", "muscl", 0.45, "overlap"), ("p2p", "muscl", 0.45, "plain"), ("staged", "muscl", 0.45, "overlap"),
    ("p2p", "hllc", 0.9, "overlap"), ("p2p", "waf", 0.45, "overlap"), ("staged", "hllc", 0.9, "plain")])
def test_two_processes_one_gpu_dist_solver(transport, scheme, cfl, schedule):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29700 + os.getpid() % 90
    ps = [ctx.Process(target=_worker, args=(r, 2, port, transport, scheme, cfl, schedule, q)) for r in range(2)]
    for p in ps:
        p.start()
    try:
        res = sorted(q.get(timeout=600) for _ in ps)
        for p in ps:
            p.join(120)
    finally:
        for p in ps:
            if p.is_alive():
                p.kill()
    assert all(r[2] == "" for r in res), [r[2] for r in res]
    assert res[0][1] is True


@pytest.mark.parametrize("extra", [[], ["--transport", "staged", "--schedule", "plain", "--scheme", "hllc", "--layers", "1"]])
def test_bench_line_of_the_distributed_arm(extra):
    """bench.py at N = 2 (two ranks on this GPU, gloo): the contract line of the strong-scaling arm."""
    import json
    import subprocess
    env = dict(os.environ, SWE_DIST_GLOO="1")
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        env.pop(k, None)
    port = 29800 + os.getpid() % 90
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "5",
           "--warmup", "3", "--workload", "c3t", "--e2e-steps", "2"] + extra
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT, env=env)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                   # rank 0 only
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "strong" and d["steps"] == 5 and d["unit"] == "cell-updates/s"
    assert d["value"] > 0 and abs(d["value"] - d["config"]["cells"] * 5 / (d["ms_per_step"] * 5e-3)) < 1e-6 * d["value"]
    assert d["config"]["zones"] == 2 and "ranks" in d["config"]["parallelism"] and d["config"]["halo_bytes_per_step"] > 0
    launches_per_step_per_rank = d["gpu_launches"] / (5 * 2)
    assert 4 <= launches_per_step_per_rank <= 14
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["achieved"] > 0 and r["peak"] > 0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0 and d["cpu_baseline"] is None


def _nccl_worker(port, schedule, transport, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK="0", LOCAL_RANK="0", WORLD_SIZE="1", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    os.environ.pop("SWE_DIST_GLOO", None)
    try:
        import torch.distributed as dist
        from paper_2307_16758_b200 import dist as d
        torch.cuda.set_device(0)
        dist.init_process_group(backend="nccl", rank=0, world_size=1)
        cfg = _river()
        S = d.DistSolver(cfg, nzones=4, nlayers=2, transport=transport, schedule=schedule)
        assert not S.comm.staged_host                      # the NCCL code path, not the host-staged one
        S.step(8, 0.45, "muscl")
        S.step(7, 0.9, "hllc")
        S.step(5, 0.45, "waf")
        t = S.time()
        st = S.get_state()
        # the step ran as a replayed CUDA graph (kernels + NCCL collectives), and the library's
        # counters saw the replays
        stats = sw.swe_get_stats(S.ctx)
        assert S.graph_replays == (8 - 1) + (7 - 1) + (5 - 1), S.graph_replays
        assert stats["steps"] == 20, stats
        S2 = d.DistSolver(cfg, nzones=4, nlayers=2, transport=transport, schedule=schedule, graphs=False)
        S2.step(8, 0.45, "muscl"); S2.step(7, 0.9, "hllc"); S2.step(5, 0.45, "waf")
        st_eager, t_eager = S2.get_state(), S2.time()
        stats2 = sw.swe_get_stats(S2.ctx)
        S2.close()
        assert S2.graph_replays == 0 and t_eager == t and all(np.array_equal(x, y) for x, y in zip(st, st_eager))
        assert stats2["kernel_launches"] == stats["kernel_launches"] and stats2["halo_bytes"] == stats["halo_bytes"], (stats, stats2)
        # a capture that fails half way: every rank falls back to call-by-call steps, nothing is lost
        os.environ["SWE_DIST_GRAPH_FAIL"] = "1"
        S3 = d.DistSolver(cfg, nzones=4, nlayers=2, transport=transport, schedule=schedule)
        S3.step(8, 0.45, "muscl"); S3.step(7, 0.9, "hllc"); S3.step(5, 0.45, "waf")
        del os.environ["SWE_DIST_GRAPH_FAIL"]
        st_fb, t_fb = S3.get_state(), S3.time()
        stats3 = sw.swe_get_stats(S3.ctx)
        S3.close()
        assert S3.graph_replays == 0 and S3.graphs is False and t_fb == t
        assert all(np.array_equal(x, y) for x, y in zip(st, st_fb)), "fallback after a failed capture"
        assert stats3["steps"] == 20 and stats3["kernel_launches"] == stats["kernel_launches"], (stats, stats3)
        S.set_state(*[torch.from_numpy(x.copy()) for x in st])
        S.step(3, 0.45, "muscl_ms")
        st2 = S.get_state()
        S.close()
        a = sw.create_from_config(cfg)
        sw.swe_step(a, 8, 0.45, "muscl"); sw.swe_step(a, 7, 0.9, "hllc")
        ta = sw.swe_step(a, 5, 0.45, "waf")
        ref = sw.swe_get_state(a)
        sw.swe_step(a, 3, 0.45, "muscl_ms")
        ref2 = sw.swe_get_state(a)
        sw.swe_mesh_destroy(a)
        checks = [ta == t] + [bool(np.array_equal(x, y)) for x, y in zip(ref, st)] + \
                 [bool(np.array_equal(x, y)) for x, y in zip(ref2, st2)]
        dist.destroy_process_group()
        q.put((all(checks), "" if all(checks) else "time / h hu hv after the first run / after set_state: %s (t %r vs %r)"
               % (checks, t, ta)))
    except Exception as e:
        import traceback
        q.put((False, traceback.format_exc() + str(e)))


@pytest.mark.parametrize("schedule,transport", [("overlap", "p2p"), ("plain", "staged"), ("overlap", "staged")])
def test_dist_solver_over_nccl_single_rank(schedule, transport):
    """The NCCL code path of dist.py (asynchronous all-reduces on NCCL's stream and work.wait(),
    device tensors in every collective) with the one rank one GPU allows: 4 resident zones."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    p = ctx.Process(target=_nccl_worker, args=(29600 + os.getpid() % 90, schedule, transport, q))
    p.start()
    try:
        ok, msg = q.get(timeout=600)
        p.join(120)
    finally:
        if p.is_alive():
            p.kill()
    assert msg == "", msg
    assert ok


def _mixed_worker(rank, world, port, transport, schedule, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK="0", WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port), SWE_DIST_GLOO="1")
    seq = [("muscl", 0.45, 6), ("hllc", 0.9, 5), ("waf", 0.45, 4), ("muscl_ms", 0.45, 3), ("hllc", 0.9, 1), ("muscl", 0.45, 2)]
    try:
        from paper_2307_16758_b200 import dist as d
        d.init_from_env()
        cfg = _river()
        S = d.DistSolver(cfg, nzones=8, nlayers=2, transport=transport, schedule=schedule)
        for scheme, cfl, n in seq:
            S.step(n, cfl, scheme)
        t = S.time()
        st = S.get_state()
        S.close()
        out = None
        if rank == 0:
            a = sw.create_from_config(cfg)
            for scheme, cfl, n in seq:
                ta = sw.swe_step(a, n, cfl, scheme)
            ref = sw.swe_get_state(a)
            sw.swe_mesh_destroy(a)
            out = bool(ta == t and all(np.array_equal(x, y) for x, y in zip(ref, st)))
        d.finalize()
        q.put((rank, out, ""))
    except Exception as e:
        import traceback
        q.put((rank, False, traceback.format_exc() + str(e)))


@pytest.mark.parametrize("transport,schedule", [("p2p", "overlap"), ("staged", "overlap"), ("p2p", "plain")])
def test_two_processes_scheme_changes_between_calls(transport, schedule):
    """The overlap schedule leaves an exchange and an all-reduce in flight between calls: changing the
    scheme from call to call (Heun <-> Euler, WAF's early dt) must not disturb them.  8 zones on 2
    ranks: remote and resident links together."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 90
    ps = [ctx.Process(target=_mixed_worker, args=(r, 2, port, transport, schedule, q)) for r in range(2)]
    for p in ps:
        p.start()
    try:
        res = sorted(q.get(timeout=600) for _ in ps)
        for p in ps:
            p.join(120)
    finally:
        for p in ps:
            if p.is_alive():
                p.kill()
    assert all(r[2] == "" for r in res), [r[2] for r in res]
    assert res[0][1] is True
