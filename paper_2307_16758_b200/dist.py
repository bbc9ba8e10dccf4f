"""Multi-process driver (one process per GPU, torch.distributed) -- SURVEY.md 8(e), scope row f3.

The explicit step has ONE real exchange per stage (the ghost cells of U) plus one
scalar min for dt per step.  `DistSolver` holds this rank's zones of a decomposition every rank
derives from the same mesh and drives the C-ABI calls of include/swe_b200.h ("zones distributed
over ranks"); the library never calls a communication library, this module does, and only for

  * the 8-byte all-reduce(min) of dt (which doubles as the stream-ordered barrier that orders the
    peer-memory pushes) and one more barrier per step,
  * with transport "staged": an all-to-all of the packed halo buffers (pack -> NCCL -> unpack),
  * set-up: the all-gather of the CUDA IPC handles of the state buffers (transport "p2p": the
    exchange is then ONE kernel per rank storing its send cells straight into its peers' ghost
    ranges over NVLink / NVSwitch).

Backend: nccl when CUDA is available (gloo with SWE_DIST_GLOO=1 or on CPU: tests).  With gloo,
CUDA tensors are staged through the host (test configurations only: 2 processes sharing one GPU).
Everything else here is bench.py plumbing: barrier, max-over-ranks time, sums, block sharding.
"""
import os


def init_from_env():
    """Returns (rank, world_size, local_rank); initialises torch.distributed when WORLD_SIZE > 1."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        if not dist.is_initialized():
            backend = "nccl" if torch.cuda.is_available() and not os.environ.get("SWE_DIST_GLOO") else "gloo"
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            if torch.cuda.is_available():
                torch.cuda.set_device(local % torch.cuda.device_count())
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world, local


def _active():
    try:
        import torch.distributed as dist
        return dist.is_available() and dist.is_initialized()
    except Exception:
        return False


def _reduce(x, op_name):
    if not _active():
        return float(x)
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return float(t.item())


def reduce_max(x):
    return _reduce(x, "MAX")


def reduce_sum(x):
    return _reduce(x, "SUM")


def barrier():
    if _active():
        import torch.distributed as dist
        dist.barrier()


def finalize():
    if _active():
        import torch.distributed as dist
        dist.destroy_process_group()


def shard_units(n_units, rank, world):
    """Contiguous block of `n_units` independent units (zones, replicas) owned by `rank`."""
    base, rem = divmod(int(n_units), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def zone_blocks(nzones, world):
    """zone_begin of swe_zones_create_dist: contiguous blocks of zones per rank."""
    return [shard_units(nzones, r, world)[0] for r in range(world)] + [int(nzones)]


class TorchComm:
    """The collectives DistSolver needs, over torch.distributed (nccl; gloo stages CUDA tensors
    through the host).  All calls are collective over the default group."""

    def __init__(self):
        import torch.distributed as dist
        self.dist = dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.staged_host = dist.get_backend() != "nccl"

    def allreduce_min(self, t):
        """In-place MIN all-reduce of a device tensor, ordered on the current stream."""
        if self.staged_host and t.is_cuda:
            c = t.cpu()
            self.dist.all_reduce(c, op=self.dist.ReduceOp.MIN)
            t.copy_(c)
        else:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MIN)

    def allreduce_min_async(self, t):
        """Starts the MIN all-reduce behind the work already on the current stream and returns a
        handle for wait(): later work on the current stream overlaps with it (nccl; with gloo the
        host-staged reduction is done at once and None is returned)."""
        if self.staged_host:
            self.allreduce_min(t)
            return None
        return self.dist.all_reduce(t, op=self.dist.ReduceOp.MIN, async_op=True)

    @staticmethod
    def wait(work):
        """Makes the current stream wait for an asynchronous collective (the host does not block)."""
        if work is not None:
            work.wait()

    def all_to_all(self, recv, send, recv_splits, send_splits):
        if self.staged_host and send.is_cuda:
            r = recv.cpu()
            self.dist.all_to_all_single(r, send.cpu(), recv_splits, send_splits)
            recv.copy_(r)
        else:
            self.dist.all_to_all_single(recv, send, recv_splits, send_splits)

    def all_gather_bytes(self, arr):
        """arr: numpy uint8; returns the list of every rank's array."""
        import torch
        t = torch.from_numpy(arr.copy())
        if not self.staged_host:
            t = t.cuda()
        out = [torch.empty_like(t) for _ in range(self.world)]
        self.dist.all_gather(out, t)
        return [o.cpu().numpy() for o in out]

    def allreduce_sum(self, t):
        if self.staged_host and t.is_cuda:
            c = t.cpu()
            self.dist.all_reduce(c, op=self.dist.ReduceOp.SUM)
            t.copy_(c)
        else:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)

    def host_barrier(self):
        import torch
        if torch.cuda.is_available():
            torch.cuda.synchronize()
        self.dist.barrier()


class DistSolver:
    """This rank's share of a mesh split into zones over the ranks of the default process group.

    cfg: an input dictionary of swe_inputs.configs (every rank passes the same one); nzones zones by
    recursive coordinate bisection (or zone_of_cell), rank r holding the block zone_blocks()[r:r+2];
    nlayers ghost layers (>= 2 for MUSCL / WAF / MUSCL_MS); transport "p2p" (peer-memory push, one
    kernel per exchange) or "staged" (pack -> all-to-all -> unpack).

    Streams: the solver owns a CUDA stream; the library context is created on it and every library
    call and every collective is issued under it, because the stream-ordered collectives that order
    the halo pushes against the peers' ghost reads only do so on ONE stream.  step(), exchange(),
    set_state() and the getters order that stream behind the caller's current torch stream on entry
    and the caller's stream behind it on exit, so a caller may use any stream.

    graphs=True (nccl backend): one step is captured once per (scheme, cfl) as a CUDA graph --
    kernels and collectives alike -- and replayed; the ranks agree on whether the capture worked and
    fall back to call-by-call steps together if it did not on any of them.
    """

    def __init__(self, cfg, nzones=None, nlayers=2, transport="p2p", zone_of_cell=None, comm=None,
                 schedule="overlap", graphs=True):
        import torch
        from . import binding as sw
        self.sw, self.torch = sw, torch
        self.comm = comm if comm is not None else TorchComm()
        self.rank, self.world = self.comm.rank, self.comm.world
        if transport not in ("p2p", "staged"):
            raise ValueError("transport must be 'p2p' or 'staged'")
        self.transport = transport
        if schedule not in ("plain", "overlap"):
            raise ValueError("schedule must be 'plain' or 'overlap'")
        self.schedule = schedule
        self._primed = False
        if nzones is None:
            nzones = 1
            while nzones < self.world:
                nzones *= 2
        self.nzones, self.nlayers = int(nzones), int(nlayers)
        # the library's kernels and the collectives must be ordered on ONE stream: the solver owns
        # a stream, creates the context on it and issues every library call and every collective
        # under it; step() / exchange() / set_state() order that stream behind the caller's current
        # stream on entry and the caller's stream behind it on exit
        self.tstream = torch.cuda.Stream() if torch.cuda.is_available() else None
        self.stream = self.tstream.cuda_stream if self.tstream is not None else 0
        self.graphs = bool(graphs)
        self._graph = {}                # (scheme, cfl, body) -> (CUDAGraph, launches, halo bytes, steps) of one step
        self.graph_replays = 0
        self.host_us_per_step = None    # host time of the last step() call per step (enqueue only)
        self._flux_done = None
        self.profile = False
        with self._on_stream():
            self.ctx = sw.create_from_config(cfg, cuda_stream=self.stream or None)
        self.ncell = sw.swe_mesh_info(self.ctx)["ncell"]
        sw.swe_zones_create_dist(self.ctx, self.nzones, self.nlayers, zone_of_cell, self.world, self.rank,
                                 zone_blocks(self.nzones, self.world))
        self.send_cells, self.recv_cells = sw.swe_halo_counts(self.ctx, self.world)
        dev = torch.device("cuda", torch.cuda.current_device())
        self.minbuf = torch.zeros(1, dtype=torch.float64, device=dev)
        self.token = torch.zeros(1, dtype=torch.float64, device=dev)
        if self.transport == "p2p":
            # map every peer's state buffers (CUDA IPC); if any rank cannot (no peer access between
            # two GPUs, IPC not permitted), ALL ranks take the staged transport -- said on stderr
            ok, why = 1.0, ""
            try:
                mine = sw.swe_peer_export(self.ctx)
            except sw.SweError as e:
                import numpy as np
                mine, ok, why = np.zeros(128, np.uint8), 0.0, str(e)
            handles = self.comm.all_gather_bytes(mine)
            for p in range(self.world):
                if ok and p != self.rank:
                    try:
                        sw.swe_peer_import(self.ctx, p, handles[p])
                    except sw.SweError as e:
                        ok, why = 0.0, str(e)
                        break
            flag = torch.tensor([ok], dtype=torch.float64, device=dev)
            self.comm.allreduce_min(flag)
            if float(flag.item()) < 1.0:
                import sys
                if why or self.rank == 0:
                    sys.stderr.write("[swe dist] rank %d: peer-memory transport unavailable (%s); every rank uses "
                                     "the staged transport\n" % (self.rank, why or "another rank failed"))
                self.transport = "staged"
        if self.transport == "staged":
            self.sendbuf = torch.zeros(max(1, 3 * int(self.send_cells.sum())), dtype=torch.float64, device=dev)
            self.recvbuf = torch.zeros(max(1, 3 * int(self.recv_cells.sum())), dtype=torch.float64, device=dev)
            self.ssplit = [3 * int(v) for v in self.send_cells]
            self.rsplit = [3 * int(v) for v in self.recv_cells]
        self.comm.host_barrier()

    # -- one exchange of the ghosts of state buffer `buffer` (0 = U, 1 = the Heun stage buffer) --
    def _on_stream(self):
        """Context manager: run under the solver's stream, ordered behind the caller's current
        stream on entry; the caller's stream is ordered behind the solver's on exit."""
        import contextlib
        torch = self.torch

        @contextlib.contextmanager
        def cm():
            if self.tstream is None:
                yield
                return
            cur = torch.cuda.current_stream()
            if cur.cuda_stream == self.tstream.cuda_stream:      # already inside (nested call)
                yield
                return
            self.tstream.wait_stream(cur)
            with torch.cuda.stream(self.tstream):
                yield
            cur.wait_stream(self.tstream)
        return cm()

    # -- one exchange of the ghosts of state buffer `buffer` (0 = U, 1 = the Heun stage buffer) --
    def exchange(self, buffer):
        with self._on_stream():
            self._exchange(buffer)

    def _exchange(self, buffer):
        sw = self.sw
        if self.transport == "p2p":
            sw.swe_halo_push(self.ctx, buffer)
        else:
            sw.swe_halo_pack(self.ctx, buffer, self.sendbuf)
            n_s, n_r = sum(self.ssplit), sum(self.rsplit)
            self.comm.all_to_all(self.recvbuf[:n_r], self.sendbuf[:n_s], self.rsplit, self.ssplit)
            sw.swe_halo_unpack(self.ctx, buffer, self.recvbuf)

    def barrier_stream(self):
        """Stream-ordered barrier: nobody's stream passes it before everybody's reached it."""
        with self._on_stream():
            self.comm.allreduce_min(self.token)

    def _exchange_async(self, buffer):
        self._exchange(buffer)
        return self.comm.allreduce_min_async(self.token) if self.transport == "p2p" else None

    # -- the step ---------------------------------------------------------------------------------
    # Invariant between steps ("primed"): the ghosts of buffer 0 are current on every rank and
    # minbuf holds the all-reduced minimum of R_i / lambda_i of U^n -- both collectives have been
    # waited for on the stream (a stream wait: the host never blocks).
    #
    # schedule "plain": the serial order  flux, update, exchange, barrier  per stage.
    # schedule "overlap" (scope row f2; "high overlap"): every stage updates the cells
    # on the send lists first, exchanges them, starts the barrier asynchronously and updates the
    # rest of the domain while the collective is in flight.  The all-reduce of dt is hidden too: for
    # every scheme but WAF the body is ROTATED -- it starts behind the gradient / flux pass of its
    # first stage and ends with that pass of the NEXT step, which runs while the all-reduce of the
    # minimum is in flight (dt is first needed by the update; WAF needs it in the flux and keeps the
    # unrotated order).  `_flux_done` remembers for which scheme that pass has been enqueued.
    # Hazards (buffer b = 0: U, 1: the Heun stage buffer):
    #   * a rank reads its ghosts of b only behind wait(barrier) of the exchange of b;
    #   * an exchange of b is issued behind a wait() on a collective that every rank started after
    #     its last flux pass over b, so nobody's ghosts are overwritten while still being read.
    #     Heun: the barrier of the other buffer's exchange is that collective.  Euler schemes have
    #     one buffer: they start one more barrier right after the flux pass and wait for it before
    #     the exchange.
    # With the nccl backend one step (same kernels, same collectives, same order; dt lives in
    # device memory) is captured ONCE as a CUDA graph per (scheme, cfl) and replayed: the host then
    # spends one graph launch per step instead of ~15 C calls and 3 torch.distributed calls.
    def _prime(self):
        sw, comm = self.sw, self.comm
        if self._primed:
            return
        bar = self._exchange_async(0)
        sw.swe_dist_local_min(self.ctx, self.minbuf)
        mw = comm.allreduce_min_async(self.minbuf)
        comm.wait(bar)
        comm.wait(mw)
        self._primed = True
        self._flux_done = None

    def _body_plain(self, sch, cfl):
        sw = self.sw
        heun = sch in (sw.SWE_MUSCL, sw.SWE_MUSCL_MS)
        p2p = self.transport == "p2p"
        sw.swe_dist_begin_step(self.ctx, self.minbuf, cfl)
        sw.swe_dist_stage(self.ctx, sch, 0)
        if heun:
            self._exchange(1)
            if p2p:
                self.comm.allreduce_min(self.token)    # every push of buffer 1 has landed
            sw.swe_dist_stage(self.ctx, sch, 1)
        elif p2p:
            self.comm.allreduce_min(self.token)        # everybody has read its ghosts of buffer 0
        self._exchange(0)
        sw.swe_dist_local_min(self.ctx, self.minbuf)
        self.comm.allreduce_min(self.minbuf)           # dt; with p2p also: every push of buffer 0 has landed

    def _body_overlap(self, sch, cfl):
        sw, comm = self.sw, self.comm
        heun = sch in (sw.SWE_MUSCL, sw.SWE_MUSCL_MS)
        waf = sch == sw.SWE_WAF
        p2p = self.transport == "p2p"
        if waf:
            sw.swe_dist_begin_step(self.ctx, self.minbuf, cfl)
            sw.swe_dist_flux(self.ctx, sch, 0)
        else:                                              # rotated: flux(0) is already behind us
            sw.swe_dist_begin_step(self.ctx, self.minbuf, cfl)
        if heun:
            sw.swe_dist_update(self.ctx, sch, 0, 1)            # send cells of U'
            bar1 = self._exchange_async(1)
            sw.swe_dist_update(self.ctx, sch, 0, 2)            # the rest, behind the barrier
            comm.wait(bar1)
            sw.swe_dist_flux(self.ctx, sch, 1)
            sw.swe_dist_update(self.ctx, sch, 1, 1)            # send cells of U^{n+1}
            bar = self._exchange_async(0)
            sw.swe_dist_update(self.ctx, sch, 1, 2)
        else:
            done = comm.allreduce_min_async(self.token) if p2p else None   # everybody's flux pass is over
            sw.swe_dist_update(self.ctx, sch, 0, 1)
            comm.wait(done)
            bar = self._exchange_async(0)
            sw.swe_dist_update(self.ctx, sch, 0, 2)
        sw.swe_dist_local_min(self.ctx, self.minbuf)
        mw = comm.allreduce_min_async(self.minbuf)
        comm.wait(bar)                                     # ghosts of buffer 0 are current
        if not waf:
            sw.swe_dist_flux(self.ctx, sch, 0)             # of the NEXT step, while the minimum is reduced
        comm.wait(mw)

    def step(self, nsteps, cfl, scheme):
        """nsteps time steps, asynchronous: enqueued on the solver's stream, which is ordered
        behind the caller's current stream; the caller's stream waits for it (no host sync)."""
        import time as _time
        sw = self.sw
        sch = sw.SCHEMES[scheme] if isinstance(scheme, str) else int(scheme)
        nsteps = int(nsteps)
        if nsteps <= 0:
            return
        overlap = self.schedule == "overlap"
        rotated = overlap and sch != sw.SWE_WAF
        body = self._body_overlap if overlap else self._body_plain
        t0 = _time.perf_counter()
        with self._on_stream():
            self._prime()
            if rotated and self._flux_done != sch:
                sw.swe_dist_flux(self.ctx, sch, 0)
            self._flux_done = sch if rotated else None
            done = 0
            if self.graphs and nsteps >= 2 and self.tstream is not None and not self.comm.staged_host \
                    and not self.profile:
                key = (sch, float(cfl), self.schedule)
                ent = self._graph.get(key)
                if ent is None:
                    body(sch, cfl)                         # a real step: NCCL set-up and lazy loading happen outside the capture
                    done = 1
                    ent = self._capture(body, sch, cfl)
                    # every rank or none: a rank whose capture failed has neither run nor recorded the
                    # step, the others have only recorded it, so nobody has executed anything yet and
                    # all can still fall back to enqueuing call by call together (one-time host sync)
                    ok = self.torch.tensor([1.0 if ent is not None else 0.0], dtype=self.torch.float64,
                                           device=self.minbuf.device)
                    self.comm.allreduce_min(ok)
                    if float(ok.item()) < 1.0:
                        if ent is not None:
                            import sys
                            sys.stderr.write("[swe dist] rank %d: another rank could not capture the step as a CUDA "
                                             "graph; steps are enqueued call by call\n" % self.rank)
                        ent = None
                        self.graphs = False
                    if ent is not None:
                        self._graph[key] = ent
                if ent is not None:
                    g, dl, dh, ds = ent
                    n = nsteps - done
                    for _ in range(n):
                        g.replay()
                    sw.swe_account_replays(self.ctx, n * ds, n * dl, n * dh)
                    self.graph_replays += n
                    done = nsteps
            for _ in range(nsteps - done):
                body(sch, cfl)
        self.host_us_per_step = 1e6 * (_time.perf_counter() - t0) / nsteps

    def _capture(self, body, sch, cfl):
        """One step captured as a CUDA graph on the solver's stream (kernels of the library and the
        NCCL collectives alike).  Returns None -- and says so once on stderr -- if the capture
        fails (then every step is enqueued call by call, as with gloo)."""
        torch, sw = self.torch, self.sw
        g = torch.cuda.CUDAGraph()
        self.tstream.synchronize()
        s1 = sw.swe_get_stats(self.ctx)
        try:
            with torch.cuda.graph(g, stream=self.tstream, capture_error_mode="thread_local"):
                if os.environ.get("SWE_DIST_GRAPH_FAIL"):      # test hook: a capture that breaks half way
                    self.sw.swe_dist_begin_step(self.ctx, self.minbuf, cfl)
                    raise RuntimeError("SWE_DIST_GRAPH_FAIL is set")
                body(sch, cfl)
        except Exception as e:                             # depends on the NCCL build
            import sys
            sys.stderr.write("[swe dist] rank %d: CUDA-graph capture of the step failed (%s); steps are enqueued "
                             "call by call\n" % (self.rank, str(e).splitlines()[0] if str(e) else type(e).__name__))
            self.graphs = False
            g = None
        s2 = sw.swe_get_stats(self.ctx)
        # the captured body was recorded, not run: take its counts back out of the library's statistics
        dl, dh, ds = (s2["kernel_launches"] - s1["kernel_launches"], s2["halo_bytes"] - s1["halo_bytes"],
                      s2["steps"] - s1["steps"])
        sw.swe_account_replays(self.ctx, -ds, -dl, -dh)
        return None if g is None else (g, dl, dh, ds)

    def set_profile(self, on):
        """Per-kernel CUDA events of the library (swe_set_profile); steps are then enqueued call
        by call (events cannot be recorded inside a replayed graph)."""
        self.profile = bool(on)
        with self._on_stream():
            self.sw.swe_set_profile(self.ctx, bool(on))

    def _drain(self):
        """Nothing is left in flight between steps: every collective has been waited for on the
        stream; kept for callers of the round-1 interface."""
        return None

    def time(self):
        return self.sw.swe_get_time(self.ctx)

    def set_state(self, h, hu, hv):
        self._primed = False
        self._flux_done = None
        self.comm.host_barrier()
        with self._on_stream():
            self.sw.swe_set_state(self.ctx, h, hu, hv)
        self.comm.host_barrier()

    def get_state_local(self, h, hu, hv):
        """Fills the entries of this rank's owned cells only."""
        with self._on_stream():
            self.sw.swe_get_state(self.ctx, h, hu, hv)

    def get_state(self):
        """The full state on every rank (numpy): owned cells of all ranks summed over zero arrays."""
        torch = self.torch
        out = torch.zeros(3, self.ncell, dtype=torch.float64, device=self.minbuf.device)
        with self._on_stream():
            self.sw.swe_get_state(self.ctx, out[0], out[1], out[2])
            self.comm.allreduce_sum(out)
        if self.tstream is not None:
            self.tstream.synchronize()
        return tuple(o.cpu().numpy() for o in out)

    def close(self):
        self._graph.clear()
        self.comm.host_barrier()                       # nobody still pushes into this rank's buffers
        self.sw.swe_mesh_destroy(self.ctx)
        self.ctx = None
