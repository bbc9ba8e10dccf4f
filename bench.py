#!/usr/bin/env python
"""bench.py -- headline benchmark: cell-updates/s of the fp64 MUSCL-RK2 step on the ~13 M-cell
synthetic river mesh (BASELINE.json configs[3]) on B200, with the HBM roofline of its dominant
kernel, an end-to-end figure through the C ABI with host buffers, and the CPU oracle timed beside
it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload c3|c3s|c1|c2]
                    [--scheme muscl|hllc|waf|muscl_ms] [--zones Z --layers L] [--transport p2p|staged]

One "step" = one full time step (CFL min-reduction, both Heun stages: gradient+limiter, edge flux,
cell update) over every cell of the mesh.  N > 1 (torchrun): the SAME mesh split into zones over
the N ranks (strong scaling; paper_2307_16758_b200/dist.py): per stage one halo exchange of the
ghost cells (one kernel storing into the peers' ghost ranges over NVLink peer memory, or pack ->
NCCL all-to-all -> unpack with --transport staged) and per step one all-reduce(min) of dt;
value = cells x steps / max-over-ranks device time.  --replicas runs N independent copies instead.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

ALGO_BYTES = {  # algorithmic bytes per cell (N_e = 1.5 N_c)
    "grad_limit": 156.0, "edge_flux_muscl": 252.0, "edge_flux_hllc": 140.0, "edge_flux_waf": 296.0,
    "cell_update_stage": 136.0, "cell_update_final": 168.0, "cell_update_euler": 144.0,
    "step_muscl": 1120.0, "step_hllc": 284.0, "step_waf": 440.0,
    "edge_flux_muscl_ms": 200.0, "step_muscl_ms": 704.0,   # 2 x (edge 108 + U 32 + flux 60) + 136 + 168
}
METRIC = "cell-updates/s (fp64 MUSCL-RK2, 13M cells) and achieved HBM GB/s vs ~8 TB/s"
PAPER_CONTEXT = {   # whole-simulation wall times, step counts not stated -> context only
    "muscl": "paper Table 5 (PAPER.md:483), 13 M-triangle Mille Iles mesh, MUSCL, 2 ghost layers, high overlap: "
             "326.38 s on 8 P100 ... 90.08 s on 32 P100 (whole simulation; number of steps not stated)",
    "muscl_ms": "paper Table 5 (PAPER.md:483), MUSCL (the multislope scheme is the paper's own), 2 layers, high overlap: "
                "326.38 s on 8 P100 ... 90.08 s on 32 P100 (whole simulation; number of steps not stated)",
    "hllc": "paper Table 5 (PAPER.md:481), HLLC, 1 ghost layer, high overlap: 205.26 s on 8 P100 ... 60.63 s on 32 P100 "
            "(whole simulation; number of steps not stated)",
    "waf": "paper Table 5 (PAPER.md:484), WAF, 2 ghost layers, high overlap: 329.56 s on 8 P100 ... 90.82 s on 32 P100 "
           "(whole simulation; number of steps not stated)",
}
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback


def build_workload(name):
    from swe_inputs import config1, config2, config3
    if name == "c3":
        return config3(), "configs[3]: 60 km x 8 km synthetic river mesh, ~13 M triangles, seed 3"
    if name == "c3p":
        from swe_inputs import permuted
        return permuted(config3()), "configs[3] with its ~13 M triangles listed in a random order (seed 7)"
    if name == "c3w":
        from swe_inputs import flooded
        return flooded(config3(), 18.0), "configs[3] mesh and bed, flooded to a flat surface at 18 m: no dry cell"
    if name == "dl":
        from swe_inputs import delaunay_case
        return (delaunay_case(n=3_000_000, lx=20000.0, ly=12000.0, seed=5, dam=True),
                "Delaunay triangulation of 3 M jittered points (~6 M triangles, mixed windings), dam break over bumps with dry tops, seed 5")
    if name == "c3s":
        return config3(length=6000.0), "configs[3] generator on a 6 km reach (~1.3 M triangles), seed 3"
    if name == "c3t":
        return config3(length=1600.0, half_width=600.0), "configs[3] generator, tiny reach (smoke)"
    if name == "c1":
        return config1(), "configs[1]: circular dam break, 245 000 triangles, seed 1"
    if name == "c2":
        return config2(), "configs[2]: lake at rest, ~1.0 M triangles, seed 2"
    raise ValueError(name)


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [s.strip() for s in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def traffic_table():
    """ncu DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full`
    capture, profiles/dram_traffic.csv: workload, kernel, bytes, capture): {(workload, kernel): (bytes, capture)}.
    A table captured in another run, NOT a measurement of this one: the line says so (traffic_source)."""
    out = {}
    p = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if os.path.exists(p):
        for ln in open(p):
            f = ln.strip().split(",", 3)
            if len(f) >= 3 and f[0] != "workload":
                try:
                    out[(f[0], f[1])] = (float(f[2]), f[3] if len(f) > 3 else "")
                except ValueError:
                    pass
    return out


def oracle_run(cfg, scheme, cfl, warmup, steps, budget_s=None, threads=0):
    """Times the CPU oracle as it stands (threads = 0: all host cores); returns cell-updates/s and details."""
    from oracle import pyoracle as po
    cores = po.set_threads(threads)
    o = po.Oracle.from_config(cfg)
    t0 = time.perf_counter()
    o.step(max(1, warmup), cfl, scheme)
    per = (time.perf_counter() - t0) / max(1, warmup)
    if budget_s is not None:                      # bounded sample: as many steps as fit the budget
        steps = int(max(2, min(steps, budget_s / max(per, 1e-9))))
    t0 = time.perf_counter()
    o.step(steps, cfl, scheme)
    dt = time.perf_counter() - t0
    nt = o.nt
    o.close()
    return nt * steps / dt, cores, nt, dt, steps


def run_reference(args):
    """--impl reference: the oracle on the box's host cores, on a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # the SAME workload as the GPU arm (at 13.1 M cells the oracle runs ~20 steps);
    # each step is one full time step of the whole mesh, as many of the requested steps as fit 90 s
    cfg, desc = build_workload(args.workload)
    cfl = 0.9 if args.scheme == "hllc" else 0.45
    warm = max(1, min(args.warmup, 2))
    v, cores, nt, secs, steps = oracle_run(cfg, args.scheme, cfl, warm, args.steps, budget_s=90.0)
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": "cell-updates/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": 1e3 * secs / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "cells": nt, "scheme": args.scheme, "cfl": cfl},
        "cpu_baseline": {"value": v, "unit": "cell-updates/s", "cores": cores, "kind": "oracle",
                         "sample": "%s, %d cells, %d steps of %d requested" % (desc, nt, steps, args.steps)},
        "e2e": {"value": v, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def kernel_roofline(prof, steps, scheme, cells, step_ms, peak, peak_src, workload):
    """Per-kernel figures from the CUDA-event profile of the timed step loop (swe_get_profile)."""
    kern = {}
    tot_ms = sum(v[0] for v in prof.values())
    for k, (kms, n) in prof.items():
        if n:
            kern[k] = {"ms_per_launch": kms / n, "launches_per_step": n / steps, "share": kms / tot_ms}
    # algorithmic bytes per launch of each kernel kind (averaged over its launches in a step)
    if scheme == "muscl":
        algo = {"grad_limit": ALGO_BYTES["grad_limit"], "edge_flux": ALGO_BYTES["edge_flux_muscl"],
                "cell_update": 0.5 * (ALGO_BYTES["cell_update_stage"] + ALGO_BYTES["cell_update_final"])}
    elif scheme == "muscl_ms":
        algo = {"edge_flux": ALGO_BYTES["edge_flux_muscl_ms"],
                "cell_update": 0.5 * (ALGO_BYTES["cell_update_stage"] + ALGO_BYTES["cell_update_final"])}
    elif scheme == "hllc":
        algo = {"edge_flux": ALGO_BYTES["edge_flux_hllc"], "cell_update": ALGO_BYTES["cell_update_euler"]}
    else:
        algo = {"edge_flux": ALGO_BYTES["edge_flux_waf"], "cell_update": ALGO_BYTES["cell_update_euler"]}
    for k in algo:
        if k in kern:
            kern[k]["algo_GBps"] = algo[k] * cells / (kern[k]["ms_per_launch"] * 1e-3) / 1e9
            kern[k]["frac_of_peak"] = kern[k]["algo_GBps"] / peak
    dom = max((k for k in algo if k in kern), key=lambda k: kern[k]["share"])
    tt = traffic_table()
    row = tt.get((workload, dom + "_" + scheme), tt.get((workload, dom)))
    traffic, traffic_src = (row[0], "profiles/dram_traffic.csv (ncu --set full, captured earlier: %s)" % row[1]) if row else (None, None)
    step_bytes = ALGO_BYTES["step_" + scheme]
    rate = cells / (step_ms * 1e-3)
    # physical DRAM bytes of one step from the ncu table (13.1 M-cell MUSCL-RK2 only), SURVEY 8(d)(iii)
    step_dram = None
    if scheme == "muscl" and all((workload, k) in tt for k in ("grad_limit", "edge_flux_muscl", "cell_update_muscl")):
        step_dram = 2.0 * (tt[(workload, "grad_limit")][0] + tt[(workload, "edge_flux_muscl")][0] + tt[(workload, "cell_update_muscl")][0])
    extra = {}
    if traffic:
        # what the kernel actually moved (ncu) over the time measured here: the fraction of the
        # bandwidth the kernel reaches on its own bytes, whatever the dry-cell skips leave out
        extra["frac_physical"] = traffic / (kern[dom]["ms_per_launch"] * 1e-3) / 1e9 / peak
        extra["physical_GBps"] = traffic / (kern[dom]["ms_per_launch"] * 1e-3) / 1e9
    if kern[dom]["algo_GBps"] > 0.95 * peak:
        extra["note"] = ("frac counts the FIXED algorithmic bytes of every cell and edge; the kernels skip cells / edges "
                         "without water (zero records written without reading their inputs), so on a partly dry state "
                         "the bytes actually moved are fewer: read frac_physical (ncu bytes) and all_wet (no dry cell, "
                         "where the algorithmic count is what is moved) beside it; DESIGN.md section 6")
    if step_dram:
        extra.update({"step_dram_bytes_ncu": step_dram, "step_algo_over_dram_bytes": step_bytes * cells / step_dram,
                      "step_dram_GBps": step_dram / (step_ms * 1e-3) / 1e9,
                      "step_frac_physical": step_dram / (step_ms * 1e-3) / 1e9 / peak})
    return dict(extra, **{
        "bound": "hbm", "kernel": dom, "achieved": kern[dom]["algo_GBps"], "peak": peak, "unit": "GB/s",
        "frac": kern[dom]["algo_GBps"] / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
        "algo_bytes_per_launch": algo[dom] * cells,
        "step_algo_GBps": step_bytes * rate / 1e9,
        "step_frac_of_peak": step_bytes * rate / 1e9 / peak,
        "step_frac_of_8TBps": step_bytes * rate / 1e9 / 8000.0,
        "kernels": kern,
    })


def run_dist(args, rank, world, local, cfg, desc, cfl):
    """N > 1: the mesh split into zones over the ranks (strong scaling), one halo exchange per stage
    over NVLink peer memory (or pack -> NCCL all-to-all -> unpack) and one all-reduce(min) for dt."""
    import torch
    from paper_2307_16758_b200 import dist as swdist
    import paper_2307_16758_b200 as sw

    t_setup = time.perf_counter()
    S = swdist.DistSolver(cfg, nzones=args.zones if args.zones > 0 else None, nlayers=args.layers,
                          transport=args.transport, schedule=args.schedule, graphs=not args.no_dist_graph)
    setup_s = swdist.reduce_max(time.perf_counter() - t_setup)     # host mesh + zones + upload + IPC, slowest rank
    nt = S.ncell
    info = sw.swe_mesh_info(S.ctx)
    owned = sum(sw.swe_zone_describe_counts(S.ctx, z)[0] for z in range(*swdist.shard_units(S.nzones, rank, world)))
    S.step(args.warmup, cfl, args.scheme)
    torch.cuda.synchronize()
    swdist.barrier()
    l0 = sw.swe_get_stats(S.ctx)
    clk = ClockSampler(local)
    clk.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    S.step(args.steps, cfl, args.scheme)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    l1 = sw.swe_get_stats(S.ctx)
    swdist.barrier()
    ms_max = swdist.reduce_max(ms)
    value = nt * args.steps / (ms_max * 1e-3)
    launches = swdist.reduce_sum(float(l1["kernel_launches"] - l0["kernel_launches"]))
    halo = swdist.reduce_sum(float(l1["halo_bytes"] - l0["halo_bytes"])) / args.steps

    # per-kernel CUDA events on this rank's launches (rank 0 reports its own share of the mesh)
    host_us = S.host_us_per_step                   # host time per step of the timed call (enqueue only)
    replays = S.graph_replays
    S.set_profile(True)
    S.step(args.steps, cfl, args.scheme)
    prof = sw.swe_get_profile(S.ctx)
    S.set_profile(False)
    # exposed collective time: the step's device time minus this rank's kernels (events around every launch)
    kern_ms = sum(v[0] for v in prof.values()) / args.steps
    clocks = clk.stop()
    peak, peak_src = hbm_peak()
    roofline = kernel_roofline(prof, args.steps, args.scheme, owned, ms / args.steps, peak, peak_src, args.workload)
    roofline["note"] = "rank 0's kernels over the %d cells its zones own (ghost cells not counted)" % owned

    # end to end with HOST buffers: every rank uploads the full state, steps, reads its own cells back
    e2e_steps = max(1, min(args.e2e_steps, args.steps))
    hbuf = [torch.zeros(nt, dtype=torch.float64).pin_memory() for _ in range(3)]
    full = S.get_state()
    for b, f in zip(hbuf, full):
        b.copy_(torch.from_numpy(f))
    for _ in range(2):
        S.set_state(*hbuf); S.step(1, cfl, args.scheme); S.get_state_local(*hbuf)
    torch.cuda.synchronize()
    swdist.barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        S.set_state(*hbuf)
        S.step(1, cfl, args.scheme)
        S.get_state_local(*hbuf)
    torch.cuda.synchronize()
    e2e_s = swdist.reduce_max(time.perf_counter() - t0)
    e2e = {"value": nt * e2e_steps / e2e_s, "unit": "cell-updates/s", "steps": e2e_steps,
           "h2d_bytes_per_step": 2 * 3 * 8 * nt * world, "d2h_bytes_per_step": 3 * 8 * nt * world,
           "what": "per step and rank: swe_set_state(full state, pinned host) + one distributed step + "
                   "swe_get_state(pinned host; the rank's own cells are filled, which stages the caller's "
                   "arrays through the device: a second host-to-device copy)"}
    S.close()
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "cell-updates/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "cells": nt, "edges": info["nedge"], "scheme": args.scheme, "cfl": cfl,
                       "l2": "inputs larger than L2 per rank" if nt / world > 2_000_000 else
                             "a rank's share may fit L2 at this size",
                       "parallelism": "zones over %d ranks (%d zones, %d ghost layers), halo transport %s, "
                                      "schedule %s, all-reduce(min) of dt" % (world, S.nzones, S.nlayers, S.transport,
                                                                              S.schedule),
                       "zones": S.nzones, "ghost_layers": S.nlayers, "halo_bytes_per_step": halo,
                       "transport_requested": args.transport, "transport_used": S.transport,
                       "solver_setup_s": setup_s,
                       "step_as_cuda_graph": bool(replays), "host_us_per_step": host_us,
                       "rank0_kernel_ms_per_step": kern_ms,
                       "rank0_not_in_kernels_ms_per_step": max(0.0, ms / args.steps - kern_ms),
                       "paper_context": PAPER_CONTEXT[args.scheme]},
            "roofline": roofline, "e2e": e2e, "cpu_baseline": None,
            "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(line))
    swdist.finalize()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3", choices=["c3", "c3p", "c3w", "dl", "c3s", "c3t", "c1", "c2"])
    ap.add_argument("--scheme", default="muscl", choices=["muscl", "hllc", "waf", "muscl_ms"])
    ap.add_argument("--zones", type=int, default=0)
    ap.add_argument("--layers", type=int, default=2)
    ap.add_argument("--renumber", default="hilbert", choices=["hilbert", "rcm", "none"])
    ap.add_argument("--transport", default="p2p", choices=["p2p", "staged"])
    ap.add_argument("--schedule", default="overlap", choices=["overlap", "plain"])
    ap.add_argument("--force-dist", action="store_true",
                    help="run the distributed arm (DistSolver, zones over ranks) even with a single rank")
    ap.add_argument("--no-dist-graph", action="store_true",
                    help="distributed arm: enqueue every step call by call instead of replaying it as one CUDA graph")
    ap.add_argument("--replicas", action="store_true", help="N > 1: independent replicas instead of one split mesh")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--dry-masks", action="store_true",
                    help="swe_set_dry_masks on: leave the records of cells / edges without water alone (un-zoned mesh only)")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--reps", type=int, default=5,
                    help="the timed region of K steps is run this many times; value = the median (BASELINE.md section 4)")
    ap.add_argument("--no-all-wet", action="store_true",
                    help="skip the second measurement on the flooded mesh (roofline.all_wet; workload c3, N = 1 only)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2307_16758_b200 import dist as swdist
    import paper_2307_16758_b200 as sw

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        # NCCL's communicator set-up lines (ranks, transports, NVLS) go to stderr: evidence of the N-rank run
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    rank, world, local = swdist.init_from_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    local = local % torch.cuda.device_count()      # test configurations put several ranks on one GPU
    torch.cuda.set_device(local)
    sw.lib()   # fails loudly if the CUDA extension is missing

    cfg, desc = build_workload(args.workload)
    cfl = 0.9 if args.scheme == "hllc" else 0.45
    if args.force_dist and world == 1:
        import torch.distributed as tdist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29533")
        tdist.init_process_group(backend="gloo" if os.environ.get("SWE_DIST_GLOO") else "nccl", rank=0, world_size=1)
    if (world > 1 and not args.replicas) or args.force_dist:
        return run_dist(args, rank, world, local, cfg, desc, cfl)
    ctx = sw.create_from_config(cfg, {"hilbert": sw.SWE_RENUM_HILBERT, "rcm": sw.SWE_RENUM_RCM,
                                      "none": sw.SWE_RENUM_NONE}[args.renumber])
    info = sw.swe_mesh_info(ctx)
    nt = info["ncell"]
    if args.zones > 0:
        sw.swe_zones_create(ctx, args.zones, args.layers)
    if args.dry_masks:
        sw.swe_set_dry_masks(ctx, True)

    # ---- device-resident throughput: warm-up, then exactly K timed steps, `reps` times over ----
    sw.swe_step(ctx, args.warmup, cfl, args.scheme)
    torch.cuda.synchronize()
    dry = sw.swe_dry_counts(ctx)                                  # of the state the timed region starts from
    swdist.barrier()
    l0 = sw.swe_get_stats(ctx)
    clk = ClockSampler(local)
    clk.start()
    rep_ms = []
    for _ in range(max(1, args.reps)):
        torch.cuda.synchronize()
        swdist.barrier()
        m = sw.swe_step_timed(ctx, args.steps, cfl, args.scheme)  # CUDA events on the context's stream
        torch.cuda.synchronize()
        swdist.barrier()
        rep_ms.append(swdist.reduce_max(m))
    l1 = sw.swe_get_stats(ctx)
    ms_max = float(np.median(rep_ms))
    ms = ms_max
    cells_total = swdist.reduce_sum(float(nt))
    value = cells_total * args.steps / (ms_max * 1e-3)
    launches_per_rep = (l1["kernel_launches"] - l0["kernel_launches"]) // max(1, args.reps)

    # ---- the same timed region again with per-kernel CUDA events (roofline of the dominant kernel) ----
    sw.swe_set_profile(ctx, True)
    sw.swe_step(ctx, args.steps, cfl, args.scheme)
    prof = sw.swe_get_profile(ctx)
    sw.swe_set_profile(ctx, False)
    clocks = clk.stop()
    peak, peak_src = hbm_peak()
    roofline = kernel_roofline(prof, args.steps, args.scheme, nt, ms / args.steps, peak, peak_src,
                               args.workload + ("+masks" if args.dry_masks and args.zones == 0 else ""))
    roofline["dry_state"] = {
        "cells_not_wet_frac": dry["cells_not_wet"] / dry["cells"], "cells_empty_frac": dry["cells_empty"] / dry["cells"],
        "edges_between_empty_cells_frac": dry["edges_between_empty_cells"] / max(1, dry["interior_edges"]),
        "what": "counted on the device after the warm-up steps: cells with h <= h_dry get zero gradients and interior "
                "edges between two cells with h == 0 a zero flux record without reading their inputs"}

    # ---- the same mesh with every cell wet: here the algorithmic bytes are what is moved ----
    if args.workload == "c3" and world == 1 and args.zones == 0 and not args.no_all_wet:
        from swe_inputs import flooded
        wet = flooded(cfg, 18.0)
        keep = [torch.empty(nt, dtype=torch.float64, device="cuda") for _ in range(3)]
        sw.swe_get_state(ctx, *keep)
        t_keep = sw.swe_get_time(ctx)[0]
        sw.swe_set_state(ctx, wet["h"], wet["hu"], wet["hv"])
        sw.swe_step(ctx, args.warmup, cfl, args.scheme)
        torch.cuda.synchronize()
        wdry = sw.swe_dry_counts(ctx)
        wms = float(np.median([sw.swe_step_timed(ctx, args.steps, cfl, args.scheme) for _ in range(3)]))
        sw.swe_set_profile(ctx, True)
        sw.swe_step(ctx, args.steps, cfl, args.scheme)
        wprof = sw.swe_get_profile(ctx)
        sw.swe_set_profile(ctx, False)
        wr = kernel_roofline(wprof, args.steps, args.scheme, nt, wms / args.steps, peak, peak_src, "c3w")
        roofline["all_wet"] = {
            "workload": "the same mesh and bed flooded to a flat surface at 18 m (swe_inputs.flooded), %d warm-up steps, "
                        "median of 3 x %d timed steps" % (args.warmup, args.steps),
            "cells_not_wet_frac": wdry["cells_not_wet"] / wdry["cells"],
            "ms_per_step": wms / args.steps, "value": nt * args.steps / (wms * 1e-3),
            "kernel": wr["kernel"], "frac": wr["frac"], "achieved": wr["achieved"],
            "frac_physical": wr.get("frac_physical"), "traffic": wr["traffic"], "traffic_source": wr["traffic_source"],
            "step_frac_of_peak": wr["step_frac_of_peak"], "step_frac_of_8TBps": wr["step_frac_of_8TBps"],
            "step_frac_physical": wr.get("step_frac_physical"),
            "kernels": {k: {"ms_per_launch": v["ms_per_launch"], "frac_of_peak": v.get("frac_of_peak")} for k, v in wr["kernels"].items()}}
        sw.swe_set_state(ctx, *keep)                              # back to the timed state for the e2e leg
        sw.swe_set_time(ctx, t_keep)
        del keep

    # ---- end to end through the C ABI with HOST buffers: every step copies the state host->device
    # (pinned memory), advances one step and reads the state back ----
    e2e_steps = max(1, min(args.e2e_steps, args.steps))
    hbuf = [torch.empty(nt, dtype=torch.float64).pin_memory() for _ in range(3)]
    sw.swe_get_state(ctx, *hbuf)
    for _ in range(2):
        sw.swe_set_state(ctx, *hbuf); sw.swe_step(ctx, 1, cfl, args.scheme, sync=False); sw.swe_get_state(ctx, *hbuf)
    torch.cuda.synchronize()
    swdist.barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sw.swe_set_state(ctx, *hbuf)
        sw.swe_step(ctx, 1, cfl, args.scheme, sync=False)
        sw.swe_get_state(ctx, *hbuf)
    torch.cuda.synchronize()
    e2e_s = swdist.reduce_max(time.perf_counter() - t0)
    e2e = {"value": cells_total * e2e_steps / e2e_s, "unit": "cell-updates/s", "steps": e2e_steps,
           "h2d_bytes_per_step": 3 * 8 * nt, "d2h_bytes_per_step": 3 * 8 * nt,
           "what": "per step: swe_set_state(pinned host) + swe_step(1) + swe_get_state(pinned host)"}
    zstats = sw.swe_zone_stats(ctx) if args.zones > 0 else None
    if zstats:
        zstats["setup_ms"] = sw.swe_zone_setup_ms(ctx)       # row f4: device ghost layers / zone build / whole call
        zstats["setup_detail_ms"] = sw.swe_zone_setup_detail(ctx)
    roofline["fp64_peak_TFLOPs_measured"] = sw.swe_fp64_peak(ctx)      # the other side of the roofline
    sw.swe_mesh_destroy(ctx)

    # ---- the oracle as it stands, timed on this box's host cores (rank 0, N=1 only) ----
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # all cores: the SAME workload (20 steps at 13.1 M cells; fewer if they do not
        # fit 25 s); one thread: the same generator on a 6 km reach, a few steps
        v, cores, ont, secs, osteps = oracle_run(cfg, args.scheme, cfl, 1, 20, budget_s=25.0)
        sname = "c3s" if args.workload in ("c3", "c3w", "c3p") else args.workload
        scfg, sdesc = (cfg, desc) if sname == args.workload else build_workload(sname)
        v1, _, ont1, secs1, osteps1 = oracle_run(scfg, args.scheme, cfl, 1, 50, budget_s=5.0, threads=1)
        cpu_baseline = {"value": v, "unit": "cell-updates/s", "cores": cores, "kind": "oracle",
                        "sample": "%s: %d cells x %d %s steps in %.1f s" % (desc, ont, osteps, args.scheme, secs),
                        "single_thread": {"value": v1, "cores": 1,
                                          "sample": "%s: %d cells x %d steps in %.1f s" % (sdesc, ont1, osteps1, secs1)}}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "cell-updates/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "cells": nt, "edges": info["nedge"], "scheme": args.scheme, "cfl": cfl,
                       "l2": "inputs larger than L2 (state+geometry+flux > 3 GB per stage at 13 M cells)"
                       if nt > 2_000_000 else "working set may fit L2 at this size",
                       "parallelism": "replicas x%d" % world if world > 1 else "single GPU",
                       "zones": args.zones, "ghost_layers": args.layers if args.zones else 0,
                       "renumber": args.renumber,
                       "dry_masks": args.dry_masks and args.zones == 0, "paper_context": PAPER_CONTEXT[args.scheme]},
            "roofline": roofline, "e2e": e2e, "cpu_baseline": cpu_baseline,
            "gpu_launches": int(launches_per_rep), "clocks": clocks,
            "reps": {"n": len(rep_ms), "ms_per_step": [m / args.steps for m in rep_ms],
                     "ms_per_step_min": min(rep_ms) / args.steps, "ms_per_step_max": max(rep_ms) / args.steps,
                     "value_is": "median over the repetitions of the K-step timed region"},
        }
        if zstats:
            line["config"]["zone_stats"] = zstats
        print(json.dumps(line))
    swdist.finalize()


if __name__ == "__main__":
    main()
