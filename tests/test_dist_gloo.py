"""The N > 1 plumbing of bench.py on CPU: world_size-2 gloo, barrier, max-over-ranks time, sum of
units, block sharding of independent units."""
import os
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2307_16758_b200 import dist as d
    r, w, l = d.init_from_env()
    d.barrier()
    mx = d.reduce_max(10.0 + r)
    sm = d.reduce_sum(100.0 * (r + 1))
    lo, hi = d.shard_units(33, r, w)
    d.barrier()
    d.finalize()
    q.put((r, w, mx, sm, lo, hi))


def test_gloo_world_size_2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 400
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1] and all(r[1] == 2 for r in res)
    assert all(r[2] == 11.0 and r[3] == 300.0 for r in res)
    assert (res[0][4], res[0][5], res[1][4], res[1][5]) == (0, 17, 17, 33)


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK"):
        os.environ.pop(k, None)
    from paper_2307_16758_b200 import dist as d
    assert d.init_from_env() == (0, 1, 0)
    assert d.reduce_max(3.5) == 3.5 and d.reduce_sum(2.0) == 2.0
    assert d.shard_units(5, 0, 1) == (0, 5)
    d.barrier()
