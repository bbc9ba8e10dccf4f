"""Host half of the multi-GPU driver (scope row f3), on CPU: every rank derives its
own halo lists and its peers' from the same mesh, independently -- they must agree.

 * the zones a rank holds are the zones the single-rank builder makes (same cells, same order);
 * what rank a sends to rank b is, cell for cell and in order, what rank b expects from rank a,
   and the push destination is the ghost slot of that very cell on b;
 * world_size-2 gloo: the all-to-all of dist.TorchComm with the library's split sizes delivers
   every ghost the cell it copies (the payload is the cell's user id).
"""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

import paper_2307_16758_b200 as sw
from paper_2307_16758_b200 import dist as swdist
from swe_inputs import config1, config3

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _river():
    return config3(length=3200.0, half_width=600.0, w2=30.0, n4=4, n8=3)


def _build(cfg, nz, nl, world, rank):
    h = sw.swe_host_mesh_build(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], cfg["bedge"], cfg["btag"])
    sw.swe_host_zones_build_dist(h, nz, nl, None, world, rank, swdist.zone_blocks(nz, world))
    names = ("zone_rank", "rsend_idx", "rsend_dst", "rsend_peer", "rrecv_idx", "rsend_off", "rrecv_off",
             "z:cell_user", "z:c2c", "z:c2e", "send_cells", "zone_offset", "zone_ncells", "zone_nowned", "send_idx", "recv_idx")
    out = {n: sw.swe_host_get(h, n) for n in names}
    sw.swe_host_mesh_free(h)
    return out


@pytest.mark.parametrize("world,nz,nl", [(2, 2, 2), (2, 8, 2), (4, 4, 1), (3, 8, 3), (4, 4, 2)])
def test_ranks_agree_on_the_halo_lists(world, nz, nl):
    cfg = _river()
    R = [_build(cfg, nz, nl, world, r) for r in range(world)]
    one = _build(cfg, nz, nl, 1, 0)
    blocks = swdist.zone_blocks(nz, world)
    for r in range(world):
        zr = R[r]["zone_rank"]
        assert all(zr[z] == q for q in range(world) for z in range(blocks[q], blocks[q + 1]))
        # this rank's concatenated mesh = the single-rank one restricted to its zones, in order
        lo = one["zone_offset"][blocks[r]] if blocks[r] < nz else 0
        n = int(R[r]["zone_ncells"][blocks[r]:blocks[r + 1]].sum())
        assert R[r]["z:cell_user"].size == n
        assert np.array_equal(R[r]["z:cell_user"], one["z:cell_user"][lo:lo + n])
        for z in range(nz):
            assert (R[r]["zone_offset"][z] >= 0) == (zr[z] == r)
    total_ghosts_remote = 0
    for a in range(world):
        for b in range(world):
            sa = slice(R[a]["rsend_off"][b], R[a]["rsend_off"][b + 1])
            rb = slice(R[b]["rrecv_off"][a], R[b]["rrecv_off"][a + 1])
            sent = R[a]["z:cell_user"][R[a]["rsend_idx"][sa]]        # user ids a packs for b
            want = R[b]["z:cell_user"][R[b]["rrecv_idx"][rb]]        # user ids of b's ghosts fed by a
            assert np.array_equal(sent, want)
            assert np.array_equal(R[a]["rsend_dst"][sa], R[b]["rrecv_idx"][rb])
            assert np.all(R[a]["rsend_peer"][sa] == b)
            if a == b:
                assert sent.size == 0
            total_ghosts_remote += want.size
        # the cells a rank packs are cells it owns (layer 0), the slots it fills are ghosts
        lay = R[a]["z:c2c"].reshape(-1, 4)[:, 3]
        assert np.all(lay[R[a]["rsend_idx"]] == 0) and np.all(lay[R[a]["rrecv_idx"]] > 0)
        assert np.all(lay[R[a]["send_idx"]] == 0) and np.all(lay[R[a]["recv_idx"]] > 0)
        # the overlap schedule's "send cells": every cell on a send list once, marked -1 in c2e.w
        sc = R[a]["send_cells"]
        assert np.array_equal(sc, np.unique(np.concatenate([R[a]["rsend_idx"], R[a]["send_idx"]])))
        mark = R[a]["z:c2e"].reshape(-1, 4)[:, 3]
        assert np.array_equal(np.flatnonzero(mark == -1), sc)
        assert np.array_equal(mark > 0, lay > 0) and np.all(mark[(lay == 0)] <= 0)
        # every ghost slot is fed exactly once: by a resident zone or by a peer
        fed = np.concatenate([R[a]["recv_idx"], R[a]["rrecv_idx"]])
        assert np.array_equal(np.sort(fed), np.flatnonzero(lay > 0))
    # remote + resident links together = all links of the single-rank decomposition
    assert total_ghosts_remote + sum(R[r]["recv_idx"].size for r in range(world)) == one["recv_idx"].size


def test_dist_zone_argument_errors():
    cfg = config1(n=12)
    h = sw.swe_host_mesh_build(cfg["x"], cfg["y"], cfg["zb"], cfg["tri"], cfg["bedge"], cfg["btag"])
    try:
        for args in [(4, 2, None, 2, 2, [0, 2, 4]), (4, 2, None, 2, 0, [0, 2, 3]), (4, 2, None, 2, 0, [1, 2, 4]),
                     (4, 2, None, 2, 0, [0, 3, 2]), (4, 2, None, 0, 0, [0]), (4, 2, None, 2, 0, None)]:
            with pytest.raises(sw.SweError):
                sw.swe_host_zones_build_dist(h, *args)
        sw.swe_host_zones_build_dist(h, 4, 2, None, 2, 1, [0, 4, 4])     # a rank may hold no zone
        assert sw.swe_host_get(h, "z:cell_user").size == 0
        assert sw.swe_host_get(h, "rsend_idx").size == 0 and sw.swe_host_get(h, "rrecv_idx").size == 0
    finally:
        sw.swe_host_mesh_free(h)


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), SWE_DIST_GLOO="1")
    import torch
    from paper_2307_16758_b200 import dist as d
    d.init_from_env()
    comm = d.TorchComm()
    nz, nl = 4, 2
    Z = _build(_river(), nz, nl, world, rank)
    send_cells = np.diff(Z["rsend_off"])
    recv_cells = np.diff(Z["rrecv_off"])
    # "pack": 3 values per cell, the payload is the user id of the cell (and two functions of it)
    ids = Z["z:cell_user"][Z["rsend_idx"]].astype(np.float64)
    sendbuf = torch.from_numpy(np.stack([ids, 2 * ids, -ids], axis=1).reshape(-1).copy())
    recvbuf = torch.full((3 * int(recv_cells.sum()),), -7.0, dtype=torch.float64)
    comm.all_to_all(recvbuf, sendbuf, [3 * int(v) for v in recv_cells], [3 * int(v) for v in send_cells])
    got = recvbuf.numpy().reshape(-1, 3)
    want = Z["z:cell_user"][Z["rrecv_idx"]].astype(np.float64)
    ok = bool(np.array_equal(got[:, 0], want) and np.array_equal(got[:, 1], 2 * want) and np.array_equal(got[:, 2], -want))
    t = torch.tensor([5.0 + rank], dtype=torch.float64)
    comm.allreduce_min(t)
    hs = comm.all_gather_bytes(np.full(128, rank, np.uint8))
    ok = ok and float(t) == 5.0 and all(int(hs[p][0]) == p and hs[p].size == 128 for p in range(world))
    comm.host_barrier()
    d.finalize()
    q.put((rank, ok, int(recv_cells.sum())))


def test_gloo_world_size_2_halo_all_to_all():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29900 + os.getpid() % 90
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=180) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1]
    assert all(r[1] for r in res) and all(r[2] > 0 for r in res)
