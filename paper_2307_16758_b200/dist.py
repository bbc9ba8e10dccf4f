"""Multi-process plumbing for bench.py (one process per GPU, torch.distributed).

The time step on one GPU has no data-path collective; with N > 1 ranks bench.py runs N independent
replicas ("replicas only", DESIGN.md section 'Multi-GPU') and only the timing is reduced: barrier
before and after the timed region, MAX of the per-rank device times, SUM of the units processed.
Backend: nccl when CUDA is available, else gloo (CPU tests, world_size 2).
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
            backend = "nccl" if torch.cuda.is_available() else "gloo"
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            if backend == "nccl":
                torch.cuda.set_device(local)
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
