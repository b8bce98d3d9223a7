"""Multi-GPU plumbing: bands (and k-points) are independent units (PAPER.md :436, :456, :500), so the
path shards with NO data-path collective.  One process per GPU; torch.distributed is used only for
the barrier around the timed region and the max-over-ranks of the measured time."""
import os


def _dist():
    import torch.distributed as dist
    return dist


def init(backend):
    """Join the process group described by RANK / WORLD_SIZE / MASTER_ADDR / MASTER_PORT."""
    dist = _dist()
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend)


def active():
    dist = _dist()
    return dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1


def barrier():
    if active():
        _dist().barrier()


def max_over_ranks(x):
    """max of a python float over all ranks (the slowest rank defines the step time)."""
    if not active():
        return float(x)
    import torch
    dist = _dist()
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def shutdown():
    dist = _dist()
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()


def band_shard(nband, rank, world):
    """Contiguous block [b0, b1) of rank `rank` when `nband` bands are split as evenly as possible."""
    q, r = divmod(int(nband), int(world))
    b0 = rank * q + min(rank, r)
    return b0, b0 + q + (1 if rank < r else 0)
