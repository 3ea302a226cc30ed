"""Multi-GPU plumbing: photons are independent and the geometry is read-only, so the path
shards by contiguous photon-id ranges with the geometry, tables and BVH replicated on every GPU.  The only
exchange is the sum of the integer histograms (tens of kB): one all-reduce through torch.distributed
(NCCL on GPUs, gloo in the CPU tests).  Nothing here touches the per-photon data path.
"""
from __future__ import annotations

import os


def _dist():
    import torch.distributed as d
    return d


def init_from_env(backend: str | None = None):
    """Returns (rank, world, local_rank); initialises torch.distributed when WORLD_SIZE > 1."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and not _dist().is_initialized():
        import torch
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        if backend == "nccl":
            torch.cuda.set_device(local)
        _dist().init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world, local


def active() -> bool:
    d = _dist()
    return d.is_available() and d.is_initialized() and d.get_world_size() > 1


def shard_ids(n: int, rank: int, world: int, weak: bool = True):
    """Photon-id range of a rank.  weak: every rank propagates n photons, ids [rank*n, (rank+1)*n).
    strong: n photons in total are split into contiguous ranges that differ by at most one.
    Returns (photon_id_base, n_local)."""
    if weak:
        return rank * n, n
    q, r = divmod(n, world)
    n_local = q + (1 if rank < r else 0)
    base = rank * q + min(rank, r)
    return base, n_local


def merge_hists(hist):
    """Sum of the reductions over all ranks.  `hist` has tensors chan_count, time_hist, fate_count, total_steps;
    returns a dict of NEW tensors (the local ones are left untouched so that they keep accumulating locally)."""
    out = {k: getattr(hist, k).clone() for k in ("chan_count", "time_hist", "fate_count", "total_steps")}
    if active():
        d = _dist()
        works = [d.all_reduce(t, op=d.ReduceOp.SUM, async_op=True) for t in out.values()]
        for w in works:
            w.wait()
    return out


def barrier():
    if active():
        _dist().barrier()


def max_over_ranks(x: float) -> float:
    if not active():
        return float(x)
    import torch
    d = _dist()
    dev = "cuda" if d.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    d.all_reduce(t, op=d.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: int) -> int:
    if not active():
        return int(x)
    import torch
    d = _dist()
    dev = "cuda" if d.get_backend() == "nccl" else "cpu"
    t = torch.tensor([int(x)], dtype=torch.int64, device=dev)
    d.all_reduce(t, op=d.ReduceOp.SUM)
    return int(t.item())


def finalize():
    if active():
        _dist().destroy_process_group()
