"""N > 1 host logic on CPU (gloo, world_size 2): photon-id sharding + the histogram all-reduce of
paper_2203_14354_b200.dist reproduce the single-process result bit for bit."""
import os
import socket
import sys
from pathlib import Path
from types import SimpleNamespace

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_total, q):
    sys.path.insert(0, str(ROOT))
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    from oracle import oracle as orc
    from paper_2203_14354_b200 import dist, synth
    r, w, _ = dist.init_from_env(backend="gloo")
    assert (r, w) == (rank, world) and dist.active()
    c = synth.config(1)
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    ph = c.make_photons(n_total)
    base, n_local = dist.shard_ids(n_total, rank, world, weak=False)
    out = o.propagate(ph.slice(base, base + n_local), c.seed, c.max_steps, n_bins=100, dt=1.0, nthreads=2, full=False)
    hist = SimpleNamespace(chan_count=torch.from_numpy(out["chan_count"].astype(np.int64)),
                           time_hist=torch.from_numpy(out["time_hist"].astype(np.int32)),
                           fate_count=torch.from_numpy(out["fate_count"].astype(np.int64)),
                           total_steps=torch.from_numpy(out["total_steps"].astype(np.int64)))
    local_copy = hist.chan_count.clone()
    merged = dist.merge_hists(hist)
    assert torch.equal(hist.chan_count, local_copy)            # local reductions untouched
    tmax = dist.max_over_ranks(10.0 + rank)
    ssum = dist.sum_over_ranks(int(out["total_steps"][0]))
    dist.barrier()
    if rank == 0:
        q.put(dict(chan=merged["chan_count"].numpy(), time=merged["time_hist"].numpy(), fate=merged["fate_count"].numpy(),
                   steps=int(merged["total_steps"][0]), tmax=tmax, ssum=ssum, base=base, n_local=n_local))
    dist.finalize()


def test_shard_ids_cover_the_batch_exactly():
    from paper_2203_14354_b200 import dist
    for n, w in ((10, 3), (7, 8), (1000, 4), (0, 2)):
        spans = [dist.shard_ids(n, r, w, weak=False) for r in range(w)]
        assert spans[0][0] == 0 and sum(s[1] for s in spans) == n
        for a, b in zip(spans, spans[1:]):
            assert a[0] + a[1] == b[0]
        assert max(s[1] for s in spans) - min(s[1] for s in spans) <= 1
    assert [dist.shard_ids(100, r, 4, weak=True) for r in range(4)] == [(0, 100), (100, 100), (200, 100), (300, 100)]
    assert dist.init_from_env() == (0, 1, 0) or os.environ.get("WORLD_SIZE")


def test_two_rank_gloo_merge_equals_single_process():
    import torch.multiprocessing as mp
    from oracle import oracle as orc
    from paper_2203_14354_b200 import synth
    n_total = 6001
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n_total, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = q.get(timeout=300)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    c = synth.config(1)
    ref = orc.Oracle(c.geometry, c.optics, bvh=True).propagate(c.make_photons(n_total), c.seed, c.max_steps, n_bins=100, dt=1.0, full=False)
    assert np.array_equal(res["chan"].astype(np.uint64), ref["chan_count"])
    assert np.array_equal(res["time"].astype(np.uint64), ref["time_hist"])
    assert np.array_equal(res["fate"].astype(np.uint64), ref["fate_count"])
    assert res["steps"] == int(ref["total_steps"][0]) == res["ssum"]
    assert res["tmax"] == 11.0 and res["base"] == 0 and res["n_local"] == 3001
