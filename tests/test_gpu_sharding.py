"""Two ranks through the CUDA path: each rank runs its contiguous shard of the segment table on the
GPU with the global segment ids of its range, the ranks sum tallies and counters with all_reduce_results (world 2,
gloo; both ranks use cuda:0 -- they exchange nothing until their kernels are done), and the sum must be the unsharded
GPU run: hits and counters bit for bit, the fp64 sums to rounding."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

import workloads as wl

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _run_shard(cfg, lo, hi):
    import torch
    import paper_2309_15861_b200 as c8
    seg = cfg["segments"][lo:hi]
    ctx = c8.Context(cfg["atmosphere"])
    ctx.add_telescopes(cfg["telescopes"])
    d_seg = torch.from_numpy(seg.view(np.uint8).reshape(len(seg), 48).copy()).to("cuda:0")
    ctx.propagate_segments(d_seg, dict(cfg["params"], mode=c8.MODE_TALLY), n=len(seg), first_segment_id=lo)
    tallies, counters, _ = ctx.read_tallies()
    ctx.close()
    return tallies, counters


def _worker(rank, world, port, name, n, q):
    import torch.distributed as dist
    from paper_2309_15861_b200.sharding import all_reduce_results, shard_range
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = wl.make_config(name, n_segments=n)
    lo, hi = shard_range(len(cfg["segments"]), rank, world)
    t, c = all_reduce_results(*_run_shard(cfg, lo, hi))
    if rank == 0:
        q.put((t, c))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("name,n", [("c2", 100_003), ("c4", 50_001)])
def test_two_shards_through_the_cuda_path_sum_to_the_unsharded_run(name, n):
    import torch
    assert torch.cuda.is_available()
    from paper_2309_15861_b200.build import build
    build()
    cfg = wl.make_config(name, n_segments=n)
    full_t, full_c = _run_shard(cfg, 0, len(cfg["segments"]))
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, name, n, q)) for r in range(2)]
    for p in procs:
        p.start()
    t, c = q.get(timeout=300)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert np.array_equal(t["hits"], full_t["hits"]) and int(t["hits"].sum()) > 1000
    assert c == full_c
    assert np.allclose(t["sum_w"], full_t["sum_w"], rtol=1e-12) and np.allclose(t["sum_wt"], full_t["sum_wt"], rtol=1e-9)
