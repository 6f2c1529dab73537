"""world_size-2 gloo test of the sharded run's host logic: contiguous id ranges, global
segment ids, and the final all-reduce of tallies + counters.  No GPU here, so each rank's per-shard result
comes from the oracle (tests may call it); what is under test is the partition + reduction code of
paper_2309_15861_b200.sharding, whose result must equal the unsharded run."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

import workloads as wl


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    import oracle
    import paper_2309_15861_b200 as c8
    from paper_2309_15861_b200.sharding import all_reduce_results, shard_range
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = wl.make_config("c2", n_segments=3001)
    lo, hi = shard_range(len(cfg["segments"]), rank, world)
    r = oracle.run(cfg["atmosphere"], cfg["telescopes"], cfg["segments"][lo:hi], cfg["params"], first_id=lo)
    # keyed exactly like Context.read_tallies() of the product (the oracle only supplies the per-shard numbers)
    counters = dict(zip(c8.COUNTER_NAMES, (int(v) for v in r["counters"])))
    counters["culled"] = 5 + rank                      # a value the reduction must carry
    t, c = all_reduce_results(r["tallies"], counters)
    if rank == 0:
        q.put((t, c))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_partition_matches_single_run():
    import oracle
    cfg = wl.make_config("c2", n_segments=3001)
    full = oracle.run(cfg["atmosphere"], cfg["telescopes"], cfg["segments"], cfg["params"])
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    t, c = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert np.array_equal(t["hits"], full["tallies"]["hits"])
    assert np.allclose(t["sum_w"], full["tallies"]["sum_w"], rtol=1e-12)
    assert np.allclose(t["sum_wt"], full["tallies"]["sum_wt"], rtol=1e-9)
    assert c["generated"] == int(full["counters"][1]) and c["segments"] == 3001
    assert c["culled"] == 5 + 6 and set(c) == set(__import__("paper_2309_15861_b200").COUNTER_NAMES)


def test_pack_unpack_round_trip_with_the_product_counter_names():
    """pack_results / unpack_results take and return the dict Context.read_tallies() returns ('unused')."""
    import paper_2309_15861_b200 as c8
    from paper_2309_15861_b200.sharding import pack_results, unpack_results
    t = np.zeros(3, dtype=c8.TALLY_DTYPE)
    t["hits"], t["sum_w"], t["sum_wt"] = [1, 2, 3], [0.5, 1.5, 2.5], [-1.0, 0.0, 7.0]
    counters = {name: 10 + i for i, name in enumerate(c8.COUNTER_NAMES)}
    ints, flts = pack_results(t, counters)
    t2, c2 = unpack_results(ints, flts, 3)
    assert c2 == counters and t2.tobytes() == t.tobytes()


def test_shard_ranges_cover_exactly():
    from paper_2309_15861_b200.sharding import shard_first_id, shard_range
    for n in (0, 1, 7, 1000, 10**7 + 3):
        for w in (1, 2, 3, 8):
            r = [shard_range(n, k, w) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(r[:-1], r[1:]))
    assert shard_first_id(3, 10**6) == 3 * 10**6
