"""Host-side logic of the sharded (multi-GPU) run: SURVEY.md §8(e).

Segments are independent and the random stream is keyed by the GLOBAL segment id (R20), so any
partition of the segment table gives bit-identical photons.  Each rank runs the single-GPU path on
its own contiguous id range; there is no collective on the data path.  The only exchange is the
final sum of the per-telescope tallies and counters (a few hundred bytes), done once per job with
torch.distributed (NCCL on GPUs, gloo in the CPU tests).  Photon records stay on the producing GPU.
"""
from __future__ import annotations

import numpy as np


def shard_range(n_total: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [lo, hi) of rank `rank` when n_total segments are split over `world` ranks (strong scaling)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return n_total * rank // world, n_total * (rank + 1) // world


def shard_first_id(rank: int, n_per_rank: int) -> int:
    """First global segment id of rank `rank` when every rank owns n_per_rank segments (weak scaling)."""
    return int(rank) * int(n_per_rank)


def pack_results(tallies: np.ndarray, counters: dict):
    """Flatten (tallies, counters) into two vectors for a sum all-reduce: an int64 vector (per-telescope hits, then
    the eight counters in the order of paper_2309_15861_b200.COUNTER_NAMES, the keys Context.read_tallies() returns)
    and a float64 vector (sum_w, sum_wt)."""
    from . import COUNTER_NAMES
    ints = np.concatenate([tallies["hits"].astype(np.int64),
                           np.array([counters[k] for k in COUNTER_NAMES], dtype=np.int64)])
    flts = np.concatenate([tallies["sum_w"], tallies["sum_wt"]]).astype(np.float64)
    return ints, flts


def unpack_results(ints: np.ndarray, flts: np.ndarray, n_tel: int):
    from . import COUNTER_NAMES, TALLY_DTYPE
    t = np.zeros(n_tel, dtype=TALLY_DTYPE)
    t["hits"] = ints[:n_tel].astype(np.uint64)
    t["sum_w"], t["sum_wt"] = flts[:n_tel], flts[n_tel:2 * n_tel]
    return t, dict(zip(COUNTER_NAMES, (int(v) for v in ints[n_tel:n_tel + 8])))


def all_reduce_results(tallies: np.ndarray, counters: dict, device=None):
    """Sum tallies and counters over all ranks of the default process group (no-op without one)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return tallies, counters
    ints, flts = pack_results(tallies, counters)
    ti = torch.from_numpy(ints).to(device) if device is not None else torch.from_numpy(ints)
    tf = torch.from_numpy(flts).to(device) if device is not None else torch.from_numpy(flts)
    dist.all_reduce(ti, op=dist.ReduceOp.SUM)
    dist.all_reduce(tf, op=dist.ReduceOp.SUM)
    return unpack_results(ti.cpu().numpy(), tf.cpu().numpy(), len(tallies))
