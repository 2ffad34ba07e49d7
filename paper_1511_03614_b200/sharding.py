"""Multi-GPU: shard sectors across ranks (one process per GPU), no data-path collective.

Sectors (and their epsilon orders) are independent integrals -- the paper parallelises exactly
so, over integrands (PAPER.md:130-132 thread pool, :142 MPI master/slaves) and over the GPUs of
a node (PAPER.md:184, :493 `gpu_per_node`).  Each rank runs the single-GPU path on its sectors;
the only exchange is the gather of the per-(sector, order) result records at the end (a few KB),
done with `torch.distributed` (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import numpy as np


def partition_sectors(costs, world_size):
    """Longest-processing-time assignment: sector indices per rank, each list ascending.

    costs[i] ~ work of sector i (e.g. IR ops x points).  Deterministic (ties by index)."""
    costs = np.asarray(costs, dtype=np.float64)
    order = sorted(range(len(costs)), key=lambda i: (-costs[i], i))
    load = [0.0] * world_size
    parts = [[] for _ in range(world_size)]
    for i in order:
        r = min(range(world_size), key=lambda q: (load[q], q))
        parts[r].append(i)
        load[r] += float(costs[i])
    return [sorted(p) for p in parts]


def gather_results(local, my_sectors, nsectors, dist=None, device="cpu"):
    """All ranks get the full [nsectors][K] record array.

    local: numpy record array [len(my_sectors)][K] (binding.RESULT_DTYPE) of this rank's sectors.
    One all_gather of fixed-size byte tensors (padded to the largest shard)."""
    local = np.ascontiguousarray(local)
    K = local.shape[1]
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        out = np.zeros((nsectors, K), dtype=local.dtype)
        out[np.asarray(my_sectors, dtype=np.int64)] = local
        return out
    import torch
    world = dist.get_world_size()
    rec = local.dtype.itemsize * K
    cap = (nsectors + world - 1) // world + nsectors  # upper bound on any shard (LPT can be uneven)
    cap = min(cap, nsectors)
    buf = np.zeros(8 + cap * (8 + rec), dtype=np.uint8)
    buf[:8] = np.frombuffer(np.int64(len(my_sectors)).tobytes(), dtype=np.uint8)
    idx = np.asarray(my_sectors, dtype=np.int64)
    buf[8:8 + 8 * len(idx)] = np.frombuffer(idx.tobytes(), dtype=np.uint8)
    o = 8 + 8 * cap
    buf[o:o + rec * len(idx)] = np.frombuffer(local.tobytes(), dtype=np.uint8)
    mine = torch.from_numpy(buf).to(device)
    got = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(got, mine)
    out = np.zeros((nsectors, K), dtype=local.dtype)
    for g in got:
        b = g.cpu().numpy()
        n = int(np.frombuffer(b[:8].tobytes(), dtype=np.int64)[0])
        ids = np.frombuffer(b[8:8 + 8 * n].tobytes(), dtype=np.int64)
        recs = np.frombuffer(b[o:o + rec * n].tobytes(), dtype=local.dtype).reshape(n, K)
        out[ids] = recs
    return out


def max_over_ranks(value, dist=None, device="cpu"):
    """max of a Python float over ranks (timing rule: device time, max over ranks)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
