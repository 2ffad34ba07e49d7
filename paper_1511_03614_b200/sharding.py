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


def split_shifts(n_shifts, world_size):
    """(first, count) per rank: the rule's shifts dealt out in contiguous, near-equal shares (count may be 0)."""
    base, extra = divmod(int(n_shifts), int(world_size))
    out, first = [], 0
    for r in range(world_size):
        cnt = base + (1 if r < extra else 0)
        out.append((first, cnt))
        first += cnt
    return out


def integrate_split_shifts(ctx, prog, npoints, rule, seed, sectors=None, dist=None, device="cpu"):
    """Few, huge sectors: every rank integrates ALL selected sectors, but only its share of the lattice rule's
    random shifts (the shifts are independent estimates of the same integral: no exchange until the end); one
    all_gather of the per-shift sums (KBs), then every rank runs the estimator on the device.  The result is,
    bit for bit, fiesta_integrate's on one GPU: a shift's sums do not depend on the rank that made them.

    ctx: binding.Context; prog: a Program compiled on every rank from the same sectors; rule: lattice."""
    world = dist.get_world_size() if (dist is not None and dist.is_initialized()) else 1
    rank = dist.get_rank() if world > 1 else 0
    R = int(rule.n_shifts)
    shares = split_shifts(R, world)
    first, cnt = shares[rank]
    nsel = prog.nsectors if sectors is None else len(sectors)
    mine = nf = None
    if cnt > 0:
        mine, nf = ctx.partial_sums_shifts(prog, npoints, rule, seed, first, cnt, sectors=sectors)
    if world == 1:
        return ctx.estimate_from_sums(prog, mine, npoints // R, nf, sectors=sectors, allow_nonfinite=True)
    import torch
    # fixed-size buffers padded to the largest share; a rank without a shift (more ranks than shifts) sends zeros
    row = None if mine is None else int(np.prod(mine.shape[2:]))
    rows = [None] * world
    dist.all_gather_object(rows, row)
    row = next(v for v in rows if v is not None)
    cap = max(c for _, c in shares)
    buf = np.zeros(nsel * cap * row + nsel, dtype=np.float64)
    if cnt > 0:
        buf[:nsel * cnt * row] = mine.reshape(-1)
        buf[nsel * cap * row:] = nf.astype(np.float64)         # counts < 2^53
    t = torch.from_numpy(buf).to(device)
    got = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(got, t)
    tail = mine.shape[2:] if mine is not None else None
    tails = [None] * world
    dist.all_gather_object(tails, tail)
    tail = next(v for v in tails if v is not None)
    full = np.zeros((nsel, R) + tuple(tail), dtype=np.float64)
    nf_all = np.zeros(nsel, dtype=np.uint64)
    for r, g in enumerate(got):
        f0, c = shares[r]
        if c == 0:
            continue
        b = g.cpu().numpy()
        full[:, f0:f0 + c] = b[:nsel * c * row].reshape((nsel, c) + tuple(tail))
        nf_all += b[nsel * cap * row:].astype(np.uint64)
    return ctx.estimate_from_sums(prog, full, npoints // R, nf_all, sectors=sectors, allow_nonfinite=True)
