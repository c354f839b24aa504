"""Multi-GPU regular force: target groups split among the ranks of one node.

PAPER.md:277-291 names multi-GPU as future work; this is the natural sharding of the path.  Every rank
holds all bodies and builds the identical tree (`Context.set_shard(rank, nranks)` then `build_tree`);
`regular_force` evaluates only the rank's own Morton range of groups; the one exchange step is an
all-gather of 16 B per particle, done here with `torch.distributed` (NCCL on the GPUs, gloo in the CPU
tests).  Neighbour lists stay with the rank that owns the particle: the irregular force of a particle is
computed where its list lives.

Everything in this module is host logic and plumbing; the arithmetic of the path runs in libp3t.so.
"""
from __future__ import annotations

import numpy as np

# algorithmic lane-instructions per interaction: the cost model of the balancer
COST_PP, COST_PC = 15.0, 37.0


def group_cost(count, npp, npc):
    """Work of each group: targets x (weighted list lengths).  Arrays over the groups."""
    return np.asarray(count, np.float64) * (COST_PP * np.asarray(npp, np.float64) + COST_PC * np.asarray(npc, np.float64))


def balanced_cuts(group_begin, n: int, cost, nranks: int):
    """Nominal cuts (sorted positions, int64[nranks + 1]) that give every rank the same summed cost.

    group_begin[g] = first sorted particle of group g (ascending), cost[g] >= 0.  Cut r is the start of the
    first group at which the running cost reaches r / nranks of the total; with no cost information
    (all zero) the cuts fall back to equal particle counts.  The positions refer to the tree they were
    measured on; the library re-aligns them to the group boundaries of the next tree."""
    group_begin = np.asarray(group_begin, np.int64)
    cost = np.asarray(cost, np.float64)
    assert group_begin.shape == cost.shape and nranks >= 1
    total = float(cost.sum())
    cuts = np.empty(nranks + 1, np.int64)
    cuts[0], cuts[nranks] = 0, n
    if total <= 0.0 or len(cost) == 0:
        for r in range(1, nranks):
            cuts[r] = r * n // nranks
        return cuts
    before = np.concatenate(([0.0], np.cumsum(cost)[:-1]))        # cost of the groups in front of g
    for r in range(1, nranks):
        g = int(np.searchsorted(before, total * r / nranks, side="left"))
        cuts[r] = group_begin[g] if g < len(group_begin) else n
    return np.maximum.accumulate(cuts)


def chunk_sizes(cuts):
    cuts = np.asarray(cuts, np.int64)
    return [int(cuts[r + 1] - cuts[r]) for r in range(len(cuts) - 1)]


def all_gather_chunks(local, sizes, group=None):
    """All-gather of unequal row counts: every rank passes its [sizes[rank], C] tensor and gets the list of
    all ranks' tensors.  Rows are padded to the largest chunk so that one equal-size collective does it."""
    import torch
    import torch.distributed as dist
    nr = dist.get_world_size(group)
    rank = dist.get_rank(group)
    assert len(sizes) == nr and local.shape[0] == sizes[rank]
    m = max(max(sizes), 1)
    send = local
    if local.shape[0] != m:
        send = torch.zeros((m,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
        send[: local.shape[0]] = local
    recv = [torch.empty_like(send) for _ in range(nr)]
    dist.all_gather(recv, send.contiguous(), group=group)
    return [recv[r][: sizes[r]] for r in range(nr)]


def exchange(ctx, acc_pot, cuts, group=None):
    """Completes acc_pot (CUDA float32 [n, 4], original order) on every rank: packs the owned rows, all-gathers
    the chunks and scatters those of the other ranks.  cuts = ctx.shard_cuts()[0] of the current tree."""
    import torch
    rank, nr = ctx.shard
    sizes = chunk_sizes(cuts)
    mine = torch.empty((max(sizes[rank], 1), 4), dtype=torch.float32, device=acc_pot.device)
    ctx.shard_pack(acc_pot, mine)
    chunks = all_gather_chunks(mine[: sizes[rank]], sizes, group)
    for r in range(nr):
        if r != rank and sizes[r] > 0:
            ctx.shard_unpack(r, chunks[r].contiguous(), acc_pot)
    return acc_pot


def gather_group_costs(ctx, group=None):
    """Per-group cost of the last regular_force over ALL groups: every rank knows the lengths of its own groups
    only (the others are zero), so the sum over ranks is the full vector.  Returns (group_begin, cost)."""
    import torch
    import torch.distributed as dist
    g = ctx.groups()
    npp, npc = ctx.list_lengths()
    cost = torch.from_numpy(group_cost(g["end"] - g["begin"], npp, npc))
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        if dist.get_backend(group) == "nccl":
            cost = cost.to(ctx.device)
        dist.all_reduce(cost, group=group)
        cost = cost.cpu()
    return g["begin"].astype(np.int64), cost.numpy()


def merge_neighbour_rows(counts_all, chunks, n: int):
    """Host-side logic of the neighbour exchange ("one all-gather of acc_pot and of the CSR rows"):
    counts_all[r] = per-particle row lengths of rank r (int64 [n], zero for the particles it does not own: every
    particle is owned by exactly one rank), chunks[r] = rank r's indices, rows back to back in original particle order.
    Returns the CSR of all particles (offsets int64 [n + 1], indices int32), identical to that of an unsharded context.
    Pure index arithmetic on whatever device the tensors live on (moves entries, computes nothing of the method)."""
    import torch
    dev = chunks[0].device
    total = torch.zeros(n, dtype=torch.int64, device=dev)
    for c in counts_all:
        total += c
    off = torch.zeros(n + 1, dtype=torch.int64, device=dev)
    torch.cumsum(total, 0, out=off[1:])
    out = torch.empty(int(off[-1].item()), dtype=torch.int32, device=dev)
    for c, idx in zip(counts_all, chunks):
        m = int(idx.shape[0])
        if m == 0:
            continue
        own_off = torch.cumsum(c, 0) - c                                   # this rank's own offsets
        rows = torch.repeat_interleave(torch.arange(n, device=dev), c)     # particle of every entry of the chunk
        pos = torch.arange(m, device=dev) - own_off[rows]
        out[off[rows] + pos] = idx
    return off, out


def exchange_neighbours(ctx, group=None):
    """Completes the neighbour CSR on every rank: all-gathers the ranks' row lengths and index chunks (padded to the
    largest) and merges them (merge_neighbour_rows).  Returns (offsets, indices) as tensors on the context's device."""
    import torch
    import torch.distributed as dist
    off, idx = ctx.neighbours()
    n = off.shape[0] - 1
    counts = (off[1:] - off[:-1]).contiguous()
    nr = dist.get_world_size(group)
    counts_all = [torch.empty_like(counts) for _ in range(nr)]
    dist.all_gather(counts_all, counts, group=group)
    sizes = [int(c.sum().item()) for c in counts_all]
    chunks = all_gather_chunks(idx.reshape(-1, 1), sizes, group)
    return merge_neighbour_rows(counts_all, [c.reshape(-1) for c in chunks], n)
