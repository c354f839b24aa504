"""Host-side logic of the sharded multi-GPU mode (paper_2110_11658_b200.shard): the cost-balanced
cuts, and the unequal-size all-gather on the gloo backend with world_size 2 and 3 (CPU)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from conftest import ROOT

sys.path.insert(0, str(ROOT))
from paper_2110_11658_b200 import shard  # noqa: E402


def test_balanced_cuts_equal_cost_is_equal_groups():
    gb = np.arange(0, 640, 64)
    cuts = shard.balanced_cuts(gb, 640, np.ones(10), 5)
    assert cuts.tolist() == [0, 128, 256, 384, 512, 640]


def test_balanced_cuts_no_cost_falls_back_to_particles():
    assert shard.balanced_cuts(np.arange(0, 100, 10), 100, np.zeros(10), 4).tolist() == [0, 25, 50, 75, 100]
    assert shard.balanced_cuts(np.zeros(0, np.int64), 7, np.zeros(0), 2).tolist() == [0, 3, 7]


@pytest.mark.parametrize("seed", range(20))
def test_balanced_cuts_bound_against_brute_force(seed):
    """Each rank's cost is below total / nranks + the largest single group (the greedy prefix rule), the
    cuts are ascending group starts, and every group is owned exactly once."""
    rng = np.random.default_rng(seed)
    ng = int(rng.integers(1, 200)); nr = int(rng.integers(1, 9))
    sizes = rng.integers(1, 65, ng)
    gb = np.concatenate(([0], np.cumsum(sizes)[:-1])); n = int(sizes.sum())
    cost = rng.random(ng) ** 3 * 1e6
    if seed % 5 == 0:
        cost[rng.integers(0, ng)] = cost.sum() * 3           # one dominant group
    cuts = shard.balanced_cuts(gb, n, cost, nr)
    assert cuts[0] == 0 and cuts[-1] == n and np.all(np.diff(cuts) >= 0)
    starts = set(gb.tolist()) | {n}
    assert all(int(c) in starts for c in cuts)
    owner = np.searchsorted(cuts[1:], gb, side="right")      # group g belongs to the rank whose range holds its start
    per_rank = np.array([cost[owner == r].sum() for r in range(nr)])
    assert np.isclose(per_rank.sum(), cost.sum())
    assert per_rank.max() <= cost.sum() / nr + cost.max() * (1 + 1e-12)


def test_group_cost_weights():
    c = shard.group_cost([64, 10], [100, 0], [0, 1000])
    assert c.tolist() == [64 * 15.0 * 100, 10 * 37.0 * 1000]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, sizes, q):
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2110_11658_b200 import shard as sh
    local = torch.arange(sizes[rank] * 4, dtype=torch.float32).reshape(sizes[rank], 4) + 1000.0 * rank
    got = sh.all_gather_chunks(local, sizes)
    ok = len(got) == world
    for r in range(world):
        want = torch.arange(sizes[r] * 4, dtype=torch.float32).reshape(sizes[r], 4) + 1000.0 * r
        ok = ok and got[r].shape == want.shape and bool(torch.equal(got[r], want))
    dist.barrier()
    q.put((rank, ok))
    dist.destroy_process_group()


@pytest.mark.parametrize("sizes", [[5, 9], [7, 7], [0, 3], [4, 0, 11]])
def test_all_gather_chunks_gloo(sizes):
    world = len(sizes)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, sizes, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(r, True) for r in range(world)]


def test_merge_neighbour_rows_is_the_unsharded_csr():
    """The CSR exchange of the sharded mode, host logic: random rows split among 3 owners."""
    rng = np.random.default_rng(3)
    n = 500
    lens = rng.integers(0, 9, n); lens[rng.random(n) < 0.4] = 0
    off = np.concatenate(([0], np.cumsum(lens)))
    idx = rng.integers(0, n, off[-1]).astype(np.int32)
    owner = np.sort(rng.integers(0, 3, n))                        # contiguous ownership is not required: shuffle it
    rng.shuffle(owner)
    counts_all, chunks = [], []
    for r in range(3):
        c = np.where(owner == r, lens, 0)
        counts_all.append(torch.from_numpy(c.astype(np.int64)))
        chunks.append(torch.from_numpy(np.concatenate([idx[off[i]:off[i + 1]] for i in range(n) if owner[i] == r] + [np.zeros(0, np.int32)]).astype(np.int32)))
    goff, gidx = shard.merge_neighbour_rows(counts_all, chunks, n)
    assert np.array_equal(goff.numpy(), off) and np.array_equal(gidx.numpy(), idx)
