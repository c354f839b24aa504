"""Sharded multi-GPU mode (p3t_set_shard, p3t_shard_pack / p3t_shard_unpack) on ONE
GPU: the shards of every rank are run one after the other in contexts of their own and merged the way the
ranks of a node would merge them (pack -> [all-gather] -> unpack).  The merged result must equal that of an
unsharded context BIT FOR BIT -- forces, potentials, neighbour rows -- because the tree is the same and every
group is evaluated by exactly one rank with the same kernels.  (One exception: below about 2e5 particles per
rank k_force<SPLIT> shares a work item among 2, 4 or 8 warps, chosen from the rank's particle count; where the
whole and the sharded run choose differently the fp32 partial sums are added in another order and the forces
agree to 2e-6 only -- neighbour rows and interaction counts are still identical.)  The oracle parity of the unsharded path is in
test_gpu_parity.py; a spot check against the oracle's direct sum is repeated here on the merged result."""
import numpy as np
import pytest

import oracle
import workloads
from paper_2110_11658_b200 import shard

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def p3t():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2110_11658_b200 as m
    m.lib()
    return m


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def _rows(off, idx):
    return [idx[off[i]:off[i + 1]] for i in range(len(off) - 1)]


def _run_sharded(p3t, w, nranks, r_in, nominal=None, order=2, key_bits=63):
    import torch
    pm = _cuda(w.pos_mass)
    merged = torch.full((w.n, 4), float("nan"), dtype=torch.float32, device="cuda")
    rows = [None] * w.n
    owner = np.full(w.n, -1)
    tot = dict(n_pp=0, n_pc=0)
    all_cuts = None
    costs = None
    for r in range(nranks):
        with p3t.Context(0) as ctx:
            ctx.set_multipole_order(order)
            ctx.set_shard(r, nranks, nominal)
            ctx.build_tree(pm, key_bits)
            cuts, gcuts = ctx.shard_cuts()
            if all_cuts is None:
                all_cuts = cuts
            assert np.array_equal(cuts, all_cuts)                       # every rank computes the same cuts
            g = ctx.groups()
            assert cuts[0] == 0 and cuts[-1] == w.n and np.all(np.diff(cuts) >= 0)
            assert np.array_equal(np.append(g["begin"], w.n)[gcuts], cuts)     # group aligned
            out = torch.full((w.n, 4), float("nan"), dtype=torch.float32, device="cuda")
            ctx.regular_force(w.r_out, r_in, w.theta, 0, out=out)
            size = int(cuts[r + 1] - cuts[r])
            chunk = torch.empty((max(size, 1), 4), dtype=torch.float32, device="cuda")
            ctx.shard_pack(out, chunk)
            ctx.shard_unpack(r, chunk, merged)                          # what the receiving ranks do with it
            off, idx = ctx.neighbours()
            off = off.cpu().numpy(); idx = idx.cpu().numpy()
            order_ = ctx.keys()[1].astype(np.int64)                     # sorted position -> original id
            own = order_[cuts[r]:cuts[r + 1]]
            assert np.all(owner[own] == -1)
            owner[own] = r
            rr = _rows(off, idx)
            notown = np.ones(w.n, bool); notown[own] = False
            assert np.all(np.diff(off)[notown] == 0)                    # rows of the others are empty
            for i in own:
                rows[i] = rr[i]
            st = ctx.stats()
            tot["n_pp"] += st["n_pp"]; tot["n_pc"] += st["n_pc"]
            npp, npc = ctx.list_lengths()
            c = shard.group_cost(g["end"] - g["begin"], npp, npc)
            mine = np.zeros(len(c), bool); mine[gcuts[r]:gcuts[r + 1]] = True
            assert np.all(c[~mine] == 0)
            costs = c if costs is None else costs + c
    assert np.all(owner >= 0)
    return merged.cpu().numpy(), rows, tot, all_cuts, costs


def _same(merged, whole, exact):
    if exact:
        assert np.array_equal(merged.view(np.uint32), whole.view(np.uint32))
        return
    a, b = merged.astype(np.float64), whole.astype(np.float64)
    assert np.all(np.linalg.norm(a[:, :3] - b[:, :3], axis=1) <= 2e-6 * np.linalg.norm(b[:, :3], axis=1))
    assert np.all(np.abs(a[:, 3] - b[:, 3]) <= 2e-6 * np.abs(b[:, 3]))


def _run_whole(p3t, w, r_in, order=2, key_bits=63):
    with p3t.Context(0) as ctx:
        ctx.set_multipole_order(order)
        ctx.build_tree(_cuda(w.pos_mass), key_bits)
        out = ctx.regular_force(w.r_out, r_in, w.theta, 0).cpu().numpy()
        off, idx = ctx.neighbours()
        st = ctx.stats()
        g = ctx.groups()
        npp, npc = ctx.list_lengths()
    return out, _rows(off.cpu().numpy(), idx.cpu().numpy()), st, g, shard.group_cost(g["end"] - g["begin"], npp, npc)


@pytest.mark.parametrize("cfg,n,nranks,key_bits,exact", [(1, 16384, 2, 63, True), (1, 5000, 3, 30, True), (2, 131072, 4, 63, False),
                                                         (4, 40000, 8, 63, True), (1, 100, 5, 63, True), (2, 524288, 2, 63, True)])
def test_sharded_equals_whole_bit_for_bit(p3t, cfg, n, nranks, key_bits, exact):
    w = workloads.make_config(cfg, n_override=n)
    r_in = w.r_in
    whole, wrows, wst, g, wcost = _run_whole(p3t, w, r_in, key_bits=key_bits)
    merged, rows, tot, cuts, costs = _run_sharded(p3t, w, nranks, r_in, key_bits=key_bits)
    _same(merged, whole, exact)
    assert all(np.array_equal(a, b) for a, b in zip(rows, wrows))
    assert tot["n_pp"] == wst["n_pp"] and tot["n_pc"] == wst["n_pc"]
    assert np.array_equal(costs, wcost)                                  # the summed cost vector = gather_group_costs
    # default cuts: the first group boundary at or after r n / nranks
    gb = np.append(g["begin"], w.n)
    for r in range(nranks + 1):
        assert cuts[r] == gb[np.searchsorted(gb, r * w.n // nranks if r < nranks else w.n, side="left")]


def test_cost_balanced_cuts_and_monopole(p3t):
    """Cuts from the previous step's list lengths (King model: the core groups are the expensive ones), monopole
    variant; the merged result still equals the whole one, and the balance is better than by particle count."""
    w = workloads.make_config(4, n_override=60000)
    r_in = w.r_in
    nranks = 4
    whole, wrows, wst, g, wcost = _run_whole(p3t, w, r_in, order=1)
    nominal = shard.balanced_cuts(g["begin"], w.n, wcost, nranks)
    merged, rows, tot, cuts, costs = _run_sharded(p3t, w, nranks, r_in, nominal=nominal, order=1)
    _same(merged, whole, False)
    assert all(np.array_equal(a, b) for a, b in zip(rows, wrows))
    assert np.array_equal(cuts, nominal)                                 # same tree: the nominal cuts are group starts already
    gb = g["begin"]

    def worst(c):
        own = np.searchsorted(c[1:], gb, side="right")
        return max(wcost[own == r].sum() for r in range(nranks)) / (wcost.sum() / nranks)
    by_count = np.array([r * w.n // nranks for r in range(nranks)] + [w.n])
    assert worst(cuts) <= 1.0 + wcost.max() * nranks / wcost.sum() + 1e-9
    assert worst(cuts) <= worst(by_count)


def test_merged_result_against_direct_sum(p3t):
    w = workloads.make_config(1, n_override=20000)
    r_in = w.r_in
    merged, rows, tot, cuts, costs = _run_sharded(p3t, w, 3, r_in)
    t = workloads.sample_targets(w.n, 256)
    d = oracle.direct(w.pos_mass, w.r_out, r_in, targets=t)
    a = merged[t, :3].astype(np.float64)
    err = np.linalg.norm(a - d["acc_reg"], axis=1) / np.linalg.norm(d["acc_reg"], axis=1)
    assert np.median(err) < 1e-3 and err.max() < 2e-2                   # the tree's own approximation (north_star's bound)


def test_nonmonotone_and_degenerate_cuts(p3t):
    """Caller's cuts out of order or beyond n: ranks get empty ranges, nothing is lost or done twice."""
    w = workloads.make_config(1, n_override=3000)
    r_in = w.r_in
    whole, wrows, wst, g, wcost = _run_whole(p3t, w, r_in)
    for nominal in ([0, 2000, 1000, 10 ** 9], [5, 0, 0, 3000], [0, 3000, 3000, 3000]):
        merged, rows, tot, cuts, costs = _run_sharded(p3t, w, 3, r_in, nominal=np.array(nominal))
        assert np.array_equal(merged.view(np.uint32), whole.view(np.uint32))
        assert all(np.array_equal(a, b) for a, b in zip(rows, wrows))


def test_shard_errors_and_reset(p3t):
    import torch
    w = workloads.make_config(1, n_override=2000)
    r_in = w.r_in
    pm = _cuda(w.pos_mass)
    with p3t.Context(0) as ctx:
        with pytest.raises(p3t.P3TError):
            ctx.set_shard(2, 2)
        with pytest.raises(p3t.P3TError):
            ctx.set_shard(0, 65)
        ctx.build_tree(pm)
        out = torch.zeros((w.n, 4), dtype=torch.float32, device="cuda")
        with pytest.raises(p3t.P3TError):                               # not sharded
            ctx.shard_pack(out, out)
        a = ctx.regular_force(w.r_out, r_in, w.theta).cpu().numpy()
        ctx.set_shard(1, 2)
        with pytest.raises(p3t.P3TError):                               # takes effect at the next build: force needs one
            ctx.regular_force(w.r_out, r_in, w.theta)
        ctx.build_tree(pm)
        b = ctx.regular_force(w.r_out, r_in, w.theta).cpu().numpy()
        cuts, _ = ctx.shard_cuts()
        own = ctx.keys()[1].astype(np.int64)[cuts[1]:cuts[2]]
        assert np.array_equal(a[own].view(np.uint32), b[own].view(np.uint32))
        ctx.set_shard(0, 1)                                             # back to the whole path
        ctx.build_tree(pm)
        c = ctx.regular_force(w.r_out, r_in, w.theta).cpu().numpy()
        assert np.array_equal(a.view(np.uint32), c.view(np.uint32))
