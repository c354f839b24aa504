"""GPU parity of the octupole variant (p3t_set_multipole_order(ctx, 3): k_octupoles,
k_octupole_add in p3t_octupole.cu) against the oracle's order-3 tree force (pinned in test_oracle_octupole.py),
through the C-ABI.  Same lists as order 2 (bit-exact lengths); third moments within a few fp32 ulp of the oracle's
(the CUDA build combines children by the parallel-axis rule in fp64, the oracle sums every cell's own particles:
they differ by fp64 rounding before the one rounding to fp32); force within 1e-6 of the sum of |terms| as for
order 2; against eq. 3 by direct summation the error must be smaller than with order 2."""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu
NLEAF, NCRIT = 16, 64


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


def _rel(a, ref):
    return np.linalg.norm(a - ref, axis=1) / np.linalg.norm(ref, axis=1)


def _check(p3t, w, bits=63, group_ids=None, vs_direct=True):
    T = oracle.Tree(w.pos_mass, bits, NLEAF, NCRIT)
    with p3t.Context(0) as ctx:
        ctx.set_multipole_order(3)
        ctx.build_tree(_cuda(w.pos_mass), bits)
        a3 = ctx.regular_force(w.r_out, w.r_in, w.theta, 0).cpu().numpy().astype(np.float64)
        npp, npc = ctx.list_lengths()
        oc = ctx.octupoles()
        st = ctx.stats()
        assert st["ms_octupole"] > 0
        off, idx = ctx.neighbours()
        nb3 = (off.cpu().numpy(), idx.cpu().numpy())
        ctx.set_multipole_order(2)                                  # back to the default on the same tree
        a2 = ctx.regular_force(w.r_out, w.r_in, w.theta, 0).cpu().numpy().astype(np.float64)
        off, idx = ctx.neighbours()
        assert np.array_equal(nb3[0], off.cpu().numpy()) and np.array_equal(nb3[1], idx.cpu().numpy())
    # third moments: scale of a cell = sum m |d|^3 <= M * (box diagonal)^3
    o = T.octupoles(); mo = T.moments()
    diag = np.linalg.norm(mo["chi"].astype(np.float64) - mo["clo"], axis=1)
    scale = mo["com_m"][:, 3].astype(np.float64) * diag ** 3
    assert oc.shape == o["oct32"].shape
    assert np.all(np.abs(oc.astype(np.float64) - o["oct64"]).max(axis=1) <= 2e-7 * scale + 1e-40)
    f3 = T.force(w.r_out, w.r_in, w.theta, 0, group_ids=group_ids, want_abs=True, order=3)
    if group_ids is None:
        assert np.array_equal(npp, f3["npp"]) and np.array_equal(npc, f3["npc"])
    ref = f3["acc_pot"]
    sel = ~np.isnan(ref[:, 0])
    assert sel.sum() > 0
    assert np.linalg.norm(a3[sel, :3] - ref[sel, :3]) <= 1e-6 * np.linalg.norm(ref[sel, :3])
    assert np.all(np.linalg.norm(a3[sel, :3] - ref[sel, :3], axis=1) <= 1e-6 * f3["abs_sum"][sel] + 1e-30)
    assert np.all(np.abs(a3[sel, 3] - ref[sel, 3]) <= 2e-6 * np.abs(ref[sel, 3]))
    if vs_direct:
        tg = np.flatnonzero(sel)[:: max(1, int(sel.sum()) // 2048)]
        d = oracle.direct(w.pos_mass, w.r_out, w.r_in, targets=tg)
        e3 = _rel(a3[tg, :3], d["acc_reg"]); e2 = _rel(a2[tg, :3], d["acc_reg"])
        assert np.median(e3) < 0.6 * np.median(e2) and np.percentile(e3, 99) < np.percentile(e2, 99)
        assert np.median(e3) < 2e-3 and np.percentile(e3, 99) < 2e-2
    return a3, a2


@pytest.mark.parametrize("bits", [63, 30])
def test_octupole_config1(p3t, bits):
    _check(p3t, workloads.make_config(1), bits)


def test_octupole_kroupa_128k_sampled_groups(p3t):
    w = workloads.make_config(2)
    T = oracle.Tree(w.pos_mass, 63, NLEAF, NCRIT)
    _check(p3t, w, group_ids=np.arange(0, T.n_groups, 16))


def test_octupole_king_and_large_theta(p3t):
    w = workloads.make_config(4, n_override=50000, theta=0.7)
    _check(p3t, w)


def test_octupole_full_size_1m_sampled(p3t):
    w = workloads.make_config(3)
    T = oracle.Tree(w.pos_mass, 63, NLEAF, NCRIT)
    _check(p3t, w, group_ids=np.arange(5, T.n_groups, 400), vs_direct=True)


def test_octupole_needs_a_build_and_tiny_inputs(p3t):
    w = workloads.make_config(1, n_override=700)
    pm = _cuda(w.pos_mass)
    with p3t.Context(0) as ctx:
        ctx.build_tree(pm)
        ctx.set_multipole_order(3)
        with pytest.raises(p3t.P3TError):                           # the third moments do not exist yet
            ctx.regular_force(w.r_out, w.r_in, w.theta)
        with pytest.raises(p3t.P3TError):
            ctx.octupoles()
        ctx.build_tree(pm)
        a = ctx.regular_force(w.r_out, w.r_in, w.theta).cpu().numpy()
        assert np.isfinite(a).all()
    for n in (1, 2, 17, 65):
        _check(p3t, workloads.make_config(1, n_override=n), vs_direct=False)


def test_octupole_with_kick_and_shard(p3t):
    """The kick of the fused epilogue gets the octupole's share too; a sharded context adds the term for its own groups."""
    import torch
    w = workloads.make_config(1, n_override=9000)
    pm = _cuda(w.pos_mass)
    vel0 = workloads.velocities_for(w)
    hdt = 0.01
    with p3t.Context(0) as ctx:
        ctx.set_multipole_order(3)
        ctx.build_tree(pm)
        vel = _cuda(vel0)
        a = ctx.regular_force(w.r_out, w.r_in, w.theta, 0, half_dt=hdt, vel=vel).cpu().numpy().astype(np.float64)
        v = vel.cpu().numpy().astype(np.float64)
        want = vel0[:, :3].astype(np.float64) + hdt * a[:, :3]
        assert np.all(np.abs(v[:, :3] - want) <= 4e-7 * (np.abs(want) + hdt * np.abs(a[:, :3])) + 1e-30)
        whole = ctx.regular_force(w.r_out, w.r_in, w.theta, 0).cpu().numpy()
    merged = torch.full((w.n, 4), float("nan"), dtype=torch.float32, device="cuda")
    for r in range(2):
        with p3t.Context(0) as ctx:
            ctx.set_multipole_order(3)
            ctx.set_shard(r, 2)
            ctx.build_tree(pm)
            cuts, _ = ctx.shard_cuts()
            out = ctx.regular_force(w.r_out, w.r_in, w.theta, 0)
            chunk = torch.empty((max(int(cuts[r + 1] - cuts[r]), 1), 4), dtype=torch.float32, device="cuda")
            ctx.shard_pack(out, chunk); ctx.shard_unpack(r, chunk, merged)
    assert np.array_equal(merged.cpu().numpy().view(np.uint32), whole.view(np.uint32))
