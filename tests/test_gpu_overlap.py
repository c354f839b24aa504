"""The force call's bookkeeping (p3t_force.cu: p3t_force_begin / p3t_force_finish): the list walk and the force kernel
run side by side and buffers are sized from the previous call.  Whatever a call could not do in its first pass
(groups whose lists did not fit, rows that could not be emitted, groups a force warp stopped waiting for) is redone
by the repair pass inside the same call -- with the same bits as a fresh context gives, and the velocity kicked
exactly once (eq. 12).  Capacity failures are reported by the force call itself."""
import os

import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def p3t():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2110_11658_b200 as m
    m.lib()
    return m


def _diag():
    from paper_2110_11658_b200 import pipebench
    return pipebench


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def _run(ctx, w, vel, half_dt, r_buff=0.0):
    ctx.build_tree(_cuda(w.pos_mass), 63)
    v = _cuda(vel)
    a = ctx.regular_force(w.r_out, w.r_in, w.theta, 0, r_buff=r_buff, half_dt=half_dt, vel=v).cpu().numpy()
    off, idx = ctx.neighbours()
    npp, npc = ctx.list_lengths()
    return dict(a=a, v=v.cpu().numpy(), off=off.cpu().numpy(), idx=idx.cpu().numpy(), npp=npp, npc=npc, st=ctx.stats())


def _same(x, y):
    for k in ("a", "v", "off", "idx", "npp", "npc"):
        assert np.array_equal(x[k], y[k]), k
    for k in ("n_pp", "n_pc", "nb_total", "nb_max"):
        assert x["st"][k] == y["st"][k], k


def _kicked_once(r, vel, half_dt):
    want = (np.float64(half_dt) * r["a"][:, :3].astype(np.float64) + vel[:, :3].astype(np.float64)).astype(np.float32)
    assert np.all(np.abs(r["v"][:, :3] - want) <= np.spacing(np.abs(want)))
    assert np.any(r["v"][:, :3] != vel[:, :3])


@pytest.mark.parametrize("overlap", ["1", "0"])
def test_repair_after_undersized_buffers(p3t, overlap):
    """A context sized by a tiny problem meets (a) a problem 20 x larger (list pools overflow: failed groups are
    redone) and (b) a dense King core with a long search radius (the neighbour total outgrows the index buffer: no row is
    emitted in the first pass, every group is evaluated again without a second kick).  Both with and without
    the walk / force overlap."""
    ov = overlap == "1"                                       # set on every context below (libp3t_diag.so)
    small = workloads.make_config(1, n_override=3000)
    big = workloads.make_config(2, n_override=60000, theta=0.3)
    king = workloads.make_config(4, n_override=50000)
    king.r_out = 0.06; king.r_in = 0.006
    half_dt = float(np.float32(1.0 / 512.0))
    for w in (big, king):
        vel = workloads.velocities_for(w)
        with p3t.Context(0) as ref_ctx:
            _diag().set_overlap(ref_ctx, ov)
            _run(ref_ctx, w, vel, half_dt)                   # first call of a fresh context (its own repair, if any)
            ref = _run(ref_ctx, w, vel, half_dt)             # second call: buffers fit, nothing is repaired
        _kicked_once(ref, vel, half_dt)
        with p3t.Context(0) as ctx:
            _diag().set_overlap(ctx, ov)
            _run(ctx, small, workloads.velocities_for(small), half_dt)
            got = _run(ctx, w, vel, half_dt)                 # outgrows the pools / index buffers of the small problem
            _same(got, ref)
            _kicked_once(got, vel, half_dt)
            _same(_run(ctx, w, vel, half_dt), ref)
    assert ref["st"]["nb_total"] > (1 << 20) + (1 << 18)      # beyond the first guess of the index capacity (max(4 n, 2^20))
    # against the oracle as well (the reference above is the same library)
    ooff, oidx = oracle.neighbours_grid(king.pos_mass, king.r_out)
    assert np.array_equal(ooff, ref["off"]) and np.array_equal(oidx, ref["idx"])


def test_force_warps_that_stop_waiting(p3t):
    """Fault bit 1 (p3t_diag_set_fault): every force warp gives up at once on a group whose lists are not there yet (what the
    time-out does when no walker is resident): those groups are marked failed and redone by the repair pass."""
    w = workloads.make_config(2, n_override=80000)
    vel = workloads.velocities_for(w)
    half_dt = float(np.float32(1.0 / 512.0))
    with p3t.Context(0) as ctx:
        _run(ctx, w, vel, half_dt)
        ref = _run(ctx, w, vel, half_dt)
    with p3t.Context(0) as ctx:
        _diag().set_fault(ctx, 1)
        for _ in range(2):
            got = _run(ctx, w, vel, half_dt)
            _same(got, ref)
            _kicked_once(got, vel, half_dt)
            assert got["st"]["force_flags"] & p3t.FF_REPAIRED
    T = oracle.Tree(w.pos_mass, 63, 16, 64)
    f = T.force(w.r_out, w.r_in, w.theta, 0)
    assert np.linalg.norm(ref["a"][:, :3] - f["acc_pot"][:, :3]) <= 1e-6 * np.linalg.norm(f["acc_pot"][:, :3])


def test_repair_keeps_the_octupole_term_of_finished_groups(p3t):
    """Order 3 at small N (every work item shared by several warps, so the sums go through k_force_final) with
    fault bit 1: some groups are complete after the first pass, the others are redone.  The repair pass must leave
    the finished groups alone -- their result already carries the octupole term, which the repair adds only to the
    groups it redoes -- so that acceleration and kicked velocity are those of an undisturbed call, bit for bit."""
    w = workloads.make_config(1, n_override=20000)
    vel = workloads.velocities_for(w)
    half_dt = float(np.float32(1.0 / 512.0))
    with p3t.Context(0) as ctx:
        ctx.set_multipole_order(3)
        _run(ctx, w, vel, half_dt)
        ref = _run(ctx, w, vel, half_dt)
    with p3t.Context(0) as ctx:
        quad = _run(ctx, w, vel, half_dt)
    assert np.mean(ref["a"][:, :3] != quad["a"][:, :3]) > 0.5          # the octupole term is really there
    with p3t.Context(0) as ctx:
        _diag().set_fault(ctx, 1)
        ctx.set_multipole_order(3)
        for _ in range(2):
            got = _run(ctx, w, vel, half_dt)
            _same(got, ref)                                            # acceleration AND velocity: kicked exactly as undisturbed
    # the order-3 kick is two fmas (quadrupole-order sum, then the octupole's share): a few ulp from the one-fma value
    a = ref["a"][:, :3].astype(np.float64)
    want = vel[:, :3].astype(np.float64) + np.float64(half_dt) * a
    assert np.all(np.abs(ref["v"][:, :3] - want) <= 4e-7 * (np.abs(want) + half_dt * np.abs(a)) + 1e-30)


def test_walk_stack_overflow_is_a_condition_of_one_call(p3t):
    """theta may change between calls without a rebuild (include/p3t.h): after a call whose wide-open walk overflowed
    the walk stack (P3T_ECUDA; fault bit 2 takes the spill space away so that 384 entries are all there is), a
    call on the SAME tree with a theta whose walk fits works, and gives what a fresh context gives."""
    w = workloads.make_config(1, n_override=20000)
    pm = _cuda(w.pos_mass)
    with p3t.Context(0) as ctx:
        ctx.build_tree(pm, 63)
        ref = ctx.regular_force(w.r_out, w.r_in, 1.0, 0).cpu().numpy()
        roff, ridx = [x.cpu().numpy() for x in ctx.neighbours()]
    with p3t.Context(0) as ctx:
        _diag().set_fault(ctx, 2)
        ctx.build_tree(pm, 63)
        with pytest.raises(p3t.P3TError) as e:
            ctx.regular_force(w.r_out, w.r_in, 1e-3, 0)
        assert e.value.code == p3t.ECUDA and "stack_overflow=1" in str(e.value)
        got = ctx.regular_force(w.r_out, w.r_in, 1.0, 0).cpu().numpy()
        assert np.array_equal(got, ref)
        off, idx = [x.cpu().numpy() for x in ctx.neighbours()]
        assert np.array_equal(off, roff) and np.array_equal(idx, ridx)


def test_capacity_error_comes_from_the_force_call(p3t):
    """Fault bit 2 removes the spill space of the walk stack: a wide-open walk (theta -> 0) overflows it, and
    p3t_regular_force itself returns P3T_ECUDA (not a later accessor); NaN input is reported by it too, and the
    velocities are not kicked in that case."""
    import torch
    w = workloads.make_config(1, n_override=20000)
    with p3t.Context(0) as ctx:
        _diag().set_fault(ctx, 2)
        ctx.build_tree(_cuda(w.pos_mass), 63)
        with pytest.raises(p3t.P3TError) as e:
            ctx.regular_force(w.r_out, w.r_in, 1e-3, 0)
        assert e.value.code == p3t.ECUDA and "stack_overflow" in str(e.value)
    with p3t.Context(0) as ctx:
        bad = w.pos_mass.copy(); bad[17, 2] = np.nan
        ctx.build_tree(_cuda(bad), 63)
        vel = _cuda(workloads.velocities_for(w)); v0 = vel.clone()
        with pytest.raises(p3t.P3TError) as e:
            ctx.regular_force(w.r_out, w.r_in, 0.4, 0, half_dt=0.01, vel=vel)
        assert e.value.code == p3t.EINVAL
        assert torch.equal(vel, v0)
        ctx.build_tree(_cuda(w.pos_mass), 63)                 # the context recovers
        ctx.regular_force(w.r_out, w.r_in, 0.4, 0)


def test_two_contexts_on_two_streams(p3t):
    """Two contexts used in turn on their own streams (only one overlapped call is in flight per device and process;
    the other takes the one-after-the-other order): same bits."""
    import torch
    w = workloads.make_config(2, n_override=50000)
    pm = _cuda(w.pos_mass)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with p3t.Context(0, stream=s1) as c1, p3t.Context(0, stream=s2) as c2:
        outs = []
        for c in (c1, c2, c1, c2):
            c.build_tree(pm, 63)
            outs.append(c.regular_force(w.r_out, w.r_in, w.theta, 0).clone())
        torch.cuda.synchronize()
        for o in outs[1:]:
            assert torch.equal(o, outs[0])


def test_two_host_threads_at_the_same_time(p3t):
    """One context per host thread (include/p3t.h), both threads stepping at the same time on their own streams: only
    one overlapped call is in flight per device and process (the other thread's call takes the serial order), nothing
    deadlocks and every step gives the same bits as a single-threaded run."""
    import threading
    import torch
    w = workloads.make_config(2, n_override=70000)
    pm = _cuda(w.pos_mass)
    with p3t.Context(0) as ctx:
        ctx.build_tree(pm, 63)
        ref = ctx.regular_force(w.r_out, w.r_in, w.theta, 0).clone()
        roff, ridx = ctx.neighbours()
        roff = roff.clone(); ridx = ridx.clone()
    torch.cuda.synchronize()
    errors = []

    def worker(k):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                out = torch.empty((w.n, 4), dtype=torch.float32, device="cuda")
            with p3t.Context(0, stream=st) as c:
                for _ in range(12):
                    c.build_tree(pm, 63)
                    c.regular_force(w.r_out, w.r_in, w.theta, 0, out=out)
                    off, idx = c.neighbours()
                    if not (torch.equal(out, ref) and torch.equal(off, roff) and torch.equal(idx, ridx)):
                        errors.append(f"thread {k}: result differs")
        except Exception as e:                              # noqa: BLE001 - reported by the main thread
            errors.append(f"thread {k}: {e!r}")

    threads = [threading.Thread(target=worker, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
        assert not t.is_alive(), "a thread hangs"
    assert not errors, errors


def test_step_host_as_first_call_with_repair(p3t):
    """p3t_step_host as the very first call of a context, on a dense King core whose neighbour total outgrows the first guess
    of the index capacity: the repair pass runs inside the call and the host buffers hold the final results."""
    w = workloads.make_config(4, n_override=50000)
    w.r_out = 0.06; w.r_in = 0.006
    with p3t.Context(0) as ctx:
        ctx.build_tree(_cuda(w.pos_mass), 63)
        a = ctx.regular_force(w.r_out, w.r_in, w.theta).cpu().numpy()
        a = ctx.regular_force(w.r_out, w.r_in, w.theta).cpu().numpy()
        off, idx = ctx.neighbours()
        off = off.cpu().numpy(); idx = idx.cpu().numpy()
    assert idx.shape[0] > (1 << 20) + (1 << 18)
    nb_off = np.empty(w.n + 1, dtype=np.int64); nb_idx = np.empty(idx.shape[0] + 10, dtype=np.int32)
    with p3t.Context(0) as ctx:
        acc, _, _, total = ctx.step_host(w.pos_mass, w.r_out, w.r_in, w.theta, nb_offsets=nb_off, nb_indices=nb_idx)
        assert total == idx.shape[0]
        assert np.array_equal(acc, a) and np.array_equal(nb_off, off) and np.array_equal(nb_idx[:total], idx)
        acc2, _, _, total2 = ctx.step_host(w.pos_mass, w.r_out, w.r_in, w.theta, nb_offsets=nb_off, nb_indices=nb_idx)
        assert total2 == total and np.array_equal(acc2, a) and np.array_equal(nb_idx[:total], idx)


def test_begin_wait_is_the_blocking_call_in_two_halves(p3t):
    """p3t_regular_force_begin returns with the call enqueued (the host is free: PAPER.md:89-94, the CPU integrates the
    irregular forces meanwhile), p3t_regular_force_wait completes it: same bits as the blocking call; the state rules
    of include/p3t.h hold in between; a context destroyed with a call in flight leaves the device's overlap slot free."""
    import torch
    w = workloads.make_config(1, n_override=120000)
    vel = workloads.velocities_for(w)
    half_dt = float(np.float32(1.0 / 512.0))
    pm = _cuda(w.pos_mass)
    with p3t.Context(0) as ctx:
        _run(ctx, w, vel, half_dt)
        ref = _run(ctx, w, vel, half_dt)
        assert ref["st"]["force_flags"] == p3t.FF_OVERLAPPED          # overlapped, nothing repaired
    L = p3t.lib()
    with p3t.Context(0) as ctx:
        assert L.p3t_regular_force_wait(ctx._h) == p3t.ESTATE        # nothing pending
        for k in range(2):                                           # first call of the context (repair inside wait), then a normal one
            ctx.build_tree(pm, 63)
            v = _cuda(vel)
            out = ctx.regular_force_begin(w.r_out, w.r_in, w.theta, 0, half_dt=half_dt, vel=v)
            host_work = sum(i * i for i in range(20000))             # the host is not blocked
            assert L.p3t_build_tree(ctx._h, w.n, pm.data_ptr(), 63) == p3t.ESTATE
            assert L.p3t_regular_force_begin(ctx._h, w.r_out, w.r_in, w.theta, 0, 0.0, 0.0, None, out.data_ptr()) == p3t.ESTATE
            with pytest.raises(p3t.P3TError):
                ctx.neighbours()
            ctx.regular_force_wait()
            off, idx = ctx.neighbours()
            npp, npc = ctx.list_lengths()
            got = dict(a=out.cpu().numpy(), v=v.cpu().numpy(), off=off.cpu().numpy(), idx=idx.cpu().numpy(), npp=npp, npc=npc, st=ctx.stats())
            _same(got, ref)
            assert host_work > 0
        assert got["st"]["force_flags"] == p3t.FF_OVERLAPPED
    # destroyed between begin and wait
    ctx = p3t.Context(0)
    ctx.build_tree(pm, 63)
    out = ctx.regular_force_begin(w.r_out, w.r_in, w.theta, 0)
    ctx.close()
    del out
    with p3t.Context(0) as ctx:
        got = _run(ctx, w, vel, half_dt)
        assert got["st"]["force_flags"] & p3t.FF_OVERLAPPED, "the overlap slot of the device was not given back"
        _same(got, ref)


def test_failed_step_host_gives_the_overlap_slot_back(p3t):
    """A CUDA failure inside p3t_step_host after the force call has been enqueued (fault bit 4 injects one) is
    reported, the context is drained, and the per-device overlap slot is free again: the next context still runs the
    walk beside the force kernel (it used to fall back to the serial order for the rest of the process)."""
    w = workloads.make_config(1, n_override=50000)
    pm_host = np.ascontiguousarray(w.pos_mass)
    with p3t.Context(0) as ctx:
        _diag().set_fault(ctx, 4)
        with pytest.raises(p3t.P3TError) as e:
            ctx.step_host(pm_host, w.r_out, w.r_in, w.theta, nb_offsets=np.empty(w.n + 1, np.int64))
        assert e.value.code == p3t.ECUDA
        with pytest.raises(p3t.P3TError):                         # a CUDA failure is sticky for its context
            ctx.build_tree(_cuda(w.pos_mass), 63)
    with p3t.Context(0) as ctx:
        ctx.build_tree(_cuda(w.pos_mass), 63)
        ctx.regular_force(w.r_out, w.r_in, w.theta, 0)
        assert ctx.stats()["force_flags"] & p3t.FF_OVERLAPPED, "the overlap slot of the device was not given back"
        a, off, idx, total = ctx.step_host(pm_host, w.r_out, w.r_in, w.theta, nb_offsets=np.empty(w.n + 1, np.int64))
        assert ctx.stats()["force_flags"] & p3t.FF_OVERLAPPED and total > 0
