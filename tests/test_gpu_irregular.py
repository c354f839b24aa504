"""GPU parity of p3t_irregular_force (eq. 1, 2, 5, 7 over the emitted neighbour
lists) against the fp64 oracle (oracle.irregular, pinned in test_oracle_irregular.py), through the C-ABI.

Tolerance: every term is evaluated in fp32 with IEEE sqrt and division (a few ulp each, 6e-8) and
summed in fp64: |error| <= 2e-6 x the sum of |terms| of the row.  On top of that the cutoff argument
x = (r - r_in)/(r_out - r_in) carries the rounding of r, dx ~ 7e-8, so K and K' = dW/dx move by
W' dx <= 1.5e-7 and W'' dx <= 5e-7 of the UNWEIGHTED (K = 1) term: + 1e-6 x abs_newt.  (Near x = 1
the weighted terms vanish like (1-x)^4 and that absolute floor is what is left.)"""
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


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def _check(p3t, w, targets=None, r_out=None, grid=False):
    r_out = w.r_out if r_out is None else r_out
    r_in = float(np.float32(0.1) * np.float32(r_out))
    vel = workloads.velocities_for(w)
    with p3t.Context(0) as ctx:
        ctx.build_tree(_cuda(w.pos_mass), 63)
        reg = ctx.regular_force(r_out, r_in, w.theta, 0).cpu().numpy().astype(np.float64)
        acc, jerk = ctx.irregular_force(_cuda(vel))
        acc = acc.cpu().numpy().astype(np.float64); jerk = jerk.cpu().numpy().astype(np.float64)
        off, idx = ctx.neighbours()
        off = off.cpu().numpy(); idx = idx.cpu().numpy()
        st = ctx.stats()
    # grid: every target at N = 2^20 -- the oracle tests only the candidates of its cell-grid search at 1.01 r_out
    cand = oracle.neighbours_grid(w.pos_mass, 1.01 * r_out, targets=targets) if grid else None
    o = oracle.irregular(w.pos_mass, vel, r_out, r_in, targets=targets, candidates=cand)
    sel = slice(None) if targets is None else targets
    a, j = acc[sel], jerk[sel]
    ea = np.linalg.norm(a[:, :3] - o["acc_irr"], axis=1)
    ej = np.linalg.norm(j[:, :3] - o["jerk_irr"], axis=1)
    na = np.linalg.norm(o["acc_irr"], axis=1)
    tol = 2e-6 * o["abs_jerk"] + 1e-6 * o["abs_newt"] + 1e-30
    assert np.all(ej <= tol), (ej / tol).max()
    assert np.linalg.norm(j[:, :3] - o["jerk_irr"]) <= 1e-6 * np.linalg.norm(o["jerk_irr"])
    assert np.linalg.norm(a[:, :3] - o["acc_irr"]) <= 1e-6 * np.linalg.norm(o["acc_irr"])
    has = na > 0
    if has.sum() > 10:
        assert np.median(ea[has] / na[has]) <= 1e-6
    # potential: relative to the row's unweighted sum of m_j / r (the rounding of r moves every pair
    # term by eps m K / r, which is all that is left of a pair near r_out where phi_I vanishes like (1-x)^5)
    rows = np.repeat(np.arange(w.n), np.diff(off))
    pos = w.pos_mass[:, :3].astype(np.float64)
    rij = np.linalg.norm(pos[idx] - pos[rows], axis=1)
    nz = rij > 0
    newt = np.bincount(rows[nz], weights=w.pos_mass[idx[nz], 3].astype(np.float64) / rij[nz], minlength=w.n)
    assert np.all(np.abs(a[:, 3] - o["phi_irr"]) <= 3e-6 * np.abs(o["phi_irr"]) + 3e-7 * newt[sel] + 1e-30)
    assert np.all(j[:, 3] == 0)
    # empty rows give exact zeros (lists are often empty)
    empty = np.diff(off) == 0
    assert np.all(acc[empty] == 0) and np.all(jerk[empty] == 0)
    return reg, acc, jerk, o, st


def test_config1_full(p3t):
    """Config 1 (Plummer 16k): every particle; F_I + F_R is the unsplit Newtonian force (eq. 3)."""
    w = workloads.make_config(1)
    reg, acc, jerk, o, st = _check(p3t, w)
    d = oracle.direct(w.pos_mass, w.r_out, w.r_in)
    newton = d["acc_reg"] + d["acc_irr"]
    tot = reg[:, :3] + acc[:, :3]
    err = np.linalg.norm(tot - newton, axis=1) / np.linalg.norm(newton, axis=1)
    assert np.median(err) < 2e-3 and np.percentile(err, 99) < 2e-2          # the tree error of F_R, north_star bound
    assert np.abs((reg[:, 3] + acc[:, 3]) / d["phi_newt"] - 1).max() < 1e-3
    assert st["ms_irregular"] > 0


def test_larger_radius_long_rows(p3t):
    """Rows longer than a warp (the warp-cooperative branch): 4 x the configured radius."""
    w = workloads.make_config(1, n_override=6000)
    reg, acc, jerk, o, st = _check(p3t, w, r_out=4 * w.r_out)
    assert st["nb_max"] > 32


def test_king_core_sampled(p3t):
    """Config 4 recipe (King W0 = 9, Kroupa masses) at N = 2^17: long rows in the core, sampled targets."""
    w = workloads.make_config(4, n_override=131072)
    t = workloads.sample_targets(w.n, 4096)
    _check(p3t, w, targets=t)


def test_king_core_full_size(p3t):
    """Config 4 itself (King W0 = 9, N = 2^20, 1.66e7 list entries, rows of up to ~500): EVERY particle."""
    w = workloads.make_config(4)
    reg, acc, jerk, o, st = _check(p3t, w, grid=True)
    assert st["nb_max"] > 256 and st["nb_total"] > 1.5e7


def test_state_and_arguments(p3t):
    import torch
    w = workloads.make_config(1, n_override=2000)
    vel = _cuda(workloads.velocities_for(w))
    with p3t.Context(0) as ctx:
        ctx.build_tree(_cuda(w.pos_mass), 63)
        with pytest.raises(p3t.P3TError) as e:
            ctx.irregular_force(vel)                       # no regular force yet: no lists
        assert e.value.code == -2
        ctx.regular_force(w.r_out, w.r_in, w.theta, 0)
        a1, j1 = ctx.irregular_force(vel)
        a2, j2 = ctx.irregular_force(vel)                  # deterministic
        assert torch.equal(a1, a2) and torch.equal(j1, j2)
        # zero velocities: zero jerk, same acceleration
        a0, j0 = ctx.irregular_force(torch.zeros_like(vel))
        assert torch.equal(a0, a1) and torch.count_nonzero(j0) == 0


# ---- buffered search radius and the fused leapfrog half-kick ----
def test_buffered_lists_and_kick(p3t):
    """r_list = r_out + r_buff: neighbour CSR bit-exact against brute force at r_list, interaction lists and
    force against the oracle tree with the widened opening clause; eq. 12 kick = one fma on the returned a."""
    import torch
    w = workloads.make_config(1)
    r_buff = float(np.float32(3.0 * w.r_out))                       # large enough for the clause to bite
    r_list = float(np.float32(w.r_out) + np.float32(r_buff))
    vel = workloads.velocities_for(w)
    half_dt = float(np.float32(1.0 / 256.0))
    T = oracle.Tree(w.pos_mass, 63, 16, 64)
    with p3t.Context(0) as ctx:
        ctx.build_tree(_cuda(w.pos_mass), 63)
        v_dev = _cuda(vel)
        out = ctx.regular_force(w.r_out, w.r_in, w.theta, 0, r_buff=r_buff, half_dt=half_dt, vel=v_dev)
        a32 = out.cpu().numpy()
        a = a32.astype(np.float64)
        npp, npc = ctx.list_lengths()
        off, idx = ctx.neighbours()
        off = off.cpu().numpy(); idx = idx.cpu().numpy()
        f = T.force(w.r_out, w.r_in, w.theta, 0, want_abs=True, r_list=r_list)
        assert np.array_equal(npp, f["npp"]) and np.array_equal(npc, f["npc"]), "interaction lists differ"
        ref = f["acc_pot"]
        assert np.linalg.norm(a[:, :3] - ref[:, :3]) <= 1e-6 * np.linalg.norm(ref[:, :3])
        assert np.all(np.linalg.norm(a[:, :3] - ref[:, :3], axis=1) <= 1e-6 * f["abs_sum"] + 1e-30)
        assert np.all(np.abs(a[:, 3] - ref[:, 3]) <= 2e-6 * np.abs(ref[:, 3]))
        ooff, oidx = oracle.neighbours(w.pos_mass, r_list)
        assert np.array_equal(ooff, off) and np.array_equal(oidx, idx), "buffered neighbour CSR differs"
        o0, _ = oracle.neighbours(w.pos_mass, w.r_out)
        assert off[-1] > 5 * o0[-1]                                  # the buffer shell is populated
        # kick: v' = fma(half_dt, a, v) in fp32; exact product + one rounding, emulated in fp64 (the product
        # of two fp32 is exact in fp64; the sum may round twice: allow 1 ulp)
        v1 = v_dev.cpu().numpy()
        want = (np.float64(half_dt) * a32[:, :3].astype(np.float64) + vel[:, :3].astype(np.float64)).astype(np.float32)
        ulp = np.spacing(np.abs(want))
        assert np.all(np.abs(v1[:, :3] - want) <= ulp) and np.mean(v1[:, :3] == want) > 0.999
        assert np.array_equal(v1[:, 3], vel[:, 3])
        # the irregular force over the buffered lists: shell members (r >= r_out) contribute nothing
        acc, jerk = ctx.irregular_force(_cuda(vel))
        o = oracle.irregular(w.pos_mass, vel, w.r_out, w.r_in)
        acc = acc.cpu().numpy().astype(np.float64); jerk = jerk.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(acc[:, :3] - o["acc_irr"]) <= 1e-6 * np.linalg.norm(o["acc_irr"])
        assert np.all(np.linalg.norm(jerk[:, :3] - o["jerk_irr"], axis=1) <= 2e-6 * o["abs_jerk"] + 1e-6 * o["abs_newt"] + 1e-30)
        # r_buff = 0 through the _ex entry point is p3t_regular_force
        b0 = ctx.regular_force(w.r_out, w.r_in, w.theta, 0)
        b1 = ctx.regular_force(w.r_out, w.r_in, w.theta, 0, r_buff=0.0, vel=torch.zeros_like(v_dev))
        assert torch.equal(b0, b1)
        with pytest.raises(p3t.P3TError):
            ctx.regular_force(w.r_out, w.r_in, w.theta, 0, r_buff=-1.0, vel=v_dev)


@pytest.mark.parametrize("n,ncore,expect_pv", [(4000, 400, True), (60000, 300, False)])
def test_row_length_classes_and_both_gather_paths(p3t, n, ncore, expect_pv):
    """A tight clump inside r_out (rows of ncore - 1 entries: the all-lanes branch) in a Plummer halo whose rows are
    short (thread per row) or medium (eight lanes per row), with the lists at >= 4 entries per particle (packed
    position + velocity records) and below (rank indirection): every branch of k_irregular against the oracle."""
    w = workloads.make_config(1, n_override=n)
    rng = np.random.default_rng(n)
    pm = w.pos_mass.copy()
    d = rng.normal(size=(ncore, 3)); d *= (0.3 * w.r_out) * rng.random((ncore, 1)) ** (1 / 3) / np.linalg.norm(d, axis=1, keepdims=True)
    pm[:ncore, :3] = (np.array([0.2, -0.1, 0.05]) + d).astype(np.float32)
    w.pos_mass = pm
    # a second, looser clump gives rows of 33 .. 256 entries
    d2 = rng.normal(size=(120, 3)); d2 *= (0.45 * w.r_out) / np.linalg.norm(d2, axis=1, keepdims=True) * rng.random((120, 1)) ** (1 / 3)
    pm[ncore:ncore + 120, :3] = (np.array([-0.3, 0.2, 0.1]) + d2).astype(np.float32)
    reg, acc, jerk, o, st = _check(p3t, w)
    assert st["nb_max"] > 256
    assert (st["nb_total"] >= 4 * n) == expect_pv
