"""Pins of the oracle's octupole term and order-3 tree force (the octupole variant for the
accuracy-throughput curve; oracle/p3t_oracle_walk.c: p3t_o_pc_octupole, p3t_o_tree_force_order(order = 3)).

The paper evaluates monopole + quadrupole (Bonsai); the octupole is the next term of the same Taylor
expansion of 1/|r - d|.  It is pinned against things other than itself:
  * the textbook axial multipole expansion phi = -sum_l (sum m d^l) P_l(cos t) / R^(l+1), P_3(c) = (5c^3 - 3c)/2;
  * the exact potential and force of a small cluster: the residual of monopole + quadrupole + octupole must fall
    like R^-5 (potential) and R^-6 (force), one power faster than without the octupole -- a wrong coefficient
    anywhere leaves an R^-4 / R^-5 residual;
  * a = -grad phi by central differences;
  * the tree's third moments against the definition written with numpy, and the parallel-axis rule the CUDA build
    uses to combine children;
  * the order-3 tree force against the direct sum: more accurate than order 2 with the same lists."""
import numpy as np
import pytest

import oracle
import workloads

IDX = [(0, 0, 0), (1, 1, 1), (2, 2, 2), (0, 0, 1), (0, 0, 2), (0, 1, 1), (1, 1, 2), (0, 2, 2), (1, 2, 2), (0, 1, 2)]


def _moments(d, m):
    """fp64 M, traceless Q [6], raw third moment T [10] of masses m at offsets d (about the origin)."""
    d2 = (d * d).sum(1)
    Q = np.array([(m * (3 * d[:, 0] ** 2 - d2)).sum(), (m * (3 * d[:, 1] ** 2 - d2)).sum(), (m * (3 * d[:, 2] ** 2 - d2)).sum(),
                  (3 * m * d[:, 0] * d[:, 1]).sum(), (3 * m * d[:, 0] * d[:, 2]).sum(), (3 * m * d[:, 1] * d[:, 2]).sum()])
    T = np.array([(m * d[:, a] * d[:, b] * d[:, c]).sum() for a, b, c in IDX])
    return m.sum(), Q, T


def _cluster(seed, n=12, eps=0.05):
    """Masses k/1024 (their sum is exact in fp32) at random offsets within eps, centre of mass moved to the origin."""
    rng = np.random.default_rng(seed)
    m = rng.integers(1, 64, n) / 1024.0
    d = rng.normal(size=(n, 3)); d *= eps * rng.random((n, 1)) ** (1 / 3) / np.linalg.norm(d, axis=1, keepdims=True)
    d -= (m[:, None] * d).sum(0) / m.sum()
    return d, m


def _exact(x, d, m):
    r = x[None, :] - d
    R = np.linalg.norm(r, axis=1)
    return np.append(-(m[:, None] * r / R[:, None] ** 3).sum(0), -(m / R).sum())


def _expansion(x, M, Q, T, order):
    com_m = np.array([0, 0, 0, M], np.float32)
    out = oracle.pc_term(x, com_m, Q if order >= 2 else np.zeros(6))
    if order >= 3:
        out = out + oracle.pc_octupole(x, com_m, T)
    return out


@pytest.mark.parametrize("c", [1.0, 0.0, -1.0, 0.5, -0.3, 0.8])
def test_axial_distribution_is_legendre_p3(c):
    """Two masses on the x axis, centre of mass at the origin: phi_3 = -T_xxx P_3(cos t) / R^4 (textbook)."""
    m = np.array([3.0, 1.0]); dx = np.array([0.01, -0.03])
    d = np.zeros((2, 3)); d[:, 0] = dx
    _, _, T = _moments(d, m)
    assert T[0] == pytest.approx(3.0 * 0.01 ** 3 - 0.03 ** 3) and np.allclose(T[1:], 0)
    R = 0.7
    x = R * np.array([c, np.sqrt(1 - c * c), 0.0])
    o = oracle.pc_octupole(x, np.array([0, 0, 0, 4.0], np.float32), T)
    Tx = float(np.float32(T[0]))
    assert o[3] == pytest.approx(-Tx * (5 * c ** 3 - 3 * c) / 2 / R ** 4, rel=1e-12, abs=1e-22)
    if c == 1.0:                                                   # on the axis: a_x = -d phi / dR = -4 T / R^5
        assert o[0] == pytest.approx(-4 * Tx / R ** 5, rel=1e-12) and abs(o[1]) < 1e-20
    if c == 0.0:                                                   # broadside: phi_3 = 0, a_x = -(3/2) T / R^5
        assert abs(o[3]) < 1e-20 and o[0] == pytest.approx(-1.5 * Tx / R ** 5, rel=1e-12)


@pytest.mark.parametrize("seed", range(6))
def test_residual_falls_one_power_faster_with_the_octupole(seed):
    d, m = _cluster(seed, eps=0.02)                                # eps / R = 1/40, 1/80: the next order is a few per cent
    M, Q, T = _moments(d, m)
    rng = np.random.default_rng(100 + seed)
    us = rng.normal(size=(16, 3)); us /= np.linalg.norm(us, axis=1, keepdims=True)
    res = {}
    for order in (2, 3):
        e = []
        for D in (0.8, 1.6):                                       # r.m.s. over 16 directions: one direction can sit on a
            diff = np.array([_expansion(D * u, M, Q, T, order) - _exact(D * u, d, m) for u in us])   # node of the next harmonic
            e.append((np.sqrt((diff[:, :3] ** 2).sum(1).mean()), np.sqrt((diff[:, 3] ** 2).mean())))
        res[order] = (np.log2(e[0][0] / e[1][0]), np.log2(e[0][1] / e[1][1]), e[0][0])
    # force residual ~ R^-(order+3), potential ~ R^-(order+2); the fp32 rounding of Q and T sits far below
    assert res[2][0] == pytest.approx(5.0, abs=0.35) and res[2][1] == pytest.approx(4.0, abs=0.35)
    assert res[3][0] == pytest.approx(6.0, abs=0.35) and res[3][1] == pytest.approx(5.0, abs=0.35)
    assert res[3][2] < 0.25 * res[2][2]


@pytest.mark.parametrize("seed", range(4))
def test_octupole_acceleration_is_minus_gradient(seed):
    d, m = _cluster(seed, eps=0.2)
    M, _, T = _moments(d, m)
    cm = np.array([0.1, -0.2, 0.05, M], np.float32)
    x = np.array([0.9, 0.4, -0.7]) * (1 + 0.1 * seed)
    a = oracle.pc_octupole(x, cm, T)[:3]
    h = 1e-5
    g = np.array([(oracle.pc_octupole(x + h * e, cm, T)[3] - oracle.pc_octupole(x - h * e, cm, T)[3]) / (2 * h) for e in np.eye(3)])
    assert np.allclose(a, -g, rtol=1e-7, atol=1e-9 * np.linalg.norm(a))


def test_inversion_symmetric_cluster_has_no_octupole():
    rng = np.random.default_rng(3)
    h = rng.normal(size=(8, 3)) * 0.05
    d = np.vstack([h, -h]); m = np.tile(rng.integers(1, 9, 8) / 16.0, 2)
    M, Q, T = _moments(d, m)
    assert np.abs(T).max() < 1e-18
    x = np.array([0.3, 0.5, -0.4])
    assert np.abs(oracle.pc_octupole(x, np.array([0, 0, 0, M], np.float32), T)).max() < 1e-12


def test_tree_third_moments_match_the_definition_and_the_parallel_axis_rule():
    w = workloads.make_config(1, n_override=3000)
    t = oracle.Tree(w.pos_mass, 63)
    nd = t.nodes(); m64 = t.moments64(); oc = t.octupoles()
    order = t.keys()[1].astype(np.int64)
    spm = w.pos_mass[order].astype(np.float64)
    rng = np.random.default_rng(0)
    internal = np.flatnonzero(nd["n_child"] > 0)
    for k in list(rng.choice(len(nd["begin"]), 40)) + [0] + list(rng.choice(internal, 20)):
        b, e = nd["begin"][k], nd["end"][k]
        dd = spm[b:e, :3] - m64["com"][k]; mm = spm[b:e, 3]
        T = np.einsum("i,ia,ib,ic->abc", mm, dd, dd, dd)
        want = np.array([T[a] for a in IDX])
        scale = (mm[:, None] * np.abs(dd) ** 3).sum() + 1e-300
        assert np.abs(oc["oct64"][k] - want).max() <= 1e-12 * scale
        assert np.array_equal(oc["oct32"][k], oc["oct64"][k].astype(np.float32))
    # parallel-axis rule (what the CUDA build does): T_parent = sum_k T_k + sym(s S_k) + M_k s s s, s = COM_k - COM_parent
    for k in rng.choice(internal, 20):
        tot = np.zeros((3, 3, 3))
        for c in range(nd["first_child"][k], nd["first_child"][k] + nd["n_child"][k]):
            b, e = nd["begin"][c], nd["end"][c]
            dd = spm[b:e, :3] - m64["com"][c]; mm = spm[b:e, 3]
            S = np.einsum("i,ia,ib->ab", mm, dd, dd)
            Tc = np.zeros((3, 3, 3))
            for q, (a1, a2, a3) in enumerate(IDX):
                for perm in {(a1, a2, a3), (a1, a3, a2), (a2, a1, a3), (a2, a3, a1), (a3, a1, a2), (a3, a2, a1)}:
                    Tc[perm] = oc["oct64"][c][q]
            s = m64["com"][c] - m64["com"][k]
            tot += Tc + np.einsum("a,bc->abc", s, S) + np.einsum("b,ac->abc", s, S) + np.einsum("c,ab->abc", s, S) \
                + m64["mass"][c] * np.einsum("a,b,c->abc", s, s, s)
        want = np.array([tot[a] for a in IDX])
        b, e = nd["begin"][k], nd["end"][k]
        scale = (spm[b:e, 3][:, None] * np.abs(spm[b:e, :3] - m64["com"][k]) ** 3).sum()
        assert np.abs(oc["oct64"][k] - want).max() <= 1e-11 * scale


def test_order3_tree_force_is_more_accurate_with_the_same_lists():
    w = workloads.make_config(1, n_override=8192)
    t = oracle.Tree(w.pos_mass, 63)
    theta = 0.6
    f2 = t.force(w.r_out, w.r_in, theta, order=2)
    f3 = t.force(w.r_out, w.r_in, theta, order=3)
    assert np.array_equal(f2["npp"], f3["npp"]) and np.array_equal(f2["npc"], f3["npc"])
    d = oracle.direct(w.pos_mass, w.r_out, w.r_in)
    n = np.linalg.norm(d["acc_reg"], axis=1)
    e2 = np.linalg.norm(f2["acc_pot"][:, :3] - d["acc_reg"], axis=1) / n
    e3 = np.linalg.norm(f3["acc_pot"][:, :3] - d["acc_reg"], axis=1) / n
    assert np.median(e3) < 0.5 * np.median(e2) and np.percentile(e3, 99) < 0.6 * np.percentile(e2, 99)
    p2 = np.abs(f2["acc_pot"][:, 3] - d["phi_reg"]) / np.abs(d["phi_reg"])
    p3 = np.abs(f3["acc_pot"][:, 3] - d["phi_reg"]) / np.abs(d["phi_reg"])
    assert np.median(p3) < 0.5 * np.median(p2)
    # theta -> 0: everything is particle-particle and the order does not matter
    g = np.arange(0, t.n_groups, 7)
    a = t.force(w.r_out, w.r_in, 1e-3, order=3, group_ids=g)["acc_pot"]
    b = t.force(w.r_out, w.r_in, 1e-3, order=2, group_ids=g)["acc_pot"]
    assert np.array_equal(np.nan_to_num(a), np.nan_to_num(b))
