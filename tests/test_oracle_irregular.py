"""Pins of the oracle's irregular force and jerk (eq. 1, 2, 5, 7).

The paper's eq. 2 / eq. 7 are garbled (reading R2): the oracle takes Fdot_I to be the exact
time derivative of eq. 1.  That reading is pinned here by what the mathematics fixes:
finite differences of F_I along the motion, the Newtonian jerk inside r_in, zero beyond r_out, the
radial and tangential special cases of the transition zone, and consistency with the (separately
pinned) direct split sums."""
import numpy as np

import oracle
import workloads

R_OUT, R_IN = 0.25, 0.025


def _dyadic_cluster(n=160, seed=11):
    """Positions on a 2^-10 grid inside a box of edge 0.5, velocities on a 2^-4 grid: x + k h v is exactly
    representable in fp32 for h = 2^-12, |k| <= 2, so the finite differences below see no input rounding."""
    u = workloads.uniform(seed, 0, 3 * n).reshape(n, 3)
    pos = np.round(u * 0.5 * 1024) / 1024
    v = np.round((workloads.uniform(seed, 1, 3 * n).reshape(n, 3) * 2 - 1) * 16) / 16
    m = 0.5 + workloads.uniform(seed, 2, n)
    pm = np.zeros((n, 4), np.float32); pm[:, :3] = pos; pm[:, 3] = m / m.sum()
    vel = np.zeros((n, 4), np.float32); vel[:, :3] = v
    return pm, vel


def test_jerk_is_the_time_derivative_of_eq1():
    pm, vel = _dyadic_cluster()
    h = 2.0 ** -12

    def acc_at(k):
        p = pm.copy()
        p[:, :3] = (pm[:, :3].astype(np.float64) + k * h * vel[:, :3].astype(np.float64)).astype(np.float32)
        assert np.array_equal(p[:, :3].astype(np.float64), pm[:, :3].astype(np.float64) + k * h * vel[:, :3])
        return oracle.irregular(p, vel, R_OUT, R_IN)["acc_irr"]

    r = oracle.irregular(pm, vel, R_OUT, R_IN)
    assert r["coincident"] == 0
    # fourth-order central difference: error O((h v / r)^4)
    fd = (8.0 * (acc_at(1) - acc_at(-1)) - (acc_at(2) - acc_at(-2))) / (12.0 * h)
    err = np.linalg.norm(fd - r["jerk_irr"], axis=1)
    rel = err / np.maximum(r["abs_jerk"], 1e-300)
    # the closest pairs (r ~ 3e-3) limit the difference quotient to (h v / r)^4 ~ 1e-4; the bulk is far better
    assert rel.max() <= 3e-4 and np.median(rel) <= 1e-6, (rel.max(), np.median(rel))
    # the pairs do sample all three zones
    d = np.linalg.norm(pm[None, :, :3].astype(np.float64) - pm[:, None, :3], axis=2)
    iu = np.triu_indices(pm.shape[0], 1)
    assert (d[iu] < R_IN).sum() > 3 and ((d[iu] > R_IN) & (d[iu] < R_OUT)).sum() > 100 and (d[iu] > R_OUT).sum() > 100


def _pair(d, v, m=0.25):
    pm = np.zeros((2, 4), np.float32); vel = np.zeros((2, 4), np.float32)
    pm[1, :3] = d; pm[:, 3] = m; vel[1, :3] = v
    r = oracle.irregular(pm, vel, R_OUT, R_IN, targets=[0])
    return r["acc_irr"][0], r["jerk_irr"][0], r["phi_irr"][0]


def test_newtonian_jerk_inside_r_in():
    d = np.array([0.0078125, -0.015625, 0.00390625]); v = np.array([0.5, 0.25, -1.0]); m = 0.25
    r = np.linalg.norm(d)
    assert r < R_IN
    a, j, phi = _pair(d, v, m)
    assert np.allclose(a, m * d / r ** 3, rtol=1e-14)
    assert np.allclose(j, m * (v / r ** 3 - 3 * d.dot(v) * d / r ** 5), rtol=1e-13)     # textbook Hermite jerk
    # phi_I = -m/r - m psi(r_in): the unsplit pair potential minus the (constant) regular part
    assert np.isclose(phi, m * (-1 / r - oracle.psi(R_IN, R_OUT, R_IN)), rtol=1e-14)


def test_nothing_beyond_r_out():
    a, j, phi = _pair(np.array([0.25, 0.0, 0.0]), np.array([1.0, 2.0, 3.0]))
    assert np.all(a == 0) and np.all(j == 0) and phi == 0
    a, j, phi = _pair(np.array([0.2, 0.2, 0.0]), np.array([1.0, 2.0, 3.0]))
    assert np.all(a == 0) and np.all(j == 0) and phi == 0


def test_transition_zone_radial_and_tangential_motion():
    m = 0.25
    for r in (0.0625, 0.125, 0.1875):
        x = (r - R_IN) / (R_OUT - R_IN)
        K, dW = 1 - oracle.W(x), oracle.dW(x)
        d = np.array([r, 0.0, 0.0])
        # tangential: r.v = 0, so K does not change: jerk = m K v / r^3
        v = np.array([0.0, 0.5, -0.25])
        a, j, _ = _pair(d, v, m)
        assert np.allclose(a, [m * K / r ** 2, 0, 0], rtol=1e-13)
        assert np.allclose(j, m * K * v / r ** 3, rtol=1e-13)
        # radial: a = m K(x(r)) / r^2, so jerk = m rdot d/dr [K / r^2] = m rdot ( -W'(x) / (D r^2) - 2 K / r^3 )
        rdot = 0.75
        a, j, _ = _pair(d, np.array([rdot, 0.0, 0.0]), m)
        assert np.allclose(j, [m * rdot * (-dW / ((R_OUT - R_IN) * r ** 2) - 2 * K / r ** 3), 0, 0], rtol=1e-12)
    # K' of eq. 7 uses the polynomial -140x^6 + 420x^5 - 420x^4 + 140x^3 = 140 x^3 (1-x)^3 = dW/dx
    for x in (0.1, 0.35, 0.5, 0.9):
        assert np.isclose(oracle.dW(x), 140 * x ** 3 * (1 - x) ** 3, rtol=1e-13)
        assert np.isclose(oracle.dW(x), (oracle.W(x + 1e-6) - oracle.W(x - 1e-6)) / 2e-6, rtol=1e-8)


def test_consistent_with_the_direct_split_sums():
    w = workloads.make_config(1, n_override=1500)
    vel = workloads.velocities_for(w)
    r = oracle.irregular(w.pos_mass, vel, w.r_out, w.r_in)
    d = oracle.direct(w.pos_mass, w.r_out, w.r_in)
    assert np.abs(r["acc_irr"] - d["acc_irr"]).max() <= 1e-13 * np.abs(d["acc_irr"]).max()
    assert np.abs(r["phi_irr"] - (d["phi_newt"] - d["phi_reg"])).max() <= 1e-12 * np.abs(d["phi_newt"]).max()
    # momentum: sum_i m_i Fdot_I,i = 0 (pair antisymmetry of eq. 2 under i <-> j)
    mj = w.pos_mass[:, 3].astype(np.float64)
    assert np.abs((mj[:, None] * r["jerk_irr"]).sum(axis=0)).max() <= 1e-12 * (mj * r["abs_jerk"]).sum()


def test_velocity_generator_is_virialised():
    w = workloads.make_config(1)
    v = workloads.velocities_for(w)[:, :3].astype(np.float64)
    # Plummer sphere in Henon units: <v^2> = 2 T / M = 1/2 (E = -1/4); isotropic
    assert abs((v * v).sum(axis=1).mean() - 0.5) < 0.02
    assert np.abs(v.mean(axis=0)).max() < 0.02


def test_candidate_rows_give_the_same_sums():
    """oracle.irregular(candidates=grid rows at 1.01 r_out) == the scan over every j (which the pins above fix):
    identical bits, since the pairs inside r_out are visited in the same (ascending j) order."""
    w = workloads.make_config(4, n_override=6000)
    vel = workloads.velocities_for(w)
    r_out, r_in = 0.05, 0.005
    full = oracle.irregular(w.pos_mass, vel, r_out, r_in)
    cand = oracle.neighbours_grid(w.pos_mass, 1.01 * r_out)
    part = oracle.irregular(w.pos_mass, vel, r_out, r_in, candidates=cand)
    for k in ("acc_irr", "jerk_irr", "phi_irr", "abs_jerk", "abs_newt"):
        assert np.array_equal(full[k], part[k]), k
    assert full["coincident"] == part["coincident"]
    tg = workloads.sample_targets(w.n, 500)
    cand_t = oracle.neighbours_grid(w.pos_mass, 1.01 * r_out, targets=tg)
    sub = oracle.irregular(w.pos_mass, vel, r_out, r_in, targets=tg, candidates=cand_t)
    assert np.array_equal(sub["jerk_irr"], full["jerk_irr"][tg])
