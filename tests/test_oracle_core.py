"""Pins of the oracle's sampled 6-nearest-neighbour densities and core quantities (
PAPER.md:134, :245; Casertano & Hut 1985 as cited by the paper; readings R17-R19)."""
import numpy as np
from scipy.special import beta

import oracle
import workloads


def _points(n, seed):
    u = workloads.uniform(seed, 0, 3 * n).reshape(n, 3)
    pm = np.zeros((n, 4), np.float32); pm[:, :3] = u; pm[:, 3] = 1.0 / n
    return pm


def test_knn_against_sorted_distances():
    pm = _points(3000, 21)
    sample = np.arange(0, 3000, 7, dtype=np.int32)
    r = oracle.knn_density(pm, sample, 6)
    pos = pm[:, :3].astype(np.float64)
    for s, i in enumerate(sample):
        d2 = ((pos - pos[i]) ** 2).sum(axis=1); d2[i] = np.inf
        o = np.argsort(d2, kind="stable")
        if d2[o[6]] - d2[o[5]] > 1e-6 * d2[o[5]] and np.all(np.diff(d2[o[:6]]) > 1e-6 * d2[o[5]]):   # no near-tie
            assert np.array_equal(r["nbr"][s], o[:6])
        assert abs(r["d2k"][s] / d2[o[5]] - 1) < 1e-6
        m5 = pm[o[:5], 3].astype(np.float64).sum()
        assert np.isclose(r["rho"][s], m5 / (4 * np.pi / 3 * float(r["d2k"][s]) ** 1.5), rtol=1e-12)


def test_ties_go_to_the_smaller_index():
    # a cubic lattice: the 6 face neighbours are all at the same distance, then 12 edge neighbours
    g = np.arange(5, dtype=np.float32)
    x, y, z = np.meshgrid(g, g, g, indexing="ij")
    pm = np.zeros((125, 4), np.float32); pm[:, 0] = x.ravel(); pm[:, 1] = y.ravel(); pm[:, 2] = z.ravel(); pm[:, 3] = 1
    c = 2 * 25 + 2 * 5 + 2                                     # the centre
    r = oracle.knn_density(pm, np.array([c], np.int32), 6)
    assert sorted(r["nbr"][0]) == sorted([c - 25, c + 25, c - 5, c + 5, c - 1, c + 1]) and r["d2k"][0] == 1.0
    assert np.array_equal(r["nbr"][0], np.sort(r["nbr"][0]))    # equal d2: ascending index
    r4 = oracle.knn_density(pm, np.array([c], np.int32), 4)     # only 4 of the 6 equidistant: the 4 smallest ids
    assert np.array_equal(r4["nbr"][0], np.sort([c - 25, c + 25, c - 5, c + 5, c - 1, c + 1])[:4])
    assert np.isclose(r["rho"][0], 5.0 / (4 * np.pi / 3))       # (K-1) m / V(r_K), r_K = 1


def test_uniform_density_is_recovered():
    n = 40000
    pm = _points(n, 22)
    inner = np.flatnonzero(np.all(np.abs(pm[:, :3] - 0.5) < 0.35, axis=1)).astype(np.int32)[:3000]
    r = oracle.knn_density(pm, inner, 6)
    # Casertano & Hut: rho = (K-1) m / V(r_K) is unbiased; relative scatter 1/sqrt(K-2) = 0.5 per particle
    assert abs(r["rho"].mean() - 1.0) < 0.04


def test_core_quantities_hand_case():
    pm = np.zeros((4, 4), np.float32); pm[1, 0] = 1.0; pm[:, 3] = 0.25
    q = oracle.core_quantities(pm, np.array([0, 1], np.int32), np.array([1.0, 3.0]))
    assert np.allclose(q["center"], [0.75, 0, 0]) and np.isclose(q["rho_core"], 2.5)
    assert np.isclose(q["r_core"], np.sqrt((1 * 0.5625 + 9 * 0.0625) / 10))
    assert q["n_core"] == 1 * 4 / 2                               # one of the two samples inside, scaled by N / ns


def test_plummer_core_against_the_analytic_moments():
    """Samples are drawn with probability ~ rho, so sum rho^2 / sum rho -> int rho^3 / int rho^2 and
    R_core^2 -> int rho^3 r^2 / int rho^3; for rho ~ (1 + r^2/a^2)^(-5/2):
    int_0^inf x^(2k) (1+x^2)^(-p) dx = B(k + 1/2, p - k - 1/2) / 2.  The estimator's own scatter (rho ~ 1/V,
    K = 6) inflates <rho^2> by about (K-1)/(K-2) = 1.25."""
    w = workloads.make_config(1)
    n = w.n
    ns = int(min(n, np.sqrt(5000.0 * n)))
    sample = workloads.sample_targets(n, ns).astype(np.int32)
    r = oracle.knn_density(w.pos_mass, sample, 6)
    q = oracle.core_quantities(w.pos_mass, sample, r["rho"])
    a = workloads.PLUMMER_A
    mt = 1.0 / (10.0 ** 3 / (1 + 10.0 ** 2) ** 1.5)               # masses renormalised after the truncation at 10 a
    rho0 = 3.0 / (4 * np.pi * a ** 3) * mt
    rho_core_th = rho0 * beta(1.5, 6.0) / beta(1.5, 3.5)          # int rho^3 / int rho^2
    r_core_th = a * np.sqrt(beta(2.5, 5.0) / beta(1.5, 6.0))      # sqrt(int rho^3 r^2 / int rho^3)
    assert np.linalg.norm(q["center"]) < 0.05
    assert 0.9 < q["rho_core"] / rho_core_th < 1.6
    assert 0.8 < q["r_core"] / r_core_th < 1.15
    mass_inside = ((w.pos_mass[:, :3].astype(np.float64) - q["center"]) ** 2).sum(axis=1) < q["r_core"] ** 2
    assert abs(q["n_core"] / mass_inside.sum() - 1) < 0.1         # the scaled sample count estimates the true count
