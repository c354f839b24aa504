"""The seeded input generators: shape statistics of the synthetic stand-ins (DESIGN.md input recipe)."""
import math

import numpy as np
import pytest

import workloads


def test_uniform_is_counter_based_and_uniform():
    a = workloads.uniform(3, 0, 1000)
    b = workloads.uniform(3, 0, 500, start=500)
    assert np.array_equal(a[500:], b)
    assert not np.array_equal(a, workloads.uniform(4, 0, 1000)) and not np.array_equal(a, workloads.uniform(3, 1, 1000))
    u = workloads.uniform(11, 2, 200000)
    assert 0.0 < u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 3e-3 and abs(u.var() - 1 / 12) < 2e-3


def test_plummer_shape():
    w = workloads.make_config(1)
    assert w.pos_mass.dtype == np.float32 and w.pos_mass.shape == (16384, 4)
    assert w.r_out == pytest.approx(0.05) and w.r_in == pytest.approx(0.005) and w.theta == 0.4
    r = np.linalg.norm(w.pos_mass[:, :3].astype(np.float64), axis=1)
    a = workloads.PLUMMER_A
    assert r.max() <= 10 * a * (1 + 1e-6)
    # half-mass radius of the truncated Plummer model: m(r)/m_t = 1/2
    mt = 1000 / 101 ** 1.5
    rh = a / math.sqrt((0.5 * mt) ** (-2 / 3) - 1)
    assert np.median(r) == pytest.approx(rh, rel=0.03)
    assert np.all(w.pos_mass[:, 3] == np.float32(1 / 16384))
    assert np.abs(w.pos_mass[:, :3].mean(0)).max() < 0.05
    assert np.array_equal(w.pos_mass, workloads.make_config(1).pos_mass)        # deterministic


def test_radius_law():
    assert workloads.r_out_for_n(16384) == 0.05
    assert workloads.r_out_for_n(131072) == pytest.approx(0.025) and workloads.r_out_for_n(1048576) == pytest.approx(0.0125)
    assert workloads.r_out_for_n(4194304) == pytest.approx(0.05 / 256 ** (1 / 3))


def test_kroupa_masses():
    m = workloads.kroupa_masses(2, 200000)
    assert m.sum() == pytest.approx(1.0, rel=1e-12)
    ratio = m.max() / m.min()
    assert 100 < ratio <= 100 / 0.08 * (1 + 1e-9)
    msun = m / m.min() * 0.08                                  # approximately in solar masses
    frac_low = (msun < 0.5).mean()
    # number fraction below the break from the two power laws
    n1 = (0.5 ** -0.3 - 0.08 ** -0.3) / -0.3
    n2 = 0.5 * (100 ** -1.3 - 0.5 ** -1.3) / -1.3
    assert frac_low == pytest.approx(n1 / (n1 + n2), abs=0.01)
    assert 100 < m.max() / m.mean() < 300


def test_king_w0_9_model():
    r, m, scale = workloads.king_model(9.0)
    assert math.log10(r[-1]) == pytest.approx(2.12, abs=0.01)          # concentration of a W0 = 9 King model
    assert m[0] == 0.0 and m[-1] == 1.0 and np.all(np.diff(m) >= 0)
    pos = workloads.king_positions(4, 100000)
    rr = np.linalg.norm(pos, axis=1)
    assert rr.max() <= r[-1] * scale * (1 + 1e-9)
    # virial scaling: potential energy -1/2 with M = 1 => <1/r>-weighted check through the tabulated model
    mid_r = 0.5 * (r[1:] + r[:-1]) * scale
    mid_m = 0.5 * (m[1:] + m[:-1])
    assert np.sum(mid_m * np.diff(m) / mid_r) == pytest.approx(0.5, rel=1e-9)
    assert np.median(rr) == pytest.approx(np.interp(0.5, m, r) * scale, rel=0.02)


def test_sample_targets():
    s = workloads.sample_targets(1000, 10)
    assert list(s) == list(range(0, 1000, 100)) and s.dtype == np.int64
    assert len(workloads.sample_targets(5, 10)) == 5


def test_two_component_spectrum_eq26():
    """eq. 26: every tenth particle ten times heavier, total mass 1, half the mass in 10 %."""
    w = workloads.make_config(6)
    m = w.pos_mass[:, 3].astype(np.float64)
    assert w.n == 65536 and abs(m.sum() - 1.0) < 1e-4           # exactly 1 only when 10 divides N
    assert np.allclose(m[::10] / m[1], 10.0, rtol=1e-6) and np.allclose(m[1:10], m[1], rtol=1e-7)
    assert abs(m[::10].sum() - 10.0 / 19.0) < 1e-3               # 'approximately half of the system's mass'
