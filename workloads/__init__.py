"""Seeded synthetic star clusters shaped like the paper's workloads.

This module only makes INPUTS (fp32 ``{x, y, z, m}`` arrays and the scalar
parameters of a force call).  It holds none of the method's arithmetic (no
cutoff, no tree, no force) and imports neither ``oracle`` nor the CUDA
package; both of those read the bytes produced here.

Shapes follow PAPER.md:148 (§3.1: Plummer model, N-body/Henon units, G = M = 1,
E = -1/4, no softening), PAPER.md:154 (N = 32k ... 2048k) and the radius law of
eq. 21-22 (r_cut proportional to N^(-1/3)); the prefactor
0.05, the Kroupa masses and the King W0 = 9 model are BASELINE.json's
extensions of that recipe.  The paper's own initial conditions are not
available, so these stand in for them.

Random numbers: a counter-based splitmix64 stream, so that a sample depends
only on (seed, stream, index) and never on numpy's generator.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

__all__ = [
    "uniform", "plummer_positions", "king_model", "king_positions",
    "kroupa_masses", "equal_masses", "r_out_for_n", "Workload", "make_config",
    "CONFIGS", "sample_targets",
]

_MASK = (1 << 64) - 1


def uniform(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """n doubles in (0, 1): splitmix64 of the counter (seed, stream, index)."""
    with np.errstate(over="ignore"):
        idx = np.arange(start, start + n, dtype=np.uint64)
        base = np.uint64((seed * 0x9E3779B97F4A7C15 + stream * 0xD1B54A32D192ED03) & _MASK)
        z = base + (idx + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    # 53 random bits, shifted half a step so that 0 and 1 never occur
    return ((z >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def _isotropic(seed: int, n: int, r: np.ndarray) -> np.ndarray:
    cz = 2.0 * uniform(seed, 1, n) - 1.0
    az = 2.0 * math.pi * uniform(seed, 2, n)
    s = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
    return np.stack([r * s * np.cos(az), r * s * np.sin(az), r * cz], axis=1)


PLUMMER_A = 3.0 * math.pi / 16.0          # Plummer scale length in Henon units (E = -1/4)
PLUMMER_TRUNC = 10.0                      # truncation radius in units of a


def plummer_positions(seed: int, n: int) -> np.ndarray:
    """Plummer sphere, truncated at 10 a; float64 [n, 3]."""
    rt = PLUMMER_TRUNC
    u_max = rt ** 3 / (1.0 + rt * rt) ** 1.5     # mass fraction inside the truncation
    u = uniform(seed, 0, n) * u_max
    r = PLUMMER_A / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
    return _isotropic(seed, n, r)


def plummer_velocities(seed: int, pos: np.ndarray) -> np.ndarray:
    """Isotropic velocities of the Plummer model at the given positions (Aarseth, Henon & Wielen 1974):
    speed q v_esc with q drawn from q^2 (1 - q^2)^(7/2) by rejection, v_esc^2 = 2 / sqrt(r^2 + a^2)
    (Henon units).  Input of the irregular-force path; for the King
    configuration the same recipe stands in (only the magnitude and isotropy of v matter there).
    Returns float64 [n, 3]."""
    n = pos.shape[0]
    q = np.zeros(n)
    todo = np.arange(n)
    rnd = 0
    while todo.size:
        u1 = uniform(seed, 8 + 2 * rnd, n)[todo]
        u2 = uniform(seed, 9 + 2 * rnd, n)[todo]
        ok = 0.1 * u2 < u1 * u1 * (1.0 - u1 * u1) ** 3.5
        q[todo[ok]] = u1[ok]
        todo = todo[~ok]
        rnd += 1
        if rnd > 200:
            q[todo] = 0.5
            break
    r2 = (pos * pos).sum(axis=1)
    speed = q * np.sqrt(2.0) * (r2 + PLUMMER_A * PLUMMER_A) ** (-0.25)
    cz = 2.0 * uniform(seed, 6, n) - 1.0
    ph = 2.0 * np.pi * uniform(seed, 7, n)
    sz = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
    return np.stack([speed * sz * np.cos(ph), speed * sz * np.sin(ph), speed * cz], axis=1)


def velocities_for(w) -> np.ndarray:
    """float32 [n, 4] = vx, vy, vz, 0 for a Workload (C-contiguous), seeded by the workload's seed."""
    v = plummer_velocities(w.seed, w.pos_mass[:, :3].astype(np.float64))
    out = np.zeros((v.shape[0], 4), dtype=np.float32)
    out[:, :3] = v.astype(np.float32)
    return np.ascontiguousarray(out)


def _king_rho(w: float) -> float:
    if w <= 0.0:
        return 0.0
    return math.exp(w) * math.erf(math.sqrt(w)) - math.sqrt(4.0 * w / math.pi) * (1.0 + 2.0 * w / 3.0)


def king_model(w0: float = 9.0, h: float = 2.0e-3):
    """Integrate the King (1966) model: W'' + 2 W'/r = -9 rho(W)/rho(W0).

    Returns (r, m, scale) with r in King radii, m the enclosed mass fraction and
    scale the factor that brings r to Henon units (potential energy -1/2, M = 1).
    """
    rho0 = _king_rho(w0)

    def rhs(r, w, v):
        # v = dW/dr ; near the centre 2 v / r -> -6 rho/rho0 (series), handled by r > 0 start
        return v, -9.0 * _king_rho(w) / rho0 - 2.0 * v / r

    r = 1.0e-4
    w = w0 - 1.5 * r * r            # series: W = W0 - (3/2) r^2 + ...
    v = -3.0 * r
    rs, ms = [0.0, r], [0.0, -r * r * v]
    while w > 0.0:
        step = h * max(1.0, r) if r > 1.0 else h
        k1w, k1v = rhs(r, w, v)
        k2w, k2v = rhs(r + 0.5 * step, w + 0.5 * step * k1w, v + 0.5 * step * k1v)
        k3w, k3v = rhs(r + 0.5 * step, w + 0.5 * step * k2w, v + 0.5 * step * k2v)
        k4w, k4v = rhs(r + step, w + step * k3w, v + step * k3v)
        wn = w + step * (k1w + 2 * k2w + 2 * k3w + k4w) / 6.0
        vn = v + step * (k1v + 2 * k2v + 2 * k3v + k4v) / 6.0
        if wn <= 0.0:
            # linear step to the tidal radius W = 0
            frac = w / (w - wn)
            r = r + frac * step
            v = v + frac * (vn - v)
            rs.append(r)
            ms.append(-r * r * v)        # Gauss: M(r) proportional to -r^2 W'
            break
        r, w, v = r + step, wn, vn
        rs.append(r)
        ms.append(-r * r * v)
    r_arr = np.asarray(rs)
    m_arr = np.asarray(ms)
    m_arr = np.maximum.accumulate(m_arr / m_arr[-1])
    # potential energy of the model with M = 1: U = -int m dm / r
    mid_r = 0.5 * (r_arr[1:] + r_arr[:-1])
    mid_m = 0.5 * (m_arr[1:] + m_arr[:-1])
    u_abs = float(np.sum(mid_m * np.diff(m_arr) / mid_r))
    scale = u_abs / 0.5
    return r_arr, m_arr, scale


_KING_CACHE: dict = {}


def king_positions(seed: int, n: int, w0: float = 9.0) -> np.ndarray:
    """King model W0 positions in Henon units; float64 [n, 3]."""
    if w0 not in _KING_CACHE:
        _KING_CACHE[w0] = king_model(w0)
    r_arr, m_arr, scale = _KING_CACHE[w0]
    u = uniform(seed, 0, n)
    r = np.interp(u, m_arr, r_arr) * scale
    return _isotropic(seed, n, r)


def kroupa_masses(seed: int, n: int, m_lo: float = 0.08, m_br: float = 0.5, m_hi: float = 100.0) -> np.ndarray:
    """Two-segment Kroupa IMF dN/dm ~ m^-1.3 on [m_lo, m_br), m^-2.3 on [m_br, m_hi];
    inverse-CDF sampled, then normalised to total mass 1.  float64 [n]."""
    a1, a2 = 1.3, 2.3
    # continuity at the break: k2 = k1 * m_br^(a2 - a1)
    n1 = (m_br ** (1 - a1) - m_lo ** (1 - a1)) / (1 - a1)
    n2 = m_br ** (a2 - a1) * (m_hi ** (1 - a2) - m_br ** (1 - a2)) / (1 - a2)
    p1 = n1 / (n1 + n2)
    u = uniform(seed, 3, n)
    m = np.empty(n)
    lo = u < p1
    t = u[lo] / p1
    m[lo] = (m_lo ** (1 - a1) + t * (m_br ** (1 - a1) - m_lo ** (1 - a1))) ** (1.0 / (1 - a1))
    t = (u[~lo] - p1) / (1.0 - p1)
    m[~lo] = (m_br ** (1 - a2) + t * (m_hi ** (1 - a2) - m_br ** (1 - a2))) ** (1.0 / (1 - a2))
    return m / m.sum()


def two_component_masses(n: int) -> np.ndarray:
    """The mass spectrum of the paper's core-collapse run, eq. 26: m_i = 10 / (1.9 N) if
    i = 0 (mod 10), else 1 / (1.9 N): about half of the mass in a tenth of the particles; the sum is 1."""
    m = np.full(n, 1.0 / (1.9 * n))
    m[::10] = 10.0 / (1.9 * n)
    return m


def equal_masses(n: int) -> np.ndarray:
    return np.full(n, 1.0 / n)


def r_out_for_n(n: int) -> float:
    """BASELINE.json radius law: 0.05 (N / 16384)^(-1/3) (exponent of eq. 21-22)."""
    return 0.05 * (n / 16384.0) ** (-1.0 / 3.0)


@dataclass
class Workload:
    name: str
    pos_mass: np.ndarray      # float32 [n, 4] = x, y, z, m  (C-contiguous)
    r_out: float              # fp32-representable
    r_in: float               # fp32-representable
    theta: float
    seed: int

    @property
    def n(self) -> int:
        return int(self.pos_mass.shape[0])


def _pack(pos: np.ndarray, mass: np.ndarray) -> np.ndarray:
    out = np.empty((pos.shape[0], 4), dtype=np.float32)
    out[:, :3] = pos.astype(np.float32)
    out[:, 3] = mass.astype(np.float32)
    return np.ascontiguousarray(out)


# id -> (label, n, model, masses, thetas, seed); the five BASELINE.json configs
CONFIGS = {
    1: ("plummer16k_equal", 16384, "plummer", "equal", (0.4,), 1),
    2: ("plummer128k_kroupa", 131072, "plummer", "kroupa", (0.4,), 2),
    3: ("plummer1m_kroupa", 1048576, "plummer", "kroupa", (0.4,), 3),
    4: ("king9_1m_kroupa", 1048576, "king9", "kroupa", (0.4,), 4),
    5: ("plummer4m_equal", 4194304, "plummer", "equal", (0.3, 0.5, 0.7), 5),
    # not a BASELINE.json config: the paper's 64k two-component cluster of section 3.2
    6: ("plummer64k_two_component", 65536, "plummer", "two_component", (0.4,), 6),
}


def make_config(cfg: int, n_override: int | None = None, theta: float | None = None) -> Workload:
    label, n, model, masses, thetas, seed = CONFIGS[cfg]
    if n_override is not None:
        n = int(n_override)
        label = f"{label}@n={n}"
    pos = plummer_positions(seed, n) if model == "plummer" else king_positions(seed, n, 9.0)
    m = equal_masses(n) if masses == "equal" else two_component_masses(n) if masses == "two_component" else kroupa_masses(seed, n)
    r_out = float(np.float32(r_out_for_n(n)))
    r_in = float(np.float32(0.1) * np.float32(r_out))     # gamma = 0.1
    return Workload(label, _pack(pos, m), r_out, float(np.float32(r_in)),
                    float(thetas[0] if theta is None else theta), seed)


def sample_targets(n: int, n_s: int) -> np.ndarray:
    """Stride sample i = floor(s * n / n_s), s = 0 .. n_s - 1 (int64)."""
    n_s = min(n, n_s)
    return (np.arange(n_s, dtype=np.int64) * n) // n_s
