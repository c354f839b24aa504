"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes binding of the plain fp64 CPU statement of the P3T regular-force path
(oracle/p3t_oracle_*.c, written from /root/reference/PAPER.md).  Only tests/,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this package; the product (paper_2110_11658_b200) never does,
and this package never imports the product.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SOURCES = ["p3t_oracle_direct.c", "p3t_oracle_grid.c", "p3t_oracle_tree.c", "p3t_oracle_walk.c"]
_HEADERS = ["p3t_oracle.h", "p3t_oracle_tree_priv.h"]
_LIB = _HERE / "libp3t_oracle.so"
NLEAF_DEFAULT = 16
NCRIT_DEFAULT = 64


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (no fast-math, no FMA contraction)."""
    srcs = [_HERE / s for s in _SOURCES]
    deps = srcs + [_HERE / h for h in _HEADERS]
    if not force and _LIB.exists() and all(_LIB.stat().st_mtime >= d.stat().st_mtime for d in deps):
        return _LIB
    tmp = _LIB.with_suffix(f".{os.getpid()}.tmp.so")
    cmd = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
           "-o", str(tmp)] + [str(s) for s in srcs] + ["-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        d, i64, f32 = C.c_double, C.c_int64, C.c_float
        vp = C.c_void_p
        _lib.p3t_o_W.restype = d; _lib.p3t_o_W.argtypes = [d]
        _lib.p3t_o_dW.restype = d; _lib.p3t_o_dW.argtypes = [d]
        _lib.p3t_o_psi.restype = d; _lib.p3t_o_psi.argtypes = [d, d, d]
        _lib.p3t_o_direct.restype = i64
        _lib.p3t_o_direct.argtypes = [i64, vp, d, d, i64, vp, vp, vp, vp, vp]
        _lib.p3t_o_irregular.restype = i64
        _lib.p3t_o_irregular.argtypes = [i64, vp, vp, d, d, i64, vp, vp, vp, vp, vp, vp]
        _lib.p3t_o_irregular_cand.restype = i64
        _lib.p3t_o_irregular_cand.argtypes = [i64, vp, vp, d, d, i64, vp, vp, vp, vp, vp, vp, vp, vp]
        _lib.p3t_o_knn_density.restype = None
        _lib.p3t_o_knn_density.argtypes = [i64, vp, i64, vp, C.c_int, vp, vp, vp]
        _lib.p3t_o_core_quantities.restype = None
        _lib.p3t_o_core_quantities.argtypes = [i64, vp, i64, vp, vp, vp]
        _lib.p3t_o_neighbours.restype = i64
        _lib.p3t_o_neighbours.argtypes = [i64, vp, f32, C.c_int, i64, vp, vp, vp]
        _lib.p3t_o_neighbours_grid.restype = i64
        _lib.p3t_o_neighbours_grid.argtypes = [i64, vp, f32, i64, vp, vp, vp]
        _lib.p3t_o_tree_build.restype = vp
        _lib.p3t_o_tree_build.argtypes = [i64, vp, C.c_int, C.c_int, C.c_int]
        _lib.p3t_o_tree_free.restype = None; _lib.p3t_o_tree_free.argtypes = [vp]
        for name, nargs in [("sizes", 2), ("cube", 3), ("keys", 3), ("nodes", 6), ("moments", 6),
                            ("moments64", 4), ("groups", 5)]:
            f = getattr(_lib, "p3t_o_tree_" + name)
            f.restype = None; f.argtypes = [vp] * nargs
        _lib.p3t_o_tree_force.restype = None
        _lib.p3t_o_tree_force.argtypes = [vp, f32, f32, f32, C.c_int, i64, vp, vp, vp, vp, vp]
        _lib.p3t_o_tree_force_buffered.restype = None
        _lib.p3t_o_tree_force_buffered.argtypes = [vp, f32, f32, f32, f32, C.c_int, i64, vp, vp, vp, vp, vp]
        _lib.p3t_o_tree_force_order.restype = None
        _lib.p3t_o_tree_force_order.argtypes = [vp, C.c_int, f32, f32, f32, f32, C.c_int, i64, vp, vp, vp, vp, vp]
        _lib.p3t_o_pc_term.restype = None; _lib.p3t_o_pc_term.argtypes = [vp, vp, vp, vp]
        _lib.p3t_o_pc_octupole.restype = None; _lib.p3t_o_pc_octupole.argtypes = [vp, vp, vp, vp]
        _lib.p3t_o_tree_octupoles.restype = None; _lib.p3t_o_tree_octupoles.argtypes = [vp, vp, vp]
        _lib.p3t_o_open_test.restype = C.c_int
        _lib.p3t_o_open_test.argtypes = [vp, vp, vp, vp, vp, f32, f32, f32, f32]
        _lib.p3t_o_interleave.restype = C.c_uint64
        _lib.p3t_o_interleave.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, C.c_int]
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _pm(pos_mass) -> np.ndarray:
    a = np.ascontiguousarray(pos_mass, dtype=np.float32)
    assert a.ndim == 2 and a.shape[1] == 4
    return a


def omp_threads() -> int:
    """Threads the oracle's OpenMP loops use (OMP_NUM_THREADS or the core count)."""
    v = os.environ.get("OMP_NUM_THREADS")
    if v:
        return int(v.split(",")[0])
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def W(x: float) -> float:
    return lib().p3t_o_W(float(x))


def dW(x: float) -> float:
    return lib().p3t_o_dW(float(x))


def K(x: float) -> float:
    """Cutoff function of eq. 6."""
    return 1.0 - W(x)


def psi(r: float, r_out: float, r_in: float) -> float:
    return lib().p3t_o_psi(float(r), float(r_out), float(r_in))


def direct(pos_mass, r_out: float, r_in: float, targets=None):
    """Direct split sums: dict(acc_reg [nt,3], phi_reg, acc_irr, phi_newt, coincident)."""
    pm = _pm(pos_mass)
    n = pm.shape[0]
    tg = None if targets is None else np.ascontiguousarray(targets, dtype=np.int64)
    nt = n if tg is None else tg.shape[0]
    ar = np.zeros((nt, 3)); ai = np.zeros((nt, 3)); pr = np.zeros(nt); pn = np.zeros(nt)
    co = lib().p3t_o_direct(n, _p(pm), float(r_out), float(r_in), nt, _p(tg), _p(ar), _p(pr), _p(ai), _p(pn))
    return dict(acc_reg=ar, phi_reg=pr, acc_irr=ai, phi_newt=pn, coincident=int(co))


def irregular(pos_mass, vel, r_out: float, r_in: float, targets=None, candidates=None):
    """Irregular acceleration, jerk, potential over the neighbour sphere (eq. 1, 2, 5, 7); fp64 arrays.
    candidates = (offsets, indices): CSR rows over the targets that contain every target's neighbour sphere
    (e.g. neighbours_grid at a slightly larger radius); None = every j is tested."""
    pm = _pm(pos_mass); v = _pm(vel)
    t = None if targets is None else np.ascontiguousarray(targets, dtype=np.int64)
    nt = pm.shape[0] if t is None else t.shape[0]
    acc = np.zeros((nt, 3)); jerk = np.zeros((nt, 3)); phi = np.zeros(nt); ab = np.zeros(nt); an = np.zeros(nt)
    co = ci = None
    if candidates is not None:
        co = np.ascontiguousarray(candidates[0], dtype=np.int64); ci = np.ascontiguousarray(candidates[1], dtype=np.int32)
        assert co.shape[0] == nt + 1
    coinc = lib().p3t_o_irregular_cand(pm.shape[0], _p(pm), _p(v), float(r_out), float(r_in), nt, _p(t), _p(co), _p(ci),
                                       _p(acc), _p(jerk), _p(phi), _p(ab), _p(an))
    return dict(acc_irr=acc, jerk_irr=jerk, phi_irr=phi, abs_jerk=ab, abs_newt=an, coincident=int(coinc))


def knn_density(pos_mass, sample, k: int = 6):
    """K nearest neighbours of the sample particles (brute force, order (fp32 d2, index)) and their
    Casertano-Hut densities: dict(nbr [ns,k] int32, d2k [ns] float32, rho [ns] float64)."""
    pm = _pm(pos_mass); sm = np.ascontiguousarray(sample, dtype=np.int32)
    ns = sm.shape[0]
    nbr = np.zeros((ns, k), np.int32); d2k = np.zeros(ns, np.float32); rho = np.zeros(ns)
    lib().p3t_o_knn_density(pm.shape[0], _p(pm), ns, _p(sm), int(k), _p(nbr), _p(d2k), _p(rho))
    return dict(nbr=nbr, d2k=d2k, rho=rho)


def core_quantities(pos_mass, sample, rho):
    """dict(center [3], r_core, rho_core, n_core) from the sample densities (NBODY6 conventions)."""
    pm = _pm(pos_mass); sm = np.ascontiguousarray(sample, dtype=np.int32)
    r = np.ascontiguousarray(rho, dtype=np.float64); out = np.zeros(6)
    lib().p3t_o_core_quantities(pm.shape[0], _p(pm), sm.shape[0], _p(sm), _p(r), _p(out))
    return dict(center=out[:3].copy(), r_core=float(out[3]), rho_core=float(out[4]), n_core=float(out[5]))


def neighbours(pos_mass, r_out: float, targets=None, fp32_predicate: bool = True):
    """Brute-force neighbour rows: (offsets int64 [nt+1], indices int32)."""
    pm = _pm(pos_mass)
    n = pm.shape[0]
    tg = None if targets is None else np.ascontiguousarray(targets, dtype=np.int64)
    nt = n if tg is None else tg.shape[0]
    counts = np.zeros(nt, dtype=np.int64)
    total = lib().p3t_o_neighbours(n, _p(pm), float(np.float32(r_out)), int(fp32_predicate), nt, _p(tg), _p(counts), None)
    idx = np.zeros(max(int(total), 1), dtype=np.int32)
    lib().p3t_o_neighbours(n, _p(pm), float(np.float32(r_out)), int(fp32_predicate), nt, _p(tg), _p(counts), _p(idx))
    off = np.zeros(nt + 1, dtype=np.int64)
    np.cumsum(counts, out=off[1:])
    return off, idx[: int(total)]


def neighbours_grid(pos_mass, r_out: float, targets=None):
    """The rows of `neighbours` (fp32 predicate) with candidates from a uniform cell grid (large N):
    (offsets int64 [nt+1], indices int32)."""
    pm = _pm(pos_mass)
    n = pm.shape[0]
    tg = None if targets is None else np.ascontiguousarray(targets, dtype=np.int64)
    nt = n if tg is None else tg.shape[0]
    counts = np.zeros(nt, dtype=np.int64)
    total = lib().p3t_o_neighbours_grid(n, _p(pm), float(np.float32(r_out)), nt, _p(tg), _p(counts), None)
    if total < 0:
        raise ValueError("p3t_o_neighbours_grid: invalid arguments or out of memory")
    idx = np.zeros(max(int(total), 1), dtype=np.int32)
    lib().p3t_o_neighbours_grid(n, _p(pm), float(np.float32(r_out)), nt, _p(tg), _p(counts), _p(idx))
    off = np.zeros(nt + 1, dtype=np.int64)
    np.cumsum(counts, out=off[1:])
    return off, idx[: int(total)]


class Tree:
    """The reference octree (Part II)."""

    def __init__(self, pos_mass, key_bits: int = 63, nleaf: int = NLEAF_DEFAULT, ncrit: int = NCRIT_DEFAULT):
        self.pm = _pm(pos_mass)
        self._h = lib().p3t_o_tree_build(self.pm.shape[0], _p(self.pm), key_bits, nleaf, ncrit)
        if not self._h:
            raise ValueError("p3t_o_tree_build: invalid arguments")
        s = np.zeros(6, dtype=np.int64)
        lib().p3t_o_tree_sizes(self._h, _p(s))
        self.n, self.n_nodes, self.n_leaves, self.max_level, self.n_groups, self.bits = (int(v) for v in s)
        self.nleaf, self.ncrit = nleaf, ncrit

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.p3t_o_tree_free(self._h)
            self._h = None

    def cube(self):
        lo = np.zeros(3, dtype=np.float32); side = C.c_float(0)
        lib().p3t_o_tree_cube(self._h, _p(lo), C.cast(C.byref(side), C.c_void_p))
        return lo, float(side.value)

    def keys(self):
        k = np.zeros(self.n, dtype=np.uint64); o = np.zeros(self.n, dtype=np.uint32)
        lib().p3t_o_tree_keys(self._h, _p(k), _p(o))
        return k, o

    def nodes(self):
        a = [np.zeros(self.n_nodes, dtype=np.int32) for _ in range(5)]
        lib().p3t_o_tree_nodes(self._h, *[_p(x) for x in a])
        return dict(level=a[0], begin=a[1], end=a[2], first_child=a[3], n_child=a[4])

    def moments(self):
        nn = self.n_nodes
        com_m = np.zeros((nn, 4), np.float32); quad = np.zeros((nn, 6), np.float32)
        clo = np.zeros((nn, 3), np.float32); chi = np.zeros((nn, 3), np.float32); delta = np.zeros(nn, np.float32)
        lib().p3t_o_tree_moments(self._h, _p(com_m), _p(quad), _p(clo), _p(chi), _p(delta))
        return dict(com_m=com_m, quad=quad, clo=clo, chi=chi, delta=delta)

    def moments64(self):
        nn = self.n_nodes
        mass = np.zeros(nn); com = np.zeros((nn, 3)); quad = np.zeros((nn, 6))
        lib().p3t_o_tree_moments64(self._h, _p(mass), _p(com), _p(quad))
        return dict(mass=mass, com=com, quad=quad)

    def octupoles(self):
        """Raw third moments about the COM per node, order xxx yyy zzz xxy xxz xyy yyz xzz yzz xyz:
        dict(oct32 [nn,10] fp32-rounded, oct64 [nn,10])."""
        nn = self.n_nodes
        f = np.zeros((nn, 10), np.float32); d = np.zeros((nn, 10))
        lib().p3t_o_tree_octupoles(self._h, _p(f), _p(d))
        return dict(oct32=f, oct64=d)

    def groups(self):
        ng = self.n_groups
        b = np.zeros(ng, np.int32); e = np.zeros(ng, np.int32)
        glo = np.zeros((ng, 3), np.float32); ghi = np.zeros((ng, 3), np.float32)
        lib().p3t_o_tree_groups(self._h, _p(b), _p(e), _p(glo), _p(ghi))
        return dict(begin=b, end=e, glo=glo, ghi=ghi)

    def force(self, r_out: float, r_in: float, theta: float, pot_mode: int = 0, group_ids=None, want_abs: bool = False,
              r_list: float | None = None, order: int = 2):
        """dict(acc_pot [n,4] fp64 in original order (rows of unwalked groups are NaN), npp, npc, abs_sum)."""
        gi = None if group_ids is None else np.ascontiguousarray(group_ids, dtype=np.int64)
        ng = self.n_groups if gi is None else gi.shape[0]
        out = np.full((self.n, 4), np.nan)
        npp = np.zeros(ng, np.int64); npc = np.zeros(ng, np.int64)
        ab = np.full(self.n, np.nan) if want_abs else None
        rl = r_out if r_list is None else r_list          # neighbour search radius in the opening rule (NEXT-2)
        lib().p3t_o_tree_force_order(self._h, int(order), float(np.float32(rl)), float(np.float32(r_out)), float(np.float32(r_in)),
                                        float(np.float32(theta)), int(pot_mode), ng, _p(gi), _p(out), _p(npp), _p(npc), _p(ab))
        return dict(acc_pot=out, npp=npp, npc=npc, abs_sum=ab)


def pc_term(xi, com_m, quad) -> np.ndarray:
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    cm = np.ascontiguousarray(com_m, dtype=np.float32); q = np.ascontiguousarray(quad, dtype=np.float32)
    out = np.zeros(4)
    lib().p3t_o_pc_term(_p(xi), _p(cm), _p(q), _p(out))
    return out


def pc_octupole(xi, com_m, oct) -> np.ndarray:
    """The octupole term alone: {ax, ay, az, phi}."""
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    cm = np.ascontiguousarray(com_m, dtype=np.float32); t = np.ascontiguousarray(oct, dtype=np.float32)
    assert t.shape == (10,)
    out = np.zeros(4)
    lib().p3t_o_pc_octupole(_p(xi), _p(cm), _p(t), _p(out))
    return out


def open_test(glo, ghi, com, clo, chi, l, delta, theta, r_out) -> bool:
    arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in (glo, ghi, com, clo, chi)]
    return bool(lib().p3t_o_open_test(*[_p(a) for a in arrs], float(l), float(delta), float(theta), float(r_out)))


def interleave(gx: int, gy: int, gz: int, bits: int) -> int:
    return int(lib().p3t_o_interleave(gx, gy, gz, bits))
