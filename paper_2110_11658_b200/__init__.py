"""paper_2110_11658_b200 -- thin Python binding of libp3t.so (include/p3t.h).

The library is the B200-native (sm_100a) regular-force path of NBODY6+P3T
(arXiv:2110.11658): GPU Barnes-Hut tree force with the paper's 7th-order cutoff
(eq. 1-10) plus the neighbour lists inside r_out.

This module only marshals arguments: every step of the path runs in the CUDA
kernels behind the C-ABI.  PyTorch is used for device memory and streams only.
There is no CPU fallback: importing works without a GPU (so that the symbols can
be checked), but every compute call needs the built library and a CUDA device.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libp3t.so"

OK, EINVAL, ESTATE, ENOMEM, ECUDA, ERANGE, ELIMIT = 0, -1, -2, -3, -4, -5, -6
STATIC_MAX_N = 1 << 18                # p3t.h: P3T_STATIC_MAX_N, the capacity of p3t_morton_order_static

# every symbol include/p3t.h declares
SYMBOLS = [
    "p3t_create", "p3t_destroy", "p3t_set_tree_params", "p3t_set_multipole_order", "p3t_build_tree", "p3t_regular_force",
    "p3t_regular_force_ex", "p3t_irregular_force", "p3t_core_quantities", "p3t_neighbours", "p3t_neighbours_copy", "p3t_neighbours_nbody6", "p3t_step_host",
    "p3t_get_stats", "p3t_get_keys", "p3t_get_nodes", "p3t_get_moments", "p3t_get_groups",
    "p3t_get_list_lengths", "p3t_strerror", "p3t_last_error", "p3t_params_from_n",
    "p3t_set_shard", "p3t_get_shard_cuts", "p3t_shard_pack", "p3t_shard_unpack", "p3t_get_octupoles",
    "p3t_morton_order_static", "p3t_regular_force_begin", "p3t_regular_force_wait",
]
FF_OVERLAPPED, FF_REPAIRED, FF_SPIN_ABORT = 1, 2, 4           # p3t.h: bits of Stats.force_flags


class Stats(C.Structure):
    _fields_ = [
        ("n", C.c_int64), ("n_nodes", C.c_int64), ("n_leaves", C.c_int64), ("n_groups", C.c_int64),
        ("max_level", C.c_int32), ("key_bits", C.c_int32),
        ("n_pp", C.c_int64), ("n_pc", C.c_int64), ("n_pp_list", C.c_int64), ("n_pc_list", C.c_int64),
        ("nb_total", C.c_int64), ("nb_max", C.c_int32), ("input_bad", C.c_int32),
        ("cube_lo", C.c_float * 3), ("cube_side", C.c_float),
        ("ms_build", C.c_float), ("ms_force", C.c_float), ("ms_walk", C.c_float), ("ms_sort", C.c_float),
        ("ms_eval", C.c_float), ("ms_count", C.c_float), ("ms_irregular", C.c_float), ("ms_core", C.c_float),
        ("launches", C.c_int64), ("ms_octupole", C.c_float), ("force_flags", C.c_int32),
    ]

    def as_dict(self) -> dict:
        d = {}
        for name, _ in self._fields_:
            v = getattr(self, name)
            d[name] = list(v) if name == "cube_lo" else v
        return d


class P3TError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} ({code})" + (f": {detail}" if detail else ""))


_lib = None


def lib() -> C.CDLL:
    """Load libp3t.so; fails loudly when it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2110_11658_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(str(LIB_PATH))
    vp, i64, i32, f32, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_float, C.c_double
    L.p3t_create.argtypes = [C.POINTER(vp), C.c_int, vp]
    L.p3t_destroy.argtypes = [vp]
    L.p3t_set_tree_params.argtypes = [vp, C.c_int, C.c_int]
    L.p3t_set_multipole_order.argtypes = [vp, C.c_int]
    L.p3t_build_tree.argtypes = [vp, i64, vp, C.c_int]
    L.p3t_regular_force.argtypes = [vp, f32, f32, f32, C.c_int, vp]
    L.p3t_regular_force_ex.argtypes = [vp, f32, f32, f32, C.c_int, f32, f32, vp, vp]
    L.p3t_regular_force_begin.argtypes = [vp, f32, f32, f32, C.c_int, f32, f32, vp, vp]
    L.p3t_regular_force_wait.argtypes = [vp]
    L.p3t_irregular_force.argtypes = [vp, vp, vp, vp]
    L.p3t_core_quantities.argtypes = [vp, i64, vp, C.c_int, vp, vp, vp, vp]
    L.p3t_neighbours.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(i64)]
    L.p3t_neighbours_copy.argtypes = [vp, vp, vp]
    L.p3t_neighbours_nbody6.argtypes = [vp, i32, vp]
    L.p3t_step_host.argtypes = [vp, i64, vp, C.c_int, f32, f32, f32, C.c_int, vp, vp, vp, i64, C.POINTER(i64)]
    L.p3t_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.p3t_get_keys.argtypes = [vp, vp, vp]
    L.p3t_get_nodes.argtypes = [vp, vp, vp, vp, vp, vp]
    L.p3t_get_moments.argtypes = [vp, vp, vp, vp, vp, vp]
    L.p3t_get_octupoles.argtypes = [vp, vp]
    L.p3t_get_groups.argtypes = [vp, vp, vp]
    L.p3t_get_list_lengths.argtypes = [vp, vp, vp]
    L.p3t_set_shard.argtypes = [vp, C.c_int, C.c_int, vp]
    L.p3t_get_shard_cuts.argtypes = [vp, vp, vp]
    L.p3t_shard_pack.argtypes = [vp, vp, vp]
    L.p3t_shard_unpack.argtypes = [vp, C.c_int, vp, vp]
    L.p3t_morton_order_static.argtypes = [C.c_int, vp, i64, vp, C.c_int, vp, vp, vp, vp]
    L.p3t_strerror.argtypes = [C.c_int]; L.p3t_strerror.restype = C.c_char_p
    L.p3t_last_error.argtypes = [vp]; L.p3t_last_error.restype = C.c_char_p
    L.p3t_params_from_n.argtypes = [i64, dbl] + [C.POINTER(dbl)] * 5
    for s in SYMBOLS:
        if s not in ("p3t_strerror", "p3t_last_error"):
            getattr(L, s).restype = C.c_int
    _lib = L
    return L


def strerror(code: int) -> str:
    return lib().p3t_strerror(int(code)).decode()


def params_from_n(n: int, sigma: float = 2.0 ** -0.5) -> dict:
    """eq. 20-25."""
    v = [C.c_double() for _ in range(5)]
    rc = lib().p3t_params_from_n(int(n), float(sigma), *[C.byref(x) for x in v])
    if rc:
        raise P3TError(rc, "p3t_params_from_n")
    return dict(zip(["tau", "r_cut", "r_buff", "dt_reg", "dt_max"], [x.value for x in v]))


def morton_order_static(pos_mass, sorted_keys, order, key_bits: int = 63, cube=None, bad_input=None, stream=None):
    """p3t_morton_order_static: Morton keys, stable sort order and bounding cube of pos_mass (CUDA float32 [n, 4])
    for callers that must not allocate device memory -- a host code whose own arena or caching allocator already
    holds the whole device, a step loop that cannot take the device-wide stall of cudaMalloc / cudaFree, a process
    under a memory quota.  The call needs no Context and allocates nothing: its scratch is a fixed 3.5 MB array
    inside libp3t.so, good for n <= STATIC_MAX_N (262 144); a larger n raises P3TError(ELIMIT).

    The caller passes every buffer, all CUDA tensors of the same device: sorted_keys int64 [n] (the uint64 keys, bit
    for bit), order int32 [n] (sorted position -> original id), and optionally cube float32 [4] (lo x, y, z, side)
    and bad_input int32 [1].  Enqueues on `stream` (a torch.cuda.Stream; None = the legacy default stream) and does
    not synchronise.  All calls on a device share the one array: order them (one stream, or events); calls that
    overlap on the GPU race.  The first call on a device also looks up the array's device address -- make it
    outside any stream capture."""
    import torch
    n = int(pos_mass.shape[0])
    assert pos_mass.is_cuda and pos_mass.dtype == torch.float32 and pos_mass.is_contiguous() and pos_mass.shape[-1] == 4
    dev = pos_mass.device
    for t, dt, cnt in ((sorted_keys, torch.int64, n), (order, torch.int32, n), (cube, torch.float32, 4), (bad_input, torch.int32, 1)):
        assert t is None or (t.device == dev and t.dtype == dt and t.is_contiguous() and t.numel() >= cnt)
    ptr = lambda t: None if t is None else C.c_void_p(t.data_ptr())
    sp = C.c_void_p(stream.cuda_stream if stream is not None else 0)
    rc = lib().p3t_morton_order_static(dev.index if dev.index is not None else torch.cuda.current_device(), sp, n,
                                       ptr(pos_mass), key_bits, ptr(sorted_keys), ptr(order), ptr(cube), ptr(bad_input))
    if rc != OK:
        raise P3TError(rc, "p3t_morton_order_static")


def _np_ptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


class Context:
    """One p3t_ctx: a device, a stream and the library-owned scratch."""

    def __init__(self, device: int = 0, stream=None, nleaf: int = 16, ncrit: int = 64):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2110_11658_b200 needs a CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        torch.cuda.init()
        torch.zeros(1, device=self.device)          # makes sure the primary context exists
        self._stream = stream
        sp = C.c_void_p(stream.cuda_stream if stream is not None else 0)
        h = C.c_void_p()
        self._check(lib().p3t_create(C.byref(h), device, sp), "p3t_create", ctx=None)
        self._h = h
        self.n = 0
        self.shard = (0, 1)
        self._check(lib().p3t_set_tree_params(self._h, nleaf, ncrit), "p3t_set_tree_params")

    # -- plumbing --
    def _check(self, rc: int, where: str, ctx="self"):
        if rc != OK:
            detail = ""
            if ctx == "self" and getattr(self, "_h", None):
                detail = lib().p3t_last_error(self._h).decode()
            raise P3TError(rc, where, detail)

    def close(self):
        if getattr(self, "_h", None):
            lib().p3t_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _dev_f32(self, t, cols):
        torch = self._torch
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.shape[-1] == cols
        return C.c_void_p(t.data_ptr())

    # -- the three calls of the hot path --
    def build_tree(self, pos_mass, key_bits: int = 63):
        """pos_mass: CUDA float32 tensor [n, 4] = x, y, z, m."""
        self.n = int(pos_mass.shape[0])
        self._check(lib().p3t_build_tree(self._h, self.n, self._dev_f32(pos_mass, 4), key_bits), "p3t_build_tree")

    def set_multipole_order(self, order: int):
        """2 = monopole + quadrupole (default), 1 = monopole only, 3 = + octupole (needs a build_tree after the
        call)."""
        self._check(lib().p3t_set_multipole_order(self._h, order), "p3t_set_multipole_order")

    # -- multi-GPU: target groups split among ranks (the exchange is in paper_2110_11658_b200.shard) --
    def set_shard(self, rank: int, nranks: int, nominal_cuts=None):
        """This context evaluates the groups of one Morton range (rank of nranks); takes effect at the next
        build_tree.  nominal_cuts: nranks + 1 sorted positions (default r n / nranks)."""
        import numpy as np
        c = None
        if nominal_cuts is not None:
            c = np.ascontiguousarray(nominal_cuts, dtype=np.int64)
            assert c.shape == (nranks + 1,)
        self._check(lib().p3t_set_shard(self._h, rank, nranks, None if c is None else _np_ptr(c)), "p3t_set_shard")
        self.shard = (rank, nranks)

    def shard_cuts(self):
        """(cuts, group_cuts): numpy int64 / int32 [nranks + 1], the group-aligned ranges of all ranks."""
        import numpy as np
        nr = self.shard[1]
        c = np.empty(nr + 1, np.int64); g = np.empty(nr + 1, np.int32)
        self._check(lib().p3t_get_shard_cuts(self._h, _np_ptr(c), _np_ptr(g)), "p3t_get_shard_cuts")
        return c, g

    def shard_pack(self, acc_pot, chunk):
        """chunk[: cuts[rank+1] - cuts[rank]] = the owned rows of acc_pot, in sorted order."""
        self._check(lib().p3t_shard_pack(self._h, self._dev_f32(acc_pot, 4), self._dev_f32(chunk, 4)), "p3t_shard_pack")

    def shard_unpack(self, from_rank: int, chunk, acc_pot):
        """Scatter the chunk of rank from_rank into acc_pot (original order)."""
        self._check(lib().p3t_shard_unpack(self._h, from_rank, self._dev_f32(chunk, 4), self._dev_f32(acc_pot, 4)), "p3t_shard_unpack")

    def regular_force(self, r_out: float, r_in: float, theta: float, pot_mode: int = 0, out=None,
                      r_buff: float = 0.0, half_dt: float = 0.0, vel=None):
        """Returns acc_pot: CUDA float32 [n, 4] = ax, ay, az, phi in original particle order.
        r_buff > 0: neighbour lists reach r_out + r_buff; vel (CUDA float32 [n, 4]) is kicked in place by
        half_dt * F_R."""
        torch = self._torch
        if out is None:
            out = torch.empty((self.n, 4), dtype=torch.float32, device=self.device)
        if r_buff == 0.0 and vel is None:
            self._check(lib().p3t_regular_force(self._h, r_out, r_in, theta, pot_mode, self._dev_f32(out, 4)), "p3t_regular_force")
        else:
            pv = None if vel is None else self._dev_f32(vel, 4)
            self._check(lib().p3t_regular_force_ex(self._h, r_out, r_in, theta, pot_mode, r_buff, half_dt, pv, self._dev_f32(out, 4)),
                        "p3t_regular_force_ex")
        return out

    def regular_force_begin(self, r_out: float, r_in: float, theta: float, pot_mode: int = 0, out=None,
                            r_buff: float = 0.0, half_dt: float = 0.0, vel=None):
        """First half of regular_force: enqueues the whole call and returns without waiting, so that the host can do its
        own work (the irregular steps of PAPER.md:89-94) while the GPU runs.  `out` (and vel) are complete only after
        regular_force_wait(); no other call on this context in between."""
        torch = self._torch
        if out is None:
            out = torch.empty((self.n, 4), dtype=torch.float32, device=self.device)
        pv = None if vel is None else self._dev_f32(vel, 4)
        self._check(lib().p3t_regular_force_begin(self._h, r_out, r_in, theta, pot_mode, r_buff, half_dt, pv, self._dev_f32(out, 4)),
                    "p3t_regular_force_begin")
        self._pending_out = (out, vel)                               # keeps the tensors alive while the GPU writes them
        return out

    def regular_force_wait(self):
        """Second half: the call's one synchronisation and its error report."""
        self._check(lib().p3t_regular_force_wait(self._h), "p3t_regular_force_wait")
        self._pending_out = None

    def irregular_force(self, vel, acc_out=None, jerk_out=None):
        """Irregular force over the neighbour lists of the last regular_force.
        vel: CUDA float32 [n, 4] (vx, vy, vz, unused), original order.  Returns (acc_irr [n, 4] = ax, ay,
        az, phi_I; jerk_irr [n, 4] = jx, jy, jz, 0) as CUDA tensors in original order."""
        torch = self._torch
        if acc_out is None:
            acc_out = torch.empty((self.n, 4), dtype=torch.float32, device=self.device)
        if jerk_out is None:
            jerk_out = torch.empty((self.n, 4), dtype=torch.float32, device=self.device)
        self._check(lib().p3t_irregular_force(self._h, self._dev_f32(vel, 4), self._dev_f32(acc_out, 4), self._dev_f32(jerk_out, 4)),
                    "p3t_irregular_force")
        return acc_out, jerk_out

    def core_quantities(self, sample, k: int = 6):
        """Sampled k-NN densities and core quantities.  sample: CUDA int32 [ns] original ids.
        Returns dict(nbr int32 [ns, k], d2k float32 [ns], rho float64 [ns] (CUDA tensors), center [3], r_core,
        rho_core, n_core)."""
        torch = self._torch
        assert sample.is_cuda and sample.dtype == torch.int32 and sample.is_contiguous()
        ns = int(sample.shape[0])
        nbr = torch.empty((ns, k), dtype=torch.int32, device=self.device)
        d2k = torch.empty(ns, dtype=torch.float32, device=self.device)
        rho = torch.empty(ns, dtype=torch.float64, device=self.device)
        out = (C.c_double * 6)()
        self._check(lib().p3t_core_quantities(self._h, ns, sample.data_ptr(), k, nbr.data_ptr(), d2k.data_ptr(), rho.data_ptr(), out),
                    "p3t_core_quantities")
        return dict(nbr=nbr, d2k=d2k, rho=rho, center=[out[0], out[1], out[2]], r_core=out[3], rho_core=out[4], n_core=out[5])

    def neighbours(self):
        """(offsets int64 [n+1], indices int32 [total]) as CUDA tensors (copied from the library's buffers)."""
        torch = self._torch
        tot = C.c_int64()
        po, pi = C.c_void_p(), C.c_void_p()
        self._check(lib().p3t_neighbours(self._h, C.byref(po), C.byref(pi), C.byref(tot)), "p3t_neighbours")
        off = torch.empty(self.n + 1, dtype=torch.int64, device=self.device)
        idx = torch.empty(max(tot.value, 1), dtype=torch.int32, device=self.device)
        self._check(lib().p3t_neighbours_copy(self._h, C.c_void_p(off.data_ptr()), C.c_void_p(idx.data_ptr())), "p3t_neighbours_copy")
        return off, idx[: tot.value]

    def neighbours_nbody6(self, lmax: int):
        import numpy as np
        out = np.zeros((self.n, lmax + 1), dtype=np.int32)
        self._check(lib().p3t_neighbours_nbody6(self._h, lmax, _np_ptr(out)), "p3t_neighbours_nbody6")
        return out

    def step_host(self, pos_mass, r_out, r_in, theta, pot_mode=0, key_bits=63, acc_pot=None, nb_offsets=None, nb_indices=None):
        """Whole step with HOST numpy (or pinned torch CPU) buffers; returns (acc_pot, nb_offsets, nb_indices, total)."""
        import numpy as np
        n = int(pos_mass.shape[0])
        self.n = n

        def ptr(a):
            if a is None:
                return None
            return C.c_void_p(a.data_ptr()) if hasattr(a, "data_ptr") else C.c_void_p(a.ctypes.data)

        if acc_pot is None:
            acc_pot = np.empty((n, 4), dtype=np.float32)
        cap = 0 if nb_indices is None else int(nb_indices.shape[0])
        tot = C.c_int64()
        rc = lib().p3t_step_host(self._h, n, ptr(pos_mass), key_bits, r_out, r_in, theta, pot_mode,
                                 ptr(acc_pot), ptr(nb_offsets), ptr(nb_indices), cap, C.byref(tot))
        self._check(rc, "p3t_step_host")
        return acc_pot, nb_offsets, nb_indices, tot.value

    # -- accessors (parity / debug) --
    def stats(self) -> dict:
        s = Stats()
        self._check(lib().p3t_get_stats(self._h, C.byref(s)), "p3t_get_stats")
        return s.as_dict()

    def keys(self):
        import numpy as np
        k = np.empty(self.n, dtype=np.uint64); o = np.empty(self.n, dtype=np.uint32)
        self._check(lib().p3t_get_keys(self._h, _np_ptr(k), _np_ptr(o)), "p3t_get_keys")
        return k, o

    def nodes(self) -> dict:
        import numpy as np
        nn = self.stats()["n_nodes"]
        a = [np.empty(nn, dtype=np.int32) for _ in range(5)]
        self._check(lib().p3t_get_nodes(self._h, *[_np_ptr(x) for x in a]), "p3t_get_nodes")
        return dict(level=a[0], begin=a[1], end=a[2], first_child=a[3], n_child=a[4])

    def moments(self) -> dict:
        import numpy as np
        nn = self.stats()["n_nodes"]
        com_m = np.empty((nn, 4), np.float32); quad = np.empty((nn, 6), np.float32)
        clo = np.empty((nn, 3), np.float32); chi = np.empty((nn, 3), np.float32); delta = np.empty(nn, np.float32)
        self._check(lib().p3t_get_moments(self._h, *[_np_ptr(x) for x in (com_m, quad, clo, chi, delta)]), "p3t_get_moments")
        return dict(com_m=com_m, quad=quad, clo=clo, chi=chi, delta=delta)

    def octupoles(self):
        """fp32 raw third moments [n_nodes, 10] (tree built with multipole order 3)."""
        import numpy as np
        t = np.empty((self.stats()["n_nodes"], 10), np.float32)
        self._check(lib().p3t_get_octupoles(self._h, _np_ptr(t)), "p3t_get_octupoles")
        return t

    def groups(self) -> dict:
        import numpy as np
        ng = self.stats()["n_groups"]
        b = np.empty(ng, np.int32); e = np.empty(ng, np.int32)
        self._check(lib().p3t_get_groups(self._h, _np_ptr(b), _np_ptr(e)), "p3t_get_groups")
        return dict(begin=b, end=e)

    def list_lengths(self):
        import numpy as np
        ng = self.stats()["n_groups"]
        npp = np.empty(ng, np.int32); npc = np.empty(ng, np.int32)
        self._check(lib().p3t_get_list_lengths(self._h, _np_ptr(npp), _np_ptr(npc)), "p3t_get_list_lengths")
        return npp, npc
