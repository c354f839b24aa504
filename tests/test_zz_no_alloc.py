"""p3t_morton_order_static -- the one entry point of libp3t.so that allocates no device memory.

Why it exists: every other call goes through a p3t_ctx, whose scratch comes from cudaMalloc.  A host integrator that
has already given the whole device to its own arena (or to a framework's caching allocator), that cannot take the
device-wide stall of cudaMalloc / cudaFree inside its step loop, or that runs under a device-memory quota cannot use
those calls.  This one keeps its scratch in a fixed array inside the library image (3.5 MB, n <= 262 144) and takes
only the caller's input and output buffers.

What is checked: its keys, sort order and bounding cube are bit-equal to those of the context path
(p3t_build_tree + p3t_get_keys / p3t_get_stats) -- integer work, so the bar is equality, as in test_gpu_parity -- on
calls made one after the other on the same device (the array keeps the previous call's contents: a larger problem
first, then a smaller one with the other key width, then the first again); that free device memory does not move
across a call; that n beyond the limit is refused with P3T_ELIMIT and nothing else.

The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It passes alone in a fresh process and after the rest of the suite."""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def p3t():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2110_11658_b200 as m
    m.lib()                                   # fails loudly if libp3t.so is missing
    return m


def _context_path(p3t, pm, bits):
    """(sorted keys uint64, order uint32, cube float32[4]) from the allocating path."""
    with p3t.Context(0) as ctx:
        ctx.build_tree(pm, bits)
        k, o = ctx.keys()
        st = ctx.stats()
    return k, o, np.asarray(list(st["cube_lo"]) + [st["cube_side"]], np.float32)


class _Buffers:
    """Everything the static call writes, allocated once by the caller (here: by torch) before any call."""

    def __init__(self, torch, nmax):
        self.keys = torch.empty(nmax, dtype=torch.int64, device="cuda")
        self.order = torch.empty(nmax, dtype=torch.int32, device="cuda")
        self.cube = torch.empty(4, dtype=torch.float32, device="cuda")
        self.bad = torch.empty(1, dtype=torch.int32, device="cuda")

    def poison(self):
        self.keys.fill_(-1); self.order.fill_(-1); self.cube.fill_(float("nan")); self.bad.fill_(-1)

    def result(self, torch, n):
        torch.cuda.synchronize()
        return (self.keys[:n].cpu().numpy().view(np.uint64), self.order[:n].cpu().numpy().view(np.uint32),
                self.cube.cpu().numpy(), int(self.bad.item()))


def _check(p3t, torch, B, pm, bits, stream=None):
    n = pm.shape[0]
    B.poison()
    p3t.morton_order_static(pm, B.keys, B.order, bits, cube=B.cube, bad_input=B.bad, stream=stream)
    k, o, cube, bad = B.result(torch, n)
    rk, ro, rcube = _context_path(p3t, pm, bits)
    assert bad == 0
    assert np.array_equal(cube, rcube), "bounding cube differs from the context path"
    assert np.array_equal(k, rk), "sorted Morton keys differ from the context path"
    assert np.array_equal(o, ro), "sort order differs from the context path"
    assert np.array_equal(np.sort(o), np.arange(n, dtype=np.uint32)), "order is not a permutation"


def test_static_entry_point_matches_the_context_path_call_after_call(p3t):
    import torch
    B = _Buffers(torch, 60000)
    big = torch.from_numpy(workloads.make_config(1, n_override=60000).pos_mass).cuda()
    small = torch.from_numpy(workloads.make_config(2, n_override=20001).pos_mass).cuda()     # ragged last tile
    _check(p3t, torch, B, big, 63)
    _check(p3t, torch, B, small, 30)        # fewer tiles, fewer passes: the array still holds the first call's words
    _check(p3t, torch, B, big, 63)
    # two calls enqueued back to back on one side stream, nothing waited for in between
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    k2 = torch.empty_like(B.keys); o2 = torch.empty_like(B.order)
    p3t.morton_order_static(small, k2, o2, 63, stream=s)
    _check(p3t, torch, B, big, 30, stream=s)
    rk, ro, _ = _context_path(p3t, small, 63)
    assert np.array_equal(k2[:20001].cpu().numpy().view(np.uint64), rk) and np.array_equal(o2[:20001].cpu().numpy().view(np.uint32), ro)


def test_static_entry_point_takes_no_device_memory(p3t):
    import torch
    n = 50000
    pm = torch.from_numpy(workloads.make_config(1, n_override=n).pos_mass).cuda()
    B = _Buffers(torch, n)
    p3t.morton_order_static(pm, B.keys, B.order, 63, cube=B.cube, bad_input=B.bad)      # set-up and code loading, if not done yet
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        p3t.morton_order_static(pm, B.keys, B.order, 63, cube=B.cube, bad_input=B.bad)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "device memory moved across calls that are documented not to allocate"


def test_static_entry_point_limits_and_arguments(p3t):
    import ctypes as C
    import torch
    L = p3t.lib()
    nmax = p3t.STATIC_MAX_N
    pm = torch.from_numpy(workloads.make_config(1, n_override=nmax).pos_mass).cuda()
    B = _Buffers(torch, nmax + 1)
    _check(p3t, torch, B, pm, 63)                                                       # exactly the maximum fits
    B.poison()
    args = (C.c_void_p(pm.data_ptr()), 63, C.c_void_p(B.keys.data_ptr()), C.c_void_p(B.order.data_ptr()), None, None)
    assert L.p3t_morton_order_static(0, None, nmax + 1, *args) == p3t.ELIMIT            # refused ...
    torch.cuda.synchronize()
    assert int(B.keys[0].item()) == -1 and int(B.order[0].item()) == -1                 # ... and nothing was written
    assert "P3T_STATIC_MAX_N" in p3t.strerror(p3t.ELIMIT)
    with pytest.raises(p3t.P3TError, match="STATIC_MAX_N"):
        p3t.morton_order_static(torch.zeros((nmax + 1, 4), device="cuda"), B.keys, B.order)
    assert L.p3t_morton_order_static(0, None, 0, *args) == p3t.EINVAL
    assert L.p3t_morton_order_static(0, None, 10, args[0], 42, *args[2:]) == p3t.EINVAL
    assert L.p3t_morton_order_static(0, None, 10, None, 63, *args[2:]) == p3t.EINVAL
    assert L.p3t_morton_order_static(99, None, 10, *args) == p3t.EINVAL
    # a NaN position is flagged, as p3t_build_tree flags it
    bad = pm[:1000].clone(); bad[17, 1] = float("nan")
    p3t.morton_order_static(bad, B.keys, B.order, 63, bad_input=B.bad)
    torch.cuda.synchronize()
    assert int(B.bad.item()) == 1
