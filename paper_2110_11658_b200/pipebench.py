"""Diagnostics (include/p3t_diag.h, libp3t_diag.so -- not part of libp3t.so): FP32-pipe micro-benchmarks of a device
(`python -m paper_2110_11658_b200.pipebench` prints the table for cuda:0) and the measurement /
fault-injection knobs of a Context (set_overlap, set_fault), which the product library does not expose."""
from __future__ import annotations

import ctypes as C
from pathlib import Path

DIAG_PATH = Path(__file__).resolve().parent / "libp3t_diag.so"
DIAG_SYMBOLS = ["p3t_diag_pipe_bench", "p3t_diag_set_overlap", "p3t_diag_set_fault"]
LABELS = ["FFMA (reuse cache)", "FFMA2, 2 distinct register pairs", "FFMA2, 3 distinct register pairs", "FMUL2",
          "FMUL2 + FFMA (pair)", "8 FMUL2 + 2 MUFU.RSQ (group)", "MUFU.RSQ", "FFMA, 3 distinct registers",
          "FFMA2, 3 distinct register pairs, one shared with the previous instruction"]
_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        if not DIAG_PATH.exists():
            raise ImportError(f"{DIAG_PATH} is missing: build it with `python -m paper_2110_11658_b200.build`")
        _lib = C.CDLL(str(DIAG_PATH))
        _lib.p3t_diag_pipe_bench.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int)]
        _lib.p3t_diag_pipe_bench.restype = C.c_int
        _lib.p3t_diag_set_overlap.argtypes = [C.c_void_p, C.c_int, C.c_int]; _lib.p3t_diag_set_overlap.restype = C.c_int
        _lib.p3t_diag_set_fault.argtypes = [C.c_void_p, C.c_int]; _lib.p3t_diag_set_fault.restype = C.c_int
    return _lib


def set_overlap(ctx, overlap: bool, walk_ctas_per_sm: int = 0) -> None:
    """Measurement knob of a Context: overlap False runs the list walk and the force kernel one after the other;
    walk_ctas_per_sm (> 0) sets the CTAs per SM left to the walk while they overlap (default 2)."""
    if lib().p3t_diag_set_overlap(ctx._h, 1 if overlap else 0, int(walk_ctas_per_sm)) != 0:
        raise ValueError("p3t_diag_set_overlap: bad argument")


def set_fault(ctx, bits: int) -> None:
    """Fault injection for the tests (include/p3t_diag.h): 1 = force warps give up waiting at once, 2 = no walk-stack
    spill, 4 = CUDA failure inside p3t_step_host with the call in flight, 0 = off."""
    if lib().p3t_diag_set_fault(ctx._h, int(bits)) != 0:
        raise ValueError("p3t_diag_set_fault: bad argument")


def pipe_bench(device: int = 0) -> dict:
    """Cycles per SM sub-partition for each instruction pattern, and the FP32 lane-instruction peak they imply
    (32 lanes / cycles[FFMA] per sub-partition)."""
    out = (C.c_double * 9)(); mhz = C.c_double(); sms = C.c_int()
    rc = lib().p3t_diag_pipe_bench(device, out, 9, C.byref(mhz), C.byref(sms))
    if rc != 0:
        raise RuntimeError(f"p3t_diag_pipe_bench failed ({rc})")
    cyc = [float(x) for x in out]
    peak = sms.value * 4 * 32 / cyc[0] * mhz.value * 1e6
    return dict(cycles=dict(zip(LABELS, cyc)), sm_clock_mhz=mhz.value, num_sms=sms.value,
                fp32_lane_instr_per_s=peak, nominal_lane_instr_per_s=sms.value * 128 * mhz.value * 1e6)


if __name__ == "__main__":
    import json
    print(json.dumps(pipe_bench(0), indent=1))
