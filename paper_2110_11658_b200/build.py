"""Build libp3t.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2110_11658_b200.build [--force]

No torch involvement: the library is plain CUDA runtime code.  nvcc cross-compiles
without a GPU, so this also runs on the CPU-only build box.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
LIB = PKG / "libp3t.so"
SOURCES = ["p3t_api.cu", "p3t_sort.cu", "p3t_tree.cu", "p3t_walk.cu", "p3t_force.cu", "p3t_irregular.cu", "p3t_core.cu", "p3t_shard.cu", "p3t_octupole.cu"]
DIAG_LIB = PKG / "libp3t_diag.so"          # diagnostics (include/p3t_diag.h): its own library, not linked into libp3t.so
DIAG_SOURCES = ["p3t_pipebench.cu", "p3t_diagknobs.cu"]
HEADERS = [CSRC / "p3t_internal.cuh", CSRC / "p3t_cutoff.cuh", CSRC / "p3t_f32x2.cuh", ROOT / "include" / "p3t.h", ROOT / "include" / "p3t_diag.h"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC",
    "-Xptxas", "-v", "--resource-usage",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def build(force: bool = False, verbose: bool = False, checks: bool = False) -> Path:
    """checks: compile with -DP3T_CHECKS (index assertions inside the kernels; profiles/r02_sanitizer.md).  A checks build is
    always rebuilt, and so is the build that follows it."""
    srcs = [CSRC / s for s in SOURCES + DIAG_SOURCES]
    deps = srcs + HEADERS + [Path(__file__)]
    marker = PKG / "build" / "checks.on"
    if checks or marker.exists():
        force = True
    if not force and LIB.exists() and DIAG_LIB.exists() and all(min(LIB.stat().st_mtime, DIAG_LIB.stat().st_mtime) >= d.stat().st_mtime for d in deps):
        return LIB
    objdir = PKG / "build"
    objdir.mkdir(exist_ok=True)
    nvcc = _nvcc()
    flags = NVCC_FLAGS + (["-DP3T_CHECKS"] if checks else [])
    if checks:
        marker.write_text("built with -DP3T_CHECKS\n")
    elif marker.exists():
        marker.unlink()
    procs = []
    for s in srcs:
        obj = objdir / (s.stem + ".o")
        cmd = [nvcc, *flags, "-I", str(ROOT / "include"), "-I", str(CSRC), "-c", str(s), "-o", str(obj)]
        procs.append((s, obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    objs = []
    log = []
    for s, obj, p in procs:
        out, _ = p.communicate()
        log.append(f"==== {s.name}\n{out}")
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed on {s.name}:\n{out}")
        objs.append(str(obj))
    (objdir / "ptxas.log").write_text("\n".join(log))
    if verbose:
        print("\n".join(log))
    ndiag = len(DIAG_SOURCES)
    for lib, group in ((LIB, objs[:-ndiag]), (DIAG_LIB, objs[-ndiag:])):
        tmp = lib.with_suffix(f".{os.getpid()}.tmp.so")
        cmd = [nvcc, "-shared", "-o", str(tmp), *group, "-cudart", "shared", "-Xcompiler", "-fPIC"]
        r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}")
        os.replace(tmp, lib)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checks="--checks" in sys.argv))
