"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/p3t.h declares (no compute calls without a GPU); host helpers; loud failure without the library."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

from conftest import ROOT, read_golden


@pytest.fixture(scope="module")
def p3t():
    from paper_2110_11658_b200 import build
    build.build()
    import paper_2110_11658_b200 as m
    return m


def _declared_symbols():
    text = (ROOT / "include" / "p3t.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(p3t_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(p3t):
    L = p3t.lib()
    decl = _declared_symbols()
    assert len(decl) >= 15 and "p3t_build_tree" in decl and "p3t_regular_force" in decl and "p3t_neighbours" in decl
    for s in decl:
        assert hasattr(L, s), f"{s} is declared in include/p3t.h but not exported by libp3t.so"
    assert sorted(p3t.SYMBOLS) == decl, "the binding's symbol list and the header disagree"


def test_every_entry_point_cites_the_paper():
    text = (ROOT / "include" / "p3t.h").read_text()
    assert text.count("PAPER.md:") >= 10
    for name in ("p3t_build_tree", "p3t_regular_force", "p3t_neighbours", "p3t_params_from_n"):
        pos = text.index(f"int {name}(") if f"int {name}(" in text else text.index(f"int  {name}(")
        assert "PAPER.md:" in text[max(0, pos - 1500):pos], name


def test_strerror_and_argument_checks_without_gpu(p3t):
    assert p3t.strerror(0) == "ok"
    assert "order" in p3t.strerror(p3t.ESTATE) and "argument" in p3t.strerror(p3t.EINVAL)
    L = p3t.lib()
    # null pointers are rejected before any CUDA call
    assert L.p3t_create(None, 0, None) == p3t.EINVAL
    assert L.p3t_build_tree(None, 10, None, 63) == p3t.EINVAL
    assert L.p3t_regular_force(None, 0.1, 0.01, 0.4, 0, None) == p3t.EINVAL
    assert L.p3t_neighbours(None, None, None, None) == p3t.EINVAL
    assert L.p3t_destroy(None) == p3t.EINVAL


def test_params_from_n_golden(p3t):
    """eq. 20-25; fixture rows carry the citation."""
    for n, tau, r_cut, dt_reg, dt_max in read_golden("params_eq20_25.txt"):
        p = p3t.params_from_n(int(n))
        assert p["tau"] == pytest.approx(tau, rel=1e-12) and p["r_cut"] == pytest.approx(r_cut, rel=1e-12)
        assert p["dt_reg"] == dt_reg and p["dt_max"] == dt_max
        assert p["r_buff"] == pytest.approx(3 * tau / np.sqrt(2), rel=1e-12)
    p = p3t.params_from_n(100000)
    assert p["dt_reg"] <= p["tau"] < 2 * p["dt_reg"] and np.log2(p["dt_reg"]) == round(np.log2(p["dt_reg"]))
    v = [ctypes.c_double() for _ in range(5)]
    assert p3t.lib().p3t_params_from_n(0, 0.7, *[ctypes.byref(x) for x in v]) == p3t.EINVAL


def test_missing_library_fails_loudly(p3t, monkeypatch, tmp_path):
    monkeypatch.setattr(p3t, "_lib", None)
    monkeypatch.setattr(p3t, "LIB_PATH", tmp_path / "libp3t.so")
    with pytest.raises(ImportError, match="no CPU fallback"):
        p3t.lib()


def test_no_gpu_means_no_context(p3t):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        p3t.Context(0)


def test_product_never_imports_the_oracle():
    pkg = ROOT / "paper_2110_11658_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + [ROOT / "include" / "p3t.h"]:
        t = f.read_text()
        assert "import oracle" not in t and "from oracle" not in t and "p3t_oracle" not in t, f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c", ".h"):
            t = f.read_text()
            assert "import paper_2110_11658_b200" not in t and "from paper_2110_11658_b200" not in t, f
            assert '#include "p3t.h"' not in t and "p3t_internal" not in t and "libp3t.so" not in t, f


def test_diagnostics_library_is_separate(p3t):
    """include/p3t_diag.h (FP32-pipe micro-benchmarks) is exported by libp3t_diag.so, not by the product library."""
    from paper_2110_11658_b200 import pipebench
    text = re.sub(r"/\*.*?\*/", "", (ROOT / "include" / "p3t_diag.h").read_text(), flags=re.S)
    decl = sorted(set(re.findall(r"\b(p3t_[a-z0-9_]+)\s*\(", text)))
    assert decl == sorted(pipebench.DIAG_SYMBOLS)
    for s in decl:
        assert hasattr(pipebench.lib(), s) and not hasattr(p3t.lib(), s)
