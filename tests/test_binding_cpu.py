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


def test_regularisation_params_eq18_19(p3t):
    """eq. 18-19: R_min = 4 r_h / (N rho_core^(1/3)); dT_min = 0.01 sqrt(eta/0.02) sqrt(R_min^3).
    Hand case: N = 1000, r_h = 0.5, rho_core = 8 -> R_min = 4 * 0.5 / (1000 * 2) = 1e-3; dT_min = 0.01 * 1e-4.5."""
    r_min, dt_min = p3t.regularisation_params(1000, 0.5, 8.0)
    assert abs(r_min - 1e-3) < 1e-18 and abs(dt_min - 0.01 * 1e-3 ** 1.5) < 1e-20
    r2, dt2 = p3t.regularisation_params(1000, 0.5, 8.0, eta=0.08)
    assert r2 == r_min and abs(dt2 / dt_min - 2.0) < 1e-14
    assert p3t.lib().p3t_regularisation_params(0, 0.5, 8.0, 0.02, None, None) == p3t.EINVAL
    assert p3t.lib().p3t_regularisation_params(10, 0.5, -1.0, 0.02, None, None) == p3t.EINVAL
