"""GPU parity of p3t_core_quantities (sampled k-NN on the octree, Casertano-Hut
densities, core quantities) against the brute-force oracle (pinned in test_oracle_core.py).
Neighbour ids and the k-th distance: bit-exact (integer / fp32 decision taken in the same precision
and tie rule on both sides); densities: the same fp64 expression, bit-exact; the reductions run in
another (fixed) order than the oracle's index loop: 1e-12."""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def p3t():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2110_11658_b200 as m
    m.lib()
    return m


def _run(p3t, pm, sample, k=6, bits=63):
    import torch
    with p3t.Context(0) as ctx:
        ctx.build_tree(torch.from_numpy(np.ascontiguousarray(pm, np.float32)).cuda(), bits)
        r = ctx.core_quantities(torch.from_numpy(np.ascontiguousarray(sample, np.int32)).cuda(), k)
        st = ctx.stats()
    return {kk: (v.cpu().numpy() if hasattr(v, "cpu") else v) for kk, v in r.items()}, st


def _compare(pm, sample, g, k=6):
    o = oracle.knn_density(pm, sample, k)
    assert np.array_equal(g["nbr"], o["nbr"]), "neighbour ids differ"
    assert np.array_equal(g["d2k"], o["d2k"])
    assert np.array_equal(g["rho"], o["rho"])
    q = oracle.core_quantities(pm, sample, o["rho"])
    assert np.allclose(g["center"], q["center"], rtol=0, atol=1e-12)
    assert abs(g["r_core"] / q["r_core"] - 1) < 1e-12 and abs(g["rho_core"] / q["rho_core"] - 1) < 1e-12
    assert g["n_core"] == q["n_core"]
    return q


def test_config1_paper_sample(p3t):
    """Config 1, the paper's sample size min(N, sqrt(5000 N)) = 9050 of 16384, k = 6."""
    w = workloads.make_config(1)
    ns = int(min(w.n, np.sqrt(5000.0 * w.n)))
    sample = workloads.sample_targets(w.n, ns).astype(np.int32)
    g, st = _run(p3t, w.pos_mass, sample)
    q = _compare(w.pos_mass, sample, g)
    assert st["ms_core"] > 0
    assert np.linalg.norm(q["center"]) < 0.05 and 0.2 < q["r_core"] < 0.5       # Plummer: a = 0.59, R_core ~ 0.4 a ... 0.7 a


def test_king_and_kroupa_masses(p3t):
    """Config 4 recipe (King W0 = 9, Kroupa masses) at N = 2^16: a dense core, unequal masses, 30-bit keys too."""
    w = workloads.make_config(4, n_override=65536)
    sample = workloads.sample_targets(w.n, 3000).astype(np.int32)
    for bits in (63, 30):
        g, _ = _run(p3t, w.pos_mass, sample, bits=bits)
        _compare(w.pos_mass, sample, g)


def test_lattice_ties_and_other_k(p3t):
    """A cubic lattice: every particle has 6 / 12 / 8 exactly equidistant neighbours; ties by original index."""
    g1 = np.arange(12, dtype=np.float32)
    x, y, z = np.meshgrid(g1, g1, g1, indexing="ij")
    pm = np.zeros((12 ** 3, 4), np.float32); pm[:, 0] = x.ravel(); pm[:, 1] = y.ravel(); pm[:, 2] = z.ravel(); pm[:, 3] = 1.0 / 12 ** 3
    perm = np.argsort(workloads.uniform(5, 0, pm.shape[0]))          # original ids unrelated to position
    pm = np.ascontiguousarray(pm[perm])
    sample = np.arange(0, pm.shape[0], 5, dtype=np.int32)
    for k in (2, 4, 6, 9, 16):
        g, _ = _run(p3t, pm, sample, k=k)
        _compare(pm, sample, g, k=k)


def test_arguments(p3t):
    import torch
    w = workloads.make_config(1, n_override=500)
    s = torch.arange(0, 100, dtype=torch.int32, device="cuda")
    with p3t.Context(0) as ctx:
        with pytest.raises(p3t.P3TError) as e:
            ctx.core_quantities(s)
        assert e.value.code == -2                                    # no tree yet
        ctx.build_tree(torch.from_numpy(w.pos_mass).cuda(), 63)
        with pytest.raises(p3t.P3TError):
            ctx.core_quantities(s, k=1)
        with pytest.raises(p3t.P3TError):
            ctx.core_quantities(s, k=17)
        ctx.core_quantities(s, k=6)
