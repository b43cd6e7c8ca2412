"""GPU parity at BASELINE.json's full sizes (configs 4 and 5), in the launch configuration
bench.py times: whole-array comparison against the k-d tree oracle (itself validated bitwise
against brute force on every config's distribution, tests/test_oracle_pins.py) plus sampled
outputs recomputed one by one by the O(N) brute-force definition."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_18314_b200 import binding as kc
from paper_2606_18314_b200 import workloads as wl

from _util import assert_same, dev, geoms, host

pytestmark = pytest.mark.gpu


def sampled_bruteforce_check(p, got, n_samples, seed, what):
    q = np.sort(np.random.default_rng(seed).choice(p.shape[0], n_samples, replace=False)).astype(np.int32)
    want = oracle.bruteforce_top2(p, queries=q)
    assert_same(got, want, idx=q, what=what + " (sampled brute force)")


@pytest.mark.parametrize("density", ["median", "mean"])
@pytest.mark.parametrize("cfg", ["cfg5_d2", "cfg5_d3"])
def test_config5_rebuild_and_repair_4m(cfg, density):
    """density = "median": the geometry bench.py times (reading R24), computed by each side on its own;
    "mean": the plain occupancy-2 grid of the bounding box."""
    c = wl.CONFIGS[cfg]
    p, mot = wl.make_scene(cfg)
    N = c["N"]
    P = dev(p)
    if density == "median":
        g_or, g_kc = oracle.geom_by_median_density(p), kc.kc_geom_by_median_density(P)
        assert tuple(g_or.G) == tuple(g_kc.G) and g_or.h == np.float32(g_kc.h) and g_or.inv_h == np.float32(g_kc.inv_h)
        assert list(g_or.lo) == [np.float32(g_kc.lo[k]) for k in range(3)]
        assert g_kc.G[0] < geoms(p)[1].G[0]
    else:
        g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, P)
    got = host(certs)
    want = oracle.kdtree_top2(p)
    assert_same(got, want, what=f"{cfg} rebuild 4M")
    sampled_bruteforce_check(p, got, 192, 1, cfg)
    # one random-walk step: Lemma-1 frontier, repair, compare at F
    q, _ = mot.step(p)
    Q = dev(q)
    eps = kc.kc_max_displacement(P, Q)
    assert eps.cpu().numpy().view(np.uint32)[0] == np.array([oracle.max_displacement(p, q)]).view(np.uint32)[0]
    flags, F, nF = kc.kc_frontier_classify(certs.c, eps)
    wf, wF = oracle.frontier(want.c, oracle.max_displacement(p, q))
    assert np.array_equal(flags.cpu().numpy(), wf) and int(nF.item()) == wF.size
    kc.kc_frontier_repair(grid, Q, F, nF, certs)
    post = oracle.kdtree_top2(q)
    got = host(certs)
    assert_same(got, post, idx=wF, what=f"{cfg} repair 4M")
    rest = np.flatnonzero(wf == 0)
    assert np.array_equal(got.nn[rest], post.nn[rest])            # Lemma 1
    H, m, C = kc.kc_frontier_entropy(grid, F, nF)
    wH, wm, wC = oracle.entropy(oracle.cell_ids(q, g_or), wF, g_or.n_cells)
    assert abs(float(H.item()) - wH) <= 1e-6 and int(m.item()) == wm and int(C.item()) == wC
    # thin frontiers on the grid resident at q (4 M points: d = 3 sweeps from N/32 on, d = 2 from N/4 on, so
    # these two sizes take the list kernels in the plane and the compacting sweep in space)
    rng = np.random.default_rng(17)
    for f in (0.04, 0.15):
        ids = np.sort(rng.choice(N, int(N * f), replace=False)).astype(np.int32)
        out = kc.Certs.empty(N, "cuda")
        out.nn.fill_(-7)
        kc.kc_frontier_search(grid, Q, dev(ids), dev(np.array([ids.size], np.int32)), out)
        assert_same(out, post, idx=ids, what=f"{cfg} frontier of {f:.0%}")
        torch.cuda.synchronize()
        assert np.array_equal(np.flatnonzero(out.nn.cpu().numpy() != -7), ids)


@pytest.mark.parametrize("d", [2, 3])
def test_config5_allpairs_1m(d):
    p = wl.make_points(f"cfg5_d{d}", N=1048576)
    got = host(kc.kc_cert_allpairs(dev(p)))
    assert_same(got, oracle.kdtree_top2(p), what=f"allpairs 1M d{d}")
    sampled_bruteforce_check(p, got, 256, 2, f"allpairs 1M d{d}")


@pytest.mark.parametrize("ball", [False, True])
def test_config4_sweep_points(ball):
    N = wl.CONFIGS["cfg4"]["N"]
    for f in (0.001, 0.1, 1.0):
        p, mot = wl.make_scene("cfg4", "fraction", fraction=f, ball=ball)
        g_or, g_kc = geoms(p)
        grid = kc.Grid(N, g_kc)
        certs = kc.kc_cert_grid_rebuild(grid, dev(p))
        assert_same(certs, oracle.kdtree_top2(p), what="cfg4 pre")
        q, movers = mot.step(p)
        F, nF = dev(movers), dev(np.array([movers.size], np.int32))
        kc.kc_frontier_repair(grid, dev(q), F, nF, certs, movers=F, n_movers=nF)
        post = oracle.kdtree_top2(q)
        assert_same(certs, post, idx=movers, what=f"cfg4 f={f} ball={ball}")
        assert_same(kc.kc_cert_grid_rebuild(grid, dev(q)), post, what="cfg4 rebuild post")
