"""Straggler hand-off: on grids of >= 200,000 points a query whose ring
search has scanned radius 24 (d=2) / 8 (d=3) without meeting its bound is finished by the brute-force
pass behind the search kernel.  Scenes: a dense block plus isolated points that need tens to hundreds
of rings; whole-set search, list repair (one warp per query), slot sweep on an updated grid with chain
residents, and a hand-off list that overflows.  Everything bit-exact against the CPU oracle."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_18314_b200 import binding as kc
from _util import assert_same, dev

pytestmark = pytest.mark.gpu


def _scene(d, n_block, side, n_out, seed, pairs=6):
    """n_block points uniform in [0, side]^d, n_out isolated points in the rest of the unit box, a few
    of them in close pairs (first neighbour near, second far)."""
    rng = np.random.default_rng(seed)
    block = rng.random((n_block, d)) * side
    out = side + 0.1 + rng.random((n_out, d)) * (0.9 - side)
    out[:pairs] = out[pairs:2 * pairs] + rng.uniform(-1e-4, 1e-4, (pairs, d))
    p = np.concatenate([block, out]).astype(np.float32)
    p[0] = 0.0
    return p[rng.permutation(p.shape[0])]


@pytest.mark.parametrize("d,side", [(2, 0.1), (3, 0.2)])
def test_isolated_points_are_handed_to_the_brute_force_pass(d, side):
    p = _scene(d, 1000000, side, 60 if d == 2 else 30, 40 + d)
    N = p.shape[0]
    grid = kc.Grid(N, kc.kc_geom_for(dev(p)))
    want = oracle.kdtree_top2(p)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    assert_same(certs, want, what=f"d{d} rebuild with isolated points")
    info = grid.info()
    assert info.n_handed >= 10 and info.n_stragglers >= 10        # the far points went through the pass
    # the list is empty again: a second search hands the same queries over once more, same bits
    assert_same(kc.kc_cert_grid_search(grid, kc.Certs.empty(N, "cuda")), want, what="second search")
    assert grid.info().n_handed == 2 * info.n_handed
    # what the pass wrote is the brute-force definition for those queries
    far = np.flatnonzero((p > side + 0.05).all(axis=1)).astype(np.int32)
    assert_same(certs, oracle.bruteforce_top2(p, queries=far), idx=far, what="isolated points, definition")


@pytest.mark.parametrize("d,side", [(2, 0.1), (3, 0.2)])
def test_handoff_in_the_repair_paths(d, side):
    """List repair (warp per query: 32 lanes hand one query over) and the slot sweep on an updated grid;
    isolated points that changed cell live in chains and must be found by the pass as candidates."""
    rng = np.random.default_rng(50 + d)
    p = _scene(d, 1000000, side, 60 if d == 2 else 30, 60 + d)
    N = p.shape[0]
    iso = np.flatnonzero((p > side + 0.05).all(axis=1)).astype(np.int32)
    g_kc = kc.kc_geom_for(dev(p))
    # (1) short list: the isolated points and some block points move by a few cells
    grid = kc.Grid(N, g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    movers = np.unique(np.concatenate([iso, rng.choice(N, 2000, replace=False).astype(np.int32)]))
    q = p.copy()
    q[movers] += rng.uniform(-3, 3, (movers.size, d)).astype(np.float32) * np.float32(g_kc.h)
    q = np.clip(q, 0, 1).astype(np.float32)
    handed0 = grid.info().n_handed
    F, nF = dev(movers), dev(np.array([movers.size], np.int32))
    kc.kc_frontier_repair(grid, dev(q), F, nF, certs, movers=F, n_movers=nF)
    post = oracle.kdtree_top2(q)
    assert_same(certs, post, idx=movers, what=f"d{d} list repair")
    info = grid.info()
    assert info.dirty == 1 and info.n_misfiled > 0 and info.n_handed - handed0 >= 10
    # (2) sweep: every point is a query on the updated grid (chains in place)
    allq = np.arange(N, dtype=np.int32)
    kc.kc_frontier_search(grid, dev(q), dev(allq), dev(np.array([N], np.int32)), certs)
    assert_same(certs, post, what=f"d{d} sweep on the updated grid")
    assert grid.info().n_handed - info.n_handed >= 10


def test_a_full_handoff_list_leaves_the_rest_to_the_rings():
    """More isolated points than the list holds (1,024): the overflow continues with the rings."""
    rng = np.random.default_rng(9)
    n_block, side = 2000000, 0.05
    block = rng.random((n_block, 2)) * side
    k = np.arange(36)
    lat = np.stack(np.meshgrid(k, k, indexing="ij"), -1).reshape(-1, 2) * 0.026 + 0.06       # 26 cell widths apart
    lat = lat[(lat > side + 0.026).any(axis=1)]
    p = np.concatenate([block, lat + rng.uniform(-1e-4, 1e-4, lat.shape)]).astype(np.float32)
    p = p[rng.permutation(p.shape[0])]
    N = p.shape[0]
    grid = kc.Grid(N, kc.kc_geom_for(dev(p)))
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    info = grid.info()
    assert lat.shape[0] > 1024 + 200 and info.n_handed == 1024 and info.n_stragglers > 1024 + 200
    assert_same(certs, oracle.kdtree_top2(p), what="overflowing hand-off list")


def test_small_grids_do_not_hand_off():
    rng = np.random.default_rng(3)
    p = np.concatenate([rng.random((50000, 2)) * 0.1, 0.3 + 0.7 * rng.random((20, 2))]).astype(np.float32)
    grid = kc.Grid(p.shape[0], kc.kc_geom_for(dev(p)))
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    assert grid.info().n_handed == 0 and grid.info().n_stragglers >= 15
    assert_same(certs, oracle.kdtree_top2(p), what="small grid, rings only")
