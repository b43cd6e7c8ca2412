"""Slot sweep of A7 (Alg. 1 l.4-7) at every frontier density.  On grids of >= 200,000
points a frontier of >= N/8 points is served in slot order; in d = 3 a frontier of less than 45 % of the
points is served by the compacting instantiation (a warp owns 64-256 slots and serves the marked ones 32
at a time), a denser one slot by slot.  Scenes with subdivided cells and a ragged tail; fresh grid and
incrementally updated grid (tombstones, chains); untouched entries stay untouched and the marks are all
clear afterwards (a second call with another list must not re-serve the first one's ids).  Bit-exact
against the CPU oracle (exact k-d tree, validated against brute force in the CPU suite)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_18314_b200 import binding as kc
from _util import assert_same, dev

pytestmark = pytest.mark.gpu

SENTINEL = -7


def _points(d, N, seed):
    """Half uniform, half in 12 tight clusters (cells of thousands of records -> second level)."""
    rng = np.random.default_rng(seed)
    nb = N // 2
    cen = rng.random((12, d)) * 0.8 + 0.1
    cl = cen[rng.integers(0, 12, N - nb)] + rng.standard_normal((N - nb, d)) * 0.004
    p = np.concatenate([rng.random((nb, d)), cl]).astype(np.float32)
    return p[rng.permutation(N)]


def _marked(certs, N):
    torch.cuda.synchronize()
    return np.flatnonzero(certs.nn.cpu().numpy() != SENTINEL)


@pytest.mark.parametrize("d,N", [(3, 300007), (2, 262147)])
def test_sweep_at_every_density_on_a_fresh_grid(d, N):
    p = _points(d, N, 70 + d)
    grid = kc.Grid(N, kc.kc_geom_for(dev(p)))
    kc.kc_grid_build(grid, dev(p))
    if d == 3:
        assert grid.info().n_heavy > 0
    want = oracle.kdtree_top2(p)
    rng = np.random.default_rng(5)
    # 12.6 % ... 100 %: sweep spans of 7, 5, 3, 2 and 1 x 32 slots per warp (d = 3); below N/8: the list kernel
    for f in (0.126, 0.17, 0.29, 0.44, 0.46, 0.7, 1.0, 0.06):
        ids = np.sort(rng.choice(N, int(N * f), replace=False)).astype(np.int32)
        certs = kc.Certs.empty(N, "cuda")
        certs.nn.fill_(SENTINEL)
        kc.kc_frontier_search(grid, dev(p), dev(ids), dev(np.array([ids.size], np.int32)), certs)
        assert_same(certs, want, idx=ids, what=f"d{d} sweep at {f:.0%}")
        assert np.array_equal(_marked(certs, N), ids), f"d{d} sweep at {f:.0%}: entries outside the list written"
    # a list that is clustered in slot order (one spatial region): warps with 0, a few and all slots marked
    near = np.flatnonzero(np.abs(p[:, 0] - 0.5) < 0.09).astype(np.int32)
    assert near.size * 8 >= N
    certs = kc.Certs.empty(N, "cuda")
    certs.nn.fill_(SENTINEL)
    kc.kc_frontier_search(grid, dev(p), dev(near), dev(np.array([near.size], np.int32)), certs)
    assert_same(certs, want, idx=near, what=f"d{d} sweep of a slab")
    assert np.array_equal(_marked(certs, N), near)


@pytest.mark.parametrize("d,N", [(3, 300007), (2, 262147)])
def test_sweep_at_every_density_on_an_updated_grid(d, N):
    """2 % of the points move by up to two cell widths first (tombstones, chains, sub-cell changes); the
    frontier lists mix movers and resting points."""
    p = _points(d, N, 80 + d)
    g_kc = kc.kc_geom_for(dev(p))
    grid = kc.Grid(N, g_kc)
    kc.kc_grid_build(grid, dev(p))
    rng = np.random.default_rng(6)
    movers = np.sort(rng.choice(N, N // 50, replace=False)).astype(np.int32)
    q = p.copy()
    q[movers] += rng.uniform(-2, 2, (movers.size, d)).astype(np.float32) * np.float32(g_kc.h)
    q = np.clip(q, 0, 1).astype(np.float32)
    kc.kc_grid_update(grid, dev(q), dev(movers))
    info = grid.info()
    assert info.dirty == 1 and info.n_misfiled > 0
    want = oracle.kdtree_top2(q)
    for f in (0.13, 0.22, 0.4, 0.5, 1.0):
        rest = rng.choice(N, int(N * f), replace=False).astype(np.int32)
        ids = np.union1d(rest, movers[::2]).astype(np.int32)
        certs = kc.Certs.empty(N, "cuda")
        certs.nn.fill_(SENTINEL)
        kc.kc_frontier_search(grid, dev(q), dev(ids), dev(np.array([ids.size], np.int32)), certs)
        assert_same(certs, want, idx=ids, what=f"d{d} sweep on the updated grid at {f:.0%}")
        assert np.array_equal(_marked(certs, N), ids), f"d{d} updated grid at {f:.0%}: entries outside the list written"


def test_device_count_decides_the_sweep_shape():
    """nF_max is only a bound: the same call shape (list buffer of N ids) with device counts of 3 %, 20 %
    and 90 % of the points goes to the list kernel, the compacting sweep and the direct sweep."""
    d, N = 3, 300007
    p = _points(d, N, 91)
    grid = kc.Grid(N, kc.kc_geom_for(dev(p)))
    kc.kc_grid_build(grid, dev(p))
    want = oracle.kdtree_top2(p)
    rng = np.random.default_rng(7)
    perm = rng.permutation(N).astype(np.int32)
    F = dev(perm)
    for f in (0.03, 0.2, 0.9, 0.2):
        n = int(N * f)
        certs = kc.Certs.empty(N, "cuda")
        certs.nn.fill_(SENTINEL)
        kc.kc_frontier_search(grid, dev(p), F, dev(np.array([n], np.int32)), certs, nF_max=N)
        ids = np.sort(perm[:n])
        assert_same(certs, want, idx=ids, what=f"device count {f:.0%} of a full-length buffer")
        assert np.array_equal(_marked(certs, N), ids)
