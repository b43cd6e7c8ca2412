"""Two-level index ("a hierarchical GPU index ... could lower its constant further"):
structure of the build and exactness of the searches on scenes with very dense cells."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_18314_b200 import binding as kc
from paper_2606_18314_b200 import workloads as wl

from _util import assert_same, dev, geoms, host, ref_certs

pytestmark = pytest.mark.gpu


def blob_scene(N, d, seed, n_blobs, sigma, frac=0.7):
    """Uniform background + a few very tight Gaussian blobs: cells with thousands of records."""
    rng = np.random.default_rng(seed)
    nb = int(N * (1 - frac))
    bg = rng.random((nb, d))
    c = rng.random((n_blobs, d))
    lab = rng.integers(0, n_blobs, N - nb)
    p = np.concatenate([bg, c[lab] + sigma * rng.standard_normal((N - nb, d))])
    rng.shuffle(p, axis=0)
    return p.astype(np.float32)


def check_structure(grid, p, g_or):
    """Level 0 unchanged (cell_start, permutation); inside a subdivided cell the leaves tile the
    cell's range and every record lies in the box of its sub-cell (up to rounding)."""
    N, d = p.shape
    info = grid.info()
    cid = oracle.cell_ids(p, g_or)
    counts = np.bincount(cid, minlength=g_or.n_cells)
    start = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    assert np.array_equal(grid.export(1).cpu().numpy(), start)
    sidx = grid.export(2).cpu().numpy()
    slot = grid.export(3).cpu().numpy()
    assert np.array_equal(np.sort(sidx), np.arange(N)) and np.array_equal(slot[sidx], np.arange(N))
    assert np.array_equal(cid[sidx], np.repeat(np.arange(g_or.n_cells), counts))
    heavy = np.flatnonzero(counts >= info.heavy_T)
    assert info.n_heavy == heavy.size
    if heavy.size == 0:
        return info
    sub = grid.export(5).cpu().numpy().reshape(-1, 2)
    leaf_start = grid.export(6).cpu().numpy()[: info.n_leaves + 1]
    assert leaf_start[0] == 0 and leaf_start[-1] == N and np.all(np.diff(leaf_start) >= 0)
    S = sub[:, 0]
    assert np.all(S[heavy] >= 2) and np.all(S[counts < info.heavy_T] == 0)
    nleaf = np.where(S > 0, S.astype(np.int64) ** d, 1)
    assert np.array_equal(sub[:, 1], np.concatenate([[0], np.cumsum(nleaf)[:-1]]))
    assert info.n_leaves == nleaf.sum()
    assert np.all(S[heavy].astype(np.int64) ** d <= np.maximum(counts[heavy], 2 ** d))
    G = np.array(g_or.G[:d])
    lo = np.array(g_or.lo[:d], np.float64)
    h = float(g_or.h)
    for c in heavy[np.argsort(-counts[heavy])[:40]]:
        s, first = int(S[c]), int(sub[c, 1])
        ls = leaf_start[first: first + s ** d + 1]
        assert ls[0] == start[c] and ls[-1] == start[c + 1]
        k = np.array([c % G[0], (c // G[0]) % G[1]] + ([c // (G[0] * G[1])] if d == 3 else []))
        for u in np.random.default_rng(c).choice(s ** d, min(s ** d, 30), replace=False):
            ids = sidx[ls[u]: ls[u + 1]]
            if ids.size == 0:
                continue
            uu = np.array([u % s, (u // s) % s] + ([u // (s * s)] if d == 3 else []))
            f = (p[ids].astype(np.float64) - lo) / h - k            # position inside the cell, in [0, 1)
            inside = (f * s >= uu - 1e-3) & (f * s <= uu + 1 + 1e-3)
            # points outside the grid box are clamped into boundary cells and boundary sub-cells
            clamped = ((uu == 0) & (f * s < uu)) | ((uu == s - 1) & (f * s > uu + 1))
            assert np.all(inside | clamped), (c, u)
    return info


@pytest.mark.parametrize("index", [None, (1, 1), (1, 2), (64, 8)])
@pytest.mark.parametrize("d,N,n_blobs,sigma", [(2, 40000, 3, 2e-3), (3, 40000, 2, 4e-3), (3, 9000, 1, 1e-4),
                                              (2, 9000, 1, 1e-5)])
def test_two_level_build_and_search_dense_cells(d, N, n_blobs, sigma, index):
    p = blob_scene(N, d, 100 + d + N, n_blobs, sigma)
    g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    if index is not None:                                   # (heavy_T, sub_occ): many small sub-grids ... few large ones
        grid.set_index(*index)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    info = check_structure(grid, p, g_or)
    assert info.max_occ >= 2000
    # the second level is on by default for d = 3 only (d = 2: kc_grid_set_index switches it on)
    assert (info.n_heavy >= 1) == (d == 3 or index is not None)
    assert_same(certs, ref_certs(p), what=f"dense cells d={d} N={N}")


@pytest.mark.parametrize("d", [2, 3])
def test_every_point_in_one_cell(d):
    """The geometry is fitted to a far larger box: all N points fall into ONE level-0 cell, which the
    second level subdivides (S^d sub-cells at ~2 records each)."""
    N = 12000
    p = (0.5 + 1e-3 * np.random.default_rng(7 + d).random((N, d))).astype(np.float32)
    g_or, g_kc = geoms(p, lo=np.zeros(d, np.float32), hi=np.full(d, 64.0, np.float32))
    grid = kc.Grid(N, g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    grid.set_index(64, 2)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    info = check_structure(grid, p, g_or)
    assert info.max_occ == N and info.c_occ == 1 and info.n_heavy == 1
    assert_same(certs, ref_certs(p), what=f"one cell d={d}")
    # duplicates and exact ties inside a subdivided cell
    q = np.round(p * 4096) / 4096
    q = q.astype(np.float32)
    assert_same(kc.kc_cert_grid_rebuild(grid, dev(q)), ref_certs(q), what=f"one cell, lattice-snapped d={d}")


@pytest.mark.parametrize("d", [2, 3])
def test_repair_on_subdivided_cells(d):
    """A6 + A7 on a grid with subdivided cells: a mover that leaves its sub-cell is re-filed (chain
    of its level-0 cell) even when the level-0 cell is unchanged; repaired entries are exact."""
    N = 30000
    p = blob_scene(N, d, 55 + d, 4, 3e-3)
    g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    grid.set_index(16, 2)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    rng = np.random.default_rng(9)
    for step in range(3):
        movers = np.sort(rng.choice(N, N // 5, replace=False)).astype(np.int32)
        q = p.copy()
        q[movers] += rng.uniform(-2e-4, 2e-4, (movers.size, d)).astype(np.float32)
        F = np.sort(rng.choice(N, N // 2, replace=False)).astype(np.int32)
        Fd, nF = dev(F), dev(np.array([F.size], np.int32))
        kc.kc_frontier_repair(grid, dev(q), Fd, nF, certs, movers=dev(movers))
        post = ref_certs(q)
        assert_same(certs, post, idx=F, what=f"repair step {step}")
        assert np.array_equal(grid.export(0).cpu().numpy(), oracle.cell_ids(q, g_or))
        certs = kc.Certs(*(dev(x) for x in (post.nn, post.nn2, post.d1, post.d2, post.c)))
        p = q
    assert grid.info().n_misfiled > 0


@pytest.mark.parametrize("cfg", ["cfg3", "cfg5_d2", "cfg5_d3"])
def test_index_parameters_never_change_a_result(cfg):
    """Config scenes with the second level forced on everywhere it can apply (small thresholds)
    and switched off: rebuild and a sweep-sized repair are bit-exact either way."""
    N = 250_000 if cfg != "cfg3" else 16000
    p, mot = wl.make_scene(cfg, "cluster_drift" if cfg == "cfg3" else None, N=N)
    q, _ = mot.step(p)
    want, post = ref_certs(p), ref_certs(q)
    F = np.sort(np.random.default_rng(3).choice(N, N // 2, replace=False)).astype(np.int32)
    movers = np.sort(np.random.default_rng(4).choice(N, N // 12, replace=False)).astype(np.int32)
    q2 = p.copy(); q2[movers] = q[movers]
    post2 = ref_certs(q2)
    for index in [(1, 1), (1, 4), (32, 2), (10 ** 9, 4)]:
        grid = kc.Grid(N, geoms(p)[1])
        grid.set_index(*index)
        certs = kc.kc_cert_grid_rebuild(grid, dev(p))
        assert_same(certs, want, what=f"{cfg} index={index}")
        kc.kc_frontier_repair(grid, dev(q2), dev(F), dev(np.array([F.size], np.int32)), certs, movers=dev(movers))
        assert_same(certs, post2, idx=F, what=f"{cfg} index={index} repair")


def test_set_index_arguments():
    p = wl.uniform_points(1000, 3, 1)
    grid = kc.Grid(1000, geoms(p)[1])
    for bad in [(0, 4), (16, 0), (16, 65), (-3, 2)]:
        with pytest.raises(kc.KcError) as e:
            grid.set_index(*bad)
        assert e.value.status == kc.KC_EINVAL
    grid.set_index(1, 1)                       # raised to sub_occ * 2^(d+1)
    kc.kc_grid_build(grid, dev(p))
    assert grid.info().heavy_T == 16
    grid.set_index(5, 4)
    with pytest.raises(kc.RebuildRequired):    # takes effect with the next build: not built until then
        kc.kc_cert_grid_search(grid, kc.Certs.empty(1000))


@pytest.mark.parametrize("d", [2, 3])
@pytest.mark.parametrize("N", [2, 3, 5, 17, 33, 64, 129])
def test_tiny_sets_in_one_subdivided_cell(d, N):
    """Few points, one level-0 cell, second level forced on: short lists (N = 2: d2 = +inf), duplicates,
    empty sub-cells, windows clipped on every side."""
    rng = np.random.default_rng(100 * d + N)
    p = (0.25 + 0.01 * rng.random((N, d))).astype(np.float32)
    if N >= 5:
        p[3] = p[1]                                         # a coincident pair
    g_or, g_kc = geoms(p, lo=np.zeros(d, np.float32), hi=np.ones(d, np.float32), occ=float(N))
    assert g_kc.n_cells == 1
    grid = kc.Grid(N, g_kc)
    grid.set_index(1, 1)
    assert_same(kc.kc_cert_grid_rebuild(grid, dev(p)), oracle.bruteforce_top2(p), what=f"tiny d={d} N={N}")


@pytest.mark.parametrize("offset", [0.0, 4096.5, -3.0e5])
def test_dense_cells_far_from_origin_and_outside_the_box(offset):
    """The ball's index box (R22) rests on the monotonicity of the filing functions only:
    dense blobs far from the origin (coarse float spacing, many exact ties and duplicates after the
    cast) and a geometry fitted to the central part of the points (the rest is clamped into boundary
    cells and boundary sub-cells)."""
    p = blob_scene(30000, 3, 71, 3, 2e-3).astype(np.float64) + offset
    p = p.astype(np.float32)
    want = ref_certs(p)
    lo, hi = p.min(0), p.max(0)
    for shrink in (0.0, 0.3):
        g_or, g_kc = geoms(p, lo=lo + shrink * (hi - lo), hi=hi - shrink * (hi - lo))
        for index in [None, (16, 1), (64, 4)]:
            grid = kc.Grid(p.shape[0], g_kc)
            if index is not None:
                grid.set_index(*index)
            assert_same(kc.kc_cert_grid_rebuild(grid, dev(p)), want, what=f"offset {offset} shrink {shrink} index {index}")
