"""The second kernel of the d = 3 leaf search (DESIGN.md section 5 A3): on grids of >= 100,000 points with
subdivided cells, queries whose ball reaches beyond what phase 1 served go to a list and are finished by
ball_finish_kernel.  Exactness of the whole-set search, of the slot sweep on a fresh and on an updated
grid (chains, tombstones), and of consecutive calls (the list is emptied by the kernel itself)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_18314_b200 import binding as kc

from _util import assert_same, dev, geoms, ref_certs

pytestmark = pytest.mark.gpu


def blob_scene(N, seed, n_blobs, sigma, frac=0.6, far=0):
    """Uniform background + tight Gaussian blobs (subdivided cells next to undivided dense ones), optionally
    a few isolated points far outside (ring search / hand-off inside a deferring grid)."""
    rng = np.random.default_rng(seed)
    nb = int(N * (1 - frac)) - far
    bg = rng.random((nb, 3))
    c = 0.1 + 0.8 * rng.random((n_blobs, 3))
    lab = rng.integers(0, n_blobs, N - nb - far)
    parts = [bg, c[lab] + sigma * rng.standard_normal((N - nb - far, 3))]
    if far:
        parts.append(1.5 + rng.random((far, 3)))
    p = np.concatenate(parts)
    rng.shuffle(p, axis=0)
    return p.astype(np.float32)


@pytest.mark.parametrize("index", [None, (32, 2), (64, 8), (1024, 4)])
@pytest.mark.parametrize("N,n_blobs,sigma", [(150_003, 6, 4e-3), (262_144, 40, 2e-3), (120_000, 1, 5e-4)])
def test_whole_set_search_through_the_second_kernel(N, n_blobs, sigma, index):
    p = blob_scene(N, 11 + N % 97, n_blobs, sigma)
    g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    if index is not None:
        grid.set_index(*index)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    info = grid.info()
    want = ref_certs(p)
    assert_same(certs, want, what=f"N={N} index={index}")
    assert info.n_heavy >= 1
    if info.n_heavy * info.heavy_T * 32 >= N:
        assert info.n_deferred > 0                           # the second kernel has served queries
    # a second search on the same grid: the list was emptied, the count doubles, the bits are the same
    again = kc.kc_cert_grid_search(grid, kc.Certs.empty(N))
    assert_same(again, want, what="second search")
    assert grid.info().n_deferred == 2 * info.n_deferred


def test_uniform_grid_defers_nothing():
    N = 200_000
    p = np.random.default_rng(3).random((N, 3)).astype(np.float32)
    _, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    assert grid.info().n_heavy == 0 and grid.info().n_deferred == 0
    assert_same(certs, ref_certs(p), what="uniform")


def test_isolated_points_on_a_deferring_grid():
    """Far points: no bound after phase 1 (ring search, hand-off) beside deferred queries in the blobs."""
    N = 210_000
    p = blob_scene(N, 5, 40, 3e-3, far=24)
    _, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    info = grid.info()
    assert info.n_deferred > 0 and info.n_stragglers > 0
    assert_same(certs, ref_certs(p), what="far points")


@pytest.mark.parametrize("frac", [0.2, 0.6, 1.0])
@pytest.mark.parametrize("updated", [False, True])
def test_sweep_through_the_second_kernel(frac, updated):
    """A7 slot sweep (direct and compacting instantiations) on a fresh grid and on an incrementally updated
    one: movers leave their sub-cells (chains, tombstones), the frontier is a random subset."""
    N = 250_000
    p = blob_scene(N, 21, 80, 3e-3)
    g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    assert grid.info().n_deferred > 0
    rng = np.random.default_rng(int(frac * 10) + updated)
    q = p.copy()
    if updated:
        movers = np.sort(rng.choice(N, N // 40, replace=False)).astype(np.int32)     # below the re-bin bound: re-filed one by one
        q[movers] += rng.uniform(-3e-4, 3e-4, (movers.size, 3)).astype(np.float32)
    else:
        movers = np.zeros(0, np.int32)
    F = np.sort(rng.choice(N, int(N * frac), replace=False)).astype(np.int32)
    F = np.union1d(F, movers).astype(np.int32)
    Fd, nF = dev(F), dev(np.array([F.size], np.int32))
    before = grid.info().n_deferred
    if updated:
        kc.kc_frontier_repair(grid, dev(q), Fd, nF, certs, movers=dev(movers))
    else:
        kc.kc_frontier_search(grid, dev(q), Fd, nF, certs)
    info = grid.info()
    assert info.dirty == int(updated) and (info.n_misfiled > 0) == updated
    assert info.n_deferred > before
    post = ref_certs(q)
    assert_same(certs, post, idx=F, what=f"sweep frac={frac} updated={updated}")
    if updated:
        assert np.array_equal(grid.export(0).cpu().numpy(), oracle.cell_ids(q, g_or))
        # and once more on the same update: the marks and both lists are clean again
        kc.kc_frontier_search(grid, dev(q), Fd, nF, certs)
        assert_same(certs, post, idx=F, what="second sweep on one update")


def test_sweep_replays_from_a_cuda_graph_with_the_second_kernel():
    N = 220_000
    p = blob_scene(N, 33, 80, 3e-3)
    _, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    P = dev(p)
    certs = kc.kc_cert_grid_rebuild(grid, P)
    assert grid.info().n_deferred > 0
    want = ref_certs(p)
    F = dev(np.arange(0, N, 2, dtype=np.int32))
    nF = dev(np.array([F.numel()], np.int32))
    out = certs.clone()
    kc.kc_frontier_search(grid, P, F, nF, out)                # warm-up outside the capture
    torch.cuda.synchronize()
    gr = torch.cuda.CUDAGraph()
    with torch.cuda.graph(gr):
        kc.kc_frontier_search(grid, P, F, nF, out)
    for _ in range(3):
        for f in ("nn", "nn2"):
            getattr(out, f).fill_(-7)
        gr.replay()
        torch.cuda.synchronize()
        assert_same(out, want, idx=F.cpu().numpy(), what="graph replay")
