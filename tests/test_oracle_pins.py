"""Pins for the CPU oracle (CPU only): the oracle is checked against what the paper and the
mathematics fix — hand-worked scenes (tests/golden), Theorem 1's tightness construction
(PAPER.md:169), lattice and entropy closed forms, Lemma 1 / Theorem 3 invariants, an independent
fp64 k-d tree (scipy), and exact rational brute force on tiny inputs — never against itself.
"""
import json
import math
import os
import struct
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2606_18314_b200 import workloads as wl


def bits(a):
    return [("%08x" % struct.unpack("<I", struct.pack("<f", float(x)))[0]) for x in a]


def load(golden_dir, name):
    with open(os.path.join(golden_dir, name)) as f:
        return json.load(f)


# ------------------------------------------------------------------ P1, P2, P2b
@pytest.mark.parametrize("name", ["p1_scene2d.json", "p2_tie_scene.json", "p2b_scene3d.json"])
@pytest.mark.parametrize("impl", ["brute", "kdtree"])
def test_hand_worked_scenes(golden_dir, name, impl):
    g = load(golden_dir, name)
    p = np.array(g["points"], np.float32)
    r = oracle.bruteforce_top2(p) if impl == "brute" else oracle.kdtree_top2(p)
    assert r.nn.tolist() == g["nn"]
    assert r.nn2.tolist() == g["nn2"]
    s1 = [float(Fraction(s)) for s in g["s1"]]
    s2 = [float(Fraction(s)) for s in g["s2"]]
    # d^2 recovers the exact rational to binary32 rounding of one sqrt
    np.testing.assert_allclose(r.d1.astype(np.float64) ** 2, s1, rtol=3e-7)
    np.testing.assert_allclose(r.d2.astype(np.float64) ** 2, s2, rtol=3e-7)
    if "d1_bits" in g:
        assert bits(r.d1) == g["d1_bits"]
        assert bits(r.d2) == g["d2_bits"]
    assert bits(r.c) == g["c_bits"]


# ------------------------------------------------------------------ P3 (Theorem 1 tightness)
def test_theorem1_tightness(golden_dir):
    g = load(golden_dir, "p3_tightness.json")
    d1, eps = g["d1"], g["eps"]
    for case in g["cases"]:
        eta = case["eta"]
        p = np.array([[0.0, 0.0], [d1, 0.0], [-(d1 + eta * eps), 0.0]], np.float32)
        q = np.array([[-eps, 0.0], [d1 + eps, 0.0], [-(d1 + eta * eps) + eps, 0.0]], np.float32)
        pre = oracle.bruteforce_top2(p)
        assert pre.nn[0] == case["nn_pre"]
        assert float(pre.c[0]) == case["c_pre"]
        e = oracle.max_displacement(p, q)
        assert float(e) == eps                                   # O3: every point moved exactly eps
        flags, F = oracle.frontier(pre.c, e)
        assert bool(flags[0]) == case["in_frontier"]             # inclusive threshold at eta = 4
        post = oracle.bruteforce_top2(q)
        assert post.nn[0] == case["nn_post"]
        assert float(post.d1[0]) == case["d1_post"]
        assert float(post.d2[0]) == case["d2_post"]
        # Definition 2 / Table 1 audit on the same scene: only i can fail (a and k keep nn = i and
        # have clearance ~d1 >> 4 eps); eta = 3 fails and is detected, eta = 4 is flagged but holds
        Ft, counts = oracle.failure_audit(pre.nn, post.nn, flags)
        want = {3: ([0], [1, 1, 0, 0]), 4: ([], [0, 0, 0, 1]), 5: ([], [0, 0, 0, 0])}[eta]
        assert Ft.tolist() == want[0] and counts.tolist() == want[1]


# ------------------------------------------------------------------ O1 against exact rationals
def test_sqdist_is_left_to_right_separately_rounded():
    rng = np.random.default_rng(11)
    f32 = np.float32
    for d in (2, 3):
        for _ in range(200):
            a = rng.standard_normal(d).astype(f32)
            b = (a + rng.standard_normal(d).astype(f32) * f32(1e-3)).astype(f32)
            # exact rational evaluation with a binary32 rounding after every operation
            def rnd(x):
                return Fraction(float(f32(float(x))))
            dx = [rnd(Fraction(float(a[k])) - Fraction(float(b[k]))) for k in range(d)]
            sq = [rnd(v * v) for v in dx]
            acc = rnd(sq[0] + sq[1])
            if d == 3:
                acc = rnd(acc + sq[2])
            assert Fraction(float(oracle.sqdist(a, b))) == acc


def test_sqdist_no_fma_witness():
    # dx*dx + dy*dy with a fused multiply-add differs from separately rounded ops here:
    # dx = 1+2^-12 -> dx*dx = 1 + 2^-11 + 2^-24 (needs 25 bits; rounds to 1 + 2^-11, tie to even)
    a = np.array([1.0 + 2.0 ** -12, 2.0 ** -12], np.float32)
    b = np.zeros(2, np.float32)
    xx = np.float32(a[0]) * np.float32(a[0])
    yy = np.float32(a[1]) * np.float32(a[1])
    want = np.float32(xx + yy)
    assert oracle.sqdist(a, b) == want
    fused = np.float32(float(a[0]) * float(a[0]) + float(yy))    # what an FMA would give
    assert fused != want, "witness must separate fused from unfused evaluation"


# ------------------------------------------------------------------ P4 tiny exact brute force
def exact_top2(p):
    n = len(p)
    P = [[Fraction(float(v)) for v in row] for row in p]
    out = []
    for i in range(n):
        keys = sorted((sum((a - b) ** 2 for a, b in zip(P[i], P[j])), j) for j in range(n) if j != i)
        out.append(keys[:2])
    return out


@pytest.mark.parametrize("d", [2, 3])
@pytest.mark.parametrize("n", [2, 3, 4, 5, 31, 32, 33])
def test_tiny_against_exact_rational(n, d):
    # coordinates on a 2^-6 lattice in [0,4): every fp32 op is exact, so the fp32 key order must
    # equal the exact rational order (ties included)
    rng = np.random.default_rng(100 * n + d)
    p = (rng.integers(0, 256, (n, d)) / 64.0).astype(np.float32)
    ex = exact_top2(p)
    for r in (oracle.bruteforce_top2(p), oracle.kdtree_top2(p)):
        for i in range(n):
            assert r.nn[i] == ex[i][0][1]
            assert float(r.d1[i]) == float(np.sqrt(np.float32(float(ex[i][0][0]))))
            if n > 2:
                assert r.nn2[i] == ex[i][1][1]
                assert float(r.d2[i]) == float(np.sqrt(np.float32(float(ex[i][1][0]))))
            else:
                assert r.nn2[i] == -1 and np.isinf(r.d2[i]) and np.isinf(r.c[i])   # reading A4


def test_duplicates_are_neighbours():
    # reading A3: only j = i is excluded; coincident points are neighbours at distance 0
    p = np.array([[0.5, 0.5], [0.5, 0.5], [0.5, 0.5], [0.75, 0.5]], np.float32)
    for r in (oracle.bruteforce_top2(p), oracle.kdtree_top2(p)):
        assert r.nn.tolist() == [1, 0, 0, 0]
        assert r.nn2.tolist() == [2, 2, 1, 1]
        assert r.d1.tolist() == [0.0, 0.0, 0.0, 0.25]
        assert r.c.tolist() == [0.0, 0.0, 0.0, 0.0]


# ------------------------------------------------------------------ P5 lattice closed form
@pytest.mark.parametrize("d,side", [(2, 17), (3, 7)])
def test_lattice_closed_form(d, side):
    p = wl.lattice_points(side, d)
    for r in (oracle.bruteforce_top2(p), oracle.kdtree_top2(p)):
        assert np.all(r.d1 == np.float32(1 / 64)) and np.all(r.d2 == np.float32(1 / 64))
        assert np.all(r.c == 0)
        # smallest-index axis neighbour: index strides are side^(d-1-axis); the -stride of the
        # slowest axis is the smallest index when it exists
        idx = np.arange(side ** d).reshape((side,) * d)
        for i in (0, side ** d - 1, (side ** d) // 2):
            coord = np.unravel_index(i, (side,) * d)
            nb = []
            for a in range(d):
                for s in (-1, 1):
                    cc = list(coord)
                    cc[a] += s
                    if 0 <= cc[a] < side:
                        nb.append(int(idx[tuple(cc)]))
            nb.sort()
            assert r.nn[i] == nb[0] and r.nn2[i] == nb[1]
    flags, F = oracle.frontier(r.c, 0.0)
    assert F.size == side ** d                                   # c = 0 <= 4*0: everyone, even eps=0


# ------------------------------------------------------------------ P9 / P10 statistical agreement
@pytest.mark.parametrize("cfg,N", [("cfg1", 1000), ("cfg2", 4000), ("cfg3", 4000), ("cfg5_d2", 6000), ("cfg5_d3", 6000)])
def test_brute_kdtree_scipy_agree(cfg, N):
    from scipy.spatial import cKDTree
    p = wl.make_points(cfg, N=N)
    b = oracle.bruteforce_top2(p)
    k = oracle.kdtree_top2(p)
    for f in ("nn", "nn2"):
        assert np.array_equal(getattr(b, f), getattr(k, f))
    for f in ("d1", "d2", "c"):
        assert np.array_equal(getattr(b, f).view(np.uint32), getattr(k, f).view(np.uint32))
    # independent fp64 k-d tree: same neighbours wherever the fp64 gap is not a near-tie
    dd, ii = cKDTree(p.astype(np.float64)).query(p.astype(np.float64), k=3)
    clear = (dd[:, 2] - dd[:, 1]) > 1e-6 * dd[:, 2]
    clear1 = (dd[:, 1] > 0) & clear
    assert np.array_equal(b.nn[clear1], ii[clear1, 1])
    np.testing.assert_allclose(b.d1, dd[:, 1], rtol=2e-6, atol=1e-9)
    np.testing.assert_allclose(b.d2, dd[:, 2], rtol=2e-6, atol=1e-9)
    # invariants (P9)
    assert np.all(b.d1 <= b.d2) and np.all(b.c >= 0)
    assert np.all(b.d1[b.nn] <= b.d1)
    i0 = int(np.argmin(b.d1))
    assert b.nn[b.nn[i0]] == i0 or b.d1[b.nn[i0]] == b.d1[i0]
    # s(i, nn_i) recomputed by O1 gives d1
    for i in range(0, N, 97):
        assert np.sqrt(oracle.sqdist(p[i], p[b.nn[i]])) == b.d1[i]
        assert np.sqrt(oracle.sqdist(p[i], p[b.nn2[i]])) == b.d2[i]


def test_subset_queries_match_full():
    p = wl.make_points("cfg3", N=3000)
    full = oracle.bruteforce_top2(p)
    q = np.array([0, 5, 17, 2999, 1500], np.int32)
    for r in (oracle.bruteforce_top2(p, queries=q), oracle.kdtree_top2(p, queries=q)):
        assert np.array_equal(r.nn, full.nn[q]) and np.array_equal(r.nn2, full.nn2[q])
        assert np.array_equal(r.c, full.c[q])


# ------------------------------------------------------------------ P11 far outlier
def test_far_outlier_kdtree():
    rng = np.random.default_rng(5)
    p = (0.5 + 0.01 * rng.standard_normal((2000, 2))).astype(np.float32)
    p[777] = (40.0, -35.0)
    b = oracle.bruteforce_top2(p)
    k = oracle.kdtree_top2(p)
    assert np.array_equal(b.nn, k.nn) and np.array_equal(b.c, k.c)
    assert b.d1[777] > 40.0


# ------------------------------------------------------------------ O3 / O4
def test_max_displacement_and_frontier_threshold():
    p = np.zeros((5, 2), np.float32)
    q = p.copy()
    q[3] = (3 / 1024, 4 / 1024)                                  # norm exactly 5/1024
    q[1] = (1 / 1024, 0)
    assert float(oracle.max_displacement(p, q)) == 5 / 1024
    assert float(oracle.max_displacement(p, p)) == 0.0
    c = np.array([0.0, 4 * 5 / 1024, np.nextafter(np.float32(20 / 1024), np.float32(1)), np.inf, 1e-9],
                 np.float32)
    flags, F = oracle.frontier(c, np.float32(5 / 1024))
    assert flags.tolist() == [1, 1, 0, 0, 1] and F.tolist() == [0, 1, 4]


# ------------------------------------------------------------------ O5 / A6 geometry
def test_geometry_rule():
    # G = smallest integer with G^d >= ceil(N/2): values of SURVEY.md §8 grid table
    for N, d, G in [(1000, 2, 23), (16000, 2, 90), (16000, 3, 20), (262144, 3, 51),
                    (4194304, 2, 1449), (4194304, 3, 128), (1048576, 2, 725), (1048576, 3, 81)]:
        g = oracle.geom_from_bbox(N, d, np.zeros(3, np.float32), np.ones(3, np.float32), 2.0)
        assert g.G[0] == G and g.G[1] == G and g.G[2] == (G if d == 3 else 1)
        assert (G - 1) ** d < math.ceil(N / 2) <= G ** d
        assert float(g.h) == float(np.float32(1.0 / G * (1 + 2.0 ** -20)))
        assert float(g.inv_h) == float(np.float32(1.0 / float(g.h)))


def _heap_scene(d, R, m, N, seed=0):
    """N points in [0,1]^d whose coarse R^d histogram is known: m points inside every coarse cell (well
    away from its faces), the remaining N - m R^d in one cell; the two box corners are among them."""
    rng = np.random.default_rng(seed)
    cells = np.stack(np.meshgrid(*[np.arange(R)] * d, indexing="ij"), -1).reshape(-1, d)
    base = (np.repeat(cells, m, axis=0) + rng.uniform(0.2, 0.8, (cells.shape[0] * m, d))) / R
    heap = (np.full((N - base.shape[0], d), R // 2) + rng.uniform(0.2, 0.8, (N - base.shape[0], d))) / R
    p = np.concatenate([base, heap]).astype(np.float32)
    p[0] = 0.0                                                    # cell (0,..,0) keeps its m points
    p[base.shape[0] - 1] = 1.0                                    # so does cell (R-1,..,R-1)
    return p[rng.permutation(N)]


@pytest.mark.parametrize("d,R,G_of_k", [(2, 8, {0: 46, 1: 32, 2: 23}), (3, 4, {0: 13, 1: 11, 2: 8})])
def test_geometry_by_median_density_hand_worked(d, R, G_of_k):
    # Reading R24.  N = 4096 = 64 R^d, so the coarse grid has R cells per axis; with m points in every
    # coarse cell and the rest heaped into one, the lower median of the occupied counts is m and
    # N / n_eff = 64 / m.  k = that ratio's log2 rounded to the nearest integer, clamped to 0..2 (the
    # boundaries are sqrt(2) = 1.414 and 2 sqrt(2) = 2.828), and the grid is the occupancy-2 grid of
    # ceil(N / 2^k) points: G = smallest integer with G^d >= 2048 / 1024 / 512, written out by hand.
    N = 4096
    for m, k in [(64, 0), (49, 0), (46, 0), (45, 1), (32, 1), (23, 1), (22, 2), (16, 2), (4, 2)]:
        g = oracle.geom_by_median_density(_heap_scene(d, R, m, N), 2.0)
        G = G_of_k[k]
        assert g.G == (G, G, G if d == 3 else 1), (m, k, g.G)
        assert float(g.h) == float(np.float32(1.0 / G * (1 + 2.0 ** -20)))
        assert g.lo[:d] == (np.float32(0),) * d


def test_geometry_by_median_density_limits():
    # a uniform set: exactly the mean-occupancy geometry (k = 0)
    for N, d in [(1000, 2), (16000, 2), (16000, 3), (262144, 3)]:
        p = wl.uniform_points(N, d, 3)
        assert oracle.geom_by_median_density(p) == oracle.geom_for(p)
    # too few points for an estimate (R < 2): the mean-occupancy geometry, whatever the set looks like
    p = _heap_scene(2, 2, 1, 255)
    assert oracle.geom_by_median_density(p) == oracle.geom_for(p)
    # config 5's mixture (half of the points in 256 clusters of negligible volume): the background has
    # half the mean density, the cells are those of a set half the size
    for d in (2, 3):
        p = wl.mixture_points(262144, d, 5)
        lo, hi = oracle.bbox(p)
        assert oracle.geom_by_median_density(p) == oracle.geom_from_bbox(131072, d, lo, hi, 2.0)


def test_cell_ids_closed_form():
    # dyadic geometry: lo = 0, h = 1/8 exactly, G = 8 -> cell of x is floor(8x), faces go up
    g = oracle.Geom(2, (8, 8, 1), (np.float32(0), np.float32(0), np.float32(0)), np.float32(0.125), np.float32(8))
    p = np.array([[0, 0], [0.125, 0], [0.1249999, 0.999], [1.0, 1.0], [-3.0, 0.5], [0.5, 7.0], [0.374, 0.376]],
                 np.float32)
    assert oracle.cell_ids(p, g).tolist() == [0, 1, 7 * 8 + 0, 7 * 8 + 7, 4 * 8 + 0, 7 * 8 + 4, 3 * 8 + 2]
    g3 = oracle.Geom(3, (4, 4, 4), (np.float32(0),) * 3, np.float32(0.25), np.float32(4))
    p3 = np.array([[0.3, 0.6, 0.9], [0.99, 0.0, 0.26]], np.float32)
    assert oracle.cell_ids(p3, g3).tolist() == [(3 * 4 + 2) * 4 + 1, (1 * 4 + 0) * 4 + 3]
    # the bbox maximum always lands inside the grid without clamping doing the work elsewhere
    p = wl.uniform_points(5000, 3, 9)
    gg = oracle.geom_for(p)
    cid = oracle.cell_ids(p, gg)
    assert cid.min() >= 0 and cid.max() < gg.n_cells
    k = np.floor((p.astype(np.float64) - np.array(gg.lo, np.float64)) * float(gg.inv_h)).astype(int)
    lin = (k[:, 2] * gg.G[1] + k[:, 1]) * gg.G[0] + k[:, 0]
    assert np.mean(lin == cid) > 0.999                           # fp64 restatement agrees off the faces


# ------------------------------------------------------------------ P6 / P7 entropy
def test_entropy_closed_forms(golden_dir):
    g = load(golden_dir, "p6_entropy.json")
    for case in g["cases"]:
        counts, Cocc = case["counts"], case["C"]
        n_cells = Cocc + 3                                       # a few empty cells too
        cell_all, F = [], []
        for cix in range(Cocc):
            k = counts[cix] if cix < len(counts) else 0
            for t in range(max(k, 1)):                           # every one of the C cells is occupied
                if t < k:
                    F.append(len(cell_all))
                cell_all.append(cix)
            cell_all.append(cix)                                 # plus one non-frontier point
        H, m, Cc = oracle.entropy(np.array(cell_all, np.int32), np.array(F, np.int32), n_cells)
        assert Cc == Cocc and m == case["m"]
        assert abs(H - case["H"]) < 1e-12


def test_entropy_theorem3_and_limits():
    rng = np.random.default_rng(3)
    p = wl.uniform_points(20000, 2, 1)
    g = oracle.geom_for(p)
    cid = oracle.cell_ids(p, g)
    for frac in (0.001, 0.05, 0.5, 1.0):
        F = np.sort(rng.choice(p.shape[0], max(1, int(frac * p.shape[0])), replace=False)).astype(np.int32)
        H, m, Cc = oracle.entropy(cid, F, g.n_cells)
        assert 0.0 <= H <= 1.0
        assert m >= Cc ** H * (1 - 1e-12)                        # Theorem 3
        assert m == np.unique(cid[F]).size and Cc == np.unique(cid).size
    # localized: all frontier points from one cell -> H = 0
    one = np.flatnonzero(cid == cid[0]).astype(np.int32)
    assert oracle.entropy(cid, one, g.n_cells)[0] == 0.0
    # diffuse: one frontier point in every occupied cell -> H = 1
    _, first = np.unique(cid, return_index=True)
    assert abs(oracle.entropy(cid, np.sort(first).astype(np.int32), g.n_cells)[0] - 1.0) < 1e-12


# ------------------------------------------------------------------ P8 Lemma 1 (miss = 0)
@pytest.mark.parametrize("cfg,fam", [("cfg2", f) for f in wl.CONFIGS["cfg2"]["families"]] +
                         [("cfg3", f) for f in wl.CONFIGS["cfg3"]["families"]])
def test_lemma1_no_missed_failure(cfg, fam):
    p, mot = wl.make_scene(cfg, fam, N=3000)
    pre = oracle.kdtree_top2(p)
    for _ in range(3):
        q, movers = mot.step(p)
        eps_t = oracle.max_displacement(p, q)
        assert 0 < float(eps_t) <= wl.CONFIGS[cfg]["eps"] * 1.02 + 2e-5
        if movers is not None:
            still = np.setdiff1d(np.arange(p.shape[0]), movers)
            assert np.array_equal(p[still], q[still])
        flags, F = oracle.frontier(pre.c, eps_t)
        post = oracle.kdtree_top2(q)
        changed = np.flatnonzero(pre.nn != post.nn)
        assert np.all(flags[changed] == 1)                       # Table 1 "miss (safe)" = 0
        Ft, counts = oracle.failure_audit(pre.nn, post.nn, flags)
        assert np.array_equal(Ft, changed) and counts[2] == 0
        assert counts[0] == counts[1] == changed.size and counts[1] + counts[3] == F.size
        p, pre = q, post


# ------------------------------------------------------------------ NEXT #3: cumulative clock (A.2)
def test_clock_rule_hand_worked():
    """Appendix A.2: valid while S - S_i < c_i/4.  eps = 2^-10 per step (dyadic, exact):
    c = 10 eps expires at step 3 (4*3 eps >= 10 eps), c = 8 eps at step 2 (inclusive), c = 4 eps at
    step 1, c = 4.5 eps at step 2; a point re-stamped at step 2 with c = 8 eps expires again at step 4."""
    eps = np.float32(2.0 ** -10)
    c = np.array([10, 8, 4, 4.5, 1000], np.float32) * eps
    stamp = np.zeros(5, np.float32)
    S = 0.0
    seen = []
    for step in (1, 2, 3, 4):
        S, flags, F = oracle.clock_frontier(c, stamp, S, eps)
        assert S == step * float(eps)
        seen.append(F.tolist())
        stamp[F] = oracle.clock_stamp(S)
    assert seen == [[2], [1, 2, 3], [0, 2], [1, 2, 3]]
    # stamps round DOWN: the elapsed clock is never under-estimated
    for S in (0.1, 1.0 / 3.0, 1e-7, 123.456789):
        st = oracle.clock_stamp(S)
        assert float(st) <= S < float(np.nextafter(st, np.float32(np.inf)))


@pytest.mark.parametrize("cfg,fam", [("cfg2", "walk"), ("cfg2", "shear"), ("cfg3", "cluster_drift"), ("cfg3", "vortex")])
def test_clock_maintenance_keeps_nn_exact(cfg, fam):
    """The rule itself (Theorem 1 on cumulative displacement): recomputing only the expired points
    keeps every nearest neighbour exact over many steps, although most d1, d2 go stale."""
    p, mot = wl.make_scene(cfg, fam, N=2500)
    N = p.shape[0]
    cert = oracle.kdtree_top2(p)
    nn, c = cert.nn.copy(), cert.c.copy()
    stamp = np.zeros(N, np.float32)
    S, skipped = 0.0, 0
    for _ in range(12):
        q, _ = mot.step(p)
        S, flags, F = oracle.clock_frontier(c, stamp, S, oracle.max_displacement(p, q))
        post = oracle.kdtree_top2(q)
        nn[F], c[F] = post.nn[F], post.c[F]
        stamp[F] = oracle.clock_stamp(S)
        assert np.array_equal(nn, post.nn)
        skipped += N - F.size
        p = q
    assert skipped > 0


# ------------------------------------------------------------------ NEXT #2: local motion budget
def test_local_budget_hand_worked():
    """One far mover: Lemma 1's global rule flags every low-clearance certificate, the per-point
    budget only those whose block holds the mover.  Dyadic scene, h = 1/8."""
    p = np.array([[0.0, 0.0], [1 / 64, 0.0], [-5 / 256, 0.0],          # i, a, k: c_i = 1/256
                  [0.875, 0.875], [0.875 + 1 / 64, 0.875], [0.875, 0.875 - 5 / 256],   # the mover and two bystanders
                  [1.0, 1.0], [-0.0625, -0.0625]], np.float32)
    q = p.copy()
    q[3] += np.float32(1 / 256)                                        # eps = sqrt(2)/256 ~ 0.00552
    g = oracle.geom_from_bbox(8, 2, np.array([-0.0625, -0.0625, 0], np.float32), np.array([1, 1, 0], np.float32), 0.125)
    assert tuple(g.G[:2]) == (8, 8)
    pre = oracle.bruteforce_top2(p)
    eps = oracle.max_displacement(p, q)
    gflags, _ = oracle.frontier(pre.c, eps)
    lflags, LF = oracle.local_frontier(p, q, g, pre.nn, pre.d1, pre.c, eps)
    assert float(pre.c[0]) == 1 / 256 and gflags[0] == 1               # 4 eps ~ 0.022 > c_i
    assert lflags[0] == 0 and lflags[1] == 0 and lflags[2] == 0        # nothing moved in their block
    # the mover's block: c_3 = 0.0039 <= 3 eps, c_4 = 0.0094 and c_5 = 0.0055 <= d_a + D_B = 2 eps = 0.011
    assert lflags[3] == 1 and lflags[4] == 1 and lflags[5] == 1
    assert np.all(lflags <= gflags)


@pytest.mark.parametrize("cfg,fam", [("cfg2", f) for f in wl.CONFIGS["cfg2"]["families"]] +
                         [("cfg3", f) for f in wl.CONFIGS["cfg3"]["families"]])
def test_local_budget_never_misses(cfg, fam):
    """No-miss guarantee of the per-point budget and F_local subset of Lemma 1's set, on all ten
    families; on the partial-motion families the local frontier is several times smaller."""
    p, mot = wl.make_scene(cfg, fam, N=4000)
    pre = oracle.kdtree_top2(p)
    ratio = []
    for _ in range(3):
        q, movers = mot.step(p)
        g = oracle.geom_for(p)
        eps = oracle.max_displacement(p, q)
        gflags, GF = oracle.frontier(pre.c, eps)
        lflags, LF = oracle.local_frontier(p, q, g, pre.nn, pre.d1, pre.c, eps)
        post = oracle.kdtree_top2(q)
        changed = np.flatnonzero(pre.nn != post.nn)
        assert np.all(lflags[changed] == 1)
        assert np.all(lflags <= gflags)
        ratio.append(LF.size / max(GF.size, 1))
        p, pre = q, post
    if fam in ("local", "diffuse5", "ball5"):
        assert max(ratio) < 0.5


# ------------------------------------------------------------------ NEXT #4: K-list certificates
def test_topk_hand_worked(golden_dir):
    """Reading R20 on the hand-worked scenes (lists, distance bits, clearance bits, tie rule)."""
    for g in load(golden_dir, "p7_topk_lists.json")["scenes"]:
        p = np.array(g["points"], np.float32)
        nnk, dk, ck = oracle.bruteforce_topk(p, g["K"])
        assert nnk.tolist() == g["nnk"]
        assert [[b for b in bits(row)] for row in dk] == g["dk_bits"]
        assert [b for b in bits(ck)] == g["ck_bits"]


def numpy_topk(p, K):
    """Independent restatement with library routines: float32 numpy arithmetic (one rounding per
    operation, left to right) and a lexicographic sort of the keys (s, j)."""
    p = np.asarray(p, np.float32)
    N, d = p.shape
    ids = np.empty((N, K), np.int32)
    dist = np.empty((N, K), np.float32)
    for i in range(N):
        df = p[i] - p
        sq = df * df
        s = sq[:, 0] + sq[:, 1]
        if d == 3:
            s = s + sq[:, 2]
        j = np.delete(np.arange(N), i)
        s = np.delete(s, i)
        o = np.lexsort((j, s))[:K]
        ids[i], dist[i] = j[o], np.sqrt(s[o])
    return ids, dist, dist[:, K - 1] - dist[:, K - 2]


@pytest.mark.parametrize("d", [2, 3])
@pytest.mark.parametrize("K", [2, 3, 5, 8])
def test_topk_against_numpy_lexsort(d, K):
    rng = np.random.default_rng(100 * d + K)
    scenes = [rng.random((400, d)).astype(np.float32),
              (rng.integers(0, 6, (300, d)) / 8).astype(np.float32)]        # lattice: ties and duplicates
    for p in scenes:
        nnk, dk, ck = oracle.bruteforce_topk(p, K)
        ids, dist, c = numpy_topk(p, K)
        assert np.array_equal(nnk, ids)
        assert np.array_equal(dk.view(np.uint32), dist.view(np.uint32))
        assert np.array_equal(ck.view(np.uint32), c.view(np.uint32))
    q = np.array([7, 0, 399, 7], np.int32)
    a = oracle.bruteforce_topk(scenes[0], K, queries=q)
    for x, y in zip(a, oracle.bruteforce_topk(scenes[0], K)):
        assert np.array_equal(x, y[q])


@pytest.mark.parametrize("cfg", ["cfg1", "cfg3"])
def test_topk_with_K2_is_definition_1(cfg):
    """K = 2 is the paper's certificate: same nn, nn2, d1, d2, c as the pinned top-2 oracle."""
    p = wl.make_points(cfg, N=1500)
    nnk, dk, ck = oracle.bruteforce_topk(p, 2)
    ref = oracle.bruteforce_top2(p)
    assert np.array_equal(nnk[:, 0], ref.nn) and np.array_equal(nnk[:, 1], ref.nn2)
    assert np.array_equal(bits(dk[:, 0]), bits(ref.d1)) and np.array_equal(bits(dk[:, 1]), bits(ref.d2))
    assert np.array_equal(bits(ck), bits(ref.c))


def test_topk_short_lists():
    """Fewer than K other points: missing entries are (-1, +inf), ck = +inf."""
    p = np.array([[0, 0], [1, 0], [0, 2]], np.float32)
    nnk, dk, ck = oracle.bruteforce_topk(p, 4)
    assert nnk.tolist() == [[1, 2, -1, -1], [0, 2, -1, -1], [0, 1, -1, -1]]
    assert np.all(np.isinf(dk[:, 2:])) and np.all(np.isinf(ck))
    nnk, dk, ck = oracle.bruteforce_topk(p, 3)
    assert np.all(nnk[:, 2] == -1) and np.all(np.isinf(ck))


@pytest.mark.parametrize("cfg,fam", [("cfg2", "walk"), ("cfg2", "shear"), ("cfg3", "walk"), ("cfg3", "cluster_drift")])
@pytest.mark.parametrize("K", [3, 5])
def test_topk_set_is_stable_beyond_4eps(cfg, fam, K):
    """Lemma 1's argument for the K-list: if dk[K-1] - dk[K-2] > 4 eps the SET of the
    K-1 nearest neighbours survives the step (its order may change)."""
    p, mot = wl.make_scene(cfg, fam, N=1500)
    pre = oracle.bruteforce_topk(p, K)
    for _ in range(3):
        q, _ = mot.step(p)
        eps = oracle.max_displacement(p, q)
        post = oracle.bruteforce_topk(q, K)
        safe = np.flatnonzero(pre[2] > np.float32(4) * eps)
        a = np.sort(pre[0][safe, :K - 1], axis=1)
        b = np.sort(post[0][safe, :K - 1], axis=1)
        assert np.array_equal(a, b)
        assert safe.size > 0
        p, pre = q, post
