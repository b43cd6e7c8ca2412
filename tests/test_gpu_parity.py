"""GPU parity (B200): every C-ABI entry point against the CPU oracle, element by element,
bit-exact for indices / flags / fp32 certificates, 1e-6 absolute for H (north_star)."""
import json
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2606_18314_b200 import binding as kc
from paper_2606_18314_b200 import workloads as wl

from _util import assert_same, dev, geoms, host, ref_certs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    kc.lib()


def scenes_small():
    rng = np.random.default_rng(7)
    out = {}
    for n in (2, 3, 4, 5, 31, 32, 33, 127, 129):
        for d in (2, 3):
            out[f"rand{n}_d{d}"] = rng.random((n, d)).astype(np.float32)
            out[f"lat{n}_d{d}"] = (rng.integers(0, 8, (n, d)) / 8.0).astype(np.float32)   # ties + duplicates
    out["lattice2"] = wl.lattice_points(33, 2)
    out["lattice3"] = wl.lattice_points(9, 3)
    out["dups"] = np.repeat(rng.random((50, 3)).astype(np.float32), 3, axis=0)
    out["onepoint"] = np.full((300, 2), 0.375, np.float32)
    pts = (0.5 + 0.01 * rng.standard_normal((3000, 2))).astype(np.float32)
    pts[1234] = (9.0, -7.0)
    out["outlier2"] = pts
    pts = (0.5 + 0.01 * rng.standard_normal((3000, 3))).astype(np.float32)
    pts[17] = (3.0, 2.0, -4.0)
    out["outlier3"] = pts
    out["cfg1"] = wl.make_points("cfg1")
    out["ragged5003_d2"] = wl.uniform_points(5003, 2, 21)
    out["ragged4099_d3"] = wl.uniform_points(4099, 3, 22)
    out["clusters3b"] = wl.cluster_points(6000, 3, 23, 32, 0.02)[0]
    out["mix_d2"] = wl.mixture_points(9000, 2, 24, 16, 0.005)
    out["mix_d3"] = wl.mixture_points(9000, 3, 25, 16, 0.005)
    return out


SMALL = scenes_small()


@pytest.mark.parametrize("name", ["p1_scene2d.json", "p2_tie_scene.json", "p2b_scene3d.json"])
def test_golden_scenes_on_gpu(golden_dir, name):
    g = json.load(open(os.path.join(golden_dir, name)))
    p = np.array(g["points"], np.float32)
    for got in (kc.kc_cert_allpairs(dev(p)), kc.kc_cert_grid_rebuild(kc.Grid(len(p), geoms(p)[1]), dev(p))):
        h = host(got)
        assert h.nn.tolist() == g["nn"] and h.nn2.tolist() == g["nn2"]
        assert ["%08x" % v for v in h.c.view(np.uint32)] == g["c_bits"]


@pytest.mark.parametrize("name", sorted(SMALL))
def test_allpairs_small(name):
    p = SMALL[name]
    assert_same(kc.kc_cert_allpairs(dev(p)), oracle.bruteforce_top2(p), what=name)


@pytest.mark.parametrize("name", sorted(SMALL))
def test_allpairs_small_warm_starts(name):
    """The seeded and the bounded start on the tiny / degenerate scenes (N = 2 has nn2 = -1 and
    d2 = inf; ties; duplicates; one point repeated)."""
    p = SMALL[name]
    want = oracle.bruteforce_top2(p)
    P = dev(p)
    assert_same(kc.kc_cert_allpairs(P, seed1=dev(want.nn), seed2=dev(want.nn2)), want, what=name + " seeded")
    eps = dev(np.zeros(1, np.float32))
    assert_same(kc.kc_cert_allpairs(P, d2_prev=dev(want.d2), eps=eps), want, what=name + " bounded")


@pytest.mark.parametrize("name", sorted(SMALL))
def test_grid_rebuild_small(name):
    p = SMALL[name]
    g_or, g_kc = geoms(p)
    grid = kc.Grid(p.shape[0], g_kc)
    got = kc.kc_cert_grid_rebuild(grid, dev(p))
    assert_same(got, oracle.bruteforce_top2(p), what=name)
    # A2 index work, bit-exact: cell ids, histogram scan, permutation
    cid = oracle.cell_ids(p, g_or)
    assert np.array_equal(grid.export(0).cpu().numpy(), cid)
    counts = np.bincount(cid, minlength=g_or.n_cells)
    assert np.array_equal(grid.export(4).cpu().numpy(), counts)
    start = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    assert np.array_equal(grid.export(1).cpu().numpy(), start)
    sidx = grid.export(2).cpu().numpy()
    slot = grid.export(3).cpu().numpy()
    assert np.array_equal(np.sort(sidx), np.arange(p.shape[0]))
    assert np.array_equal(sidx[slot], np.arange(p.shape[0]))
    assert np.all(np.diff(cid[sidx]) >= 0)                      # slots are cell-sorted
    info = grid.info()
    assert info.c_occ == np.count_nonzero(counts) and info.max_occ == counts.max()


@pytest.mark.parametrize("cfg,N", [("cfg2", 16000), ("cfg3", 16000), ("cfg4", 80000), ("cfg4", 262144),
                                   ("cfg5_d2", 310000), ("cfg5_d3", 310000)])
def test_allpairs_and_rebuild_configs(cfg, N):
    p = wl.make_points(cfg, N=N)
    want = ref_certs(p)
    P = dev(p)
    assert_same(kc.kc_cert_allpairs(P), want, what=f"allpairs {cfg} {N}")
    grid = kc.Grid(N, geoms(p)[1])
    assert_same(kc.kc_cert_grid_rebuild(grid, P), want, what=f"rebuild {cfg} {N}")


@pytest.mark.parametrize("cfg,N", [("cfg1", 1000), ("cfg2", 16000), ("cfg3", 16000), ("cfg4", 100000)])
def test_allpairs_bounded_is_exact_for_any_bound(cfg, N):
    """kc_cert_allpairs_bounded (kinetic bound d2_prev + 2 eps, Lemma 1's triangle inequality,
    PAPER.md:33): same bits as the oracle for a true bound, a useless one, a wrong one and NaN."""
    p, mot = wl.make_scene(cfg) if cfg != "cfg4" else (wl.make_points(cfg, N=N), None)
    if mot is None:
        q = (p + np.float32(1e-4) * wl.uniform_points(N, p.shape[1], 5)).astype(np.float32)
    else:
        q, _ = mot.step(p)
    pre, want = ref_certs(p), ref_certs(q)
    Q = dev(q)
    eps = dev(np.array([oracle.max_displacement(p, q)], np.float32))
    rng = np.random.default_rng(3)
    wrong = pre.d2.copy()
    k = rng.choice(N, N // 7, replace=False)
    wrong[k] = 0.0                                     # no candidate inside: recomputed from scratch
    wrong[rng.choice(N, 50, replace=False)] = np.nan
    half = np.maximum(want.d1 - 2 * eps.cpu().numpy()[0], 0).astype(np.float32)   # admits only the nearest
    bounds = {"kinetic": pre.d2, "inf": np.full(N, np.inf, np.float32), "huge": np.full(N, 10.0, np.float32),
              "zero": np.zeros(N, np.float32), "mixed": wrong, "one_candidate": half}
    for name, b in bounds.items():
        got = kc.kc_cert_allpairs(Q, d2_prev=dev(b), eps=eps)
        assert_same(got, want, what=f"bounded allpairs {cfg} bound={name}")


@pytest.mark.parametrize("d", [2, 3])
@pytest.mark.parametrize("offset", [0.0, 1000.0, -4096.5, 3.0e5])
def test_grid_far_from_origin_and_on_cell_faces(d, offset):
    """Pruning / ring bounds under coarse coordinates: boxes far from the origin (fp32 spacing up
    to h/30), points exactly on computed cell faces, dense and sparse cells mixed; rebuild and
    repair (both search kernels) against brute force."""
    rng = np.random.default_rng(int(abs(offset)) + d)
    N = 24000
    base = wl.mixture_points(N, d, 60 + d, 12, 0.004).astype(np.float64)
    p = (base + offset).astype(np.float32)
    g_or, g_kc = geoms(p)
    # a tenth of the points snapped onto cell faces of the grid actually used
    k = rng.choice(N, N // 10, replace=False)
    lo = np.array(list(g_or.lo)[:d], np.float32)
    p[k] = (lo + np.round((p[k] - lo) / g_or.h).astype(np.float32) * g_or.h).astype(np.float32)
    g_or, g_kc = geoms(p)
    want = oracle.bruteforce_top2(p)
    grid = kc.Grid(N, g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    assert_same(certs, want, what=f"offset {offset} d{d} rebuild")
    step = np.float32(g_or.h * 0.3)
    q = (p + (rng.random((N, d)).astype(np.float32) - np.float32(0.5)) * step).astype(np.float32)
    post = oracle.bruteforce_top2(q)
    for F in (np.arange(N, dtype=np.int32), np.sort(rng.choice(N, 900, replace=False)).astype(np.int32)):
        kc.kc_grid_build(grid, dev(p))
        work = kc.Certs.empty(N)
        kc.kc_frontier_repair(grid, dev(q), dev(F), dev(np.array([F.size], np.int32)), work)
        assert_same(work, post, idx=F, what=f"offset {offset} d{d} repair |F|={F.size}")


@pytest.mark.parametrize("cfg,N", [("cfg1", 1000), ("cfg2", 16000), ("cfg3", 16000), ("cfg4", 100000)])
def test_allpairs_seeded_is_exact_for_any_seeds(cfg, N):
    """kc_cert_allpairs_seeded: same bits as the oracle whether the seeds are the previous
    neighbours, the true new ones, random ids, or garbage (self, duplicates, out of range)."""
    p, mot = wl.make_scene(cfg) if cfg != "cfg4" else (wl.make_points(cfg, N=N), None)
    if mot is None:
        q = (p + np.float32(1e-4) * wl.uniform_points(N, p.shape[1], 5)).astype(np.float32)
    else:
        q, _ = mot.step(p)
    pre, want = ref_certs(p), ref_certs(q)
    Q = dev(q)
    rng = np.random.default_rng(11)
    ids = np.arange(N, dtype=np.int32)
    garbage1 = rng.integers(-5, N + 5, N).astype(np.int32)
    garbage2 = garbage1.copy()
    garbage2[::3] = rng.integers(0, N, garbage2[::3].size)
    seeds = {"previous": (pre.nn, pre.nn2), "true": (want.nn, want.nn2), "swapped": (want.nn2, want.nn),
             "random": (rng.integers(0, N, N).astype(np.int32), rng.integers(0, N, N).astype(np.int32)),
             "self": (ids, ids), "none": (np.full(N, -1, np.int32), np.full(N, -1, np.int32)),
             "garbage": (garbage1, garbage2), "one": (want.nn, np.full(N, -1, np.int32))}
    for name, (s1, s2) in seeds.items():
        got = kc.kc_cert_allpairs(Q, seed1=dev(s1), seed2=dev(s2))
        assert_same(got, want, what=f"seeded allpairs {cfg} seeds={name}")


@pytest.mark.parametrize("cfg,N", [("cfg2", 16000), ("cfg3", 5000)])
def test_allpairs_workspace_is_reusable(cfg, N):
    """Workspace contract (kc.h): zero-filled once, then any sequence of start modes and sizes on
    the same workspace — cold, seeded, bounded, a query subset, another N, everything beyond the
    ticket area scribbled over in between — and the same launch replayed from a CUDA graph."""
    p = wl.make_points(cfg, N=N)
    d = p.shape[1]
    want = ref_certs(p)
    small = np.ascontiguousarray(p[: N // 3])
    want_small = ref_certs(small)
    P, S = dev(p), dev(small)
    need = max(kc.lib().kc_cert_allpairs_workspace(N, d), kc.lib().kc_frontier_oracle_workspace(N, d, N))
    ws = torch.zeros(need + 64, dtype=torch.uint8, device="cuda")
    gen = torch.Generator(device="cuda").manual_seed(5)
    eps = dev(np.array([1e-4], np.float32))
    head = 16 + 148 * 8 * 8 * 4                                   # KC_AP_TICKET_BYTES + 16
    q = np.sort(np.random.default_rng(2).choice(N, N // 7, replace=False)).astype(np.int32)
    for rnd in range(3):
        assert_same(kc.kc_cert_allpairs(P, workspace=ws), want, what=f"cold, round {rnd}")
        assert_same(kc.kc_cert_allpairs(S, workspace=ws), want_small, what=f"cold, other N, round {rnd}")
        assert_same(kc.kc_cert_allpairs(P, workspace=ws, seed1=dev(want.nn), seed2=dev(want.nn2)), want,
                    what=f"seeded, round {rnd}")
        ws[head:] = torch.randint(0, 256, (ws.numel() - head,), dtype=torch.uint8, device="cuda", generator=gen)
        assert_same(kc.kc_cert_allpairs(P, workspace=ws, d2_prev=dev(want.d2), eps=eps), want, what=f"bounded, round {rnd}")
        out = kc.Certs.empty(N)
        kc.kc_frontier_oracle(P, dev(q), dev(np.array([q.size], np.int32)), out, workspace=ws)
        assert_same(out, want, idx=q, what=f"query subset, round {rnd}")
    out = kc.Certs.empty(N)
    s1, s2 = dev(want.nn), dev(want.nn2)
    kc.kc_cert_allpairs(P, out, ws, seed1=s1, seed2=s2)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        kc.kc_cert_allpairs(P, out, ws, seed1=s1, seed2=s2)
    for rnd in range(4):
        out.buf.zero_()
        g.replay()
        assert_same(out, want, what=f"graph replay {rnd}")


def test_grid_with_points_outside_the_box():
    # geometry fitted to the central half of the points: the rest is clamped into boundary cells
    p = wl.uniform_points(20000, 3, 31)
    g_or, g_kc = geoms(p, lo=np.full(3, 0.25, np.float32), hi=np.full(3, 0.75, np.float32))
    grid = kc.Grid(p.shape[0], g_kc)
    assert_same(kc.kc_cert_grid_rebuild(grid, dev(p)), oracle.bruteforce_top2(p), what="clamped")
    assert np.array_equal(grid.export(0).cpu().numpy(), oracle.cell_ids(p, g_or))
    p2 = wl.uniform_points(20000, 2, 32)
    g_or, g_kc = geoms(p2, occ=0.5, lo=np.full(2, 0.4, np.float32), hi=np.full(2, 0.6, np.float32))
    assert_same(kc.kc_cert_grid_rebuild(kc.Grid(p2.shape[0], g_kc), dev(p2)), oracle.bruteforce_top2(p2),
                what="clamped2")


@pytest.mark.parametrize("occ", [0.25, 1.0, 8.0, 64.0])
def test_grid_any_occupancy(occ):
    for d in (2, 3):
        p = wl.mixture_points(12000, d, 40 + d, 8, 0.01)
        grid = kc.Grid(p.shape[0], geoms(p, occ=occ)[1])
        assert_same(kc.kc_cert_grid_rebuild(grid, dev(p)), oracle.bruteforce_top2(p), what=f"occ{occ} d{d}")


def test_frontier_oracle_subset():
    for cfg in ("cfg2", "cfg3"):
        p = wl.make_points(cfg)
        want = oracle.bruteforce_top2(p)
        for nq in (1, 77, 5000):
            q = np.sort(np.random.default_rng(nq).choice(p.shape[0], nq, replace=False)).astype(np.int32)
            certs = kc.Certs.empty(p.shape[0])
            for t in (certs.nn, certs.nn2):
                t.fill_(-7)
            for t in (certs.d1, certs.d2, certs.c):
                t.fill_(-7.0)
            kc.kc_frontier_oracle(dev(p), dev(q), dev(np.array([nq], np.int32)), certs)
            assert_same(certs, want, idx=q, what=f"oracle {cfg} {nq}")
            rest = np.setdiff1d(np.arange(p.shape[0]), q)
            assert np.all(host(certs).nn[rest] == -7) and np.all(host(certs).c[rest] == -7.0)


def test_empty_and_degenerate_frontiers():
    """Empty id lists leave everything untouched (repair, frontier oracle, audit, entropy); a step that
    moves nothing has eps = 0 and its frontier is exactly the points with c = 0 (ties, duplicates)."""
    p = wl.make_points("cfg2", N=3000)
    p[10] = p[11]                                             # a duplicate pair: d1 = 0
    p[20], p[21], p[22] = (0.5, 0.5), (0.5 + 2.0 ** -8, 0.5), (0.5 - 2.0 ** -8, 0.5)   # point 20: d1 = d2
    want = oracle.bruteforce_top2(p)
    P = dev(p)
    _, g_kc = geoms(p)
    grid = kc.Grid(p.shape[0], g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, P)
    assert_same(certs, want, what="degenerate scene")
    eps = kc.kc_max_displacement(P, P)
    flags, F, nF = kc.kc_frontier_classify(certs.c, eps)
    wf, wF = oracle.frontier(want.c, np.float32(0))
    assert float(eps.item()) == 0.0 and np.array_equal(flags.cpu().numpy(), wf)
    assert int(nF.item()) == wF.size and 20 in wF and want.c[20] == 0
    before = certs.clone()
    zero = dev(np.array([0], np.int32))
    nothing = dev(np.zeros(1, np.int32))                       # a valid pointer, zero entries
    kc.kc_frontier_repair(grid, P, nothing, zero, certs)
    kc.kc_frontier_oracle(P, nothing, zero, certs)
    assert_same(certs, host(before), what="empty frontier leaves the certificates alone")
    H, m, C = kc.kc_frontier_entropy(grid, nothing, zero)
    assert float(H.item()) == 0.0 and int(m.item()) == 0 and int(C.item()) > 0
    # the zero-motion frontier repaired in place gives the same certificates back
    kc.kc_frontier_repair(grid, P, F, nF, certs)
    assert_same(certs, want, what="repair of the c = 0 frontier")


def test_max_displacement_and_classify():
    for cfg in ("cfg1", "cfg2", "cfg3"):
        for fam in wl.CONFIGS[cfg]["families"]:
            p, mot = wl.make_scene(cfg, fam)
            q, _ = mot.step(p)
            eps = kc.kc_max_displacement(dev(p), dev(q))
            want_eps = oracle.max_displacement(p, q)
            assert eps.cpu().numpy().view(np.uint32)[0] == np.array([want_eps]).view(np.uint32)[0]
            c = oracle.kdtree_top2(p).c
            flags, F, nF = kc.kc_frontier_classify(dev(c), eps)
            wf, wF = oracle.frontier(c, want_eps)
            assert np.array_equal(flags.cpu().numpy(), wf)
            n = int(nF.item())
            assert n == wF.size
            assert np.array_equal(np.sort(F[:n].cpu().numpy()), wF)
    # ragged sizes and the inclusive threshold
    for N in (1, 3, 4, 5, 1023, 1024, 1025, 4097):
        c = np.random.default_rng(N).random(N).astype(np.float32)
        e = np.float32(0.125)
        c[0] = 0.5                                                # == 4*eps exactly: in F
        flags, F, nF = kc.kc_frontier_classify(dev(c), dev(np.array([e])))
        wf, wF = oracle.frontier(c, e)
        assert np.array_equal(flags.cpu().numpy(), wf) and int(nF.item()) == wF.size
        assert np.array_equal(np.sort(F[:wF.size].cpu().numpy()), wF)
    z = kc.kc_max_displacement(dev(p), dev(p))
    assert float(z.item()) == 0.0


def test_entropy_matches_oracle():
    rng = np.random.default_rng(5)
    for cfg, N in (("cfg1", 1000), ("cfg2", 16000), ("cfg3", 16000), ("cfg5_d3", 50000)):
        p = wl.make_points(cfg, N=N)
        g_or, g_kc = geoms(p)
        grid = kc.Grid(N, g_kc)
        kc.kc_grid_build(grid, dev(p))
        cid = oracle.cell_ids(p, g_or)
        lists = [np.arange(N), np.zeros(0, np.int64), np.flatnonzero(cid == cid[0]),
                 rng.choice(N, N // 10, replace=False), np.unique(cid, return_index=True)[1]]
        for F in lists:
            F = np.sort(F).astype(np.int32)
            Fd = dev(F) if F.size else torch.zeros(1, dtype=torch.int32, device="cuda")
            for rep in range(2):                                  # scratch must be left clean
                H, m, C = kc.kc_frontier_entropy(grid, Fd, dev(np.array([F.size], np.int32)), nF_max=max(F.size, 1))
                wH, wm, wC = oracle.entropy(cid, F, g_or.n_cells)
                assert abs(float(H.item()) - wH) <= 1e-6, (cfg, F.size, float(H.item()), wH)
                assert int(m.item()) == wm and int(C.item()) == wC
                assert F.size == 0 or wm >= wC ** wH * (1 - 1e-9)   # Theorem 3


def run_repair_steps(cfg, fam, N, steps, use_movers, frontier="lemma", **kw):
    p, mot = wl.make_scene(cfg, fam, N=N, **kw)
    g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    pre = ref_certs(p)
    assert_same(certs, pre, what="pre")
    for t in range(steps):
        q, movers = mot.step(p)
        Q = dev(q)
        eps = kc.kc_max_displacement(dev(p), Q)
        if frontier == "lemma":
            flags, F, nF = kc.kc_frontier_classify(certs.c, eps)
        elif frontier == "all":
            F, nF = dev(np.arange(N, dtype=np.int32)), dev(np.array([N], np.int32))
        else:                                                     # the mover list as the frontier (A12)
            mv = movers if movers is not None else np.arange(N, dtype=np.int32)
            F, nF = dev(mv), dev(np.array([mv.size], np.int32))
        mv_d = dev(movers) if (use_movers and movers is not None and movers.size) else None
        if use_movers and movers is not None and movers.size == 0:
            mv_d, nmv = torch.zeros(1, dtype=torch.int32, device="cuda"), dev(np.array([0], np.int32))
            kc.kc_frontier_repair(grid, Q, F, nF, certs, movers=mv_d, n_movers=nmv, n_movers_max=0)
        else:
            kc.kc_frontier_repair(grid, Q, F, nF, certs, movers=mv_d)
        post = ref_certs(q)
        n = int(nF.item())
        Fh = np.sort(F[:n].cpu().numpy())
        got = host(certs)
        # O8: repaired entries equal the exact post-step certificates, bit for bit
        assert_same(got, post, idx=Fh, what=f"{cfg}/{fam} step {t} repaired")
        rest = np.setdiff1d(np.arange(N), Fh)
        if frontier == "lemma":
            # Lemma 1: nn of every skipped point is still exact; d1,d2,c keep pre-step values
            assert np.array_equal(got.nn[rest], post.nn[rest])
            assert_same(got, pre, idx=rest, what=f"{cfg}/{fam} step {t} untouched", nn2=False)
        # entropy and cells on the updated filing
        cid = oracle.cell_ids(q, g_or)
        assert np.array_equal(grid.export(0).cpu().numpy(), cid)
        H, m, C = kc.kc_frontier_entropy(grid, F, nF)
        wH, wm, wC = oracle.entropy(cid, Fh.astype(np.int32), g_or.n_cells)
        assert abs(float(H.item()) - wH) <= 1e-6 and int(m.item()) == wm and int(C.item()) == wC
        # per-transition protocol (A13): next step starts from exact certificates
        certs = kc.Certs(*(dev(x) for x in (post.nn, post.nn2, post.d1, post.d2, post.c)))
        p, pre = q, post
    info = grid.info()
    return info


@pytest.mark.parametrize("cfg,fam", [("cfg2", f) for f in wl.CONFIGS["cfg2"]["families"]] +
                         [("cfg3", f) for f in wl.CONFIGS["cfg3"]["families"]])
def test_repair_per_family(cfg, fam):
    info = run_repair_steps(cfg, fam, 16000, 4, use_movers=True)
    assert info.dirty == 1


@pytest.mark.parametrize("d_cfg", ["cfg2", "cfg3"])
def test_repair_long_run_chains_accumulate(d_cfg):
    # 12 steps without a rebuild in between: misfiled points accumulate and move again
    info = run_repair_steps(d_cfg, "walk", 6000, 12, use_movers=False, frontier="all")
    assert info.n_misfiled > 150


def test_repair_mover_list_as_frontier_cfg4_style():
    for ball in (False, True):
        for f in (0.001, 0.03, 1.0):
            run_repair_steps("cfg4", "fraction", 40000, 2, use_movers=True, frontier="movers", fraction=f, ball=ball)


@pytest.mark.parametrize("cfg,fam", [("cfg2", "walk"), ("cfg2", "local"), ("cfg3", "cluster_drift"), ("cfg3", "ball5")])
def test_failure_audit_and_true_frontier_entropy(cfg, fam):
    """NEXT #2: F_t = {nn changed} (Definition 2), the Lemma-1 audit counts (Table 1) and H(F_t)."""
    p, mot = wl.make_scene(cfg, fam)
    q, _ = mot.step(p)
    N = p.shape[0]
    g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    pre = kc.kc_cert_grid_rebuild(grid, dev(p))
    eps = kc.kc_max_displacement(dev(p), dev(q))
    flags, F, nF = kc.kc_frontier_classify(pre.c, eps)
    post = kc.kc_cert_grid_rebuild(grid, dev(q))
    counts, Ft = kc.kc_failure_audit(pre.nn, post.nn, flags)
    o_pre, o_post = oracle.bruteforce_top2(p), oracle.bruteforce_top2(q)
    o_flags, _ = oracle.frontier(o_pre.c, oracle.max_displacement(p, q))
    wFt, wcounts = oracle.failure_audit(o_pre.nn, o_post.nn, o_flags)
    assert counts.cpu().numpy().tolist() == wcounts.tolist() and wcounts[2] == 0
    assert np.array_equal(np.sort(Ft.cpu().numpy()[: int(wcounts[0])]), wFt)
    H, m, C = kc.kc_frontier_entropy(grid, Ft, counts[:1])
    wH, wm, wC = oracle.entropy(oracle.cell_ids(q, g_or), wFt, g_or.n_cells)
    assert abs(float(H.item()) - wH) <= 1e-6 and int(m.item()) == wm and int(C.item()) == wC


@pytest.mark.parametrize("tree", [False, True])
@pytest.mark.parametrize("cfg,fam", [("cfg2", "walk"), ("cfg2", "local"), ("cfg3", "cluster_drift"), ("cfg3", "vortex")])
def test_clock_maintenance_multi_step(cfg, fam, tree):
    """NEXT #3 (Appendix A.2): 15 steps without a rebuild; every step the expired set equals the
    oracle's clock rule, repaired certificates are exact, and nn is exact for ALL points.  tree: the
    expired set comes from the expiry tournament tree (Theorem 2) instead of the flat test."""
    from paper_2606_18314_b200.driver import ClockMaintainer
    p, mot = wl.make_scene(cfg, fam, N=6000)
    N = p.shape[0]
    m = ClockMaintainer(dev(p), tree=tree)
    o = oracle.bruteforce_top2(p)
    o_c, o_stamp, o_S = o.c.copy(), np.zeros(N, np.float32), 0.0
    for step in range(15):
        q, movers = mot.step(p)
        F, nF = m.step(dev(q), movers=None if movers is None else dev(movers))
        o_S, o_flags, o_F = oracle.clock_frontier(o_c, o_stamp, o_S, oracle.max_displacement(p, q))
        post = oracle.bruteforce_top2(q)
        got = host(m.certs)
        assert float(m.S[0].item()) == o_S
        if not tree:
            assert np.array_equal(m.flags.cpu().numpy(), o_flags), f"step {step}: expired set differs"
        assert np.array_equal(np.sort(F.cpu().numpy()[: int(nF.item())]), o_F)
        assert_same(got, post, idx=o_F, what=f"clock {cfg}/{fam} step {step}")
        assert np.array_equal(got.nn, post.nn), f"step {step}: a stale certificate holds a wrong nn"
        o_c[o_F] = post.c[o_F]
        o_stamp[o_F] = oracle.clock_stamp(o_S)
        assert np.array_equal(m.stamp.cpu().numpy().view(np.uint32), o_stamp.view(np.uint32))
        p = q


@pytest.mark.parametrize("cfg,fam", [("cfg2", "walk"), ("cfg2", "local"), ("cfg3", "cluster_drift"), ("cfg3", "diffuse5"),
                                     ("cfg3", "ball5"), ("cfg4", "fraction")])
def test_local_motion_budget_frontier(cfg, fam):
    """NEXT #2: kc_frontier_classify_local, flags bit-exact against the oracle's
    float32 restatement, F as a set, and the repaired certificates keep nn exact for all points."""
    if cfg == "cfg4":
        p, mot = wl.make_scene("cfg4", "fraction", fraction=0.01, ball=False, N=60000)
    else:
        p, mot = wl.make_scene(cfg, fam)
    q, movers = mot.step(p)
    N = p.shape[0]
    g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    P, Q = dev(p), dev(q)
    certs = kc.kc_cert_grid_rebuild(grid, P)
    eps = kc.kc_max_displacement(P, Q)
    flags, F, nF = kc.kc_frontier_classify_local(grid, P, Q, certs, eps)
    pre = ref_certs(p)
    wflags, wF = oracle.local_frontier(p, q, g_or, pre.nn, pre.d1, pre.c, oracle.max_displacement(p, q))
    assert np.array_equal(flags.cpu().numpy(), wflags)
    assert int(nF.item()) == wF.size and np.array_equal(np.sort(F.cpu().numpy()[: wF.size]), wF)
    kc.kc_frontier_repair(grid, Q, F, nF, certs, movers=None if movers is None else dev(movers))
    post = ref_certs(q)
    got = host(certs)
    assert_same(got, post, idx=wF, what=f"local budget repair {cfg}/{fam}")
    assert np.array_equal(got.nn, post.nn)                       # no missed failure


@pytest.mark.parametrize("overlap", [True, False])
@pytest.mark.parametrize("cfg,fam", [("cfg1", "walk"), ("cfg2", "walk"), ("cfg2", "local"), ("cfg3", "cluster_drift")])
def test_graphed_step_matches_the_oracle(cfg, fam, overlap):
    """The CUDA-graph form of the step (driver.GraphMaintainer): 5 replayed transitions, every
    output bit-exact against the oracle, and identical to the eager step."""
    from paper_2606_18314_b200.driver import GraphMaintainer, Maintainer
    p, mot = wl.make_scene(cfg, fam)
    g_or, _ = geoms(p)
    gm, em = GraphMaintainer(dev(p), overlap_allpairs=overlap), Maintainer(dev(p))
    pre = oracle.bruteforce_top2(p)
    for step in range(5):
        q, movers = mot.step(p)
        res = gm.step(dev(q))
        ref = em.step(dev(q), movers=None if movers is None else dev(movers))
        post = oracle.bruteforce_top2(q)
        eps = oracle.max_displacement(p, q)
        flags, F = oracle.frontier(pre.c, eps)
        assert float(res.eps.item()) == float(eps) and int(res.nF.item()) == F.size
        assert_same(res.rebuilt, post, what=f"graph rebuilt {step}")
        assert_same(res.certified, post, what=f"graph allpairs {step}")
        assert_same(res.repaired, post, idx=F, what=f"graph repaired {step}")
        H, mm, C = oracle.entropy(oracle.cell_ids(q, g_or), F, g_or.n_cells)
        assert abs(float(res.H.item()) - H) <= 1e-6 and int(res.m_cells.item()) == mm and int(res.C_occ.item()) == C
        for f in ("nn", "nn2", "d1", "d2", "c"):
            assert torch.equal(getattr(res.rebuilt, f), getattr(ref.rebuilt, f))
        assert gm.launches_per_step(0) > 0
        p, pre = q, post


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_randomized_scenes(seed):
    """Random scenes (uniform / Gaussian / lattice with ties / tight clusters / mixtures; scaled and
    shifted; occupancy 0.25-50; box sometimes smaller than the data): all-pairs, rebuild, two
    successive repairs of a random id list (the second over overflow chains), seeded all-pairs,
    rebuild again, each bit-exact against brute force."""
    rng = np.random.default_rng(seed)
    for it in range(60):
        d = int(rng.integers(2, 4))
        N = int(rng.integers(2, 3000))
        kind = int(rng.integers(0, 5))
        if kind == 0:
            p = rng.random((N, d))
        elif kind == 1:
            p = 0.5 + 0.02 * rng.standard_normal((N, d))
        elif kind == 2:
            p = rng.integers(0, 12, (N, d)) / 12.0
        elif kind == 3:
            k = max(1, N // 50)
            p = rng.random((k, d))[rng.integers(0, k, N)] + rng.choice([1e-4, 1e-2]) * rng.standard_normal((N, d))
        else:
            p = np.concatenate([rng.random((N - N // 2, d)), 0.3 + 1e-3 * rng.standard_normal((N // 2, d))])
        p = (p * rng.choice([1.0, 100.0, 1e-3]) + rng.choice([0.0, 0.0, 1000.0, -77.7])).astype(np.float32)
        tag = f"seed {seed} scene {it} (d={d}, N={N}, kind={kind})"
        lo, hi = np.zeros(3, np.float32), np.zeros(3, np.float32)
        lo[:d], hi[:d] = p.min(0), p.max(0)
        if rng.random() < 0.2:
            c = (lo + hi) / 2
            lo, hi = (c - (c - lo) * 0.5).astype(np.float32), (c + (hi - c) * 0.5).astype(np.float32)
        g_or, g_kc = geoms(p, occ=float(rng.choice([0.25, 1, 2, 2, 2, 8, 50])), lo=lo[:d], hi=hi[:d])
        grid = kc.Grid(N, g_kc)
        want = oracle.bruteforce_top2(p)
        assert_same(kc.kc_cert_allpairs(dev(p)), want, what=tag + " allpairs")
        certs = kc.kc_cert_grid_rebuild(grid, dev(p))
        assert_same(certs, want, what=tag + " rebuild")
        step = float(rng.choice([1e-4, 1e-2, 0.3])) * float(max(hi.max() - lo.min(), 1e-6)) / max(1, int(round(N ** (1 / d))))
        F = np.sort(rng.choice(N, int(rng.integers(1, N + 1)), replace=False)).astype(np.int32)
        q = p
        for rep in range(2):
            q = (q + step * (rng.random((N, d)) - 0.5)).astype(np.float32)
            post = oracle.bruteforce_top2(q)
            kc.kc_frontier_repair(grid, dev(q), dev(F), dev(np.array([F.size], np.int32)), certs)
            assert_same(certs, post, idx=F, what=tag + f" repair {rep}")
        assert_same(kc.kc_cert_allpairs(dev(q), seed1=certs.nn, seed2=certs.nn2), post, what=tag + " seeded")
        assert_same(kc.kc_cert_grid_rebuild(grid, dev(q)), post, what=tag + " rebuild 2")


def test_search_refused_on_dirty_grid():
    p, mot = wl.make_scene("cfg1")
    grid = kc.Grid(p.shape[0], geoms(p)[1])
    with pytest.raises(kc.RebuildRequired):
        kc.kc_cert_grid_search(grid, kc.Certs.empty(p.shape[0]))
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    q, _ = mot.step(p)
    F = dev(np.arange(p.shape[0], dtype=np.int32))
    kc.kc_frontier_repair(grid, dev(q), F, dev(np.array([p.shape[0]], np.int32)), certs)
    assert_same(certs, oracle.bruteforce_top2(q), what="cfg1 full-frontier repair")
    with pytest.raises(kc.RebuildRequired):
        kc.kc_cert_grid_search(grid, certs)
    with pytest.raises(kc.RebuildRequired):
        kc.kc_frontier_repair(grid, dev(q[:500]), F, dev(np.array([10], np.int32)), certs)
    assert_same(kc.kc_cert_grid_rebuild(grid, dev(q)), oracle.bruteforce_top2(q), what="rebuild after repair")


def test_bbox_device():
    p = (np.random.default_rng(1).standard_normal((10007, 3)) * 5).astype(np.float32)
    b = kc.kc_bbox(dev(p)).cpu().numpy()
    assert np.array_equal(b[:3], p.min(0)) and np.array_equal(b[3:], p.max(0))
    lo, hi = oracle.bbox(p)
    assert np.array_equal(b[:3], lo) and np.array_equal(b[3:], hi)


def test_allpairs_dirty_workspace_is_reported_not_trapped():
    """A workspace that was never zero-filled (kc.h, workspace contract) must not poison the CUDA
    context: the kernel reports through the error word, the NEXT all-pairs call returns KC_EINVAL
    after clearing the counters, and the call after that is exact again."""
    p = wl.make_points("cfg2")
    N, d = p.shape
    want = ref_certs(p)
    P = dev(p)
    need = kc.lib().kc_cert_allpairs_workspace(N, d)
    ws = torch.full((need + 64,), 0x7f, dtype=torch.uint8, device="cuda")      # counters hold 0x7f7f7f7f
    kc.kc_cert_allpairs(P, workspace=ws, seed1=dev(want.nn), seed2=dev(want.nn2))   # j-split launch
    torch.cuda.synchronize()                                     # the context is still alive
    with pytest.raises(kc.KcError) as e:
        kc.kc_cert_allpairs(P, workspace=ws)
    assert e.value.status == kc.KC_EINVAL and "zero-filled" in str(e.value)
    assert_same(kc.kc_cert_allpairs(P, workspace=ws), want, what="after the report")
    assert_same(kc.kc_cert_allpairs(P, workspace=ws, seed1=dev(want.nn), seed2=dev(want.nn2)), want,
                what="seeded after the report")


def test_frontier_search_twice_on_one_update():
    """Two sweep-sized kc_frontier_search calls after ONE kc_grid_update: the second must not
    replay the chain residents of the first (entries outside its list stay untouched)."""
    N = 230_000
    p = wl.uniform_points(N, 2, 77)
    rng = np.random.default_rng(78)
    q = (p + rng.uniform(-2e-3, 2e-3, p.shape)).astype(np.float32)      # many points change cell
    movers = np.sort(rng.choice(N, N // 10, replace=False)).astype(np.int32)   # below the re-bin bound N/8
    still = np.setdiff1d(np.arange(N), movers)
    q[still] = p[still]
    grid = kc.Grid(N, geoms(p)[1])
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    Q = dev(q)
    kc.kc_grid_update(grid, Q, movers=dev(movers))
    assert grid.info().n_misfiled > N // 200 and grid.info().dirty == 1
    post = ref_certs(q)
    perm = rng.permutation(N).astype(np.int32)
    F1, F2 = np.sort(perm[: N // 2]), np.sort(perm[N // 2: N // 2 + N // 4])
    sentinel = kc.Certs.empty(N)
    for name in ("nn", "nn2"):
        getattr(sentinel, name).fill_(-7)
    for name in ("d1", "d2", "c"):
        getattr(sentinel, name).fill_(-7.0)
    for F in (F1, F2, F1):
        out = sentinel.clone()
        kc.kc_frontier_search(grid, Q, dev(F), dev(np.array([F.size], np.int32)), out)
        got = host(out)
        assert_same(got, post, idx=F, what="searched entries")
        rest = np.setdiff1d(np.arange(N), F)
        assert np.all(got.nn[rest] == -7) and np.all(got.c[rest] == -7.0), "entries outside F were written"


@pytest.mark.parametrize("N", [1001, 1002, 1003])
def test_maintainer_any_N(N):
    """Certs.empty keeps every row 16-byte aligned for N that is not a multiple of 4."""
    from paper_2606_18314_b200.driver import Maintainer
    p, mot = wl.make_scene("cfg1", N=N)
    q, _ = mot.step(p)
    m = Maintainer(dev(p))
    res = m.step(dev(q))
    post = ref_certs(q)
    assert_same(res.rebuilt, post, what="rebuilt")
    assert_same(res.certified, post, what="certified")
    F = oracle.frontier(ref_certs(p).c, oracle.max_displacement(p, q))[1]
    assert int(res.nF.item()) == F.size
    assert_same(res.repaired, post, idx=F, what="repaired")


def test_update_rebins_when_most_points_move():
    """kc_grid_update on a large grid with every point a potential mover re-bins (A2) instead of
    re-filing: no chains, the grid counts as fresh, the frontier search that follows is exact."""
    N = 150_000
    p = wl.mixture_points(N, 3, 91, 16, 0.01)
    rng = np.random.default_rng(92)
    q = (p + rng.uniform(-1e-3, 1e-3, p.shape)).astype(np.float32)
    g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    certs = kc.kc_cert_grid_rebuild(grid, dev(p))
    kc.kc_grid_update(grid, dev(q))
    info = grid.info()
    assert info.n_misfiled == 0 and info.dirty == 0
    assert np.array_equal(grid.export(0).cpu().numpy(), oracle.cell_ids(q, g_or))
    F = np.sort(rng.choice(N, N // 3, replace=False)).astype(np.int32)
    kc.kc_frontier_search(grid, dev(q), dev(F), dev(np.array([F.size], np.int32)), certs)
    post = ref_certs(q)
    assert_same(certs, post, idx=F, what="after a re-binning update")
    rest = np.setdiff1d(np.arange(N), F)
    assert_same(certs, ref_certs(p), idx=rest, what="untouched")


def test_sweep_path_replays_from_a_cuda_graph():
    """The slot sweep keeps no host-side counter: update + classify + sweep captured once at
    N = 262,144 and replayed on new positions is exact every time."""
    N = 262_144
    p = wl.uniform_points(N, 3, 93)
    rng = np.random.default_rng(94)
    g_or, g_kc = geoms(p)
    grid = kc.Grid(N, g_kc)
    P, Q = dev(p), dev(p)
    certs = kc.kc_cert_grid_rebuild(grid, P)
    eps = torch.zeros(1, device="cuda")
    flags = torch.empty(N, dtype=torch.uint8, device="cuda")
    F = torch.empty(N, dtype=torch.int32, device="cuda")
    nF = torch.zeros(1, dtype=torch.int32, device="cuda")
    work = kc.Certs.empty(N)

    def body():
        work.buf.copy_(certs.buf)
        kc.kc_max_displacement(P, Q, eps)
        kc.kc_frontier_classify(work.c, eps, flags, F, nF)
        kc.kc_grid_build(grid, P)                              # the grid resident at p ...
        kc.kc_frontier_repair(grid, Q, F, nF, work)            # ... updated to q, F re-searched

    q0 = (p + rng.uniform(-5e-4, 5e-4, p.shape)).astype(np.float32)
    Q.copy_(dev(q0))
    body()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        body()
    pre = ref_certs(p)
    for rnd in range(3):
        q = (p + rng.uniform(-5e-4, 5e-4, p.shape)).astype(np.float32)
        Q.copy_(dev(q))
        g.replay()
        torch.cuda.synchronize()
        wf, wF = oracle.frontier(pre.c, oracle.max_displacement(p, q))
        assert int(nF.item()) == wF.size and wF.size * 8 >= N          # sweep-sized
        post = ref_certs(q)
        assert_same(work, post, idx=wF, what=f"replay {rnd}")
        rest = np.flatnonzero(wf == 0)
        assert np.array_equal(host(work).nn[rest], post.nn[rest])


def _same_geom(g_or, g_kc):
    assert g_or.d == g_kc.d and tuple(g_or.G) == (g_kc.G[0], g_kc.G[1], g_kc.G[2])
    assert g_or.h == np.float32(g_kc.h) and g_or.inv_h == np.float32(g_kc.inv_h)
    assert list(g_or.lo) == [np.float32(g_kc.lo[k]) for k in range(3)]


@pytest.mark.parametrize("d", [2, 3])
def test_geometry_by_median_density_matches_the_oracle(d):
    """Reading R24: the library's coarse histogram + median and the oracle's give the same geometry,
    field by field, on uniform sets (k = 0), config 5's mixture (k = 1), sets heaped into one coarse
    cell around the rounding boundaries of k, sets too small for an estimate and a box far from the
    origin; the certificates on the coarser grid are the oracle's."""
    rng = np.random.default_rng(7 + d)
    scenes = [wl.uniform_points(20000, d, 4), wl.mixture_points(262144, d, 5), wl.uniform_points(100, d, 6),
              (wl.mixture_points(65536, d, 8, 16, 0.002).astype(np.float64) * 3.0 + 250.0).astype(np.float32)]
    R = 8 if d == 2 else 4
    cells = np.stack(np.meshgrid(*[np.arange(R)] * d, indexing="ij"), -1).reshape(-1, d)
    for m in (64, 46, 45, 32, 23, 22, 4):
        base = (np.repeat(cells, m, axis=0) + rng.uniform(0.2, 0.8, (cells.shape[0] * m, d))) / R
        heap = (np.full((4096 - base.shape[0], d), R // 2) + rng.uniform(0.2, 0.8, (4096 - base.shape[0], d))) / R
        p = np.concatenate([base, heap]).astype(np.float32)
        p[0] = 0.0
        p[base.shape[0] - 1] = 1.0
        scenes.append(p)
    for p in scenes:
        g_or = oracle.geom_by_median_density(p)
        g_kc = kc.kc_geom_by_median_density(dev(p))
        _same_geom(g_or, g_kc)
    with pytest.raises(kc.KcError):
        kc.kc_geom_by_median_density(dev(scenes[0]), occ=0.0)
    p = scenes[1]
    g_kc = kc.kc_geom_by_median_density(dev(p))
    assert g_kc.G[0] < geoms(p)[1].G[0]                            # coarser than the mean-occupancy grid
    grid = kc.Grid(p.shape[0], g_kc)
    assert_same(kc.kc_cert_grid_rebuild(grid, dev(p)), oracle.kdtree_top2(p), what=f"median-density grid d{d}")
