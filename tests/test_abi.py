"""CPU-only: libkc.so builds, loads and exports every symbol include/kc.h declares; the host-side
entry points behave; the product path fails loudly (no fallback) without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2606_18314_b200 import _build, binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    _build.build()
    return binding.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "kc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kc_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    names = declared_symbols()
    assert len(names) >= 20
    raw = ctypes.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), f"{n} declared in kc.h but not exported by libkc.so"
    assert set(names) == set(binding.EXPORTS)


def test_geom_matches_survey_table(L):
    for N, d, G in [(1000, 2, 23), (16000, 2, 90), (16000, 3, 20), (262144, 3, 51), (4194304, 2, 1449),
                    (4194304, 3, 128)]:
        g = binding.kc_geom_from_bbox(N, d, [0, 0, 0], [1, 1, 1])
        assert (g.G[0], g.G[1], g.G[2]) == (G, G, G if d == 3 else 1)
        assert g.h == np.float32(1.0 / G * (1 + 2.0 ** -20))
        assert g.inv_h == np.float32(1.0 / float(np.float32(g.h)))


def test_geom_agrees_with_oracle_bitwise(L):
    import oracle
    rng = np.random.default_rng(0)
    for _ in range(50):
        d = int(rng.integers(2, 4))
        N = int(rng.integers(2, 10 ** 6))
        lo = rng.standard_normal(3).astype(np.float32)
        hi = (lo + rng.random(3).astype(np.float32) * 3).astype(np.float32)
        occ = float(rng.choice([1.0, 2.0, 3.5]))
        a = binding.kc_geom_from_bbox(N, d, lo, hi, occ)
        b = oracle.geom_from_bbox(N, d, lo, hi, occ)
        assert (a.G[0], a.G[1], a.G[2]) == tuple(b.G)
        assert np.float32(a.h) == b.h and np.float32(a.inv_h) == b.inv_h
        assert [np.float32(a.lo[k]) for k in range(3)] == list(b.lo)


def test_bad_arguments_are_rejected(L):
    with pytest.raises(binding.KcError):
        binding.kc_geom_from_bbox(100, 4, [0, 0, 0], [1, 1, 1])
    with pytest.raises(binding.KcError):
        binding.kc_geom_from_bbox(100, 2, [0, 0, 0], [1, 1, 1], occ=0.0)
    assert L.kc_cert_allpairs_workspace(1, 2) == 0 and L.kc_cert_allpairs_workspace(1000, 2) > 0
    # NULL pointers are refused before any CUDA call
    assert L.kc_cert_allpairs(None, 100, 2, None, None, None, None, None, None, 0, None) == binding.KC_EINVAL
    assert L.kc_max_displacement(None, None, 10, 2, None, None) == binding.KC_EINVAL
    assert b"kc_max_displacement" in L.kc_last_error()
    E = binding.KC_EINVAL
    assert L.kc_cert_allpairs_bounded(None, 100, 2, None, None, None, None, None, None, None, None, 0, None) == E
    assert L.kc_cert_allpairs_seeded(None, 100, 2, None, None, None, None, None, None, None, None, 0, None) == E
    assert L.kc_frontier_oracle(None, 100, 2, None, None, 5, None, None, None, None, None, None, 0, None) == E
    assert L.kc_grid_build(None, None, 100, None) == E
    assert L.kc_cert_grid_search(None, None, None, None, None, None, None) == E
    assert L.kc_frontier_classify(None, 100, None, None, None, None, None) == E
    assert L.kc_frontier_classify_clock(None, None, 100, None, None, None, None, None, None, None) == E
    assert L.kc_frontier_classify_local(None, None, None, 100, None, None, None, None, None, None, None, None) == E
    assert L.kc_clock_stamp(None, None, 0, 100, None, None, None) == E
    assert L.kc_frontier_entropy(None, None, None, 10, None, None, None, None) == E
    assert L.kc_grid_update(None, None, 100, None, None, 0, None) == E
    assert L.kc_frontier_search(None, None, 100, None, None, 10, None, None, None, None, None, None) == E
    assert L.kc_frontier_repair(None, None, 100, None, None, 0, None, None, 10, None, None, None, None, None, None) == E
    assert L.kc_failure_audit(None, None, None, 100, None, None, None) == E
    assert L.kc_cert_allpairs_topk(None, 100, 2, 4, None, None, None, None, None, 0, None) == E
    assert L.kc_cert_grid_topk(None, 4, None, None, None, None) == E
    assert L.kc_frontier_search_topk(None, None, 100, None, None, 10, 4, None, None, None, None) == E
    assert L.kc_cert_allpairs_topk_workspace(1000, 2, 9) == 0 and L.kc_cert_allpairs_topk_workspace(1000, 2, 4) > 0
    assert L.kc_grid_destroy(None) == binding.KC_OK and L.kc_grid_bytes(None) == 0


def test_no_cpu_fallback_without_gpu(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    p = torch.zeros(8, 2)
    with pytest.raises((ValueError, RuntimeError)):
        binding.kc_cert_allpairs(p)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2606_18314_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "kc_oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "kc_oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2606_18314_b200", otxt, flags=re.M)
    assert '#include "kc' not in otxt and "include/kc.h" not in otxt


@pytest.mark.gpu
def test_full_step_through_raw_ctypes():
    """One maintenance step (A0, A4, A6+A7, A5, A2+A3, A1) driven through ctypes.CDLL alone --
    no binding.py, torch only as the owner of device memory -- and checked against the oracle."""
    import ctypes as C

    import torch

    import oracle
    from paper_2606_18314_b200 import workloads as wl
    from paper_2606_18314_b200.binding import LIB_PATH, kc_geom

    lib = C.CDLL(LIB_PATH)
    lib.kc_cert_allpairs_workspace.restype = C.c_size_t
    lib.kc_cert_allpairs_workspace.argtypes = [C.c_int64, C.c_int]
    vp = C.c_void_p
    p, mot = wl.make_scene("cfg1")
    q, _ = mot.step(p)
    N, d = p.shape
    P, Q = torch.from_numpy(p).cuda(), torch.from_numpy(q).cuda()
    lo = (C.c_float * 3)(*p.min(0), 0.0)
    hi = (C.c_float * 3)(*p.max(0), 0.0)
    geom = kc_geom()
    lib.kc_geom_from_bbox.argtypes = [C.c_int64, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_double, C.POINTER(kc_geom)]
    assert lib.kc_geom_from_bbox(N, d, lo, hi, 2.0, C.byref(geom)) == 0
    grid = vp()
    lib.kc_grid_create.argtypes = [C.POINTER(vp), C.c_int64, C.POINTER(kc_geom)]
    assert lib.kc_grid_create(C.byref(grid), N, C.byref(geom)) == 0
    i32 = lambda n: torch.empty(n, dtype=torch.int32, device="cuda")
    f32 = lambda n: torch.empty(n, dtype=torch.float32, device="cuda")
    pre = [i32(N), i32(N), f32(N), f32(N), f32(N)]          # nn, nn2, d1, d2, c
    post = [i32(N), i32(N), f32(N), f32(N), f32(N)]
    ap = [i32(N), i32(N), f32(N), f32(N), f32(N)]
    ptr = lambda t: vp(t.data_ptr())
    st = vp(torch.cuda.current_stream().cuda_stream)
    lib.kc_cert_grid_rebuild.argtypes = [vp, vp, C.c_int64, vp, vp, vp, vp, vp, vp]
    assert lib.kc_cert_grid_rebuild(grid, ptr(P), N, *map(ptr, pre), st) == 0
    eps, flags, F, nF = f32(1), torch.empty(N, dtype=torch.uint8, device="cuda"), i32(N), i32(1)
    lib.kc_max_displacement.argtypes = [vp, vp, C.c_int64, C.c_int, vp, vp]
    assert lib.kc_max_displacement(ptr(P), ptr(Q), N, d, ptr(eps), st) == 0
    lib.kc_frontier_classify.argtypes = [vp, C.c_int64, vp, vp, vp, vp, vp]
    assert lib.kc_frontier_classify(ptr(pre[4]), N, ptr(eps), ptr(flags), ptr(F), ptr(nF), st) == 0
    lib.kc_frontier_repair.argtypes = [vp, vp, C.c_int64, vp, vp, C.c_int64, vp, vp, C.c_int64, vp, vp, vp, vp, vp, vp]
    assert lib.kc_frontier_repair(grid, ptr(Q), N, None, None, 0, ptr(F), ptr(nF), N, *map(ptr, pre), st) == 0
    H = torch.empty(1, dtype=torch.float64, device="cuda")
    m, Cc = i32(1), i32(1)
    lib.kc_frontier_entropy.argtypes = [vp, vp, vp, C.c_int64, vp, vp, vp, vp]
    assert lib.kc_frontier_entropy(grid, ptr(F), ptr(nF), N, ptr(H), ptr(m), ptr(Cc), st) == 0
    assert lib.kc_cert_grid_rebuild(grid, ptr(Q), N, *map(ptr, post), st) == 0
    need = lib.kc_cert_allpairs_workspace(N, d)
    ws = torch.zeros(max(need, 16), dtype=torch.uint8, device="cuda")
    lib.kc_cert_allpairs.argtypes = [vp, C.c_int64, C.c_int, vp, vp, vp, vp, vp, vp, C.c_size_t, vp]
    assert lib.kc_cert_allpairs(ptr(Q), N, d, *map(ptr, ap), ptr(ws), ws.numel(), st) == 0
    torch.cuda.synchronize()
    want = oracle.bruteforce_top2(q)
    w_eps = oracle.max_displacement(p, q)
    wf, wF = oracle.frontier(oracle.bruteforce_top2(p).c, w_eps)
    assert eps.cpu().numpy().view(np.uint32)[0] == np.array([w_eps], np.float32).view(np.uint32)[0]
    assert int(nF.item()) == wF.size and np.array_equal(flags.cpu().numpy(), wf)
    for k, name in enumerate(("nn", "nn2", "d1", "d2", "c")):
        ref = getattr(want, name).view(np.uint32)
        assert np.array_equal(post[k].cpu().numpy().view(np.uint32), ref), name
        assert np.array_equal(ap[k].cpu().numpy().view(np.uint32), ref), name
        assert np.array_equal(pre[k].cpu().numpy().view(np.uint32)[wF], ref[wF]), name
    g_or = oracle.geom_for(p)
    wH, wm, wC = oracle.entropy(oracle.cell_ids(q, g_or), wF, g_or.n_cells)
    assert abs(float(H.item()) - wH) <= 1e-6 and int(m.item()) == wm and int(Cc.item()) == wC
    lib.kc_grid_destroy.argtypes = [vp]
    assert lib.kc_grid_destroy(grid) == 0
