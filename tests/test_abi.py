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
