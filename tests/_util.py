"""Shared helpers of the GPU parity tests (marshalling only; no method arithmetic)."""
import numpy as np
import torch

import oracle
from paper_2606_18314_b200 import binding as kc


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def geoms(p, occ=2.0, lo=None, hi=None):
    """Geometry computed independently by both sides from the same bbox; asserted identical."""
    p = np.asarray(p, np.float32)
    N, d = p.shape
    lo3 = np.zeros(3, np.float32)
    hi3 = np.zeros(3, np.float32)
    lo3[:d] = p.min(0) if lo is None else lo
    hi3[:d] = p.max(0) if hi is None else hi
    g_or = oracle.geom_from_bbox(N, d, lo3, hi3, occ)
    g_kc = kc.kc_geom_from_bbox(N, d, lo3, hi3, occ)
    assert tuple(g_or.G) == (g_kc.G[0], g_kc.G[1], g_kc.G[2])
    assert g_or.h == np.float32(g_kc.h) and g_or.inv_h == np.float32(g_kc.inv_h)
    assert list(g_or.lo) == [np.float32(g_kc.lo[k]) for k in range(3)]
    return g_or, g_kc


def host(c: kc.Certs):
    torch.cuda.synchronize()
    return oracle.Certs(c.nn.cpu().numpy(), c.nn2.cpu().numpy(), c.d1.cpu().numpy(), c.d2.cpu().numpy(),
                        c.c.cpu().numpy())


def assert_same(got, want, idx=None, what="", nn2=True):
    """Bit-exact comparison of certificate arrays (got: GPU, want: oracle)."""
    if isinstance(got, kc.Certs):
        got = host(got)
    fields = ("nn", "nn2", "d1", "d2", "c") if nn2 else ("nn", "d1", "d2", "c")
    for f in fields:
        a, b = getattr(got, f), getattr(want, f)
        if idx is not None:
            a = a[idx]
            b = b[idx] if b.shape[0] != a.shape[0] else b
        if a.dtype == np.float32:
            a, b = a.view(np.uint32), b.view(np.uint32)
        bad = np.flatnonzero(a != b)
        assert bad.size == 0, f"{what}: {f} differs at {bad.size} entries, first {bad[:5]}: {a[bad[:5]]} vs {b[bad[:5]]}"


def ref_certs(p):
    """Oracle certificates: brute force up to 20k points, the (brute-force-validated) k-d tree above."""
    p = np.asarray(p, np.float32)
    return oracle.bruteforce_top2(p) if p.shape[0] <= 20000 else oracle.kdtree_top2(p)
