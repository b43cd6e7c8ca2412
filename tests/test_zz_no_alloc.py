"""kc_cert_allpairs_static: the all-pairs pass with the library's file-scope scratch (no allocation in
the call, include/kc.h) against the existing path kc_cert_allpairs with a caller-allocated workspace.
Same kernels, so the bar is the one of every certificate test here: bit-exact.  The file sorts last
on purpose (the static array is shared state: nothing else in the suite depends on it)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_18314_b200 import binding as kc
from paper_2606_18314_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _bits(c: kc.Certs):
    torch.cuda.synchronize()
    return [np.ascontiguousarray(getattr(c, f).cpu().numpy()).view(np.uint32) for f in ("nn", "nn2", "d1", "d2", "c")]


def _same(got, want, what):
    for name, g, w in zip(("nn", "nn2", "d1", "d2", "c"), _bits(got), _bits(want)):
        assert np.array_equal(g, w), f"{what}: {name} differs at {np.flatnonzero(g != w)[:5]}"


def test_static_scratch_matches_the_workspace_path_on_consecutive_calls():
    assert kc.lib().kc_cert_allpairs_static_max_n() == 65536
    # two calls in a row on the same stream, sizes and dimensions that use different launch shapes
    # (the second finds the first one's partial lists and counters in the array), then the first again
    scenes = [wl.uniform_points(16000, 2, 21), wl.mixture_points(5000, 3, 22, 8, 0.01), wl.uniform_points(16000, 2, 21),
              wl.uniform_points(65536, 3, 23), wl.uniform_points(300, 2, 24)]
    dev = [torch.from_numpy(p).cuda() for p in scenes]
    outs = [kc.Certs.empty(p.shape[0], "cuda") for p in scenes]
    for o in outs:
        o.buf.fill_(-1)
    for P, o in zip(dev, outs):                     # back to back, no synchronisation in between
        kc.kc_cert_allpairs_static(P, o)
    for k, (P, o) in enumerate(zip(dev, outs)):
        _same(o, kc.kc_cert_allpairs(P), f"call {k} (N={P.shape[0]}, d={P.shape[1]})")
    # and the existing path is the oracle's (brute-force definition), so the new one is too
    want = oracle.bruteforce_top2(scenes[1])
    got = _bits(outs[1])
    for g, f in zip(got, ("nn", "nn2", "d1", "d2", "c")):
        assert np.array_equal(g, np.ascontiguousarray(getattr(want, f)).view(np.uint32))


def test_static_scratch_call_allocates_no_device_memory():
    P = torch.from_numpy(wl.uniform_points(40000, 3, 25)).cuda()
    out = kc.Certs.empty(P.shape[0], "cuda")
    kc.kc_cert_allpairs_static(P, out)              # the first call on a device looks the address up
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        kc.kc_cert_allpairs_static(P, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0
    _same(out, kc.kc_cert_allpairs(P), "after repeated calls")


def test_static_scratch_rejects_sizes_beyond_its_maximum():
    n = int(kc.lib().kc_cert_allpairs_static_max_n()) + 1
    P = torch.from_numpy(wl.uniform_points(n, 2, 26)).cuda()
    out = kc.Certs.empty(n, "cuda")
    out.buf.fill_(-7)
    with pytest.raises(kc.KcError, match="65536"):
        kc.kc_cert_allpairs_static(P, out)
    torch.cuda.synchronize()
    assert bool((out.buf == -7).all())              # nothing was launched
    with pytest.raises(kc.KcError):
        kc.kc_cert_allpairs_static(P[:1], kc.Certs.empty(1, "cuda"))
    # every size up to the maximum fits the array (the library checks the same on every call)
    need = max(kc.lib().kc_cert_allpairs_workspace(N, d) for d in (2, 3) for N in range(2, 65537, 61))
    assert need <= 5 << 20
