"""Thin Python binding of libkc.so: same names as include/kc.h, argument marshalling only.

Every function takes torch CUDA tensors (device memory) and passes ``data_ptr()`` plus the
current torch stream through the C-ABI; every step of the path runs in the library's own CUDA
kernels.  There is no CPU fallback: if libkc.so is missing or fails to load, importing any
entry point raises ``RuntimeError``.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

KC_OK, KC_EINVAL, KC_ENOMEM, KC_ECUDA, KC_EREBUILD = 0, -1, -2, -3, -4
_STATUS = {0: "KC_OK", -1: "KC_EINVAL", -2: "KC_ENOMEM", -3: "KC_ECUDA", -4: "KC_EREBUILD"}

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkc.so")

EXPORTS = (
    "kc_version", "kc_last_error", "kc_geom_from_bbox", "kc_bbox", "kc_geom_by_median_density",
    "kc_max_displacement",
    "kc_cert_allpairs_workspace", "kc_cert_allpairs", "kc_cert_allpairs_static_max_n", "kc_cert_allpairs_static", "kc_cert_allpairs_bounded", "kc_cert_allpairs_seeded",
    "kc_frontier_oracle_workspace",
    "kc_frontier_oracle", "kc_grid_create", "kc_grid_destroy", "kc_grid_bytes", "kc_grid_set_index", "kc_grid_build",
    "kc_cert_grid_search", "kc_cert_grid_rebuild", "kc_frontier_classify", "kc_frontier_entropy",
    "kc_frontier_repair", "kc_grid_update", "kc_frontier_search", "kc_failure_audit", "kc_frontier_classify_clock", "kc_clock_stamp", "kc_clock_tree_floats", "kc_clock_tree_build",
    "kc_frontier_classify_clock_tree", "kc_clock_tree_update", "kc_frontier_classify_local",
    "kc_cert_allpairs_topk_workspace", "kc_cert_allpairs_topk", "kc_cert_grid_topk", "kc_frontier_search_topk",
    "kc_grid_info", "kc_grid_export", "kc_fp32_probe", "kc_launch_count",
)


class KcError(RuntimeError):
    def __init__(self, status, where, msg):
        super().__init__(f"{where}: {_STATUS.get(status, status)} {msg}")
        self.status = status


class RebuildRequired(KcError):
    pass


class kc_geom(C.Structure):
    _fields_ = [("d", C.c_int32), ("G", C.c_int32 * 3), ("lo", C.c_float * 3),
                ("h", C.c_float), ("inv_h", C.c_float)]

    @property
    def n_cells(self):
        return int(self.G[0]) * int(self.G[1]) * int(self.G[2])


class kc_grid_info_t(C.Structure):
    _fields_ = [("n_points", C.c_int64), ("n_cells", C.c_int64), ("c_occ", C.c_int32),
                ("max_occ", C.c_int32), ("n_misfiled", C.c_int32), ("built", C.c_int32),
                ("dirty", C.c_int32), ("n_stragglers", C.c_int32), ("n_heavy", C.c_int32),
                ("n_leaves", C.c_int32), ("heavy_T", C.c_int32), ("n_handed", C.c_int32),
                ("n_deferred", C.c_int32)]


_lib = None


def lib():
    """Load libkc.so (fails loudly; never falls back to anything)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_18314_b200._build` "
                           "(nvcc, sm_100a). There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    vp, i64, sz, ci = C.c_void_p, C.c_int64, C.c_size_t, C.c_int
    L.kc_version.restype = C.c_char_p
    L.kc_last_error.restype = C.c_char_p
    L.kc_geom_from_bbox.argtypes = [i64, ci, C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_double,
                                    C.POINTER(kc_geom)]
    L.kc_bbox.argtypes = [vp, i64, ci, vp, vp]
    L.kc_geom_by_median_density.argtypes = [vp, i64, ci, C.c_double, vp, C.POINTER(kc_geom)]
    L.kc_max_displacement.argtypes = [vp, vp, i64, ci, vp, vp]
    L.kc_cert_allpairs_static_max_n.restype = i64
    L.kc_clock_tree_floats.restype = sz
    L.kc_clock_tree_floats.argtypes = [i64]
    L.kc_clock_tree_build.argtypes = [vp, vp, i64, vp, vp]
    L.kc_frontier_classify_clock_tree.argtypes = [vp, vp, i64, vp, vp, vp, vp, vp, vp, vp]
    L.kc_clock_tree_update.argtypes = [vp, vp, i64, vp, vp, i64, vp, vp]
    L.kc_cert_allpairs_static.argtypes = [vp, i64, ci, vp, vp, vp, vp, vp, vp]
    L.kc_cert_allpairs_workspace.restype = sz
    L.kc_cert_allpairs_workspace.argtypes = [i64, ci]
    L.kc_cert_allpairs.argtypes = [vp, i64, ci, vp, vp, vp, vp, vp, vp, sz, vp]
    L.kc_cert_allpairs_bounded.argtypes = [vp, i64, ci, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    L.kc_cert_allpairs_seeded.argtypes = [vp, i64, ci, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    L.kc_frontier_oracle_workspace.restype = sz
    L.kc_frontier_oracle_workspace.argtypes = [i64, ci, i64]
    L.kc_frontier_oracle.argtypes = [vp, i64, ci, vp, vp, i64, vp, vp, vp, vp, vp, vp, sz, vp]
    L.kc_grid_create.argtypes = [C.POINTER(vp), i64, C.POINTER(kc_geom)]
    L.kc_grid_destroy.argtypes = [vp]
    L.kc_grid_bytes.restype = sz
    L.kc_grid_bytes.argtypes = [vp]
    L.kc_grid_set_index.argtypes = [vp, ci, ci]
    L.kc_grid_build.argtypes = [vp, vp, i64, vp]
    L.kc_cert_grid_search.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    L.kc_cert_grid_rebuild.argtypes = [vp, vp, i64, vp, vp, vp, vp, vp, vp]
    L.kc_frontier_classify.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    L.kc_frontier_entropy.argtypes = [vp, vp, vp, i64, vp, vp, vp, vp]
    L.kc_frontier_repair.argtypes = [vp, vp, i64, vp, vp, i64, vp, vp, i64, vp, vp, vp, vp, vp, vp]
    L.kc_grid_update.argtypes = [vp, vp, i64, vp, vp, i64, vp]
    L.kc_frontier_search.argtypes = [vp, vp, i64, vp, vp, i64, vp, vp, vp, vp, vp, vp]
    L.kc_failure_audit.argtypes = [vp, vp, vp, i64, vp, vp, vp]
    L.kc_frontier_classify_clock.argtypes = [vp, vp, i64, vp, vp, vp, vp, vp, vp, vp]
    L.kc_clock_stamp.argtypes = [vp, vp, i64, i64, vp, vp, vp]
    L.kc_frontier_classify_local.argtypes = [vp, vp, vp, i64, vp, vp, vp, vp, vp, vp, vp, vp]
    L.kc_cert_allpairs_topk_workspace.restype = sz
    L.kc_cert_allpairs_topk_workspace.argtypes = [i64, ci, ci]
    L.kc_cert_allpairs_topk.argtypes = [vp, i64, ci, ci, vp, vp, vp, vp, vp, sz, vp]
    L.kc_cert_grid_topk.argtypes = [vp, ci, vp, vp, vp, vp]
    L.kc_frontier_search_topk.argtypes = [vp, vp, i64, vp, vp, i64, ci, vp, vp, vp, vp]
    L.kc_grid_info.argtypes = [vp, C.POINTER(kc_grid_info_t), vp]
    L.kc_grid_export.argtypes = [vp, ci, vp, i64, C.POINTER(i64), vp]
    L.kc_fp32_probe.argtypes = [ci, ci, C.POINTER(C.c_double), vp]
    L.kc_launch_count.restype = C.c_uint64
    L.kc_launch_count.argtypes = []
    for name in EXPORTS:
        fn = getattr(L, name)
        if fn.restype is C.c_int:      # default restype: all kc_status functions
            fn.restype = C.c_int
    _lib = L
    return L


def _check(status, where):
    if status != KC_OK:
        msg = lib().kc_last_error().decode()
        raise (RebuildRequired if status == KC_EREBUILD else KcError)(status, where, msg)


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t, dtype=None, name="tensor"):
    if t is None:
        return C.c_void_p(0)
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{name} must be a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"{name} must have dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _pos(p, name="p"):
    if p.dim() != 2 or p.shape[1] not in (2, 3):
        raise ValueError(f"{name} must be (N, 2) or (N, 3)")
    return _ptr(p, torch.float32, name), int(p.shape[0]), int(p.shape[1])


@dataclass
class Certs:
    """Device certificate arrays of Definition 1, indexed by point id.  ``empty``
    carves the five arrays out of one (5, N) int32 allocation (``buf``: rows nn, d1, d2, c, nn2), so
    a caller can move a certificate set with one copy (``buf[:4]`` without the runner-up index)."""
    nn: torch.Tensor
    nn2: torch.Tensor
    d1: torch.Tensor
    d2: torch.Tensor
    c: torch.Tensor
    buf: torch.Tensor | None = None

    @staticmethod
    def _views(buf, N=None):
        N = buf.shape[1] if N is None else N
        return Certs(buf[0, :N], buf[4, :N], buf[1, :N].view(torch.float32), buf[2, :N].view(torch.float32),
                     buf[3, :N].view(torch.float32), buf)

    @staticmethod
    def empty(N, device="cuda"):
        # rows padded to a multiple of 4 entries: every row starts 16-byte aligned for any N
        # (kc_frontier_classify reads c as float4)
        return Certs._views(torch.empty((5, (N + 3) // 4 * 4), dtype=torch.int32, device=device), N)

    def clone(self):
        if self.buf is not None:
            return Certs._views(self.buf.clone(), self.nn.numel())
        return Certs(self.nn.clone(), self.nn2.clone(), self.d1.clone(), self.d2.clone(), self.c.clone())

    def _ptrs(self):
        return (_ptr(self.nn, torch.int32, "nn"), _ptr(self.nn2, torch.int32, "nn2"),
                _ptr(self.d1, torch.float32, "d1"), _ptr(self.d2, torch.float32, "d2"),
                _ptr(self.c, torch.float32, "c"))


# ------------------------------------------------------------------------------------------
def kc_version() -> str:
    return lib().kc_version().decode()


def kc_geom_from_bbox(N, d, lo, hi, occ=2.0) -> kc_geom:
    """Host: grid geometry of reading A6."""
    lo3 = (C.c_float * 3)(*[float(x) for x in list(lo)[:3]] + [0.0] * (3 - len(list(lo)[:3])))
    hi3 = (C.c_float * 3)(*[float(x) for x in list(hi)[:3]] + [0.0] * (3 - len(list(hi)[:3])))
    g = kc_geom()
    _check(lib().kc_geom_from_bbox(int(N), int(d), lo3, hi3, float(occ), C.byref(g)), "kc_geom_from_bbox")
    return g


def kc_bbox(p, out=None):
    """Device bbox: returns a float32[6] CUDA tensor (min xyz, max xyz)."""
    pp, N, d = _pos(p)
    out = out if out is not None else torch.empty(6, dtype=torch.float32, device=p.device)
    _check(lib().kc_bbox(pp, N, d, _ptr(out, torch.float32), _stream()), "kc_bbox")
    return out


def kc_geom_for(p, occ=2.0) -> kc_geom:
    """Convenience: device bbox (one sync) then kc_geom_from_bbox."""
    b = kc_bbox(p).cpu().numpy()
    return kc_geom_from_bbox(p.shape[0], p.shape[1], b[:3], b[3:], occ)


def kc_geom_by_median_density(p, occ=2.0) -> kc_geom:
    """Geometry of reading R24: the occupancy is measured against the median density of
    the occupied volume (a uniform set gives the geometry of kc_geom_for).  A setup call: it syncs."""
    pp, N, d = _pos(p)
    g = kc_geom()
    _check(lib().kc_geom_by_median_density(pp, N, d, float(occ), _stream(), C.byref(g)),
           "kc_geom_by_median_density")
    return g


def kc_max_displacement(p, p2, eps_out=None):
    """A0, Algorithm 1 line 1.  Returns the device float32[1] tensor eps_t."""
    pp, N, d = _pos(p)
    pq, N2, d2 = _pos(p2, "p2")
    if (N, d) != (N2, d2):
        raise ValueError("p and p2 must have the same shape")
    eps_out = eps_out if eps_out is not None else torch.empty(1, dtype=torch.float32, device=p.device)
    _check(lib().kc_max_displacement(pp, pq, N, d, _ptr(eps_out, torch.float32), _stream()),
           "kc_max_displacement")
    return eps_out


_ws_cache = {}


def _workspace(nbytes, device, kind="allpairs"):
    """Cached scratch per device and purpose.  The all-pairs workspace is zero-filled once and then
    only ever passed to the all-pairs entry points (workspace contract, kc.h)."""
    if nbytes == 0:
        return None
    key = (str(device), kind)
    w = _ws_cache.get(key)
    if w is None or w.numel() < nbytes:
        w = torch.zeros(nbytes, dtype=torch.uint8, device=device)
        _ws_cache[key] = w
    return w


def kc_cert_allpairs_static(p, out: Certs) -> Certs:
    """A1 with the library's static scratch (no allocation anywhere in the call, kc.h): N up to
    ``lib().kc_cert_allpairs_static_max_n()``; ``out`` is the caller's, allocated beforehand."""
    pp, N, d = _pos(p)
    _check(lib().kc_cert_allpairs_static(pp, N, d, *out._ptrs(), _stream()), "kc_cert_allpairs_static")
    return out


def kc_cert_allpairs(p, out: Certs | None = None, workspace=None, d2_prev=None, eps=None,
                     seed1=None, seed2=None) -> Certs:
    """A1: exact all-pairs certificates (Table 2).  With ``d2_prev`` (float32[N]) and
    ``eps`` (float32[1]) the pass starts from the kinetic bound d2_prev + 2 eps
    (kc_cert_allpairs_bounded); with ``seed1``, ``seed2`` (int32[N], e.g. the previous nn, nn2) from
    those two points (kc_cert_allpairs_seeded); the result is the same bits in every case."""
    pp, N, d = _pos(p)
    out = out or Certs.empty(N, p.device)
    need = lib().kc_cert_allpairs_workspace(N, d)
    ws = workspace if workspace is not None else _workspace(need, p.device)
    if (d2_prev is None) != (eps is None):
        raise ValueError("d2_prev and eps go together")
    if (seed1 is None) != (seed2 is None):
        raise ValueError("seed1 and seed2 go together")
    if seed1 is not None:
        if seed1.numel() != N or seed2.numel() != N:
            raise ValueError("seeds must have N entries")
        _check(lib().kc_cert_allpairs_seeded(pp, N, d, _ptr(seed1, torch.int32, "seed1"),
                                             _ptr(seed2, torch.int32, "seed2"), *out._ptrs(), _ptr(ws),
                                             ws.numel() if ws is not None else 0, _stream()),
               "kc_cert_allpairs_seeded")
        return out
    if d2_prev is None:
        _check(lib().kc_cert_allpairs(pp, N, d, *out._ptrs(), _ptr(ws), ws.numel() if ws is not None else 0,
                                      _stream()), "kc_cert_allpairs")
    else:
        if d2_prev.numel() != N:
            raise ValueError("d2_prev must have N entries")
        _check(lib().kc_cert_allpairs_bounded(pp, N, d, _ptr(d2_prev, torch.float32, "d2_prev"),
                                              _ptr(eps, torch.float32, "eps"), *out._ptrs(), _ptr(ws),
                                              ws.numel() if ws is not None else 0, _stream()),
               "kc_cert_allpairs_bounded")
    return out


def kc_frontier_oracle(p, q, nq, certs: Certs, nq_max=None, workspace=None) -> Certs:
    """NEXT #1 (PAPER.md:69 rtx_frontier_oracle): brute-force relabel of the ids in q."""
    pp, N, d = _pos(p)
    nq_max = int(q.numel() if nq_max is None else nq_max)
    need = lib().kc_frontier_oracle_workspace(N, d, nq_max)
    ws = workspace if workspace is not None else _workspace(need, p.device)
    _check(lib().kc_frontier_oracle(pp, N, d, _ptr(q, torch.int32, "q"), _ptr(nq, torch.int32, "nq"),
                                    nq_max, *certs._ptrs(), _ptr(ws),
                                    ws.numel() if ws is not None else 0, _stream()), "kc_frontier_oracle")
    return certs


class Grid:
    """Resident uniform grid (kc_grid handle).  Owns only the handle; arrays are the library's."""

    def __init__(self, N_max: int, geom: kc_geom):
        self.geom = geom
        self.N_max = int(N_max)
        self.N = 0                      # points of the last build
        h = C.c_void_p()
        _check(lib().kc_grid_create(C.byref(h), self.N_max, C.byref(geom)), "kc_grid_create")
        self._h = h

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:      # _lib is gone at interpreter exit
            _lib.kc_grid_destroy(self._h)
        self._h = None

    __del__ = close

    @property
    def bytes(self) -> int:
        return int(lib().kc_grid_bytes(self._h))

    def set_index(self, heavy_T: int, sub_occ: int = 4):
        """Parameters of the two-level index (kc_grid_set_index); effective from the next build."""
        _check(lib().kc_grid_set_index(self._h, int(heavy_T), int(sub_occ)), "kc_grid_set_index")
        self.N = 0

    def info(self) -> kc_grid_info_t:
        out = kc_grid_info_t()
        _check(lib().kc_grid_info(self._h, C.byref(out), _stream()), "kc_grid_info")
        return out

    def export(self, what: int) -> torch.Tensor:
        """One of the grid's int32 arrays (see kc_grid_export) copied into a new CUDA tensor."""
        cnt = C.c_int64()
        _check(lib().kc_grid_export(self._h, what, C.c_void_p(0), 0, C.byref(cnt), _stream()), "kc_grid_export")
        out = torch.empty(cnt.value, dtype=torch.int32, device="cuda")
        _check(lib().kc_grid_export(self._h, what, _ptr(out), cnt.value, C.byref(cnt), _stream()), "kc_grid_export")
        return out


def kc_grid_build(grid: Grid, p):
    """A2: cell ids, histogram, scan, scatter."""
    pp, N, d = _pos(p)
    _check(lib().kc_grid_build(grid._h, pp, N, _stream()), "kc_grid_build")
    grid.N = N


def kc_cert_grid_search(grid: Grid, out: Certs | None = None, N=None) -> Certs:
    """A3 (Corollary 1): certificates of all points of a fresh grid."""
    out = out or Certs.empty(N if N is not None else grid.N_max)
    _check(lib().kc_cert_grid_search(grid._h, *out._ptrs(), _stream()), "kc_cert_grid_search")
    return out


def kc_cert_grid_rebuild(grid: Grid, p, out: Certs | None = None) -> Certs:
    """A2 + A3: the O(N) rebuild strategy (PAPER.md:69 rtx_grid_rebuild)."""
    pp, N, d = _pos(p)
    out = out or Certs.empty(N, p.device)
    _check(lib().kc_cert_grid_rebuild(grid._h, pp, N, *out._ptrs(), _stream()), "kc_cert_grid_rebuild")
    grid.N = N
    return out


def _topk_out(N, K, device):
    return (torch.empty((N, K), dtype=torch.int32, device=device),
            torch.empty((N, K), dtype=torch.float32, device=device),
            torch.empty(N, dtype=torch.float32, device=device))


def kc_cert_allpairs_topk(p, K: int, workspace=None, seed_ids=None):
    """NEXT #4: K-list certificates by the tiled N x N pass (Definition 1 :29 with K
    keys).  ``seed_ids`` (int32[N,K], optional): K known points per query to start from.  Returns
    (nnk int32[N,K], dk float32[N,K], ck float32[N])."""
    pp, N, d = _pos(p)
    if seed_ids is not None and tuple(seed_ids.shape) != (N, K):
        raise ValueError("seed_ids must be (N, K)")
    nnk, dk, ck = _topk_out(N, K, p.device)
    need = lib().kc_cert_allpairs_topk_workspace(N, d, K)
    ws = workspace if workspace is not None else _workspace(need, p.device, "topk")
    _check(lib().kc_cert_allpairs_topk(pp, N, d, K, _ptr(seed_ids, torch.int32, "seed_ids"), _ptr(nnk), _ptr(dk),
                                       _ptr(ck), _ptr(ws),
                                       ws.numel() if ws is not None else 0, _stream()), "kc_cert_allpairs_topk")
    return nnk, dk, ck


def kc_cert_grid_topk(grid: Grid, K: int, device=None):
    """NEXT #4: K-list certificates of every point of a freshly built grid (ring search, exact)."""
    if grid.N < 2:
        raise RebuildRequired(KC_EREBUILD, "kc_cert_grid_topk", "the grid has not been built")
    nnk, dk, ck = _topk_out(grid.N, K, device or torch.device("cuda"))
    _check(lib().kc_cert_grid_topk(grid._h, K, _ptr(nnk), _ptr(dk), _ptr(ck), _stream()), "kc_cert_grid_topk")
    return nnk, dk, ck


def kc_frontier_search_topk(grid: Grid, p_new, F, nF, lists, nF_max=None):
    """A7 for K-list certificates: recompute rows F of ``lists`` = (nnk, dk, ck) against the updated
    grid (call kc_grid_update first), in place."""
    pp, N, d = _pos(p_new, "p_new")
    nnk, dk, ck = lists
    K = int(nnk.shape[1])
    nF_max = int(F.numel() if nF_max is None else nF_max)
    _check(lib().kc_frontier_search_topk(grid._h, pp, N, _ptr(F, torch.int32, "F"), _ptr(nF, torch.int32, "nF"),
                                         nF_max, K, _ptr(nnk, torch.int32, "nnk"), _ptr(dk, torch.float32, "dk"),
                                         _ptr(ck, torch.float32, "ck"), _stream()), "kc_frontier_search_topk")
    return lists


def kc_frontier_classify(c, eps, flags=None, F=None, nF=None):
    """A4, Algorithm 1 line 2.  eps: device float32[1].  Returns (flags, F, nF)."""
    N = c.numel()
    flags = flags if flags is not None else torch.empty(N, dtype=torch.uint8, device=c.device)
    F = F if F is not None else torch.empty(N, dtype=torch.int32, device=c.device)
    nF = nF if nF is not None else torch.empty(1, dtype=torch.int32, device=c.device)
    _check(lib().kc_frontier_classify(_ptr(c, torch.float32, "c"), N, _ptr(eps, torch.float32, "eps"),
                                      _ptr(flags, torch.uint8, "flags"), _ptr(F, torch.int32, "F"),
                                      _ptr(nF, torch.int32, "nF"), _stream()), "kc_frontier_classify")
    return flags, F, nF


def kc_frontier_entropy(grid: Grid, F, nF, nF_max=None, out=None):
    """A5, Definition 2.  Returns device tensors (H float64[1], m int32[1], C int32[1])."""
    nF_max = int(F.numel() if nF_max is None else nF_max)
    if out is None:
        out = (torch.empty(1, dtype=torch.float64, device=F.device),
               torch.empty(1, dtype=torch.int32, device=F.device),
               torch.empty(1, dtype=torch.int32, device=F.device))
    H, m, Cc = out
    _check(lib().kc_frontier_entropy(grid._h, _ptr(F, torch.int32, "F"), _ptr(nF, torch.int32, "nF"), nF_max,
                                     _ptr(H, torch.float64, "H"), _ptr(m, torch.int32), _ptr(Cc, torch.int32),
                                     _stream()), "kc_frontier_entropy")
    return H, m, Cc


def kc_frontier_repair(grid: Grid, p_new, F, nF, certs: Certs, movers=None, n_movers=None,
                       nF_max=None, n_movers_max=None) -> Certs:
    """A6 + A7, Algorithm 1 lines 3-7: update the grid, re-search F in place."""
    pp, N, d = _pos(p_new, "p_new")
    nF_max = int(F.numel() if nF_max is None else nF_max)
    if movers is not None:
        n_movers_max = int(movers.numel() if n_movers_max is None else n_movers_max)
        if n_movers is None:
            n_movers = torch.tensor([movers.numel()], dtype=torch.int32, device=p_new.device)
    else:
        n_movers_max = 0
    _check(lib().kc_frontier_repair(grid._h, pp, N, _ptr(movers, torch.int32, "movers"),
                                    _ptr(n_movers, torch.int32, "n_movers"), n_movers_max,
                                    _ptr(F, torch.int32, "F"), _ptr(nF, torch.int32, "nF"), nF_max,
                                    *certs._ptrs(), _stream()), "kc_frontier_repair")
    return certs


def kc_grid_update(grid: Grid, p_new, movers=None, n_movers=None, n_movers_max=None):
    """A6, Algorithm 1 line 3: bring the resident grid to positions p_new."""
    pp, N, d = _pos(p_new, "p_new")
    if movers is not None:
        n_movers_max = int(movers.numel() if n_movers_max is None else n_movers_max)
        if n_movers is None:
            n_movers = torch.tensor([movers.numel()], dtype=torch.int32, device=p_new.device)
    else:
        n_movers_max = 0
    _check(lib().kc_grid_update(grid._h, pp, N, _ptr(movers, torch.int32, "movers"),
                                _ptr(n_movers, torch.int32, "n_movers"), n_movers_max, _stream()), "kc_grid_update")


def kc_frontier_search(grid: Grid, p_new, F, nF, certs: Certs, nF_max=None) -> Certs:
    """A7, Algorithm 1 lines 4-7: re-search the ids in F, in place."""
    pp, N, d = _pos(p_new, "p_new")
    nF_max = int(F.numel() if nF_max is None else nF_max)
    _check(lib().kc_frontier_search(grid._h, pp, N, _ptr(F, torch.int32, "F"), _ptr(nF, torch.int32, "nF"), nF_max,
                                    *certs._ptrs(), _stream()), "kc_frontier_search")
    return certs


def kc_frontier_classify_local(grid: Grid, p, p2, certs: Certs, eps, flags=None, F=None, nF=None):
    """NEXT #2: frontier from per-point displacements and the per-block maximum; a
    subset of the Lemma-1 frontier that shrinks with the number of movers.  Grid resident at p."""
    pp, N, d = _pos(p)
    pq, N2, d2 = _pos(p2, "p2")
    if (N, d) != (N2, d2):
        raise ValueError("p and p2 must have the same shape")
    flags = flags if flags is not None else torch.empty(N, dtype=torch.uint8, device=p.device)
    F = F if F is not None else torch.empty(N, dtype=torch.int32, device=p.device)
    nF = nF if nF is not None else torch.empty(1, dtype=torch.int32, device=p.device)
    _check(lib().kc_frontier_classify_local(grid._h, pp, pq, N, _ptr(certs.nn, torch.int32, "nn"),
                                            _ptr(certs.d1, torch.float32, "d1"), _ptr(certs.c, torch.float32, "c"),
                                            _ptr(eps, torch.float32, "eps"), _ptr(flags, torch.uint8, "flags"),
                                            _ptr(F, torch.int32, "F"), _ptr(nF, torch.int32, "nF"), _stream()),
           "kc_frontier_classify_local")
    return flags, F, nF


def kc_frontier_classify_clock(c, stamp, S_in, eps, S_out, flags=None, F=None, nF=None):
    """NEXT #3, Appendix A.2: F = {i : c_i <= 4 (S - S_i)}, S = S_in + eps -> S_out."""
    N = c.numel()
    flags = flags if flags is not None else torch.empty(N, dtype=torch.uint8, device=c.device)
    F = F if F is not None else torch.empty(N, dtype=torch.int32, device=c.device)
    nF = nF if nF is not None else torch.empty(1, dtype=torch.int32, device=c.device)
    _check(lib().kc_frontier_classify_clock(_ptr(c, torch.float32, "c"), _ptr(stamp, torch.float32, "stamp"), N,
                                            _ptr(S_in, torch.float64, "S_in"), _ptr(eps, torch.float32, "eps"),
                                            _ptr(S_out, torch.float64, "S_out"), _ptr(flags, torch.uint8, "flags"),
                                            _ptr(F, torch.int32, "F"), _ptr(nF, torch.int32, "nF"), _stream()),
           "kc_frontier_classify_clock")
    return flags, F, nF


def kc_clock_stamp(stamp, S, F=None, nF=None, nF_max=None):
    """stamp[i] = S rounded down for i in F (all points when F is None)."""
    N = stamp.numel()
    nF_max = 0 if F is None else int(F.numel() if nF_max is None else nF_max)
    _check(lib().kc_clock_stamp(_ptr(F, torch.int32, "F"), _ptr(nF, torch.int32, "nF"), nF_max, N,
                                _ptr(S, torch.float64, "S"), _ptr(stamp, torch.float32, "stamp"), _stream()),
           "kc_clock_stamp")
    return stamp


def kc_clock_tree_build(c, stamp, tree=None):
    """Expiry tournament tree of the clock (Theorem 2; kc.h) from c and stamp."""
    N = c.numel()
    if tree is None:
        tree = torch.empty(int(lib().kc_clock_tree_floats(N)), dtype=torch.float32, device=c.device)
    _check(lib().kc_clock_tree_build(_ptr(c, torch.float32, "c"), _ptr(stamp, torch.float32, "stamp"), N,
                                     _ptr(tree, torch.float32, "tree"), _stream()), "kc_clock_tree_build")
    return tree


def kc_frontier_classify_clock_tree(c, stamp, tree, S_in, eps, S_out, F=None, nF=None):
    """kc_frontier_classify_clock's F (as a set) through the expiry tree: reads N/1024 nodes + the opened ones."""
    N = c.numel()
    F = F if F is not None else torch.empty(N, dtype=torch.int32, device=c.device)
    nF = nF if nF is not None else torch.empty(1, dtype=torch.int32, device=c.device)
    _check(lib().kc_frontier_classify_clock_tree(_ptr(c, torch.float32, "c"), _ptr(stamp, torch.float32, "stamp"), N,
                                                 _ptr(tree, torch.float32, "tree"), _ptr(S_in, torch.float64, "S_in"),
                                                 _ptr(eps, torch.float32, "eps"), _ptr(S_out, torch.float64, "S_out"),
                                                 _ptr(F, torch.int32, "F"), _ptr(nF, torch.int32, "nF"), _stream()),
           "kc_frontier_classify_clock_tree")
    return F, nF


def kc_clock_tree_update(tree, c, stamp, F, nF, nF_max=None):
    """Recompute the tree nodes above the ids in F (after their certificates were re-stamped)."""
    N = c.numel()
    nF_max = int(F.numel() if nF_max is None else nF_max)
    _check(lib().kc_clock_tree_update(_ptr(F, torch.int32, "F"), _ptr(nF, torch.int32, "nF"), nF_max,
                                      _ptr(c, torch.float32, "c"), _ptr(stamp, torch.float32, "stamp"), N,
                                      _ptr(tree, torch.float32, "tree"), _stream()), "kc_clock_tree_update")
    return tree


def kc_failure_audit(nn_pre, nn_post, flags, Ft=None, counts=None, want_list=True):
    """NEXT #2, Definition 2 / Table 1: true frontier F_t = {nn changed} and
    the audit of the Lemma-1 rule.  Returns (counts int32[4] = |F_t|, detected, missed, false; Ft)."""
    N = nn_pre.numel()
    counts = counts if counts is not None else torch.empty(4, dtype=torch.int32, device=nn_pre.device)
    if Ft is None and want_list:
        Ft = torch.empty(N, dtype=torch.int32, device=nn_pre.device)
    _check(lib().kc_failure_audit(_ptr(nn_pre, torch.int32, "nn_pre"), _ptr(nn_post, torch.int32, "nn_post"),
                                  _ptr(flags, torch.uint8, "flags"), N, _ptr(Ft, torch.int32, "Ft"),
                                  _ptr(counts, torch.int32, "counts"), _stream()), "kc_failure_audit")
    return counts, Ft


def kc_launch_count() -> int:
    return int(lib().kc_launch_count())


def kc_fp32_probe(blocks=148 * 8, iters=20000) -> float:
    out = C.c_double()
    _check(lib().kc_fp32_probe(int(blocks), int(iters), C.byref(out), _stream()), "kc_fp32_probe")
    return float(out.value)
