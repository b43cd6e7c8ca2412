"""CPU oracle for the exact 2-NN certificate path — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` leg may import this package.  It shares no code with
``paper_2606_18314_b200`` (the CUDA product) and never imports it.

The arithmetic lives in ``kc_oracle.c`` (plain C, gcc, ``-ffp-contract=off``); this
module only compiles it and marshals numpy arrays through ctypes.  Every function
cites the passage of PAPER.md it restates (see the C file).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kc_oracle.c")
_LIB = os.path.join(_HERE, "libkc_oracle.so")
_lib = None

CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-std=c11"]


def build(force: bool = False) -> str:
    """Compile kc_oracle.c with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *CFLAGS, _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Geom(C.Structure):
    _fields_ = [("d", C.c_int32), ("G", C.c_int32 * 3), ("lo", C.c_float * 3),
                ("h", C.c_float), ("inv_h", C.c_float)]


@dataclass(frozen=True)
class Geom:
    """Grid geometry (reading A6): G cells per axis, origin lo, cell width h, 1/h."""
    d: int
    G: tuple
    lo: tuple
    h: np.float32
    inv_h: np.float32

    @property
    def n_cells(self) -> int:
        return int(self.G[0]) * int(self.G[1]) * int(self.G[2])

    def _c(self) -> _Geom:
        g = _Geom()
        g.d = self.d
        for a in range(3):
            g.G[a] = int(self.G[a])
            g.lo[a] = float(self.lo[a])
        g.h = float(self.h)
        g.inv_h = float(self.inv_h)
        return g


def _load():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        fp, ip, u8 = C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_uint8)
        L.orc_sqdist.restype = C.c_float
        L.orc_sqdist.argtypes = [fp, fp, C.c_int]
        L.orc_bruteforce_top2.restype = C.c_int
        L.orc_bruteforce_top2.argtypes = [fp, C.c_int64, C.c_int, ip, ip, fp, fp, fp, C.c_int]
        L.orc_bruteforce_top2_subset.restype = C.c_int
        L.orc_bruteforce_top2_subset.argtypes = [fp, C.c_int64, C.c_int, ip, C.c_int64,
                                                 ip, ip, fp, fp, fp, C.c_int]
        L.orc_bruteforce_topk.restype = C.c_int
        L.orc_bruteforce_topk.argtypes = [fp, C.c_int64, C.c_int, C.c_int, ip, C.c_int64, ip, fp, fp, C.c_int]
        L.orc_kdtree_top2.restype = C.c_int
        L.orc_kdtree_top2.argtypes = [fp, C.c_int64, C.c_int, ip, C.c_int64,
                                      ip, ip, fp, fp, fp, C.c_int]
        L.orc_max_displacement.restype = C.c_float
        L.orc_max_displacement.argtypes = [fp, fp, C.c_int64, C.c_int]
        L.orc_frontier.restype = C.c_int64
        L.orc_frontier.argtypes = [fp, C.c_int64, C.c_float, u8]
        L.orc_bbox.restype = None
        L.orc_bbox.argtypes = [fp, C.c_int64, C.c_int, fp, fp]
        L.orc_geom_from_bbox.restype = C.c_int
        L.orc_geom_from_bbox.argtypes = [C.c_int64, C.c_int, fp, fp, C.c_double, C.POINTER(_Geom)]
        L.orc_cell_ids.restype = None
        L.orc_cell_ids.argtypes = [fp, C.c_int64, C.POINTER(_Geom), ip]
        L.orc_entropy.restype = C.c_int
        L.orc_entropy.argtypes = [ip, C.c_int64, ip, C.c_int64, C.c_int64,
                                  C.POINTER(C.c_double), ip, ip]
        L.orc_num_procs.restype = C.c_int
        _lib = L
    return _lib


def num_procs() -> int:
    return int(_load().orc_num_procs())


def _f32(a, d=None):
    a = np.ascontiguousarray(a, dtype=np.float32)
    if d is not None:
        assert a.ndim == 2 and a.shape[1] == d
    return a


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


@dataclass
class Certs:
    """Certificate arrays of Definition 1 plus the runner-up index."""
    nn: np.ndarray
    nn2: np.ndarray
    d1: np.ndarray
    d2: np.ndarray
    c: np.ndarray


def _alloc(n):
    return Certs(np.empty(n, np.int32), np.empty(n, np.int32), np.empty(n, np.float32),
                 np.empty(n, np.float32), np.empty(n, np.float32))


def sqdist(a, b) -> np.float32:
    """O1: ((dx*dx)+(dy*dy))+(dz*dz) in separately rounded binary32."""
    a, b = _f32(a).ravel(), _f32(b).ravel()
    return np.float32(_load().orc_sqdist(_fp(a), _fp(b), a.size))


def bruteforce_top2(p, queries=None, nthreads: int | None = None) -> Certs:
    """O2, Definition 1: exact certificates by the O(N^2) definition."""
    p = _f32(p)
    N, d = p.shape
    nthreads = nthreads or num_procs()
    if queries is None:
        out = _alloc(N)
        rc = _load().orc_bruteforce_top2(_fp(p), N, d, _ip(out.nn), _ip(out.nn2), _fp(out.d1),
                                         _fp(out.d2), _fp(out.c), nthreads)
    else:
        q = np.ascontiguousarray(queries, dtype=np.int32)
        out = _alloc(q.size)
        rc = _load().orc_bruteforce_top2_subset(_fp(p), N, d, _ip(q), q.size, _ip(out.nn),
                                                _ip(out.nn2), _fp(out.d1), _fp(out.d2),
                                                _fp(out.c), nthreads)
    if rc != 0:
        raise ValueError(f"orc_bruteforce_top2 rc={rc}")
    return out


def bruteforce_topk(p, K: int, queries=None, nthreads: int | None = None):
    """NEXT #4, reading R20 (Definition 1 :29 generalised): the K smallest keys
    (s, j) of every query by the O(N^2) definition.  Returns (nnk int32[nq,K], dk float32[nq,K],
    ck float32[nq]) with ck = dk[:,K-1] - dk[:,K-2]."""
    p = _f32(p)
    N, d = p.shape
    nthreads = nthreads or num_procs()
    if queries is None:
        qp, nq = None, N
    else:
        q = np.ascontiguousarray(queries, dtype=np.int32)
        qp, nq = _ip(q), q.size
    nnk = np.empty((nq, K), np.int32)
    dk = np.empty((nq, K), np.float32)
    ck = np.empty(nq, np.float32)
    rc = _load().orc_bruteforce_topk(_fp(p), N, d, K, qp, nq, _ip(nnk), _fp(dk), _fp(ck), nthreads)
    if rc != 0:
        raise ValueError(f"orc_bruteforce_topk rc={rc}")
    return nnk, dk, ck


def kdtree_top2(p, queries=None, nthreads: int | None = None) -> Certs:
    """O7: the same certificates through an exact k-d tree."""
    p = _f32(p)
    N, d = p.shape
    nthreads = nthreads or num_procs()
    if queries is None:
        out = _alloc(N)
        qp, nq = None, 0
    else:
        q = np.ascontiguousarray(queries, dtype=np.int32)
        out = _alloc(q.size)
        qp, nq = _ip(q), q.size
    rc = _load().orc_kdtree_top2(_fp(p), N, d, qp, nq, _ip(out.nn), _ip(out.nn2), _fp(out.d1),
                                 _fp(out.d2), _fp(out.c), nthreads)
    if rc != 0:
        raise ValueError(f"orc_kdtree_top2 rc={rc}")
    return out


def max_displacement(p, p2) -> np.float32:
    """O3, Algorithm 1 line 1."""
    p, p2 = _f32(p), _f32(p2)
    assert p.shape == p2.shape
    return np.float32(_load().orc_max_displacement(_fp(p), _fp(p2), p.shape[0], p.shape[1]))


def frontier(c, eps):
    """O4, Algorithm 1 line 2: flags and the ascending index list."""
    c = _f32(c)
    flags = np.empty(c.size, np.uint8)
    n = _load().orc_frontier(_fp(c), c.size, C.c_float(float(eps)),
                             flags.ctypes.data_as(C.POINTER(C.c_uint8)))
    F = np.flatnonzero(flags).astype(np.int32)
    assert F.size == n
    return flags, F


def bbox(p):
    p = _f32(p)
    lo = np.zeros(3, np.float32)
    hi = np.zeros(3, np.float32)
    _load().orc_bbox(_fp(p), p.shape[0], p.shape[1], _fp(lo), _fp(hi))
    return lo, hi


def geom_from_bbox(N, d, lo, hi, occ=2.0) -> Geom:
    """Reading A6 of PAPER.md:27: grid geometry for mean occupancy ``occ``."""
    lo = np.ascontiguousarray(lo, np.float32)
    hi = np.ascontiguousarray(hi, np.float32)
    g = _Geom()
    rc = _load().orc_geom_from_bbox(int(N), int(d), _fp(lo), _fp(hi), float(occ), C.byref(g))
    if rc != 0:
        raise ValueError(f"orc_geom_from_bbox rc={rc}")
    return Geom(int(g.d), tuple(int(x) for x in g.G), tuple(np.float32(x) for x in g.lo),
                np.float32(g.h), np.float32(g.inv_h))


def geom_for(p, occ=2.0) -> Geom:
    p = _f32(p)
    lo, hi = bbox(p)
    return geom_from_bbox(p.shape[0], p.shape[1], lo, hi, occ)


def geom_by_median_density(p, occ=2.0) -> Geom:
    """Reading R24 of PAPER.md:27 ("the resolution is set so that the mean cell occupancy is a small
    constant") for point sets whose density is far from uniform: the occupancy is measured against
    the MEDIAN density of the occupied volume instead of the mean one, so that points packed into
    clusters of negligible volume do not shrink the cells of everything else.  Step by step:
      1. R = the largest integer with R^d * 64 <= N, at most 32 (d = 3) / 256 (d = 2); R < 2: no
         estimate, the result is geom_for(p, occ);
      2. a coarse grid of R cells per axis over the bounding box (geom_from_bbox(R^d, ..., occ = 1))
         and the number of points in each of its cells (the cell ids of O5);
      3. med = the lower median of the counts of the occupied coarse cells; n_eff = med * R^d is
         the size a uniform set of that density would have;
      4. k = log2(N / n_eff) rounded to the nearest integer and clamped to 0 .. 2 (decided in
         integers: k grows while 2 * (n_eff * 2^k)^2 < N^2);
      5. the result is geom_from_bbox(ceil(N / 2^k), d, lo, hi, occ): the cells of a set 2^k times
         smaller.  A uniform set gives k = 0, i.e. exactly geom_for(p, occ)."""
    p = _f32(p)
    N, d = p.shape
    lo, hi = bbox(p)
    r_max = 32 if d == 3 else 256
    R = 1
    while R + 1 <= r_max and (R + 1) ** d * 64 <= N:
        R += 1
    k = 0
    if R >= 2:
        gc = geom_from_bbox(R ** d, d, lo, hi, 1.0)
        counts = np.bincount(cell_ids(p, gc), minlength=gc.n_cells)
        occupied = np.sort(counts[counts > 0])
        med = int(occupied[(occupied.size - 1) // 2])
        n_eff = med * R ** d
        while k < 2 and 2 * (n_eff * 2 ** k) ** 2 < N * N:
            k += 1
    return geom_from_bbox(-(-N // 2 ** k), d, lo, hi, occ)


def cell_ids(p, g: Geom) -> np.ndarray:
    """O5: index cell of every point."""
    p = _f32(p, g.d)
    cell = np.empty(p.shape[0], np.int32)
    cg = g._c()
    _load().orc_cell_ids(_fp(p), p.shape[0], C.byref(cg), _ip(cell))
    return cell


def entropy(cell_all, F, n_cells):
    """O6, Definition 2: returns (H, m touched cells, C occupied cells)."""
    cell_all = np.ascontiguousarray(cell_all, np.int32)
    F = np.ascontiguousarray(F, np.int32)
    H = C.c_double()
    m = C.c_int32()
    Cc = C.c_int32()
    rc = _load().orc_entropy(_ip(cell_all), cell_all.size, _ip(F), F.size, int(n_cells),
                             C.byref(H), C.byref(m), C.byref(Cc))
    if rc != 0:
        raise ValueError(f"orc_entropy rc={rc}")
    return float(H.value), int(m.value), int(Cc.value)


def failure_audit(nn_pre, nn_post, flags):
    """Definition 2 and the audit columns of Table 1 / the dataset (PAPER.md:75-88,
    :131), written out: F_t = {i : nn changed}; returns (F_t ascending, counts) with counts =
    [|F_t|, detected = failed and flagged, missed = failed but called safe, false = flagged but
    still valid]."""
    nn_pre = np.asarray(nn_pre, np.int32)
    nn_post = np.asarray(nn_post, np.int32)
    flagged = np.asarray(flags) != 0
    failed = nn_pre != nn_post
    Ft = np.flatnonzero(failed).astype(np.int32)
    counts = np.array([failed.sum(), (failed & flagged).sum(), (failed & ~flagged).sum(),
                       (~failed & flagged).sum()], np.int32)
    return Ft, counts


def clock_stamp(S) -> np.float32:
    """Stamp of Appendix A.2's clock: S (float64) rounded toward -inf to float32, so the elapsed
    clock S - S_i is never under-estimated."""
    f = np.float32(S)
    if np.float64(f) > np.float64(S):
        f = np.nextafter(f, np.float32(-np.inf))
    return np.float32(f)


def clock_frontier(c, stamp, S_in, eps):
    """Appendix A.2: S = S_in + eps_t; a certificate last recomputed at clock S_i
    stays valid while S - S_i < c_i / 4, so F = {i : c_i <= 4 (S - S_i)} (inclusive, as Lemma 1 is
    strict).  Evaluated in float64.  Returns (S, flags, F ascending)."""
    S = np.float64(S_in) + np.float64(np.float32(eps))
    c64 = np.asarray(c, np.float32).astype(np.float64)
    st64 = np.asarray(stamp, np.float32).astype(np.float64)
    flags = (c64 <= 4.0 * (S - st64)).astype(np.uint8)
    return S, flags, np.flatnonzero(flags).astype(np.int32)


def local_frontier(p, p2, g: Geom, nn, d1, c, eps):
    """Per-point motion budget (reading R19), written out in float32:
    delta_k = ||p2_k - p_k|| (O1 arithmetic), Delta_B(i) = max delta over the points filed in the
    3^d cell block of i's cell (cells of p), a = nn_i,
      safe_local(i) = c_i > ((2 delta_i + delta_a) + Delta_B) K + m_i
                  and  R  > (((d1_i + 2 delta_i) + delta_a) + eps) K + m_i,
      K = 1 + 2^-18, m_i = (d1_i + c_i) 2^-18, R = h (1 - 2^-8) - max_axis slk,
      F = {i : not (c_i > 4 eps or safe_local(i))}.  Returns (flags, F ascending)."""
    f32 = np.float32
    p = _f32(p, g.d)
    p2 = _f32(p2, g.d)
    N, d = p.shape
    diff = (p2 - p).astype(f32)
    sq = (diff * diff).astype(f32)
    s = (sq[:, 0] + sq[:, 1]).astype(f32)
    if d == 3:
        s = (s + sq[:, 2]).astype(f32)
    delta = np.sqrt(s).astype(f32)
    cid = cell_ids(p, g)
    G = [int(x) for x in g.G]
    cellmax = np.zeros(G[0] * G[1] * G[2], f32)
    np.maximum.at(cellmax, cid, delta)
    cm = np.pad(cellmax.reshape(G[2], G[1], G[0]), 1)
    blk = np.zeros((G[2], G[1], G[0]), f32)
    for dz in (0, 1, 2):
        for dy in (0, 1, 2):
            for dx in (0, 1, 2):
                blk = np.maximum(blk, cm[dz:dz + G[2], dy:dy + G[1], dx:dx + G[0]])
    dB = blk.reshape(-1)[cid]
    slk = []
    for a in range(3):
        t = (abs(float(g.lo[a])) + G[a] * float(g.h)) / 1048576.0
        slk.append(np.nextafter(f32(t), f32(np.inf)))
    R = f32(f32(f32(g.h) * f32(0.99609375)) - max(slk))
    eps = f32(eps)
    nn = np.asarray(nn, np.int32)
    d1 = np.asarray(d1, f32)
    c = np.asarray(c, f32)
    da = np.where(nn >= 0, delta[np.maximum(nn, 0)], f32(0)).astype(f32)
    K = f32(1.0 + 2.0 ** -18)
    k18 = f32(2.0 ** -18)
    two = (f32(2) * delta).astype(f32)
    with np.errstate(invalid="ignore", over="ignore"):
        m = ((d1 + c).astype(f32) * k18).astype(f32)
        rhs1 = ((((two + da).astype(f32) + dB).astype(f32) * K).astype(f32) + m).astype(f32)
        rhs2 = (((((d1 + two).astype(f32) + da).astype(f32) + eps).astype(f32) * K).astype(f32) + m).astype(f32)
        safe = (c > f32(f32(4) * eps)) | ((c > rhs1) & (R > rhs2))
    flags = (~safe).astype(np.uint8)
    return flags, np.flatnonzero(flags).astype(np.int32)
