"""Seeded synthetic inputs: point sets and motion families of BASELINE.json's five configs.

This module holds NONE of the method's arithmetic (no distances-to-neighbours, no grid, no
frontier, no entropy): it only draws points and moves them.  It is the one module that both
the CUDA product (bench.py, driver) and the CPU oracle's tests consume, so both sides see the
same fp32 arrays ("both devices regenerate identical state from the shared
seed").  The paper's own ten families are named but not parameterised; the
recipes below are BASELINE.json's ``configs`` and are restated in DESIGN.md §inputs.

Everything is numpy on the host; positions are float32 ``(N, d)`` C-contiguous.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

F32 = np.float32

# name -> (N, d, eps, point recipe, families)
CONFIGS = {
    "cfg1": dict(N=1000, d=2, eps=1e-3, points="uniform", families=("walk",), steps=1, seed=0),
    "cfg2": dict(N=16000, d=2, eps=1e-3, points="uniform",
                 families=("walk", "translate", "rotate", "local", "shear"), steps=100, seed=2),
    "cfg3": dict(N=16000, d=3, eps=5e-4, points="uniform",
                 families=("walk", "cluster_drift", "diffuse5", "ball5", "vortex"), steps=100, seed=3),
    "cfg4": dict(N=262144, d=3, eps=1e-3, points="uniform", families=("fraction",), steps=1, seed=4),
    "cfg5_d2": dict(N=4194304, d=2, eps=2e-4, points="mixture", families=("walk",), steps=20, seed=5),
    "cfg5_d3": dict(N=4194304, d=3, eps=2e-4, points="mixture", families=("walk",), steps=20, seed=6),
}
CFG4_FRACTIONS = (0.001, 0.003, 0.01, 0.03, 0.1, 0.3, 1.0)


def _unit_vectors(rng, n, d):
    v = rng.standard_normal((n, d))
    v /= np.maximum(np.linalg.norm(v, axis=1, keepdims=True), 1e-300)
    return v


def in_ball(rng, n, d, radius):
    """n vectors uniform in the d-ball of the given radius (float64)."""
    r = radius * rng.random(n) ** (1.0 / d)
    return _unit_vectors(rng, n, d) * r[:, None]


def uniform_points(N, d, seed):
    rng = np.random.default_rng(seed)
    return rng.random((N, d)).astype(F32)


def cluster_points(N, d, seed, n_clusters, sigma):
    """N points from n_clusters isotropic Gaussians with centres uniform in [0,1]^d.
    Returns (points, cluster label of every point)."""
    rng = np.random.default_rng(seed)
    centres = rng.random((n_clusters, d))
    lab = rng.integers(0, n_clusters, N)
    p = centres[lab] + sigma * rng.standard_normal((N, d))
    return p.astype(F32), lab.astype(np.int32)


def mixture_points(N, d, seed, n_clusters=256, sigma=0.005):
    """Config 5: 50 % uniform background + 50 % from 256 Gaussian clusters, shuffled so that
    the point index carries no spatial information."""
    rng = np.random.default_rng(seed)
    nb = N // 2
    bg = rng.random((nb, d))
    centres = rng.random((n_clusters, d))
    lab = rng.integers(0, n_clusters, N - nb)
    cl = centres[lab] + sigma * rng.standard_normal((N - nb, d))
    p = np.concatenate([bg, cl], axis=0)
    rng.shuffle(p, axis=0)
    return p.astype(F32)


def lattice_points(n_side, d, pitch=1.0 / 64):
    """Regular lattice (a*pitch, b*pitch[, c*pitch]); dyadic pitch gives exact ties."""
    ax = np.arange(n_side, dtype=np.float64) * pitch
    g = np.stack(np.meshgrid(*([ax] * d), indexing="ij"), axis=-1).reshape(-1, d)
    return g.astype(F32)


def make_points(cfg: str, N=None, seed=None):
    c = CONFIGS[cfg]
    N = N or c["N"]
    seed = c["seed"] if seed is None else seed
    if c["points"] == "uniform":
        return uniform_points(N, c["d"], seed)
    return mixture_points(N, c["d"], seed)


@dataclass
class Motion:
    """One motion family.  ``step(p)`` returns (p_new float32, movers int32 or None=all).

    Families (BASELINE.json configs 1-5):
      walk           every point displaced by a vector uniform in the eps-ball
      translate      rigid translation by eps along a fixed random direction + 1e-5 jitter
      rotate         d=2 rigid rotation about (0.5,0.5), omega = eps / r_max
      local          only points within 0.1 of a fixed random centre move, each by <= eps
      shear          v_x = eps*(2y-1)
      cluster_drift  each Gaussian cluster drifts rigidly by eps along its own direction
      diffuse5       5 % of points, drawn uniformly each step, move by exactly eps
      ball5          the same count, the points nearest a random centre, move by exactly eps
      vortex         differential rotation about the z-axis through (0.5,0.5), max step eps
      fraction       a fraction f of points (scattered or one ball) moves by exactly eps
    """
    family: str
    d: int
    eps: float
    seed: int
    labels: np.ndarray | None = None     # cluster labels for cluster_drift
    fraction: float = 0.05
    ball: bool = False

    def __post_init__(self):
        self.rng = np.random.default_rng(self.seed)
        self.t = 0
        d = self.d
        if self.family == "translate":
            self.dir = _unit_vectors(self.rng, 1, d)[0]
        if self.family == "local":
            self.centre = 0.2 + 0.6 * self.rng.random(d)
        if self.family == "cluster_drift":
            assert self.labels is not None
            self.cdir = _unit_vectors(self.rng, int(self.labels.max()) + 1, d)

    def step(self, p: np.ndarray):
        N, d = p.shape
        rng, eps, fam = self.rng, self.eps, self.family
        q = p.astype(np.float64)
        movers = None
        if fam == "walk":
            q += in_ball(rng, N, d, eps)
        elif fam == "translate":
            q += eps * self.dir + in_ball(rng, N, d, 1e-5)
        elif fam == "rotate":
            ctr = np.full(2, 0.5)
            r = q[:, :2] - ctr
            rmax = np.sqrt((r * r).sum(1).max())
            w = eps / rmax
            cw, sw = np.cos(w), np.sin(w)
            q[:, 0] = ctr[0] + cw * r[:, 0] - sw * r[:, 1]
            q[:, 1] = ctr[1] + sw * r[:, 0] + cw * r[:, 1]
        elif fam == "local":
            sel = np.flatnonzero(((q - self.centre) ** 2).sum(1) <= 0.1 ** 2)
            q[sel] += in_ball(rng, sel.size, d, eps)
            movers = sel
        elif fam == "shear":
            q[:, 0] += eps * (2.0 * q[:, 1] - 1.0)
        elif fam == "cluster_drift":
            q += eps * self.cdir[self.labels]
        elif fam in ("diffuse5", "ball5", "fraction"):
            k = max(1, int(round(self.fraction * N)))
            if fam == "ball5" or (fam == "fraction" and self.ball):
                ctr = 0.25 + 0.5 * rng.random(d)
                d2c = ((q - ctr) ** 2).sum(1)
                sel = np.argpartition(d2c, k - 1)[:k] if k < N else np.arange(N)
            else:
                sel = rng.choice(N, size=k, replace=False) if k < N else np.arange(N)
            sel = np.sort(sel)
            q[sel] += eps * _unit_vectors(rng, sel.size, d)
            movers = sel
        elif fam == "vortex":
            r0 = 0.25
            rx, ry = q[:, 0] - 0.5, q[:, 1] - 0.5
            r = np.sqrt(rx * rx + ry * ry)
            arc = eps * (r / r0) * np.exp(1.0 - r / r0)          # <= eps, max at r = r0
            th = np.where(r > 0, arc / np.maximum(r, 1e-300), 0.0)
            cw, sw = np.cos(th), np.sin(th)
            q[:, 0] = 0.5 + cw * rx - sw * ry
            q[:, 1] = 0.5 + sw * rx + cw * ry
        else:
            raise ValueError(f"unknown motion family {fam!r}")
        self.t += 1
        return q.astype(F32), (None if movers is None else movers.astype(np.int32))


def make_scene(cfg: str, family: str | None = None, N=None, seed=None, **kw):
    """Points + Motion for one config/family.  Returns (p0 float32 (N,d), Motion)."""
    c = CONFIGS[cfg]
    family = family or c["families"][0]
    seed = c["seed"] if seed is None else seed
    labels = None
    if family == "cluster_drift":
        p0, labels = cluster_points(N or c["N"], c["d"], seed, 32, 0.02)
    else:
        p0 = make_points(cfg, N, seed)
    fam_id = sum(ord(ch) for ch in family)
    mot = Motion(family, c["d"], c["eps"], seed * 1000 + fam_id, labels=labels, **kw)
    return p0, mot
