"""A8 step driver: one maintenance step of Algorithm 1 on the GPU, both ways.

Per transition p -> p' (the per-transition protocol of reading A13: every step starts from exact
certificates and a grid resident at p, like the paper's independently labelled transitions,
PAPER.md:69-73):

    A0  eps_t = max_i ||p'_i - p_i||                         kc_max_displacement   (Alg. 1 l.1)
    A4  F = {i : c_i <= 4 eps_t}                             kc_frontier_classify  (Alg. 1 l.2)
    A6+A7  REPAIR path: incremental cell update + search of F  kc_frontier_repair  (Alg. 1 l.3-7)
    A5  H(F), m, C on the updated filing                     kc_frontier_entropy   (Def. 2)
    A2+A3  REBUILD path: O(N) grid rebuild at p'             kc_cert_grid_rebuild
    A1  all-pairs certification at p'                        kc_cert_allpairs[_bounded]

This module is host orchestration only: every arithmetic step runs in libkc's kernels.  It owns
the device buffers (torch tensors) and hands pointers to the C-ABI through :mod:`.binding`.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

from . import binding as kc

PHASES = ("maxdisp", "classify", "repair", "entropy", "rebuild", "allpairs")


@dataclass
class StepResult:
    """Device-side results of one step (no host sync was made to produce them)."""
    eps: torch.Tensor          # float32[1]
    nF: torch.Tensor           # int32[1]
    H: torch.Tensor            # float64[1]
    m_cells: torch.Tensor      # int32[1]
    C_occ: torch.Tensor        # int32[1]
    repaired: kc.Certs         # pre-step certificates with F re-searched (repair path); this buffer
                               # is reused by the NEXT step's rebuild
    rebuilt: kc.Certs          # exact certificates at p' from the grid rebuild
    certified: kc.Certs | None # exact certificates at p' from the all-pairs pass
    phase_ms: dict = field(default_factory=dict)
    audit: torch.Tensor | None = None   # int32[4]: |F_t|, detected, missed, false (kc_failure_audit)
    Ft: torch.Tensor | None = None      # ids of the true frontier F_t (audit[0] entries)


class Maintainer:
    """Resident state for N points: grid, certificates, frontier buffers."""

    def __init__(self, p0: torch.Tensor, occ: float = 2.0, geom: kc.kc_geom | None = None,
                 allpairs: bool = True):
        assert p0.is_cuda and p0.dtype == torch.float32 and p0.dim() == 2
        self.N, self.d = int(p0.shape[0]), int(p0.shape[1])
        self.geom = geom if geom is not None else kc.kc_geom_for(p0, occ)
        self.grid = kc.Grid(self.N, self.geom)
        dev = p0.device
        N = self.N
        self.certs = kc.Certs.empty(N, dev)        # current exact certificates (pre-step)
        self.other = kc.Certs.empty(N, dev)        # ping-pong partner: the rebuild writes here
        self.ap = kc.Certs.empty(N, dev) if allpairs else None
        self.flags = torch.empty(N, dtype=torch.uint8, device=dev)
        self.F = torch.empty(N, dtype=torch.int32, device=dev)
        # the step's scalar results share one 24-byte allocation (one device-to-host copy reads them all)
        self.scalars = torch.zeros(24, dtype=torch.uint8, device=dev)
        self.eps = self.scalars[0:4].view(torch.float32)
        self.nF = self.scalars[4:8].view(torch.int32)
        self.H = self.scalars[8:16].view(torch.float64)
        self.m = self.scalars[16:20].view(torch.int32)
        self.C = self.scalars[20:24].view(torch.int32)
        need = kc.lib().kc_cert_allpairs_workspace(N, self.d) if allpairs else 0
        self.ws = torch.zeros(max(need, 16), dtype=torch.uint8, device=dev)   # zero-filled once (kc.h)
        self.p = p0
        kc.kc_cert_grid_rebuild(self.grid, p0, self.certs)

    def step(self, p_next: torch.Tensor, movers: torch.Tensor | None = None,
             frontier: torch.Tensor | None = None, time_phases: bool = False,
             do_allpairs: bool = True, bounded_allpairs: bool = True, seeded_allpairs: bool = True,
             audit: bool = False) -> StepResult:
        """One transition p -> p_next through every row of the hot path.

        ``movers``: optional int32 id list of the points that moved (None = all may have moved).
        ``frontier``: optional int32 id list to repair instead of the Lemma-1 set (reading A12:
        the sweep's controlled frontier is the mover list)."""
        ev = {}

        def mark(name):
            if time_phases:
                e = torch.cuda.Event(enable_timing=True)
                e.record()
                ev[name] = e

        nn_pre = self.certs.nn.clone() if audit else None    # the repair below overwrites nn at F
        mark("t0")
        kc.kc_max_displacement(self.p, p_next, self.eps)
        mark("maxdisp")
        if frontier is None:
            kc.kc_frontier_classify(self.certs.c, self.eps, self.flags, self.F, self.nF)
            F, nF, nF_max = self.F, self.nF, self.N
        else:
            kc.kc_frontier_classify(self.certs.c, self.eps, self.flags, self.F, self.nF)
            F, nF_max = frontier, int(frontier.numel())
            nF = torch.full((1,), nF_max, dtype=torch.int32, device=F.device)
        mark("classify")
        # repair path: in place on the pre-step certificates (Alg. 1 returns "updated certificates");
        # the rebuild path writes the ping-pong partner, so neither strategy sees the other's output
        repaired = self.certs
        kc.kc_frontier_repair(self.grid, p_next, F, nF, repaired, movers=movers, nF_max=nF_max)
        mark("repair")
        kc.kc_frontier_entropy(self.grid, F, nF, nF_max=nF_max, out=(self.H, self.m, self.C))
        mark("entropy")
        kc.kc_cert_grid_rebuild(self.grid, p_next, self.other)
        self.certs, self.other = self.other, self.certs
        mark("rebuild")
        if do_allpairs and self.ap is not None:
            # the maintained certificates bound the new second-neighbour distance by d2 + 2 eps_t
            # (Lemma 1's triangle inequality; entries repaired above already hold the
            # new d2); the pass is exact whatever the bound (kc_cert_allpairs_bounded)
            if seeded_allpairs:
                # ... or, tighter and without eps_t: the maintained neighbours themselves are two
                # known points, their new distances bound the new d2 (kc_cert_allpairs_seeded)
                kc.kc_cert_allpairs(p_next, self.ap, self.ws, seed1=repaired.nn, seed2=repaired.nn2)
            elif bounded_allpairs:
                kc.kc_cert_allpairs(p_next, self.ap, self.ws, d2_prev=repaired.d2, eps=self.eps)
            else:
                kc.kc_cert_allpairs(p_next, self.ap, self.ws)
        mark("allpairs")
        self.p = p_next
        res = StepResult(self.eps, nF, self.H, self.m, self.C, repaired, self.certs,
                         self.ap if do_allpairs else None)
        if time_phases:
            res.phase_ms = ev
        if audit:
            # Definition 2: the true frontier F_t and the Lemma-1 audit, from the exact
            # certificates before and after the step (outside the timed phases)
            res.audit, res.Ft = kc.kc_failure_audit(nn_pre, self.certs.nn, self.flags)
        return res

    @staticmethod
    def phase_times(ev: dict) -> dict:
        """Milliseconds per phase from the events of a finished step (call after a sync)."""
        order = ["t0", "maxdisp", "classify", "repair", "entropy", "rebuild", "allpairs"]
        out = {}
        for a, b in zip(order[:-1], order[1:]):
            out[b] = ev[a].elapsed_time(ev[b])
        return out


def crossover_fraction(fracs, t_repair, t_rebuild):
    """Smallest mover fraction f* with t_repair(f*) >= t_rebuild, by linear interpolation in log f
    between the bracketing sweep points (Proposition 1).  None if repair always wins
    inside the sweep, 0.0 if it never does."""
    fracs = np.asarray(fracs, float)
    r = np.asarray(t_repair, float) / np.asarray(t_rebuild, float)
    if r[0] >= 1.0:
        return 0.0
    for k in range(1, len(fracs)):
        if r[k] >= 1.0:
            a, b = np.log(fracs[k - 1]), np.log(fracs[k])
            w = (1.0 - r[k - 1]) / (r[k] - r[k - 1])
            return float(np.exp(a + w * (b - a)))
    return None


class ClockMaintainer:
    """NEXT #3: multi-step maintenance with the cumulative clock of Appendix A.2.

    No rebuild between steps: the clock S accumulates the per-step maxima eps_s, a certificate last
    recomputed at clock S_i is revisited when c_i <= 4 (S - S_i), and only those points are
    re-searched against the incrementally updated grid.  Nearest neighbours stay exact for every
    point (Theorem 1 on cumulative displacement); d1, d2, c are exact for the points revisited in
    the current step and stale for the rest, by design."""

    def __init__(self, p0: torch.Tensor, occ: float = 2.0, rebin_every: int = 4, tree: bool = False,
                 geom: kc.kc_geom | None = None):
        assert p0.is_cuda and p0.dtype == torch.float32 and p0.dim() == 2
        self.N = int(p0.shape[0])
        dev = p0.device
        # tree: the expired set comes from the expiry tournament tree (Theorem 2's heap, kc.h) instead
        # of the flat test of all N certificates: same set, no flags array
        self.tree = torch.empty(int(kc.lib().kc_clock_tree_floats(self.N)), dtype=torch.float32, device=dev) if tree else None
        # every `rebin_every` steps the grid is re-binned at the new positions (A2 only: O(N), no
        # certificate is recomputed) instead of updated incrementally, so the overflow chains of
        # re-filed points never grow long; 0 = never
        self.rebin_every = int(rebin_every)
        self.k = 0
        self.none = torch.zeros(1, dtype=torch.int32, device=dev)
        self.geom = geom if geom is not None else kc.kc_geom_for(p0, occ)
        self.grid = kc.Grid(self.N, self.geom)
        self.certs = kc.Certs.empty(self.N, dev)
        self.stamp = torch.zeros(self.N, dtype=torch.float32, device=dev)
        self.S = [torch.zeros(1, dtype=torch.float64, device=dev), torch.zeros(1, dtype=torch.float64, device=dev)]
        self.flags = torch.empty(self.N, dtype=torch.uint8, device=dev)
        self.F = torch.empty(self.N, dtype=torch.int32, device=dev)
        self.nF = torch.zeros(1, dtype=torch.int32, device=dev)
        self.eps = torch.zeros(1, dtype=torch.float32, device=dev)
        self.rebuild(p0)

    def rebuild(self, p: torch.Tensor):
        """Fresh grid and exact certificates at p; every stamp is set to the current clock."""
        kc.kc_cert_grid_rebuild(self.grid, p, self.certs)
        kc.kc_clock_stamp(self.stamp, self.S[0])
        if self.tree is not None:
            kc.kc_clock_tree_build(self.certs.c, self.stamp, self.tree)
        self.p = p

    def step(self, p_next: torch.Tensor, movers: torch.Tensor | None = None):
        """p -> p_next: A0, clock classify, A6 + A7 on the expired certificates, re-stamp.  No host
        sync.  Returns (F, nF) of this step (device tensors)."""
        kc.kc_max_displacement(self.p, p_next, self.eps)
        if self.tree is not None:
            kc.kc_frontier_classify_clock_tree(self.certs.c, self.stamp, self.tree, self.S[0], self.eps, self.S[1],
                                               self.F, self.nF)
        else:
            kc.kc_frontier_classify_clock(self.certs.c, self.stamp, self.S[0], self.eps, self.S[1],
                                          self.flags, self.F, self.nF)
        self.S.reverse()
        self.k += 1
        if self.rebin_every and self.k % self.rebin_every == 0:
            kc.kc_grid_build(self.grid, p_next)
            movers, n_movers = self.F, self.none          # nothing left to refresh
        else:
            n_movers = None
        kc.kc_frontier_repair(self.grid, p_next, self.F, self.nF, self.certs, movers=movers,
                              n_movers=n_movers, nF_max=self.N)
        kc.kc_clock_stamp(self.stamp, self.S[0], self.F, self.nF, self.N)
        if self.tree is not None:
            kc.kc_clock_tree_update(self.tree, self.certs.c, self.stamp, self.F, self.nF, self.N)
        self.p = p_next
        return self.F, self.nF


class GraphMaintainer:
    """The step of :class:`Maintainer` captured in CUDA graphs (small N is launch-bound: ~20 short
    kernels per step).  Per ping-pong parity:
      graph A  = A0, A4, A6, A7 || A5 on the grid resident at p, beside them (second stream, fork /
                 join inside the graph) A2+A3 of p' into a second grid, then a snapshot of the new nn,
                 nn2 as the NEXT step's all-pairs seeds;
      graph B  = the all-pairs certification of p' started from every point's previous nn, nn2
                 (kc_cert_allpairs_seeded; the ids are the snapshot the previous step left).
    B depends on nothing A computes, so (overlap_allpairs) it runs on its own stream beside A,
    B still bracketed by CUDA events; the short latency-bound kernels of A fill the issue slots the
    N x N pass leaves free.  With overlap_allpairs=False B is replayed after A on the same stream.

    Device pointers are fixed: positions live in two library-side buffers (the caller's p_next is
    copied in, 4 d N bytes), certificates and grids ping-pong.  Every point is treated as a
    potential mover (no mover list: its length varies from step to step), which changes no
    result.  Only for grids below the sweep threshold of kc_frontier_search (its epoch is a
    host-side counter); larger problems are not launch-bound and use :class:`Maintainer`."""

    MAX_N = 199_999

    def __init__(self, p0: torch.Tensor, occ: float = 2.0, overlap_allpairs: bool = True):
        assert int(p0.shape[0]) <= self.MAX_N, "GraphMaintainer is for launch-bound (small) problems"
        self.overlap = bool(overlap_allpairs)
        self.m = Maintainer(p0, occ)
        self.N = self.m.N
        dev = p0.device
        self.grid = [self.m.grid, kc.Grid(self.N, self.m.geom)]
        self.side = torch.cuda.Stream(device=dev)
        self.side2 = torch.cuda.Stream(device=dev)
        self.side_ap = torch.cuda.Stream(device=dev)
        self.pos = [p0.clone(), torch.empty_like(p0)]
        self.cert = [self.m.certs, self.m.other]
        # seed1/2[k]: two known points per query at pos[k] (its exact neighbours there)
        self.seed1 = [self.cert[0].nn.clone(), torch.empty(self.N, dtype=torch.int32, device=dev)]
        self.seed2 = [self.cert[0].nn2.clone(), torch.empty(self.N, dtype=torch.int32, device=dev)]
        self.k = 0
        self.graphs = [None, None]
        self.launches = [0, 0]
        self.ap_events = None

    def _body_a(self, k):
        m, cur, nxt = self.m, self.pos[k], self.pos[1 - k]
        certs, other = self.cert[k], self.cert[1 - k]
        main = torch.cuda.current_stream()
        self.side.wait_stream(main)
        with torch.cuda.stream(self.side):                 # rebuild path: needs only p'
            kc.kc_cert_grid_rebuild(self.grid[1 - k], nxt, other)
            self.seed1[1 - k].copy_(other.nn)              # the next step's all-pairs seeds
            self.seed2[1 - k].copy_(other.nn2)
        kc.kc_max_displacement(cur, nxt, m.eps)            # repair path, on the grid resident at p
        kc.kc_frontier_classify(certs.c, m.eps, m.flags, m.F, m.nF)
        kc.kc_grid_update(self.grid[k], nxt)
        self.side2.wait_stream(main)
        with torch.cuda.stream(self.side2):                # A5 and A7 touch disjoint state
            kc.kc_frontier_entropy(self.grid[k], m.F, m.nF, nF_max=self.N, out=(m.H, m.m, m.C))
        kc.kc_frontier_search(self.grid[k], nxt, m.F, m.nF, certs, nF_max=self.N)
        main.wait_stream(self.side2)
        main.wait_stream(self.side)

    def _body_b(self, k):
        m = self.m
        kc.kc_cert_allpairs(self.pos[1 - k], m.ap, m.ws, seed1=self.seed1[k], seed2=self.seed2[k])

    def _capture(self, k):
        n0 = kc.kc_launch_count()
        ga, gb = torch.cuda.CUDAGraph(), torch.cuda.CUDAGraph()
        with torch.cuda.graph(ga):
            self._body_a(k)
        with torch.cuda.graph(gb):
            self._body_b(k)
        self.graphs[k] = (ga, gb)
        self.launches[k] = kc.kc_launch_count() - n0

    def _replay_b(self, gb, timed):
        if timed:
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            e0.record()
            gb.replay()
            e1.record()
            self.ap_events = (e0, e1)
        else:
            gb.replay()

    def step(self, p_next: torch.Tensor | None, time_allpairs: bool = False, a_first: bool = False) -> StepResult:
        """One transition; returns the same StepResult as Maintainer.step (no host sync).  With
        ``time_allpairs`` two CUDA events bracket the all-pairs graph (``self.ap_events``).
        ``p_next`` None: the caller has already written the new positions into next_buffer().
        ``a_first``: replay graph A before graph B.  The N x N pass takes every CTA slot once it is
        resident, so A's first kernels should be in before it; worth ~2 us when the host runs ahead
        of the device (steps queued back to back), but when every step is synchronised the host-side
        launch of the 20-node graph A then delays the pass, so the default launches B first."""
        k, m = self.k, self.m
        if p_next is not None:
            self.pos[1 - k].copy_(p_next, non_blocking=True)
        if self.graphs[k] is None:
            torch.cuda.synchronize()
            self._capture(k)
        ga, gb = self.graphs[k]
        main = torch.cuda.current_stream()
        if self.overlap:
            self.side_ap.wait_stream(main)
            if a_first:
                ga.replay()
            with torch.cuda.stream(self.side_ap):
                self._replay_b(gb, time_allpairs)
            if not a_first:
                ga.replay()
            main.wait_stream(self.side_ap)
        else:
            ga.replay()
            self._replay_b(gb, time_allpairs)
        self.k = 1 - k
        return StepResult(m.eps, m.nF, m.H, m.m, m.C, self.cert[k], self.cert[1 - k], m.ap)

    def next_buffer(self) -> torch.Tensor:
        """The device buffer the next step reads p' from (for callers that upload straight into it)."""
        return self.pos[1 - self.k]

    def launches_per_step(self, k=None):
        """Kernels of this library launched by one replayed step (counted at capture)."""
        return self.launches[self.k if k is None else k]
