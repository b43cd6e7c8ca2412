#!/usr/bin/env python
"""bench.py — certified points/s of the whole hot path.

    python bench.py --gpus 1 --steps K --warmup W            # this repo's CUDA path
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands

Default workload: BASELINE.json config 5 ("Scale"), N = 4,194,304 points in d = 3 (``--workload
cfg5_d2`` for d = 2): 50 % uniform background + 50 % from 256 Gaussian clusters, random-walk steps
with eps = 2e-4.  A "step" is one maintenance transition p -> p' through every row of the hot path:
max displacement (A0), Lemma-1 classify (A4), incremental repair (A6+A7), frontier entropy (A5),
O(N) grid rebuild (A2+A3) at all 4,194,304 points, and the all-pairs oracle pass (A1) at the
first 1,048,576 points of p' (1.1e12 pair evaluations).  ``--workload cfg2 / cfg3`` runs the small
launch-bound configurations (N = 16,000, five motion families) as CUDA graphs.
Prints ONE JSON line (rank 0).  Details of every field: DESIGN.md §6.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_18314_b200 import workloads as wl  # noqa: E402

METRIC = "certified_points_per_s"
UNIT = "points/s"
L2_FLUSH_BYTES = int(os.environ.get("KC_FLUSH_MB", "256")) << 20
FP32_LANES = 148 * 128          # B200: 148 SMs x 128 FP32 lanes, one non-fused op / lane / clk
N_ALLPAIRS = 1 << 20            # config 5: the all-pairs oracle pass runs on the first 2^20 points
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the named kernel, from the committed
# ncu --set full captures (profiles/, file named beside each figure); None where no capture exists
NCU_TRAFFIC_BYTES = {
    ("cfg2", "allpairs_kernel"): 279552,            # profiles/r1f_allpairs_cfg2_full.txt
    ("cfg5_d3", "allpairs_kernel"): 165806848,      # profiles/r2_allpairs_1m_cfg5_d3_full.txt (read + written)
    ("cfg5_d2", "allpairs_kernel"): 145646592,      # profiles/r2_allpairs_1m_cfg5_d2_full.txt
    # A2 + A3, summed over the kernels of one kc_cert_grid_rebuild call (build_prep, cellid_hist, scan_cells,
    # leafid_hist, lscan, scatter, search_leaf + ball_finish / search_tiled): profiles/r2_grid_cfg5_d3_full.txt
    # (591 MB read + 387 MB written) / r2_grid_cfg5_d2_full.txt (420 + 663 MB)
    ("cfg5_d3", "rebuild"): 978100000,
    ("cfg5_d2", "rebuild"): 1082500000,
}
# algorithmic bytes per point of the O(N) rebuild (A2 + A3) with this layout
REBUILD_BYTES_PER_POINT = {2: 76.0, 3: 90.0}
BUILD_BYTES_PER_POINT = {2: 46.0, 3: 56.0}          # A2 alone
SEARCH_BYTES_PER_POINT = {2: 36.0, 3: 40.0}         # A3 alone (compulsory traffic)


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def build_trajectories(cfg, n_per_family, seed_shift=0):
    """Host-side positions for every family: {family: (list of (N,d) float32, list of movers)}."""
    c = wl.CONFIGS[cfg]
    out = {}
    for fam in c["families"]:
        p, mot = wl.make_scene(cfg, fam, seed=c["seed"] + 7919 * seed_shift)
        ps, mv = [p], [None]
        for _ in range(n_per_family):
            q, movers = mot.step(ps[-1])
            ps.append(q)
            mv.append(movers)
        out[fam] = (ps, mv)
    return out


def schedule(cfg, K):
    """K steps split evenly (round-robin remainder) over the config's families, family by family."""
    fams = wl.CONFIGS[cfg]["families"]
    per = [K // len(fams) + (1 if i < K % len(fams) else 0) for i in range(len(fams))]
    return fams, per


# ------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline and --impl reference): the oracle as it stands, never tuned.
def oracle_step(oracle, p, q, pre_c, geom, brute_queries=None):
    """The oracle's restatement of one step: O3, O4, O5+O6, and the certificates by definition
    (brute force; a bounded query sample when asked)."""
    eps = oracle.max_displacement(p, q)
    flags, F = oracle.frontier(pre_c, eps)
    cid = oracle.cell_ids(q, geom)
    H, m, C = oracle.entropy(cid, F, geom.n_cells)
    post = oracle.kdtree_top2(q)                                   # the O(N log N) exact relabel
    bf = oracle.bruteforce_top2(q, queries=brute_queries)          # the O(N^2) definition
    return post, bf, (float(eps), F.size, H)


def run_oracle_arm(cfg, K, W, time_budget_s=None, pair_budget=1.5e11):
    import oracle
    oracle.build()
    c = wl.CONFIGS[cfg]
    N = c["N"]
    fams, per = schedule(cfg, K)
    nq = int(min(N, max(64, pair_budget // max(1, K * N))))
    queries = None if nq >= N else np.sort(np.random.default_rng(0).choice(N, nq, replace=False)).astype(np.int32)
    traj = build_trajectories(cfg, max(per) + W)
    p0 = traj[fams[0]][0][0]
    geom = oracle.geom_for(p0)
    done, t_total = 0, 0.0
    for fi, fam in enumerate(fams):
        ps, _ = traj[fam]
        pre = oracle.kdtree_top2(ps[0])
        n_warm = W if fi == 0 else 0
        for t in range(per[fi] + n_warm):
            t0 = time.perf_counter()
            post, bf, _ = oracle_step(oracle, ps[t], ps[t + 1], pre.c, geom, queries)
            dt = time.perf_counter() - t0
            pre = post
            if t >= n_warm:
                t_total += dt
                done += 1
            if time_budget_s is not None and t_total > time_budget_s:
                break
        if time_budget_s is not None and t_total > time_budget_s:
            break
    frac = 1.0 if queries is None else nq / N
    sample = (f"{done} full steps of {cfg} (families {','.join(fams)} in order); per step: max displacement, "
              f"Lemma-1 frontier, cell ids + entropy, k-d tree relabel of all {N} points, brute-force "
              f"definition for {nq if queries is not None else N} of {N} query points")
    # points certified per step by the O(N^2) definition, as in the GPU arm's all-pairs row
    value = (N * frac) * done / t_total
    return dict(value=value, steps=done, seconds=t_total, cores=oracle.num_procs(), sample=sample,
                ms_per_step=1e3 * t_total / max(done, 1))


def scale_workload_text(cfg):
    """config.workload of the headline (the same string in both arms)."""
    c = wl.CONFIGS[cfg]
    N, d, n_ap = c["N"], c["d"], min(N_ALLPAIRS, c["N"])
    return (f"{cfg} (BASELINE.json config 5, Scale): N={N}, d={d}, 50% uniform + 50% from 256 Gaussian clusters "
            f"(sigma=0.005), random-walk steps eps={c['eps']}, grid occupancy 2 against the median density (DESIGN.md R24); every step = A0, A4, A6+A7 (Lemma-1 "
            f"frontier), A5, A2+A3 at all {N} points, and the all-pairs oracle pass A1 on the first {n_ap} points of p' "
            f"({n_ap * (n_ap - 1):.3e} pairs)")


def oracle_scale_step(oracle, p, q, pre_c, geom, n_ap, n_bf):
    """Config 5, the oracle's restatement of one step at full size: O3, O4, O5+O6, the exact k-d
    tree relabel of all N points (all cores), and for the all-pairs row the k-d tree on the first
    n_ap points plus the brute-force definition for n_bf sampled queries (1.1e12 pairs on the CPU
    are not run)."""
    eps = oracle.max_displacement(p, q)
    flags, F = oracle.frontier(pre_c, eps)
    cid = oracle.cell_ids(q, geom)
    H, m, C = oracle.entropy(cid, F, geom.n_cells)
    post = oracle.kdtree_top2(q)
    qa = np.ascontiguousarray(q[:n_ap])
    ap = oracle.kdtree_top2(qa)
    qs = np.sort(np.random.default_rng(11).choice(n_ap, n_bf, replace=False)).astype(np.int32)
    bf = oracle.bruteforce_top2(qa, queries=qs)
    return dict(eps=eps, flags=flags, F=F, cid=cid, H=H, m=m, C=C, post=post, ap=ap, bf=bf, qs=qs)


def run_oracle_scale(cfg, K, W, time_budget_s=150.0):
    """--impl reference on config 5: K steps of oracle_scale_step (W capped at one untimed step),
    stopped early when the time budget is spent (the number of steps done is reported)."""
    import oracle
    oracle.build()
    c = wl.CONFIGS[cfg]
    N = c["N"]
    p, mot = wl.make_scene(cfg)
    geom = oracle.geom_by_median_density(p)
    pre = oracle.kdtree_top2(p)
    done, t_total = 0, 0.0
    for t in range(min(W, 1) + K):
        q, _ = mot.step(p)
        t0 = time.perf_counter()
        r = oracle_scale_step(oracle, p, q, pre.c, geom, N_ALLPAIRS, 64)
        dt = time.perf_counter() - t0
        p, pre = q, r["post"]
        if t >= min(W, 1):
            t_total += dt
            done += 1
            if t_total > time_budget_s:
                break
    sample = (f"{done} full steps of {cfg}: per step max displacement, Lemma-1 frontier, cell ids + entropy, exact "
              f"k-d tree relabel of all {N} points, k-d tree on the first {N_ALLPAIRS} points and the brute-force "
              f"definition for 64 of them")
    return dict(value=N * done / t_total, steps=done, seconds=t_total, cores=oracle.num_procs(), sample=sample,
                ms_per_step=1e3 * t_total / max(done, 1))


# ------------------------------------------------------------------------------------------
def aggregate_over_ranks(local_ms, local_units, device):
    """Replicas only (multi-GPU): the job's time is the MAX of the ranks' device times,
    its work the SUM of their units.  Works on any initialised process group (nccl on the GPU
    box, gloo in the CPU tests); without one it is the identity."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(local_ms), int(local_units)
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())


class ClockSampler:
    """SM clock / throttle reasons sampled through NVML from a thread DURING the timed region
    (the region is tens of milliseconds: an nvidia-smi subprocess would not even start in time)."""

    def __init__(self, index, period_s=0.002):
        import threading
        self.samples, self.reasons, self.err = [], set(), None
        self._stop = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:                                    # noqa: BLE001
            self.nv, self.err = None, repr(e)
            return
        self.period = period_s
        self.t = threading.Thread(target=self._run, daemon=True)
        self.t.start()

    def _sample(self):
        nv = self.nv
        sm = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
        pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
        r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
            else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        self.samples.append((sm, pw))
        for name, bit in (("hw_slowdown", 0x8), ("sw_power_cap", 0x4), ("sw_thermal_slowdown", 0x20),
                          ("hw_thermal_slowdown", 0x40), ("hw_power_brake_slowdown", 0x80)):
            if r & bit:
                self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._sample()
            except Exception as e:                                # noqa: BLE001
                self.err = repr(e)
                return
            time.sleep(self.period)

    def stop(self):
        if self.nv is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=[f"nvml unavailable: {self.err}"])
        self._stop.set()
        self.t.join(timeout=2)
        if not self.samples:
            try:
                self._sample()
            except Exception as e:                                # noqa: BLE001
                return dict(sm_mhz=None, sm_max_mhz=self.max_mhz, reasons=[f"nvml error: {e!r}"])
        sm = [s[0] for s in self.samples]
        return dict(sm_mhz=float(np.median(sm)), sm_min_mhz=float(min(sm)), sm_max_mhz=self.max_mhz,
                    power_w_max=float(max(s[1] for s in self.samples)), samples=len(sm),
                    reasons=sorted(self.reasons))


# ------------------------------------------------------------------------------------------
def run_gpu_arm(args):
    import torch
    import torch.distributed as dist

    from paper_2606_18314_b200 import binding as kc
    from paper_2606_18314_b200.driver import GraphMaintainer, Maintainer, crossover_fraction

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    kc.lib()
    dev = torch.device("cuda", local)
    cfg, K, W = args.workload, args.steps, args.warmup
    c = wl.CONFIGS[cfg]
    N, d = c["N"], c["d"]
    fams, per = schedule(cfg, K)
    # replicas only: every rank runs its own seeded copy of the workload
    traj = build_trajectories(cfg, 2 * max(per) + W, seed_shift=rank)
    flush = torch.empty(L2_FLUSH_BYTES // 4, dtype=torch.float32, device=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # device-resident inputs for `value`: every position array uploaded before the timed region
    dev_traj = {f: [torch.from_numpy(p).to(dev) for p in traj[f][0][: per[i] + W + 1]] for i, f in enumerate(fams)}
    dev_mv = {f: [None if m is None else torch.from_numpy(m).to(dev) for m in traj[f][1][: per[i] + W + 1]]
              for i, f in enumerate(fams)}
    # the step is launch-bound at this N (~20 short kernels): it runs as two CUDA graphs per step
    # (everything but all-pairs | all-pairs, so that the dominant kernel is still bracketed by
    # events); --no-graph issues the same calls eagerly
    use_graph = (not args.no_graph) and N <= GraphMaintainer.MAX_N
    ov = bool(int(os.environ.get('KC_BENCH_OVERLAP', '1')))     # all-pairs graph beside graph A
    maint = {f: (GraphMaintainer(dev_traj[f][0], overlap_allpairs=ov) if use_graph else Maintainer(dev_traj[f][0])) for f in fams}
    torch.cuda.synchronize()

    def do_step(f, t, timed):
        if use_graph:
            return maint[f].step(dev_traj[f][t], time_allpairs=timed, a_first=True)   # steps are queued back to back
        return maint[f].step(dev_traj[f][t], movers=dev_mv[f][t], time_phases=timed)

    phase_sum = {ph: 0.0 for ph in ("maxdisp", "classify", "repair", "entropy", "rebuild", "allpairs")}
    fam_stats = {f: dict(steps=0, repair_ms=0.0, rebuild_ms=0.0, frontier=0, H=0.0) for f in fams}
    step_events, step_info = [], []
    # warm-up, untimed: W steps of every family (graphs of both ping-pong parities get captured here)
    for f in fams:
        for t in range(W):
            do_step(f, t + 1, False)
    barrier()
    sampler = ClockSampler(local)
    launches0 = kc.kc_launch_count()
    graph_launches = 0
    t_wall0 = time.perf_counter()
    for fi, f in enumerate(fams):
        for t in range(per[fi]):
            flush.zero_()                                            # L2 flush between timed steps
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            if use_graph:
                graph_launches += maint[f].launches_per_step()
            e0.record()
            res = do_step(f, W + t + 1, True)
            e1.record()
            step_events.append((e0, e1))
            step_info.append((f, maint[f].ap_events if use_graph else res.phase_ms, res.nF.clone(), res.H.clone()))
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = kc.kc_launch_count() - launches0 + graph_launches
    clocks = sampler.stop()
    dev_ms = sum(a.elapsed_time(b) for a, b in step_events)
    ap_ms_sum = 0.0
    for f, ev, nF, H in step_info:
        s = fam_stats[f]
        s["steps"] += 1; s["frontier"] += int(nF.item()); s["H"] += float(H.item())
        if use_graph:
            ap_ms_sum += ev[0].elapsed_time(ev[1])
        else:
            pt = Maintainer.phase_times(ev)
            ap_ms_sum += pt["allpairs"]
    # per-phase times: an eager pass of the same steps outside the timed region (events between
    # the calls; inside a graph there is nothing to bracket)
    ph_steps = 0
    em = {f: Maintainer(dev_traj[f][0]) for f in fams}
    for fi, f in enumerate(fams):
        for t in range(W + min(per[fi], 10)):
            if t >= W:
                flush.zero_()
            r = em[f].step(dev_traj[f][t + 1], movers=dev_mv[f][t + 1], time_phases=t >= W)
            if t >= W:
                torch.cuda.synchronize()
                pt = Maintainer.phase_times(r.phase_ms)
                for ph in phase_sum:
                    phase_sum[ph] += pt[ph]
                ph_steps += 1
                fs = fam_stats[f]
                fs["repair_ms"] += pt["repair"] + pt["classify"] + pt["maxdisp"]; fs["rebuild_ms"] += pt["rebuild"]
                fs["ph_steps"] = fs.get("ph_steps", 0) + 1
    del em
    dev_ms_max, units = aggregate_over_ranks(dev_ms, N * K, dev)
    value = units / (dev_ms_max * 1e-3)

    # ---- end to end through the public API: pinned host inputs, H2D + step + D2H per step ----
    host_next = {f: [torch.from_numpy(p).pin_memory() for p in traj[f][0]] for f in fams}
    # results come back as two copies: the certificate set (nn, d1, d2, c: the first four rows of one
    # allocation) and the 24 bytes of scalars (eps_t, |F|, H, m, C)
    host_out = dict(certs=torch.empty((4, N), dtype=torch.int32).pin_memory(),
                    scalars=torch.empty(24, dtype=torch.uint8).pin_memory())
    bufs = [torch.empty(N, d, device=dev), torch.empty(N, d, device=dev)]
    h2d = N * d * 4
    d2h = 4 * N * 4 + 24
    e2e_events = []
    barrier()
    k = 0
    for fi, f in enumerate(fams):
        base = per[fi] + W                            # continue each family's trajectory
        m = maint[f]
        for t in range(per[fi]):
            flush.zero_()
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            e0.record()
            buf = m.next_buffer() if use_graph else bufs[k & 1]
            k += 1
            buf.copy_(host_next[f][base + t + 1], non_blocking=True)
            mv = traj[f][1][base + t + 1]
            mvd = None if mv is None else torch.from_numpy(mv).to(dev, non_blocking=True)
            res = m.step(None) if use_graph else m.step(buf, movers=mvd)
            host_out["certs"].copy_(res.rebuilt.buf[:4], non_blocking=True)
            host_out["scalars"].copy_(m.m.scalars if use_graph else m.scalars, non_blocking=True)
            e1.record()
            e1.synchronize()                                         # the user reads the result here
            e2e_events.append((e0, e1))
    barrier()
    e2e_ms = sum(a.elapsed_time(b) for a, b in e2e_events)
    e2e_ms_max, units = aggregate_over_ranks(e2e_ms, N * K, dev)
    e2e_value = units / (e2e_ms_max * 1e-3)

    out = None
    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        # ---- parity of the timed outputs against the CPU oracle (outside the timed region) ----
        certified, audit = verify_against_oracle(kc, Maintainer, torch, dev, cfg, traj, fams,
                                                 graph_cls=GraphMaintainer if use_graph else None)
        # ---- roofline of the dominant kernel (all-pairs; FP32 ALU bound) ----
        ops_per_pair = 5 if d == 2 else 8
        ap_ms = ap_ms_sum / K                      # live CUDA events around the kernel's launch, timed region
        ap_alone_ms = None
        if use_graph:                              # the same graph with nothing beside it, for comparison
            gm0 = maint[fams[0]]
            gb = gm0.graphs[gm0.k][1] if gm0.graphs[gm0.k] is not None else None
            if gb is not None:
                ap_alone_ms = _median_ms(torch, gb.replay, 9, flush=flush)
        achieved = N * (N - 1) * ops_per_pair / (ap_ms * 1e-3) / 1e12
        sm_max = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
        peak = FP32_LANES * sm_max * 1e6 / 1e12
        probe = kc.kc_fp32_probe() / 1e12
        roofline = dict(bound="alu", kernel="allpairs_kernel", achieved=achieved, peak=peak, unit="TFLOP/s",
                        frac=achieved / peak, traffic=NCU_TRAFFIC_BYTES.get((cfg, "allpairs_kernel")),
                        note=(f"{ops_per_pair} separately rounded FP32 ops per ordered pair (no FMA by contract); peak = "
                              f"148 SM x 128 lanes x {sm_max:.0f} MHz (derived, DESIGN.md); measured non-fused "
                              f"FADD/FMUL chain rate {probe:.2f} Top/s; kernel share of step = "
                              f"{ap_ms / (dev_ms_max / K):.2f}"),
                        pairs_per_s=N * (N - 1) / (ap_ms * 1e-3), ms_per_launch=ap_ms, fp32_probe_tops=probe,
                        # the same launch with the GPU to itself (the timed one shares it with graph A)
                        ms_per_launch_alone=ap_alone_ms,
                        frac_alone=None if not ap_alone_ms else N * (N - 1) * ops_per_pair / (ap_alone_ms * 1e-3) / 1e12 / peak)
        cpu = run_oracle_arm(cfg, K=30, W=0, time_budget_s=25.0)
        cpu_baseline = dict(value=cpu["value"], unit=UNIT, cores=cpu["cores"], kind="oracle", sample=cpu["sample"],
                            ms_per_step=cpu["ms_per_step"])
        extras = {}
        if not args.no_extras:
            extras = run_extras(kc, Maintainer, crossover_fraction, torch, dev, peaks, skip_cfg=cfg)
        families = {f: dict(steps=s["steps"], frontier_frac=s["frontier"] / max(1, s["steps"]) / N,
                            H=s["H"] / max(1, s["steps"]),
                            repair_path_ms=s["repair_ms"] / max(1, s.get("ph_steps", 0)),
                            rebuild_path_ms=s["rebuild_ms"] / max(1, s.get("ph_steps", 0)),
                            repair_over_rebuild=s["repair_ms"] / max(s["rebuild_ms"], 1e-12),
                            # Definition 2 / Table 1 on the certified transitions: P_t = |F_t|/N,
                            # fraction re-validated although still valid, Lemma-1 misses (must be 0)
                            pressure_true=audit[f]["pressure"], false_frac=audit[f]["false_frac"],
                            missed_safe=audit[f]["missed"])
                    for f, s in fam_stats.items()}
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": dev_ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{cfg}: N={N}, d={d}, eps={c['eps']}, families {','.join(fams)} "
                                   f"({'/'.join(map(str, per))} steps), grid occupancy 2, every step = A0,A4,A6+A7,A5,A2+A3,A1 "
                                   f"(A1 = the full N(N-1)-pair pass, started from each point's previous two neighbours, "
                                   f"kc_cert_allpairs_seeded)",
                       "l2": "flushed between timed steps (256 MiB write); per-step CUDA-event times summed",
                       "launch": ("CUDA graphs per step (all rows but A1 | A1), replayed; A1 on its own "
                                  "stream beside the other rows, bracketed by events"
                                  if use_graph else "eager stream launches"),
                       "multi_gpu": "replicas only: each rank runs its own seeded copy, no collective on the data path",
                       "certified": certified},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "cpu_baseline": cpu_baseline,
            # eager (ungraphed) pass of the same steps outside the timed region
            "phases_ms_per_step": {ph: v / max(ph_steps, 1) for ph, v in phase_sum.items()},
            "paths_points_per_s": {"allpairs": N / (ap_ms * 1e-3),
                                   "grid_rebuild": N / (phase_sum["rebuild"] / max(ph_steps, 1) * 1e-3),
                                   "frontier_repair": N / ((phase_sum["repair"] + phase_sum["classify"] + phase_sum["maxdisp"]) / max(ph_steps, 1) * 1e-3)},
            "families": families,
            "wall_s_timed_region": t_wall,
            "extras": extras,
        }
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return out


def run_gpu_arm_scale(args):
    """Config 5 (the headline): N = 4,194,304 points, random-walk steps, every row of the hot path
    per step; the all-pairs row on the first 2^20 points of p'.  Grids of this size are not
    launch-bound: the calls are issued eagerly through the public API."""
    import torch
    import torch.distributed as dist

    from paper_2606_18314_b200 import binding as kc
    from paper_2606_18314_b200.driver import Maintainer, crossover_fraction

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    kc.lib()
    dev = torch.device("cuda", local)
    cfg, K, W = args.workload, args.steps, args.warmup
    c = wl.CONFIGS[cfg]
    N, d = c["N"], c["d"]
    n_ap = min(N_ALLPAIRS, N)
    # default: replicas only, every rank runs its own seeded copy of the workload;
    # --shard queries: ONE copy, the N x N pass split by query over the ranks
    sharded = args.shard == "queries"
    p0, mot = wl.make_scene(cfg, seed=c["seed"] + (0 if sharded else 7919 * rank))
    host = [p0]
    for _ in range(W + K):
        host.append(mot.step(host[-1])[0])
    flush = torch.empty(L2_FLUSH_BYTES // 4, dtype=torch.float32, device=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    dev_traj = [torch.from_numpy(p).to(dev) for p in host]         # resident before the timed region
    geom = kc.kc_geom_by_median_density(dev_traj[0])               # reading R24 (both arms)
    m = Maintainer(dev_traj[0], geom=geom, allpairs=False)
    ap = kc.Certs.empty(n_ap, dev)
    ws = torch.zeros(max(16, kc.lib().kc_cert_allpairs_workspace(n_ap, d)), dtype=torch.uint8, device=dev)
    if sharded:
        from paper_2606_18314_b200.sharding import gather_columns, query_slice
        q_lo, q_hi = query_slice(n_ap, rank, world)
        q_ids = torch.arange(q_lo, q_hi, dtype=torch.int32, device=dev)
        q_n = torch.tensor([q_hi - q_lo], dtype=torch.int32, device=dev)
        ws_q = torch.zeros(max(16, kc.lib().kc_frontier_oracle_workspace(n_ap, d, q_hi - q_lo)), dtype=torch.uint8, device=dev)

    def step(mm, p_next, timed):
        res = mm.step(p_next, time_phases=timed, do_allpairs=False)
        ev = None
        if timed:
            ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
            ev[0].record()
        if sharded:
            # A1 by query: this rank's ids against all 2^20 points, then the certificate columns of the
            # other ranks (20 B per point, one all-gather)
            kc.kc_frontier_oracle(p_next[:n_ap], q_ids, q_n, ap, workspace=ws_q)
            gather_columns(ap.buf, n_ap)
        else:
            kc.kc_cert_allpairs(p_next[:n_ap], ap, ws)              # A1: the oracle pass, 2^20 points of p'
        if timed:
            ev[1].record()
        return res, ev

    for t in range(W):
        step(m, dev_traj[t + 1], False)
    barrier()
    sampler = ClockSampler(local, period_s=0.02)
    launches0 = kc.kc_launch_count()
    t_wall0 = time.perf_counter()
    step_events, infos = [], []
    for t in range(K):
        flush.zero_()                                                # L2 flush between timed steps
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        res, ev = step(m, dev_traj[W + t + 1], True)
        e1.record()
        step_events.append((e0, e1))
        infos.append((res.phase_ms, ev, res.nF.clone(), res.H.clone()))
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = kc.kc_launch_count() - launches0
    clocks = sampler.stop()
    dev_ms = sum(a.elapsed_time(b) for a, b in step_events)
    phase_sum = {ph: 0.0 for ph in ("maxdisp", "classify", "repair", "entropy", "rebuild", "allpairs")}
    nF_sum, H_sum = 0, 0.0
    for ph_ev, ev, nF, H in infos:
        pt = Maintainer.phase_times(ph_ev)
        for ph in ("maxdisp", "classify", "repair", "entropy", "rebuild"):
            phase_sum[ph] += pt[ph]
        phase_sum["allpairs"] += ev[0].elapsed_time(ev[1])
        nF_sum += int(nF.item()); H_sum += float(H.item())
    dev_ms_max, units = aggregate_over_ranks(dev_ms, N * K, dev)
    if sharded:
        units = N * K                                                # one job: every rank certified the same points
    value = units / (dev_ms_max * 1e-3)
    info = m.grid.info()
    del m

    # ---- end to end through the public API: pinned host inputs, H2D + step + D2H per step ----
    pinned = [torch.from_numpy(p).pin_memory() for p in host[: K + 1]]
    m2 = Maintainer(dev_traj[0], geom=geom, allpairs=False)
    n_pad = m2.certs.buf.shape[1]
    host_certs = torch.empty((5, n_pad), dtype=torch.int32).pin_memory()     # nn, d1, d2, c, nn2 of all N points
    host_scal = torch.empty(24, dtype=torch.uint8).pin_memory()
    bufs = [torch.empty(N, d, device=dev), torch.empty(N, d, device=dev)]
    h2d, d2h = N * d * 4, 5 * N * 4 + 24
    e2e_events = []
    barrier()
    for t in range(K):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        buf = bufs[t & 1]
        buf.copy_(pinned[t + 1], non_blocking=True)
        res, _ = step(m2, buf, False)
        host_certs.copy_(res.rebuilt.buf, non_blocking=True)
        host_scal.copy_(m2.scalars, non_blocking=True)
        e1.record()
        e1.synchronize()                                             # the user reads the result here
        e2e_events.append((e0, e1))
    barrier()
    e2e_ms = sum(a.elapsed_time(b) for a, b in e2e_events)
    e2e_ms_max, units = aggregate_over_ranks(e2e_ms, N * K, dev)
    if sharded:
        units = N * K
    e2e_value = units / (e2e_ms_max * 1e-3)
    del m2, pinned, bufs

    out = None
    if rank == 0:
        import oracle
        oracle.build()
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        hbm = float(peaks.get("hbm_gbs", 6650.0))
        hbm_src = "measured (MEASURED_PEAKS.json)" if "hbm_gbs" in peaks else "fallback (B200_PROFILING.md)"
        # ---- certified: the first transition recomputed by the CPU oracle (k-d tree at this size,
        # itself validated bitwise against brute force; brute-force definition on sampled queries);
        # the oracle's wall time for that step is the cpu_baseline (the oracle as it stands)
        g_or = oracle.geom_by_median_density(host[0])
        pre = oracle.kdtree_top2(host[0])
        t0 = time.perf_counter()
        w = oracle_scale_step(oracle, host[0], host[1], pre.c, g_or, n_ap, 64)
        t_cpu = time.perf_counter() - t0
        m3 = Maintainer(dev_traj[0], geom=geom, allpairs=False)
        u32 = lambda a: np.ascontiguousarray(a).view(np.uint32)
        ok = all(np.array_equal(u32(getattr(m3.certs, f).cpu().numpy()), u32(getattr(pre, f)))
                 for f in ("nn", "nn2", "d1", "d2", "c"))
        res, _ = step(m3, dev_traj[1], False)
        torch.cuda.synchronize()
        ok &= u32(res.eps.cpu().numpy())[0] == u32(np.array([w["eps"]], np.float32))[0]
        ok &= int(res.nF.item()) == w["F"].size
        F = w["F"]
        for f in ("nn", "nn2", "d1", "d2", "c"):
            want = u32(getattr(w["post"], f))
            ok &= bool(np.array_equal(u32(getattr(res.rebuilt, f).cpu().numpy()), want))
            ok &= bool(np.array_equal(u32(getattr(res.repaired, f).cpu().numpy())[F], want[F]))
            gap = u32(getattr(ap, f).cpu().numpy())
            ok &= bool(np.array_equal(gap, u32(getattr(w["ap"], f))))
            ok &= bool(np.array_equal(gap[w["qs"]], u32(getattr(w["bf"], f))))
        rest = np.flatnonzero(w["flags"] == 0)
        ok &= bool(np.array_equal(res.repaired.nn.cpu().numpy()[rest], w["post"].nn[rest]))      # Lemma 1
        ok &= abs(float(res.H.item()) - w["H"]) <= 1e-6 and int(res.m_cells.item()) == w["m"] and \
            int(res.C_occ.item()) == w["C"]
        if not ok:
            raise RuntimeError(f"parity failure against the CPU oracle: {cfg} step 0")
        certified = (f"1 transition at N={N}: rebuild (all points), repair (at F), all-pairs ({n_ap} points), eps, |F|, "
                     f"Lemma-1 nn bit-exact vs the CPU k-d tree oracle (+ 64 brute-force queries), H within 1e-6")
        del m3
        cpu_baseline = dict(value=N / t_cpu, unit=UNIT, cores=oracle.num_procs(), kind="oracle",
                            algorithm="exact k-d tree over all points, all cores (PAPER.md:106, Table 2's 149 ms row)",
                            sample=(f"1 full step at N={N}: max displacement, Lemma-1 frontier, cell ids + entropy, k-d tree "
                                    f"relabel of all points, k-d tree on the first {n_ap} points + 64 brute-force queries"),
                            ms_per_step=1e3 * t_cpu)
        # ---- rooflines
        ms = {ph: v / K for ph, v in phase_sum.items()}
        sm_max = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
        ops_per_pair = 5 if d == 2 else 8
        alu_peak = FP32_LANES * sm_max * 1e6 / 1e12
        probe = kc.kc_fp32_probe() / 1e12
        ap_achieved = n_ap * (n_ap - 1) * ops_per_pair / (ms["allpairs"] * 1e-3) / 1e12
        step_ms = dev_ms_max / K
        roofline = dict(bound="alu", kernel="allpairs_kernel", achieved=ap_achieved, peak=alu_peak, unit="TFLOP/s",
                        frac=ap_achieved / alu_peak, traffic=NCU_TRAFFIC_BYTES.get((cfg, "allpairs_kernel")),
                        note=(f"dominant kernel of the step by time (share {ms['allpairs'] / step_ms:.3f}): {ops_per_pair} separately "
                              f"rounded FP32 ops per ordered pair (no FMA by contract) x {n_ap}*({n_ap}-1) pairs per launch; peak = "
                              f"148 SM x 128 lanes x {sm_max:.0f} MHz (derived, DESIGN.md §5); measured non-fused FADD/FMUL "
                              f"chain rate {probe:.2f} Top/s"),
                        pairs_per_s=n_ap * (n_ap - 1) / (ms["allpairs"] * 1e-3), ms_per_launch=ms["allpairs"],
                        fp32_probe_tops=probe)
        reb_bytes = REBUILD_BYTES_PER_POINT[d] * N
        reb_gbs = reb_bytes / (ms["rebuild"] * 1e-3) / 1e9
        roofline_rebuild = dict(bound="hbm", kernel=f"kc_cert_grid_rebuild (A2 + A3: build kernels + {'search_leaf_kernel + ball_finish_kernel' if d == 3 else 'search_tiled_kernel'})",
                                achieved=reb_gbs, peak=hbm, unit="GB/s", frac=reb_gbs / hbm,
                                traffic=NCU_TRAFFIC_BYTES.get((cfg, "rebuild")),
                                note=(f"{REBUILD_BYTES_PER_POINT[d]:.0f} algorithmic B/point (SURVEY.md §8(d)) x {N} points / "
                                      f"{ms['rebuild']:.4f} ms (CUDA events around the call inside the timed steps); peak {hbm_src}; "
                                      f"the search is issue/latency-bound, not HBM-bound (DESIGN.md §5)"),
                                ms_per_call=ms["rebuild"])
        frontier_frac = nF_sum / K / N
        paths = {"allpairs": n_ap / (ms["allpairs"] * 1e-3), "grid_rebuild": N / (ms["rebuild"] * 1e-3),
                 "frontier_repair": N / ((ms["repair"] + ms["classify"] + ms["maxdisp"]) * 1e-3)}
        extras = {}
        if not args.no_extras:
            extras = run_extras(kc, Maintainer, crossover_fraction, torch, dev, peaks, skip_cfg=cfg)
            extras["mover_sweep_" + cfg] = mover_sweep_scale(kc, Maintainer, crossover_fraction, torch, dev, cfg, flush)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": step_ms, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": scale_workload_text(cfg),
                       "l2": "flushed between timed steps (256 MiB write); per-step CUDA-event times summed",
                       "launch": "eager stream launches through the C-ABI (a grid of this size is not launch-bound)",
                       "multi_gpu": ("query-partitioned all-pairs pass (SURVEY.md §8(e)): one copy of the workload, rank r "
                                     "runs kc_frontier_oracle on its contiguous share of the 2^20 queries, one all-gather of the "
                                     "certificate columns (20 B/point); the O(N) rows run replicated" if sharded else
                                     "replicas only: each rank runs its own seeded copy, no collective on the data path"),
                       "certified": certified},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms_max / K},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "roofline_rebuild": roofline_rebuild,
            "cpu_baseline": cpu_baseline,
            "phases_ms_per_step": ms,
            "paths_points_per_s": paths,
            "repair_over_rebuild": (ms["repair"] + ms["classify"] + ms["maxdisp"]) / ms["rebuild"],
            "lemma1_frontier_frac": frontier_frac, "H_mean": H_sum / K,
            "grid": {"max_cell_occupancy": int(info.max_occ), "occupied_cells": int(info.c_occ),
                     "subdivided_cells": int(info.n_heavy), "leaves": int(info.n_leaves)},
            "wall_s_timed_region": t_wall,
            "extras": extras,
        }
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return out

def verify_against_oracle(kc, Maintainer, torch, dev, cfg, traj, fams, steps_per_family=2, graph_cls=None):
    """'Certified' = the outputs of the timed configuration equal the CPU oracle's bit for bit
    (H within 1e-6).  Checked outside the timed region on the first transitions of every family;
    raises on any mismatch."""
    import oracle
    N = wl.CONFIGS[cfg]["N"]
    checked = 0
    audit = {}
    for f in fams:
        ps, mvs = traj[f]
        m = (graph_cls or Maintainer)(torch.from_numpy(ps[0]).to(dev))
        g = oracle.geom_for(ps[0])
        pre = oracle.bruteforce_top2(ps[0])
        for t in range(steps_per_family):
            q = ps[t + 1]
            mv = None if mvs[t + 1] is None else torch.from_numpy(mvs[t + 1]).to(dev)
            if graph_cls is not None:                      # the launch configuration the bench times
                nn_pre = m.cert[m.k].nn.clone()
                res = m.step(torch.from_numpy(q).to(dev))
                res.audit, res.Ft = kc.kc_failure_audit(nn_pre, res.rebuilt.nn, m.m.flags)
            else:
                res = m.step(torch.from_numpy(q).to(dev), movers=mv, audit=True)
            torch.cuda.synchronize()
            post = oracle.bruteforce_top2(q)
            eps = oracle.max_displacement(ps[t], q)
            flags, F = oracle.frontier(pre.c, eps)
            ok = res.eps.cpu().numpy().view(np.uint32)[0] == np.array([eps]).view(np.uint32)[0]
            ok &= int(res.nF.item()) == F.size
            for name in ("nn", "nn2", "d1", "d2", "c"):
                want = getattr(post, name)
                for got in (res.rebuilt, res.certified):
                    ok &= bool(np.array_equal(getattr(got, name).cpu().numpy().view(np.uint32), want.view(np.uint32)))
                ok &= bool(np.array_equal(getattr(res.repaired, name).cpu().numpy().view(np.uint32)[F], want.view(np.uint32)[F]))
            H, mm, C = oracle.entropy(oracle.cell_ids(q, g), F, g.n_cells)
            ok &= abs(float(res.H.item()) - H) <= 1e-6 and int(res.m_cells.item()) == mm and int(res.C_occ.item()) == C
            wFt, wcounts = oracle.failure_audit(pre.nn, post.nn, flags)
            got_counts = res.audit.cpu().numpy()
            ok &= got_counts.tolist() == wcounts.tolist() and int(wcounts[2]) == 0
            a = audit.setdefault(f, dict(pressure=0.0, false_frac=0.0, missed=0, n=0))
            a["pressure"] += float(wcounts[0]) / N; a["false_frac"] += float(wcounts[3]) / N
            a["missed"] += int(got_counts[2]); a["n"] += 1
            if not ok:
                raise RuntimeError(f"parity failure against the CPU oracle: {cfg}/{f} step {t}")
            pre = post
            checked += 1
    for a in audit.values():
        a["pressure"] /= a["n"]; a["false_frac"] /= a["n"]
    return (f"{checked} transitions ({steps_per_family} per family) bit-exact vs CPU oracle, H within 1e-6",
            audit)


def _median_ms(torch, fn, reps, setup=None, flush=None):
    ts = []
    for _ in range(reps):
        if setup is not None:
            setup()
        if flush is not None:
            flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1))
    return float(np.median(ts))


def family_table(kc, Maintainer, torch, dev, cfg, flush, steps=8):
    """Configs 2 / 3 (N = 16,000, five motion families each): per family the Lemma-1 frontier
    fraction, H(F), and the repair-path and rebuild-path time of a step (eager calls, medians).
    Config 3's diffuse5 / ball5 pair is the equal-size, different-entropy control of the paper's
    Fig. 2: the same number of movers, scattered or from one ball; the mover
    list is the controlled frontier there (reading R12)."""
    c = wl.CONFIGS[cfg]
    N = c["N"]
    rows = {}
    for fam in c["families"]:
        p, mot = wl.make_scene(cfg, fam)
        m = Maintainer(torch.from_numpy(p).to(dev), allpairs=False)
        rep_ms, reb_ms, fr, Hs, mvH, mv_ms = [], [], [], [], [], []
        for t in range(steps + 2):
            q, movers = mot.step(p)
            Q = torch.from_numpy(q).to(dev)
            mv = None if movers is None else torch.from_numpy(movers).to(dev)
            if t >= 2:
                flush.zero_()
            r = m.step(Q, movers=mv, time_phases=True, do_allpairs=False)
            torch.cuda.synchronize()
            if t >= 2:
                pt = Maintainer.phase_times(r.phase_ms)
                rep_ms.append(pt["maxdisp"] + pt["classify"] + pt["repair"]); reb_ms.append(pt["rebuild"])
                fr.append(int(r.nF.item()) / N); Hs.append(float(r.H.item()))
            p = q
        row = dict(lemma1_frontier_frac=float(np.mean(fr)), H=float(np.mean(Hs)), repair_path_ms=float(np.median(rep_ms)),
                   rebuild_path_ms=float(np.median(reb_ms)),
                   repair_over_rebuild=float(np.median(rep_ms) / np.median(reb_ms)))
        if fam in ("diffuse5", "ball5", "local"):
            # the mover list as the frontier: A0 + A6 + A7 at the movers only, and H of that list
            p, mot = wl.make_scene(cfg, fam)
            m = Maintainer(torch.from_numpy(p).to(dev), allpairs=False)
            H = torch.zeros(1, dtype=torch.float64, device=dev)
            for t in range(steps + 2):
                q, movers = mot.step(p)
                Q = torch.from_numpy(q).to(dev)
                mv = torch.from_numpy(movers).to(dev)
                nmv = torch.tensor([movers.size], dtype=torch.int32, device=dev)
                if t >= 2:
                    flush.zero_()
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record()
                kc.kc_max_displacement(m.p, Q, m.eps)
                kc.kc_frontier_repair(m.grid, Q, mv, nmv, m.certs, movers=mv, n_movers=nmv)
                e1.record()
                kc.kc_frontier_entropy(m.grid, mv, nmv, out=(H, m.m, m.C))
                kc.kc_cert_grid_rebuild(m.grid, Q, m.certs)
                m.p = Q
                torch.cuda.synchronize()
                if t >= 2:
                    mv_ms.append(e0.elapsed_time(e1)); mvH.append(float(H.item()))
                p = q
            row.update(movers=int(movers.size), mover_frontier_H=float(np.mean(mvH)), mover_repair_ms=float(np.median(mv_ms)),
                       mover_repair_over_rebuild=float(np.median(mv_ms) / np.median(reb_ms)))
        rows[fam] = row
        del m
    return rows


def mover_sweep_scale(kc, Maintainer, crossover_fraction, torch, dev, cfg, flush,
                      fractions=(0.001, 0.01, 0.03, 0.1, 0.3, 1.0)):
    """Config 5's points with config 4's protocol: a fraction f of the 4,194,304 points (scattered)
    moves by exactly eps; the mover list is the controlled frontier (reading R12).  Repair = A0 + A4 +
    A6 + A7 at the movers against the rebuild A2 + A3, and the crossover f* (Prop. 1)."""
    c = wl.CONFIGS[cfg]
    N, d = c["N"], c["d"]
    p = wl.make_points(cfg)
    P = torch.from_numpy(p).to(dev)
    m = Maintainer(P, geom=kc.kc_geom_by_median_density(P), allpairs=False)
    certs = m.certs.clone()
    eps = torch.zeros(1, device=dev)
    H = torch.zeros(1, dtype=torch.float64, device=dev)
    rows = []
    for f in fractions:
        mot = wl.Motion("fraction", d, c["eps"], c["seed"] * 1000 + int(f * 1e6), fraction=f, ball=False)
        q, movers = mot.step(p)
        Q, MV = torch.from_numpy(q).to(dev), torch.from_numpy(movers).to(dev)
        nMV = torch.tensor([movers.size], dtype=torch.int32, device=dev)

        def repair():
            kc.kc_max_displacement(P, Q, eps)
            kc.kc_frontier_classify(certs.c, eps, m.flags, m.F, m.nF)
            kc.kc_frontier_repair(m.grid, Q, MV, nMV, certs, movers=MV, n_movers=nMV)

        t_rep = _median_ms(torch, repair, 3, setup=lambda: kc.kc_grid_build(m.grid, P), flush=flush)
        kc.kc_frontier_entropy(m.grid, MV, nMV, out=(H, m.m, m.C))
        t_reb = _median_ms(torch, lambda: kc.kc_cert_grid_rebuild(m.grid, Q, m.other), 3, flush=flush)
        rows.append(dict(f=f, movers=int(movers.size), repair_ms=t_rep, rebuild_ms=t_reb, H=float(H.item())))
        del Q, MV
    fs = [r["f"] for r in rows]
    return dict(rows=rows, crossover_f=crossover_fraction(fs, [r["repair_ms"] for r in rows], [r["rebuild_ms"] for r in rows]))


def run_extras(kc, Maintainer, crossover_fraction, torch, dev, peaks, skip_cfg=None):
    """Other configs, reported beside the headline (not part of `value`): configs 2 / 3 per
    family, config 4 repair-vs-rebuild sweep (crossover per entropy class), the other dimension of
    config 5."""
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    flush = torch.empty(L2_FLUSH_BYTES // 4, dtype=torch.float32, device=dev)
    ex = {"hbm_peak_gbs": hbm, "hbm_peak_source": "measured" if "hbm_gbs" in peaks else "fallback"}
    if skip_cfg not in ("cfg2", "cfg3"):
        ex["cfg2_families"] = family_table(kc, Maintainer, torch, dev, "cfg2", flush)
        ex["cfg3_families"] = family_table(kc, Maintainer, torch, dev, "cfg3", flush)
    # ---------------- config 4: N=262,144, d=3, mover fraction sweep, scattered vs one ball
    c4 = wl.CONFIGS["cfg4"]
    N = c4["N"]
    sweep = {}
    for ball in (False, True):
        rows = []
        for f in wl.CFG4_FRACTIONS:
            p, mot = wl.make_scene("cfg4", "fraction", fraction=f, ball=ball)
            q, movers = mot.step(p)
            P, Q, MV = (torch.from_numpy(x).to(dev) for x in (p, q, movers))
            nMV = torch.tensor([movers.size], dtype=torch.int32, device=dev)
            m = Maintainer(P, allpairs=False)
            certs = m.certs.clone()
            eps = torch.zeros(1, device=dev)
            H = torch.zeros(1, dtype=torch.float64, device=dev)
            mc = torch.zeros(1, dtype=torch.int32, device=dev)
            Cc = torch.zeros(1, dtype=torch.int32, device=dev)

            def reset():
                kc.kc_grid_build(m.grid, P)

            def repair():
                kc.kc_max_displacement(P, Q, eps)
                kc.kc_frontier_classify(certs.c, eps, m.flags, m.F, m.nF)
                kc.kc_frontier_repair(m.grid, Q, MV, nMV, certs, movers=MV, n_movers=nMV)

            def rebuild():
                kc.kc_cert_grid_rebuild(m.grid, Q, m.other)

            def repair_local():        # NEXT #2: the provable frontier of the per-point budget
                kc.kc_max_displacement(P, Q, eps)
                kc.kc_frontier_classify_local(m.grid, P, Q, certs0, eps, m.flags, m.F, m.nF)
                kc.kc_frontier_repair(m.grid, Q, m.F, m.nF, certs, movers=MV, n_movers=nMV)

            certs0 = m.certs.clone()
            t_rep = _median_ms(torch, repair, 7, setup=reset, flush=flush)
            lemma = int(m.nF.item())
            t_loc = _median_ms(torch, repair_local, 7, setup=reset, flush=flush)
            local_frac = int(m.nF.item()) / N
            t_reb = _median_ms(torch, rebuild, 7, flush=flush)
            kc.kc_frontier_entropy(m.grid, MV, nMV, out=(H, mc, Cc))
            rows.append(dict(f=f, movers=int(movers.size), repair_ms=t_rep, rebuild_ms=t_reb, H=float(H.item()),
                             m_cells=int(mc.item()), lemma1_frontier_frac=lemma / N,
                             local_frontier_frac=local_frac, repair_local_ms=t_loc))
            del m
        fs = [r["f"] for r in rows]
        sweep["ball" if ball else "scattered"] = dict(
            rows=rows, crossover_f=crossover_fraction(fs, [r["repair_ms"] for r in rows], [r["rebuild_ms"] for r in rows]),
            crossover_f_local=crossover_fraction(fs, [r["repair_local_ms"] for r in rows], [r["rebuild_ms"] for r in rows]))
    ex["cfg4_sweep"] = sweep
    # ---------------- NEXT #3: multi-step maintenance with the cumulative clock (Appendix A.2):
    # 40 steps with no rebuild in between, against a rebuild every step
    from paper_2606_18314_b200.driver import ClockMaintainer
    clock = {}
    for cfg, fam in (("cfg2", "walk"), ("cfg2", "local"), ("cfg3", "walk"), ("cfg3", "ball5")):
        p, mot = wl.make_scene(cfg, fam)
        Ncl = p.shape[0]
        ps, mv = [p], [None]
        for _ in range(40):
            q, movers = mot.step(ps[-1])
            ps.append(q); mv.append(movers)
        dps = [torch.from_numpy(x).to(dev) for x in ps]
        dmv = [None if m_ is None else torch.from_numpy(m_).to(dev) for m_ in mv]
        cm = ClockMaintainer(dps[0])
        fsum = torch.zeros(1, dtype=torch.int64, device=dev)
        for t in range(1, 6):
            _, nF = cm.step(dps[t], movers=dmv[t])
            fsum += nF                                   # also loads this torch kernel before the timing
        fsum.zero_()
        torch.cuda.synchronize()
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for t in range(6, 41):
            _, nF = cm.step(dps[t], movers=dmv[t])
            fsum += nF
        e1.record(); e1.synchronize()
        t_clock = e0.elapsed_time(e1) / 35
        other = kc.Certs.empty(Ncl, dev)
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for t in range(6, 41):
            kc.kc_cert_grid_rebuild(cm.grid, dps[t], other)
        e1.record(); e1.synchronize()
        clock[f"{cfg}/{fam}"] = dict(steps=35, clock_step_ms=t_clock, rebuild_step_ms=e0.elapsed_time(e1) / 35,
                                     mean_revisited_frac=float(fsum.item()) / 35 / Ncl,
                                     points_per_s=Ncl / (t_clock * 1e-3))
        del cm
    ex["clock_loop"] = clock
    # the same loop at 4,194,304 points (config 5's d = 3 set, random walk) for three step sizes: the
    # expired set through the expiry tree (Theorem 2, kc_frontier_classify_clock_tree) and through the
    # flat test; the step follows the revisited fraction, the tree's classify the number of opened nodes
    if skip_cfg != "clock4m":
        c5 = wl.CONFIGS["cfg5_d3"]
        p0 = wl.make_points("cfg5_d3")
        P0 = torch.from_numpy(p0).to(dev)
        geom5 = kc.kc_geom_by_median_density(P0)
        rows = []
        for eps_w in (2e-8, 2e-7, 2e-6, 2e-4):
            mot = wl.Motion("walk", c5["d"], eps_w, 4242)
            hp = [p0]
            for _ in range(7):
                hp.append(mot.step(hp[-1])[0])
            dp = [torch.from_numpy(x).to(dev) for x in hp]
            row = dict(eps=eps_w, N=c5["N"])
            for tree in (True, False):
                cm = ClockMaintainer(dp[0], tree=tree, geom=geom5)
                fsum = torch.zeros(1, dtype=torch.int64, device=dev)
                for t in (1, 2):
                    cm.step(dp[t])
                torch.cuda.synchronize()
                flush.zero_()
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record()
                for t in range(3, 8):
                    _, nF = cm.step(dp[t])
                    fsum += nF
                e1.record(); e1.synchronize()
                key = "tree" if tree else "flat"
                row[f"clock_step_ms_{key}"] = e0.elapsed_time(e1) / 5
                row["mean_revisited_frac"] = float(fsum.item()) / 5 / c5["N"]
                # the classify alone, on the state the loop has reached (it changes neither c nor the stamps)
                Sx = torch.zeros(1, dtype=torch.float64, device=dev)
                if tree:
                    fn = lambda: kc.kc_frontier_classify_clock_tree(cm.certs.c, cm.stamp, cm.tree, cm.S[0], cm.eps, Sx, cm.F, cm.nF)
                else:
                    fn = lambda: kc.kc_frontier_classify_clock(cm.certs.c, cm.stamp, cm.S[0], cm.eps, Sx, cm.flags, cm.F, cm.nF)
                row[f"classify_ms_{key}"] = _median_ms(torch, fn, 7, flush=flush)
                del cm
            other = kc.Certs.empty(c5["N"], dev)
            g5 = kc.Grid(c5["N"], geom5)
            row["rebuild_step_ms"] = _median_ms(torch, lambda: kc.kc_cert_grid_rebuild(g5, dp[7], other), 5, flush=flush)
            del g5, other, dp
            rows.append(row)
        ex["clock_loop_cfg5_d3"] = rows
    # ---------------- NEXT #4: K-list certificates (K = 4): all-pairs pass and grid search
    topk = {}
    for cfg, n_sub in (("cfg2", None), ("cfg4", 131072)):
        ck_ = wl.CONFIGS[cfg]
        p = wl.make_points(cfg)
        P = torch.from_numpy(p).to(dev)
        Nk, dk_ = p.shape
        K = 4
        lo_hi = kc.kc_geom_for(P)
        gk = kc.Grid(Nk, lo_hi)
        kc.kc_grid_build(gk, P)
        t_grid = _median_ms(torch, lambda: kc.kc_cert_grid_topk(gk, K), 5, flush=flush)
        PA = P if n_sub is None else P[:n_sub].contiguous()
        na = PA.shape[0]
        t_ap = _median_ms(torch, lambda: kc.kc_cert_allpairs_topk(PA, K), 3, flush=flush)
        # the same pass started from the grid's lists (certifying them): no cold lists in the j-chunks
        if n_sub is None:
            sd = kc.kc_cert_grid_topk(gk, K)[0]
        else:
            gs = kc.Grid(na, kc.kc_geom_for(PA))
            kc.kc_grid_build(gs, PA)
            sd = kc.kc_cert_grid_topk(gs, K)[0]
        t_aps = _median_ms(torch, lambda: kc.kc_cert_allpairs_topk(PA, K, seed_ids=sd), 3, flush=flush)
        ops = 5 if dk_ == 2 else 8
        topk[cfg] = dict(K=K, N=Nk, grid_topk_ms=t_grid, grid_topk_points_per_s=Nk / (t_grid * 1e-3),
                         allpairs_topk_N=na, allpairs_topk_ms=t_ap,
                         allpairs_topk_pairs_per_s=na * (na - 1) / (t_ap * 1e-3),
                         allpairs_topk_seeded_ms=t_aps, allpairs_topk_seeded_pairs_per_s=na * (na - 1) / (t_aps * 1e-3),
                         allpairs_topk_tflops=na * (na - 1) * ops / (t_ap * 1e-3) / 1e12)
        del gk
    ex["topk"] = topk
    # ---------------- the sizes of the paper's Table 2 (54 ... 2,095 ms on an RTX PRO 6000,
    # 30 -> 19 G pairs/s; context, another machine): one cold all-pairs pass per N, uniform points
    t2 = {}
    for dd in (2, 3):
        rows = []
        for n2 in (40000, 80000, 120000, 160000, 200000):
            PT = torch.from_numpy(wl.uniform_points(n2, dd, 1000 + n2 // 1000 + dd)).to(dev)
            out2 = kc.Certs.empty(n2, dev)
            ws2 = torch.zeros(max(16, kc.lib().kc_cert_allpairs_workspace(n2, dd)), dtype=torch.uint8, device=dev)
            t_ms = _median_ms(torch, lambda: kc.kc_cert_allpairs(PT, out2, ws2), 3, flush=flush)
            rows.append(dict(N=n2, ms=t_ms, pairs_per_s=n2 * (n2 - 1) / (t_ms * 1e-3),
                             resident_bytes=int(PT.numel() * 4 + out2.buf.numel() * 4 + ws2.numel())))
        t2[f"d{dd}"] = rows
    ex["table2_sizes"] = t2
    # ---------------- config 5: 4,194,304 points, rebuild + Lemma-1 repair; all-pairs at 2^20
    for cfg in ("cfg5_d2", "cfg5_d3"):
        if cfg == skip_cfg:
            continue
        c5 = wl.CONFIGS[cfg]
        N, d = c5["N"], c5["d"]
        p, mot = wl.make_scene(cfg)
        q, _ = mot.step(p)
        P, Q = torch.from_numpy(p).to(dev), torch.from_numpy(q).to(dev)
        m = Maintainer(P, geom=kc.kc_geom_by_median_density(P), allpairs=False)
        t_build = _median_ms(torch, lambda: kc.kc_grid_build(m.grid, Q), 5, flush=flush)
        t_reb = _median_ms(torch, lambda: kc.kc_cert_grid_rebuild(m.grid, Q, m.other), 5, flush=flush)
        info = m.grid.info()
        kc.kc_cert_grid_rebuild(m.grid, P, m.certs)
        eps = kc.kc_max_displacement(P, Q)
        kc.kc_frontier_classify(m.certs.c, eps, m.flags, m.F, m.nF)
        nF = int(m.nF.item())
        certs = m.certs.clone()
        t_rep = _median_ms(torch, lambda: kc.kc_frontier_repair(m.grid, Q, m.F, m.nF, certs), 3,
                           setup=lambda: kc.kc_grid_build(m.grid, P), flush=flush)
        # NEXT #2 at scale: 1 % scattered movers, frontier from the per-point motion budget
        pf, motf = wl.make_scene(cfg, "fraction", fraction=0.01, ball=False)
        qf, mvf = motf.step(pf)
        Qf, MVf = torch.from_numpy(qf).to(dev), torch.from_numpy(mvf).to(dev)
        nMVf = torch.tensor([mvf.size], dtype=torch.int32, device=dev)
        epsf = torch.zeros(1, device=dev)
        kc.kc_cert_grid_rebuild(m.grid, P, m.certs)
        scratch = m.certs.clone()

        def repair_local():
            kc.kc_max_displacement(P, Qf, epsf)
            kc.kc_frontier_classify_local(m.grid, P, Qf, m.certs, epsf, m.flags, m.F, m.nF)
            kc.kc_frontier_repair(m.grid, Qf, m.F, m.nF, scratch, movers=MVf, n_movers=nMVf)

        t_loc = _median_ms(torch, repair_local, 3, setup=lambda: kc.kc_grid_build(m.grid, P), flush=flush)
        local_frac = int(m.nF.item()) / N
        bpp = REBUILD_BYTES_PER_POINT[d]
        n_ap = 1 << 20
        PA = P[:n_ap].contiguous()
        ap = kc.Certs.empty(n_ap, dev)
        ws = torch.zeros(max(16, kc.lib().kc_cert_allpairs_workspace(n_ap, d)), dtype=torch.uint8, device=dev)
        t_ap = _median_ms(torch, lambda: kc.kc_cert_allpairs(PA, ap, ws), 2, flush=flush)
        ops = 5 if d == 2 else 8
        ex[cfg] = dict(N=N, grid_build_ms=t_build, grid_build_frac_of_hbm=N * BUILD_BYTES_PER_POINT[d] / (t_build * 1e-3) / 1e9 / hbm,
                       rebuild_ms=t_reb, rebuild_points_per_s=N / (t_reb * 1e-3),
                       rebuild_alg_bytes_per_point=bpp, rebuild_gbs=N * bpp / (t_reb * 1e-3) / 1e9,
                       rebuild_frac_of_hbm=N * bpp / (t_reb * 1e-3) / 1e9 / hbm,
                       max_cell_occupancy=int(info.max_occ), occupied_cells=int(info.c_occ),
                       lemma1_frontier_frac=nF / N, repair_ms=t_rep, repair_points_per_s=nF / (t_rep * 1e-3),
                       local_budget_1pct_movers=dict(frontier_frac=local_frac, repair_ms=t_loc,
                                                     repair_over_rebuild=t_loc / t_reb),
                       allpairs_N=n_ap, allpairs_ms=t_ap, allpairs_pairs_per_s=n_ap * (n_ap - 1) / (t_ap * 1e-3),
                       allpairs_points_per_s=n_ap / (t_ap * 1e-3),
                       allpairs_tflops=n_ap * (n_ap - 1) * ops / (t_ap * 1e-3) / 1e12)
        del m
    return ex


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", default="cfg5_d3", choices=["cfg5_d3", "cfg5_d2", "cfg2", "cfg3"])
    ap.add_argument("--shard", choices=["none", "queries"], default="none",
                    help="multi-GPU mode of the config 5 workloads: replicas (default) or the all-pairs pass split by query")
    ap.add_argument("--no-extras", action="store_true", help="skip the config 4 / config 5 side measurements")
    ap.add_argument("--no-graph", action="store_true", help="issue the step eagerly instead of replaying CUDA graphs")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    rank = int(os.environ.get("RANK", "0"))
    if args.impl == "reference":
        if rank != 0:
            return
        scale = args.workload.startswith("cfg5")
        r = run_oracle_scale(args.workload, args.steps, args.warmup) if scale else \
            run_oracle_arm(args.workload, args.steps, args.warmup)
        c = wl.CONFIGS[args.workload]
        line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT,
                "n_gpus": args.gpus, "steps": r["steps"], "warmup": args.warmup, "ms_per_step": r["ms_per_step"],
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic",
                "config": {"workload": scale_workload_text(args.workload) if scale else
                           f"{args.workload}: N={c['N']}, d={c['d']}, eps={c['eps']} (CPU oracle arm)"},
                "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                                 "sample": r["sample"]},
                "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line), flush=True)
        return
    out = run_gpu_arm_scale(args) if args.workload.startswith("cfg5") else run_gpu_arm(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
