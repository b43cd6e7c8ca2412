#!/usr/bin/env python
"""bench.py — certified points/s of the whole hot path.

    python bench.py --gpus 1 --steps K --warmup W            # this repo's CUDA path
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands

A "step" is one maintenance transition p -> p' through every row of the hot path (max
displacement, Lemma-1 classify, incremental repair, frontier entropy, O(N) grid rebuild, all-pairs
certification) on BASELINE.json configs[1] (N=16,000, d=2, five motion families, eps=1e-3).
Prints ONE JSON line (rank 0).  Details of every field: DESIGN.md §measurement.
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
# dram__bytes_read.sum + dram__bytes_write.sum of one allpairs_kernel launch, from the committed ncu
# --set full capture of this command (profiles/r1e_allpairs_cfg2_full.txt); null for other workloads
AP_TRAFFIC_BYTES = {("cfg2", 16000): 279552}   # profiles/r1f_allpairs_cfg2_full.txt: dram read + write per launch


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
                        frac=achieved / peak, traffic=AP_TRAFFIC_BYTES.get((cfg, N)),
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
            extras = run_extras(kc, Maintainer, crossover_fraction, torch, dev, peaks)
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


def run_extras(kc, Maintainer, crossover_fraction, torch, dev, peaks):
    """Other configs, reported beside the headline (not part of `value`):
    config 4 repair-vs-rebuild sweep (crossover per entropy class) and config 5 at scale."""
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    flush = torch.empty(L2_FLUSH_BYTES // 4, dtype=torch.float32, device=dev)
    ex = {"hbm_peak_gbs": hbm, "hbm_peak_source": "measured" if "hbm_gbs" in peaks else "fallback"}
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
        c5 = wl.CONFIGS[cfg]
        N, d = c5["N"], c5["d"]
        p, mot = wl.make_scene(cfg)
        q, _ = mot.step(p)
        P, Q = torch.from_numpy(p).to(dev), torch.from_numpy(q).to(dev)
        m = Maintainer(P, allpairs=False)
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
        # algorithmic bytes per point of the rebuild: positions read twice,
        # cell+rank written and read, histogram + scan, sorted records, idx, slot, certificates
        pos = 4 * d
        rec = 8 if d == 2 else 16
        cells_per_pt = m.grid.geom.n_cells / N
        bpp = (pos + 8) + cells_per_pt * (4 + 4 + 4 + 4) + (pos + 8 + 4 + rec + 4 + 4) + (rec + (4 if d == 2 else 0) + 8 + 20)
        n_ap = 1 << 20
        PA = P[:n_ap].contiguous()
        ap = kc.Certs.empty(n_ap, dev)
        ws = torch.zeros(max(16, kc.lib().kc_cert_allpairs_workspace(n_ap, d)), dtype=torch.uint8, device=dev)
        t_ap = _median_ms(torch, lambda: kc.kc_cert_allpairs(PA, ap, ws), 2, flush=flush)
        ops = 5 if d == 2 else 8
        ex[cfg] = dict(N=N, grid_build_ms=t_build, rebuild_ms=t_reb, rebuild_points_per_s=N / (t_reb * 1e-3),
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
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", default="cfg2", choices=["cfg2", "cfg3"])
    ap.add_argument("--no-extras", action="store_true", help="skip the config 4 / config 5 side measurements")
    ap.add_argument("--no-graph", action="store_true", help="issue the step eagerly instead of replaying CUDA graphs")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    rank = int(os.environ.get("RANK", "0"))
    if args.impl == "reference":
        if rank != 0:
            return
        r = run_oracle_arm(args.workload, args.steps, args.warmup)
        c = wl.CONFIGS[args.workload]
        line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT,
                "n_gpus": args.gpus, "steps": r["steps"], "warmup": args.warmup, "ms_per_step": r["ms_per_step"],
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic",
                "config": {"workload": f"{args.workload}: N={c['N']}, d={c['d']}, eps={c['eps']} (CPU oracle arm)"},
                "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                                 "sample": r["sample"]},
                "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line), flush=True)
        return
    out = run_gpu_arm(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
