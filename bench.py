#!/usr/bin/env python
"""bench.py -- one JSON line for the Barnes-Hut hot path (bh_build + bh_potential) on B200.

A "step" is one pass of the whole hot path over one batch of synthetic input: 63-bit Morton keys ->
radix sort -> permute -> octree topology -> monopole moments -> group tree walk -> Phi scattered to
the original order.  Workload at N=1: BASELINE.json configs[3], the 256^3 turbulent medium
(16,777,216 cells, theta = 0.5) -- the configuration the north-star's 40 % FP32 / 60 % HBM bars are
stated on.  `value` = cells/s of build+walk with inputs resident in HBM; the walk's interactions/s
and the roofline of the dominant kernel (the walk) are reported beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

N > 1 (torchrun): the path is scoped to one GPU: every rank
runs an independent replica of the workload ("replicas only", weak scaling, no collective on the data
path); time = max over ranks.
--impl reference: the fp64 CPU oracle (oracle/), as it stands, on the host cores, on a bounded
sample of the same workload per step.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FLOPS_PER_INTERACTION = 13          # north-star convention (BASELINE.json)
FP32_LANES_PER_SM = 128


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d.get("hbm_gbs", 6650.0)), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [t.strip() for t in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def build_bytes_per_cell(n, n_nodes, sort_passes):
    """ALGORITHMIC HBM bytes of bh_build per cell, exactly SURVEY.md §8(d)'s table: a1 keys 36; a2 sort 8 (one
    histogram read) + 24 per executed 8-bit pass; a3 permute 84; a4 topology 8 + 24 n_nodes/n; a5 moments
    32 + 72 n_nodes/n.  What the implementation moves beyond that (its leaf_slot and c(s) arrays) is reported
    separately as IMPL_EXTRA_BYTES_PER_CELL and is not part of the roofline numerator."""
    keys = 36.0
    sort = (8.0 + 24.0 * sort_passes) if sort_passes else 0.0
    permute = 84.0
    topo = 8.0 + (n_nodes / n) * 24.0
    mom = 32.0 + (n_nodes / n) * 72.0
    return keys + sort + permute + topo + mom


IMPL_EXTRA_BYTES_PER_CELL = 9.0     # leaf_slot: 4 B written; c(s): 1 B written + 1 B read; leaf_slot read by the refit: not per build


def make_config(w, world):
    """The `config` object, identical for both arms (--impl ours / reference) so that the driver can match them."""
    return {"workload": w.name, "n_cells": w.n, "theta": w.theta, "group": 32, "mac": "eq3", "G": w.G,
            "l2": "inputs_exceed_l2 (4 x %.0f MB fp64 arrays re-read every step)" % (w.n * 8 / 1e6),
            "parallelism": "replicas x%d" % world}


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.lower().startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_step(w, orc, n_sample_groups, phi_buf, sample=None):
    """One pass of the oracle as it stands (fp64, the criterion evaluated in fp64 as the paper writes it): full
    build, then the group walk on `n_sample_groups` groups taken as 16 evenly spaced contiguous runs; walk time
    is extrapolated linearly to all groups (groups are independent).  Returns (t_build, t_walk_extrapolated,
    interactions_sampled, targets_sampled, groups walked).  `sample` (a dict) receives what the parity key needs:
    the runs, the per-group counters and the sorted permutation; phi_buf holds Phi of the walked targets."""
    import numpy as np
    t0 = time.perf_counter()
    ot = orc.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    t_build = time.perf_counter() - t0
    ng = (w.n + 31) // 32
    ns = min(n_sample_groups, ng)
    runs = 16 if ns >= 64 else 1
    per = max(ns // runs, 1)
    inter = 0
    targets = 0
    t_walk = 0.0
    spans, counts = [], []
    for r in range(runs):
        g0 = min((ng // runs) * r + (ng // runs - per) // 2, ng - per)
        t1 = time.perf_counter()
        _, cnt = ot.potential(w.theta, w.G, group=32, groups=(g0, g0 + per), want_counts=True, out=phi_buf)
        t_walk += time.perf_counter() - t1
        members = np.minimum(32, w.n - 32 * np.arange(g0, g0 + per))
        inter += int(((cnt[:, 0] + cnt[:, 1]) * members).sum())
        targets += int(members.sum())
        spans.append((g0, g0 + per))
        counts.append(cnt)
    walked = runs * per
    if sample is not None:
        sample["runs"], sample["counts"] = spans, counts
        sample["perm"] = ot.sorted_keys_perm()[1].astype(np.int64)
    del ot
    return t_build, t_walk * (ng / walked), inter, targets, walked


def parity_key(w, phi_gpu, cnt_gpu, ev_gpu, phi_orc, sample):
    """The GPU's Phi of the timed configuration against the oracle's on the groups the cpu_baseline leg walked
    (tests/parity.py's primary comparison): groups whose (accepted, leaf, opened) differ from the fp64-decision
    oracle's are flips (fp32-vs-fp64 opening decisions), counted; relative errors over the targets of the
    other groups, and separately over the flipped ones."""
    import numpy as np
    keep, flp = [], []
    flips = ng = 0
    own = True
    for (g0, g1), c64 in zip(sample["runs"], sample["counts"]):
        flipped = np.any(cnt_gpu[g0:g1] != c64, axis=1)
        own = own and bool(np.array_equal(ev_gpu[g0:g1], cnt_gpu[g0:g1, 0] + cnt_gpu[g0:g1, 1]))
        flips += int(flipped.sum())
        ng += g1 - g0
        for g in range(g0, g1):
            tg = sample["perm"][32 * g:min(32 * (g + 1), w.n)]
            ref = phi_orc[tg]
            rel = np.abs(phi_gpu[tg] - ref) / np.abs(ref)
            (flp if flipped[g - g0] else keep).append(rel)
    keep = np.concatenate(keep) if keep else np.zeros(1)
    out = {"groups": ng, "targets": int(keep.size + sum(a.size for a in flp)), "max_rel": float(keep.max()),
           "median_rel": float(np.median(keep)), "flips_fp32_vs_fp64": flips,
           "max_rel_flipped_groups": float(np.concatenate(flp).max()) if flp else None,
           "kernel_entry_counts_equal_counters": own,
           "oracle": "fp64 decisions (Eq. 3 as written); tolerance 1e-4 max / 1e-6 median on non-flipped groups",
           "pass": bool(keep.max() <= 1e-4 and np.median(keep) <= 1e-6 and own)}
    return out


def run_reference(args):
    """--impl reference: the oracle on the host cores; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import numpy as np
    import bh_workloads as wl
    import oracle as orc
    orc.build_library()
    w = wl.by_name(args.workload)
    w.theta = args.theta
    phi_buf = np.full(w.n, np.nan)
    times = []
    inter = tg = walked = 0
    for it in range(args.warmup + args.steps):
        tb, tw, inter, tg, walked = oracle_step(w, orc, args.ref_groups, phi_buf)
        if it >= args.warmup:
            times.append((tb, tw))
    tb = sum(t[0] for t in times) / len(times)
    tw = sum(t[1] for t in times) / len(times)
    value = w.n / (tb + tw)
    ng = (w.n + 31) // 32
    sample = (f"full fp64 build of {w.n} cells + group walk of {walked} of {ng} groups (16 evenly spaced runs), "
              f"walk time scaled by {ng / walked:.1f}; single thread")
    line = {
        "impl": "reference", "metric": "cells_per_s_build_plus_walk", "value": value, "unit": "cells/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": (tb + tw) * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": make_config(w, max(args.gpus, 1)), "timing": "host wall clock, single thread",
        "walk_interactions_per_s": (inter / tg) * w.n / tw,
        "cpu_baseline": {"value": value, "unit": "cells/s", "cores": 1, "kind": "oracle", "sample": sample,
                         "host_cpus": os.cpu_count(), "host_cpu_model": cpu_model()},
        "e2e": {"value": value, "unit": "cells/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_workloads_table(args):
    """--workloads-table: the five BASELINE.json workloads (config 4 = theta sweep on the AMR grid) on one GPU, one
    markdown row each: absolute numbers and achieved fraction of roofline (north_star)."""
    import numpy as np
    import torch
    import bh_workloads as wl
    import paper_1509_07370_b200 as bh
    hbm_gbs, sm_max_mhz, _ = _peaks()
    peak = st_sms(0) * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    rows = [("sphere32", 0.5), ("maclaurin128", 0.5), ("amr_core", 0.5), ("turb256", 0.5),
            ("amr_core", 0.3), ("amr_core", 0.7), ("amr_core", 1.0)]
    import oracle as orc
    orc.build_library()
    print("| workload | cells | theta | build ms | build B/cell | build % HBM | walk ms | interactions/target | interactions/s | walk % FP32 "
          f"| cells/s (build+walk) | oracle cells/s (1 core of {os.cpu_count()}, {cpu_model()}) | Phi max / median rel vs oracle (groups, flips) |")
    print("|---|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---|")
    cache = {}
    for name, theta in rows:
        if name not in cache:
            w = wl.by_name(name)
            cache = {name: (w, [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.x, w.y, w.z, w.m)])}
        w, d = cache[name]
        ctx = bh.Context(0)
        phi = torch.empty(w.n, dtype=torch.float64, device="cuda")
        tb, tw = [], []
        for r in range(args.warmup + args.steps):
            e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            e[0].record(); ctx.build(*d, w.cube); e[1].record(); ctx.potential(theta, w.G, out=phi); e[2].record()
            torch.cuda.synchronize()
            if r >= args.warmup:
                tb.append(e[0].elapsed_time(e[1])); tw.append(e[1].elapsed_time(e[2]))
        st = ctx.get_stats()
        b, t = statistics.median(tb), statistics.median(tw)
        bpc = build_bytes_per_cell(w.n, st.n_nodes, st.sort_passes)
        # the oracle on this box's host (one core), full build + a sample of the groups, and the parity of that sample
        w.theta = theta
        buf = np.full(w.n, np.nan)
        sample = {}
        tbo, two, _, _, walked = oracle_step(w, orc, min(args.ref_groups, 2048), buf, sample)
        par = parity_key(w, phi.cpu().numpy(), ctx.last_group_counts().cpu().numpy(),
                         ctx.last_group_evaluated().cpu().numpy().astype(np.int64), buf, sample)
        print(f"| {name} | {w.n} | {theta} | {b:.3f} | {bpc:.1f} | {100 * bpc * w.n / (b * 1e-3) / 1e9 / hbm_gbs:.1f} | {t:.3f} | "
              f"{st.interactions / w.n:.1f} | {st.interactions / (t * 1e-3):.3e} | "
              f"{100 * st.interactions * FLOPS_PER_INTERACTION / (t * 1e-3) / 1e12 / peak:.1f} | {w.n / ((b + t) * 1e-3):.3e} | "
              f"{w.n / (tbo + two):.3e} | {par['max_rel']:.1e} / {par['median_rel']:.1e} ({par['groups']}, {par['flips_fp32_vs_fp64']}) |")
        ctx.close()
    return 0


def run_ours(args):
    import numpy as np
    import torch
    import bh_workloads as wl
    import paper_1509_07370_b200 as bh
    from paper_1509_07370_b200 import ranks

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libbh has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    hbm_gbs, sm_max_mhz, peak_src = _peaks()
    w = wl.by_name(args.workload)
    w.theta = args.theta
    n = w.n
    dev = f"cuda:{local}"
    host = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (w.x, w.y, w.z, w.m)]
    d = [t.to(dev, non_blocking=False) for t in host]
    phi = torch.empty(n, dtype=torch.float64, device=dev)
    ctx = bh.Context(local)

    def step():
        ctx.build(d[0], d[1], d[2], d[3], w.cube)
        ctx.potential(w.theta, w.G, out=phi)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    st = ctx.get_stats()
    launches_per_step = st.launches_build + st.launches_walk

    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(local)
    sampler.start()
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(args.steps):
        ev[k][0].record()
        ctx.build(d[0], d[1], d[2], d[3], w.cube)
        ev[k][1].record()
        ctx.potential(w.theta, w.G, out=phi)
        ev[k][2].record()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    elapsed = time.perf_counter() - t0
    clocks = sampler.stop()
    dev_total = ev[0][0].elapsed_time(ev[-1][2]) / 1e3          # device time first event -> last event
    t_build = sum(e[0].elapsed_time(e[1]) for e in ev) / args.steps / 1e3
    t_walk = sum(e[1].elapsed_time(e[2]) for e in ev) / args.steps / 1e3
    per_step = sorted(e[0].elapsed_time(e[2]) for e in ev)                  # build + walk of each timed step, ms
    step_median, step_best = per_step[len(per_step) // 2], per_step[0]
    dev_total, elapsed, t_build, t_walk = ranks.max_over_ranks([dev_total, elapsed, t_build, t_walk], dev)
    st = ctx.get_stats()
    phi_timed = phi.cpu().numpy() if rank == 0 else None             # the result of the timed configuration (parity key)
    cnt_timed = ctx.last_group_counts().cpu().numpy() if rank == 0 else None
    ev_timed = ctx.last_group_evaluated().cpu().numpy().astype("int64") if rank == 0 else None

    # ---- measured FP32 denominator: register-resident FMA chains, packed (FFMA2) and scalar (own small library) ----
    from paper_1509_07370_b200 import fma_peak
    fma_packed_tflops, fma_scalar_tflops = fma_peak.measure(local)

    # ---- per-pass table of the build (BH_OPT_PASS_TIMING: one event per kernel; medians over 5 builds) ----
    ctx.set_option(bh.binding.BH_OPT_PASS_TIMING, 1)
    runs_p = []
    for _ in range(5):
        ctx.build(d[0], d[1], d[2], d[3], w.cube)
        runs_p.append(ctx.build_passes())
    st_phases = ctx.get_stats()        # the five phase times exist only under pass timing (events break the launch chain)
    ctx.set_option(bh.binding.BH_OPT_PASS_TIMING, 0)
    passes = []
    for k, (name, _, nbytes) in enumerate(runs_p[0]):
        ms = statistics.median(r[k][1] for r in runs_p)
        passes.append({"pass": name, "ms": round(ms, 5), "alg_bytes": nbytes,
                       "frac": (nbytes / (ms * 1e-3) / 1e9 / hbm_gbs) if (nbytes > 0 and ms > 0) else None})

    # ---- cold and plan-miss builds (the timed steps always hit the sort plan speculated from the previous build) ----
    def timed_build(c, arrs):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t_0 = time.perf_counter()
        a.record()
        c.build(*arrs, w.cube)
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b), (time.perf_counter() - t_0) * 1e3
    other = wl.uniform_sphere(64)                      # a different mesh: other key bits vary, the speculated plan misses
    od = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (other.x, other.y, other.z, other.m)]
    miss = []
    for _ in range(3):
        ctx.build(*od, other.cube)
        miss.append(timed_build(ctx, d))
    ms_build_miss = statistics.median(m_[0] for m_ in miss)
    cold_ctx = bh.Context(local)                       # fresh context: every buffer allocated, no plan to speculate on
    ms_build_cold, ms_build_cold_wall = timed_build(cold_ctx, d)
    ms_build_second = timed_build(cold_ctx, d)[0]
    cold_ctx.close()

    # ---- mass-only refit (bh_update_masses): same cells, new masses; keys / sort / topology reused ----
    ra, rb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ctx.update_masses(d[3])
    torch.cuda.synchronize()
    ra.record()
    for _ in range(args.steps):
        ctx.update_masses(d[3])
    rb.record()
    torch.cuda.synchronize()
    t_refit = ra.elapsed_time(rb) / args.steps / 1e3

    # ---- NEXT-1: Find Essential Nodes for a face-neighbour domain of the same size ----
    ess_box = ((w.cube[0] + w.cube[3], w.cube[1], w.cube[2]),
               (w.cube[0] + 2 * w.cube[3], w.cube[1] + w.cube[3], w.cube[2] + w.cube[3]))
    ctx.set_mac(1)                                  # Eq. 4, the paper's choice for this step
    ess = ctx.essential_nodes(ess_box[0], ess_box[1], w.theta)
    n_ess = int(ess.shape[0])
    torch.cuda.synchronize()
    ra.record()
    for _ in range(args.steps):
        ctx.essential_nodes(ess_box[0], ess_box[1], w.theta, cap=n_ess)
    rb.record()
    torch.cuda.synchronize()
    t_ess = ra.elapsed_time(rb) / args.steps / 1e3
    ctx.set_mac(0)

    # ---- NEXT-4: bh_field, Phi and g = -grad Phi from one walk (3 packed mul + 3 packed fma more per entry pair) ----
    ctx.build(*d, w.cube)
    ctx.field(w.theta, w.G)
    torch.cuda.synchronize()
    ra.record()
    for _ in range(args.steps):
        ctx.field(w.theta, w.G)
    rb.record()
    torch.cuda.synchronize()
    t_field = ra.elapsed_time(rb) / args.steps / 1e3

    # ---- NEXT-3: the same cells in a PERIODIC box (App. A): minimum-image walk + Ewald field lookup per interaction ----
    pctx = bh.Context(local)
    pctx.set_periodic(True)
    pctx.build(*d, w.cube)
    pphi_dev = pctx.potential(w.theta, w.G)                # builds the field array (once per context) and warms up
    torch.cuda.synchronize()
    ra.record()
    pphi_dev = pctx.potential(w.theta, w.G)
    rb.record()
    torch.cuda.synchronize()
    t_periodic = ra.elapsed_time(rb) / 1e3
    pst = pctx.get_stats()
    periodic_info = {"ms_walk": t_periodic * 1e3, "interactions_per_s": world * pst.interactions / t_periodic,
                     "interactions_per_target": pst.interactions / n, "ewald_grid_points_per_axis": 66, "ewald_nested_grids": 1,
                     "slowdown_vs_isolated_walk": t_periodic / t_walk,
                     "note": "every interaction adds a quadratic table lookup (one 32 B record, ~48 instructions) to the 13-flop kernel"}
    del pphi_dev
    pctx.close()

    # ---- optional (--let-domains P): the locally-essential-tree solve of P x-slab domains, one after the other on
    # this GPU (paper_1509_07370_b200/let.py, let_potential_serial): what a P-GPU run computes, without the exchange ----
    let_info = None
    if args.let_domains > 1 and world == 1:
        from paper_1509_07370_b200 import let as let_mod
        order = torch.argsort(d[0], stable=True)
        parts = []
        for c in torch.tensor_split(order, args.let_domains):
            c = torch.sort(c).values
            parts.append(tuple(t[c].contiguous() for t in d))
        let_mod.let_potential_serial(parts, w.cube, w.theta, w.G, mac=1, ctx=ctx)          # warm-up (buffers)
        torch.cuda.synchronize()
        ra.record()
        phis, sent = let_mod.let_potential_serial(parts, w.cube, w.theta, w.G, mac=1, ctx=ctx)
        rb.record()
        torch.cuda.synchronize()
        recv = [sum(sent[dd][e] for dd in range(args.let_domains)) for e in range(args.let_domains)]
        let_info = {"domains": args.let_domains, "split": "equal-count slabs along x", "mac": "eq4", "theta": w.theta,
                    "ms_all_domains_serial": ra.elapsed_time(rb), "cells_per_domain": n // args.let_domains,
                    "entries_received_mean": sum(recv) / len(recv), "entries_received_max": max(recv),
                    "entries_sent_total": sum(map(sum, sent))}
        ctx.set_mac(0)

    # ---- e2e: the public host-buffer call, copies inside the timed region ----
    e2e_steps = max(1, min(args.steps, 5))
    phi_host = torch.empty(n, dtype=torch.float64).pin_memory()
    hx = [t.numpy() for t in host]
    ctx.solve_host(hx[0], hx[1], hx[2], hx[3], w.cube, w.theta, w.G, out=phi_host.numpy())
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.solve_host(hx[0], hx[1], hx[2], hx[3], w.cube, w.theta, w.G, out=phi_host.numpy())
    torch.cuda.synchronize()
    e2e_t = time.perf_counter() - t1
    e2e_t = ranks.max_over_ranks([e2e_t], dev)[0]
    e2e_split = ctx.host_breakdown()
    # the same call with pageable (ordinary numpy) buffers
    px = [np.array(a) for a in (w.x, w.y, w.z, w.m)]
    pphi = np.empty(n)
    ctx.solve_host(*px, w.cube, w.theta, w.G, out=pphi)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    ctx.solve_host(*px, w.cube, w.theta, w.G, out=pphi)
    torch.cuda.synchronize()
    e2e_pageable_t = time.perf_counter() - t1

    # independent problems (a serving loop, not a time-stepping solver: a step there needs Phi before its next
    # positions exist): two contexts on two streams, one host thread each -- the copies of one call run under the
    # kernels of the other.  ctypes releases the GIL for the duration of bh_solve_host.
    import threading
    pair_ctx = [bh.Context(local, stream=torch.cuda.Stream(device=local)) for _ in range(2)]
    pair_out = [torch.empty(n, dtype=torch.float64).pin_memory() for _ in range(2)]

    def _serve(k, steps):
        for _ in range(steps):
            pair_ctx[k].solve_host(hx[0], hx[1], hx[2], hx[3], w.cube, w.theta, w.G, out=pair_out[k].numpy())

    for k in range(2):
        _serve(k, 1)                                           # first build of each context: allocations
    torch.cuda.synchronize()
    workers = [threading.Thread(target=_serve, args=(k, e2e_steps)) for k in range(2)]
    t1 = time.perf_counter()
    for th in workers:
        th.start()
    for th in workers:
        th.join()
    torch.cuda.synchronize()
    e2e_pair_t = time.perf_counter() - t1
    e2e_pair_t = ranks.max_over_ranks([e2e_pair_t], dev)[0]
    e2e_pair_equal = bool(np.array_equal(pair_out[0].numpy(), phi_host.numpy()) and
                          np.array_equal(pair_out[1].numpy(), phi_host.numpy()))
    for c in pair_ctx:
        c.close()
    del pair_out

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return 0

    inter = st.interactions
    fp32_peak_tflops = st_sms(local) * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    walk_tflops = inter * FLOPS_PER_INTERACTION / t_walk / 1e12
    bpc = build_bytes_per_cell(n, st.n_nodes, st.sort_passes)
    line = {
        "metric": "cells_per_s_build_plus_walk", "value": ranks.whole_job_rate(n, args.steps, dev_total, world), "unit": "cells/s",
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": dev_total / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": make_config(w, world), "timing": "cuda events, max over ranks",
        "wall_ms_per_step": elapsed / args.steps * 1e3,
        "walk_interactions_per_s": world * inter / t_walk,
        "interactions_per_target": inter / n,
        "ms_build": t_build * 1e3, "ms_walk": t_walk * 1e3, "ms_update_masses": t_refit * 1e3,
        "ms_step_median": step_median, "ms_step_best": step_best,
        "ms_build_cold": ms_build_cold, "ms_build_cold_wall": ms_build_cold_wall, "ms_build_second": ms_build_second,
        "ms_build_miss": ms_build_miss,
        "build_notes": "ms_build: the timed steps (same mesh every step: the sort plan speculated from the previous build "
                       "hits, one host round trip); ms_build_miss: previous build on another mesh (plan miss: keys, sort and "
                       "count run twice, two round trips); ms_build_cold: first build of a fresh context (allocations inside); "
                       "build_passes: a build under BH_OPT_PASS_TIMING, one event after every kernel -- the events stand "
                       "between the kernels, so that build runs without the overlap of dependent launches and its passes add "
                       "up to more than ms_build",
        "build_passes": passes,
        "field": {"ms_walk": t_field * 1e3, "interactions_per_s": world * st.interactions / t_field,
                  "flops_per_interaction": 22, "frac_fp32": st.interactions * 22 / t_field / 1e12 / (
                      st_sms(local) * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12)},
        "periodic": periodic_info,
        "essential_nodes": {"box": "face-neighbour cube of the same size", "theta": w.theta, "mac": "eq4",
                            "entries": n_ess, "ms": t_ess * 1e3},
        "build_passes_ms": {"keys": st_phases.ms_keys, "sort": st_phases.ms_sort, "count": st_phases.ms_count,
                            "assign_permute": st_phases.ms_assign, "moments": st_phases.ms_moments,
                            "note": "a build under BH_OPT_PASS_TIMING (events between the kernels: no overlap of "
                                    "dependent launches, so the phases add up to more than ms_build)"},
        "tree": {"n_nodes": st.n_nodes, "depth": st.depth, "sort_passes": st.sort_passes,
                 "exact_tests_per_group": st.n_exact_tests / ((n + 31) // 32)},
        "roofline": {"bound": "alu", "kernel": "walk_pair_kernel<false>", "achieved": walk_tflops, "peak": fp32_peak_tflops,
                     "unit": "TFLOP/s", "frac": walk_tflops / fp32_peak_tflops, "traffic": walk_traffic(w.name, w.theta),
                     "launch_ms": t_walk * 1e3, "flops_per_launch": inter * FLOPS_PER_INTERACTION,
                     "peak_measured": {"fma_chain_packed_tflops": fma_packed_tflops, "fma_chain_scalar_tflops": fma_scalar_tflops,
                                       "frac_of_measured": walk_tflops / max(fma_packed_tflops, fma_scalar_tflops),
                                       "frac_at_run_clock": walk_tflops / (fp32_peak_tflops * (clocks.get("sm_mhz") or sm_max_mhz) / sm_max_mhz)},
                     "peak_source": "nominal FP32: %d SMs x 128 lanes x 2 x %.0f MHz (sm_max_mhz, MEASURED_PEAKS.json %s); "
                                    "13 flops/interaction" % (st_sms(local), sm_max_mhz, peak_src),
                     "build_hbm": {"achieved": bpc * n / t_build / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                                   "frac": bpc * n / t_build / 1e9 / hbm_gbs, "bytes_per_cell": bpc,
                                   "bytes_per_cell_source": "SURVEY.md 8(d): 36 + 8 + 24 x %d passes + 84 + (8 + 24 nn/n) + (32 + 72 nn/n)" % st.sort_passes,
                                   "impl_extra_bytes_per_cell": IMPL_EXTRA_BYTES_PER_CELL,
                                   "frac_incl_impl_extra": (bpc + IMPL_EXTRA_BYTES_PER_CELL) * n / t_build / 1e9 / hbm_gbs,
                                   "dram_bytes_measured": build_traffic(w.name),
                                   "frac_of_measured_dram_bytes": (build_traffic(w.name) / t_build / 1e9 / hbm_gbs)
                                   if build_traffic(w.name) else None,
                                   "peak_source": peak_src}},
        "clocks": clocks,
        "e2e": {"value": ranks.whole_job_rate(n, e2e_steps, e2e_t, world), "unit": "cells/s", "h2d_bytes_per_step": 4 * 8 * n,
                "d2h_bytes_per_step": 8 * n, "steps": e2e_steps, "api": "bh_solve_host (pinned host buffers)",
                "ms_per_step": e2e_t / e2e_steps * 1e3, "split_last_call": e2e_split,
                "pageable_buffers": {"value": n / e2e_pageable_t, "ms_per_step": e2e_pageable_t * 1e3,
                                     "note": "ordinary (pageable) numpy arrays: the CUDA runtime stages the copies, no overlap with the kernels"},
                "two_contexts_two_threads": {"value": ranks.whole_job_rate(n, 2 * e2e_steps, e2e_pair_t, world),
                                             "ms_per_step": e2e_pair_t / (2 * e2e_steps) * 1e3, "calls": 2 * e2e_steps,
                                             "phi_equal_to_single_context": e2e_pair_equal,
                                             "note": "independent problems: bh_solve_host from two host threads, each with its own context and stream; one call's copies run under the other's kernels"}},
        "gpu_launches": launches_per_step * args.steps,
    }
    if let_info is not None:
        line["let_serial"] = let_info
    if not args.no_cpu_baseline and world == 1:
        import oracle as orc
        orc.build_library()
        phi_buf = np.full(n, np.nan)
        sample = {}
        tb, tw, oi, otg, walked = oracle_step(w, orc, args.ref_groups, phi_buf, sample)
        ng = (n + 31) // 32
        line["cpu_baseline"] = {
            "value": n / (tb + tw), "unit": "cells/s", "cores": 1, "kind": "oracle",
            "sample": f"full fp64 build ({tb:.1f} s) + group walk of {walked} of {ng} groups "
                      f"(16 evenly spaced runs), walk time scaled by {ng / walked:.1f} to {tw:.1f} s",
            "walk_interactions_per_s": (oi / otg) * n / tw, "host_cpus": os.cpu_count(), "host_cpu_model": cpu_model()}
        # the groups the oracle just walked, against the Phi of the timed steps
        line["parity"] = parity_key(w, phi_timed, cnt_timed, ev_timed, phi_buf, sample)
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()
    return 0


def build_traffic(workload):
    """Sum over the build kernels of dram__bytes_read.sum + dram__bytes_write.sum per build, from the committed ncu
    capture (profiles/build_traffic.csv), if one was taken on this workload; else None."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "build_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload:
                    return float(row["dram_bytes_per_build"])
    except Exception:
        pass
    return None


def walk_traffic(workload, theta):
    """dram__bytes_read.sum + dram__bytes_write.sum of one walk launch from the committed ncu --set full capture
    (profiles/walk_traffic.csv), if one was taken on this workload; else None."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "walk_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and abs(float(row["theta"]) - theta) < 1e-12:
                    return float(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


def st_sms(index):
    import torch
    return torch.cuda.get_device_properties(index).multi_processor_count


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="turb256")
    ap.add_argument("--theta", type=float, default=0.5)
    ap.add_argument("--ref-groups", type=int, default=4096, help="groups the oracle walks per step (sample)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workloads-table", action="store_true",
                    help="print one markdown row per BASELINE workload (build / walk times and roofline fractions) instead of the JSON line")
    ap.add_argument("--let-domains", type=int, default=0,
                    help="also run the locally-essential-tree solve of this many slab domains serially on the GPU")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workloads_table:
        return run_workloads_table(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
