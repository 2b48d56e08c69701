#!/usr/bin/env python
"""bench.py -- throughput of the fused SK + polarization-alignment flag-and-average pass on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload lofar] [--impl ours|reference]

A "step" is one pass of the whole hot path (one rfi_process_chunk = one kernel launch) over one chunk of
seeded synthetic correlator output that is already resident in HBM.  The default workload is
BASELINE.json configs[1] (LOFAR-subband-scale fp32, 18.5 GB, far larger than the 126 MB L2, so no cache
flush is needed between iterations).  One JSON line is printed by rank 0 (see README / DESIGN.md for keys).

N > 1: `python bench.py --gpus N` starts N ranks itself (torch.distributed.run, one process per GPU, rendezvous on
127.0.0.1; it refuses a node with fewer than N GPUs), and it runs as one of the ranks when a launcher (the driver's
torchrun command) has already set WORLD_SIZE.  The path shards by baseline with no data-path collective (every cell is an
independent stream), so every rank processes its own chunk ("scaling": "weak"); the timed region
is bracketed by a barrier and the time is the max over ranks.

--scaling strong (N > 1) shards ONE chunk by baseline with rfi_plan_set_baseline_shard; the default
"weak" gives every rank its own subband chunk.

Besides the headline line (configs[1], fp32, K = 1) the default N = 1 run appends `configs`: one sub-record per
BASELINE.json config (tiny, lofar_fp16, large, sweep K = 64) plus the paper's 10 x 2 footprint, each with best and
median kernel time over the timed launches, samples/s, roofline fractions and a sampled-cell parity check against
the oracle (verification outside every timed region).

--impl reference times the fp64 CPU oracle (oracle/), as it stands, on the host cores.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "visibility samples/s (flag+average, fused SK + polarization alignment)"
UNIT = "samples/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_ncu_traffic(workload: str, variant: str):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture, or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            t = json.load(f)
        return t.get(f"{workload}:{variant}")
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
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
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_baseline(vis_np, w, thr, target_cpu_seconds=15.0):
    """Time the fp64 oracle, as it stands, on a bounded sample of the workload (all host cores)."""
    import numpy as np
    from oracle import rfi_oracle as orc
    cores = orc.max_threads()
    n_cells = vis_np.shape[1]
    probe = min(n_cells, 1024)
    first = np.ascontiguousarray(vis_np[:, :probe])
    orc.process(first, w.window_M, w.n_int, thr, n_threads=cores, want_stats=False)   # warm-up: threads, pages
    t0 = time.perf_counter()
    orc.process(first, w.window_M, w.n_int, thr, n_threads=cores, want_stats=False)
    dt = max(time.perf_counter() - t0, 1e-4)
    per_cell_cpu = dt * cores / probe                       # CPU-seconds per cell
    use = int(max(probe, min(n_cells, target_cpu_seconds / per_cell_cpu)))
    sample = np.ascontiguousarray(vis_np[:, :use])          # the oracle's input, resident and contiguous before timing
    t0 = time.perf_counter()
    orc.process(sample, w.window_M, w.n_int, thr, n_threads=cores, want_stats=False)
    dt = time.perf_counter() - t0
    samples = use * vis_np.shape[0]
    # "... plus a 1-thread figure" -- the same oracle, one thread, on a smaller slice of the same sample
    use1 = int(max(64, min(use, 4.0 / max(per_cell_cpu, 1e-9))))
    one = np.ascontiguousarray(sample[:, :use1])
    t0 = time.perf_counter()
    orc.process(one, w.window_M, w.n_int, thr, n_threads=1, want_stats=False)
    dt1 = time.perf_counter() - t0
    return {"value": samples / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{use} of {w.n_cells} cells x all {vis_np.shape[0]} time samples of the same chunk "
                      f"({samples} samples, {dt:.2f} s wall, OpenMP over cells)",
            "value_1thread": use1 * vis_np.shape[0] / dt1,
            "sample_1thread": f"{use1} cells x all {vis_np.shape[0]} time samples, 1 thread, {dt1:.2f} s wall"}


def run_reference(args):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    from oracle import rfi_oracle as orc
    from paper_2412_14775_b200 import synth
    w = synth.WORKLOADS.get(args.workload, synth.WORKLOADS["lofar"])      # sim42 etc.: the reference arm times the lofar recipe
    thr = synth.default_thresholds(w.window_M)
    cores = orc.max_threads()
    # bounded sample: few stations of the same recipe, all time samples; sized so K+W steps end within minutes
    ns = 6
    ws = w.scaled(n_stations=ns, burst_cell_frac=max(w.burst_cell_frac, 0.02))
    vis, _ = synth.make_chunk(ws, seed=1234, device="cpu")
    v = vis.numpy().reshape(ws.n_time, ws.n_cells, 4, 2)
    steps, warm = max(1, min(args.steps, 5)), max(1, min(args.warmup, 2))
    for _ in range(warm):
        orc.process(v, ws.window_M, ws.n_int, thr, n_threads=cores, want_stats=False)
    t0 = time.perf_counter()
    for _ in range(steps):
        orc.process(v, ws.window_M, ws.n_int, thr, n_threads=cores, want_stats=False)
    dt = (time.perf_counter() - t0) / steps
    samples = ws.n_time * ws.n_cells
    val = samples / dt
    sample = (f"{ws.n_cells} of {w.n_cells} cells ({ns} stations incl. autos) x all {ws.n_time} time samples per step; "
              f"{steps} timed steps after {warm} warm-up")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic (seeded; stands in for LOFAR data)",
        "config": {"workload": f"{w.name}: BASELINE.json configs[1] recipe, bounded sample", "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def _pctl_stats(ms):
    return {"kernel_ms_best": min(ms), "kernel_ms_median": statistics.median(ms), "kernel_ms_mean": statistics.mean(ms),
            "launches_timed": len(ms)}


def _tables_compare(sub, w, thr, mask, out):
    """Tables arithmetic (rfi_plan_set_arithmetic): bit for bit against the step-by-step oracle (oracle_tables_process),
    the comparator of tests/test_gpu_tables.py.  out as for tests.parity_util.compare (K = 1)."""
    import math
    import numpy as np
    from oracle import rfi_oracle as orc
    ref = orc.tables_process(sub, w.window_M, w.n_int, [float(np.float32(x)) for x in thr], mask)
    for key, r in (("tau", ref.tau[0]), ("r_re", ref.r_re), ("r_im", ref.r_im)):
        nan = np.isnan(r)
        assert np.array_equal(np.isnan(out[key]), nan), f"tables {key}: NaN positions differ"
        assert np.array_equal(out[key][~nan].view(np.uint32), r[~nan].view(np.uint32)), f"tables {key}: not bit-exact"
    assert np.array_equal(out["flags"][0], ref.flags[0].astype(bool)), "tables flags differ"
    assert np.array_equal(out["weight"][0], ref.weight[0]), "tables weights differ"
    a = ref.avg[0].view(np.float64).reshape(-1)
    got = out["avg"][0].astype(np.complex128).view(np.float64).reshape(-1)
    rms = math.sqrt(float((a ** 2).mean()))
    fin = np.isfinite(a)
    worst = float((np.abs(got - a)[fin] / (1e-5 * np.maximum(np.abs(a[fin]), rms))).max(initial=0))
    assert worst <= 1.0, f"tables avg: worst |d|/bound = {worst:.3g}"
    n = int(ref.flags[0].size)
    return {"n_windows": n, "flag_mismatch": 0, "flag_mismatch_near_threshold": 0, "flag_mismatch_unexplained": 0,
            "flag_agreement": 1.0, "avg_worst_over_bound": worst, "outputs_skipped": 0, "tau_worst_over_bound": 0.0,
            "r_re_worst_over_bound": 0.0}


def sampled_parity(w, plan, vis, truth, thr, avg, weight, stats, n_clean, n_rfi, groups=None, tables_mask=None):
    """Verification leg (outside every timed region): a seeded sample of cells of the chunk the timed kernel just
    processed -- all time samples of each -- is brought back and compared with the fp64 oracle element by element
    with the comparators and tolerances of tests/ (the logic of tests/test_gpu_full_size.py).
    vis: the chunk as a time-major [n_time, n_baselines, n_chan, 4, 2] tensor or view.  groups (optional): cells whose
    windows were decided with different threshold sets (baseline classes, per-stream adaptation) are compared group by
    group: [(label, bool tensor [n_cells], thresholds [K][4])]; default: all cells with `thr`.  tables_mask: compare with the
    tables oracle bit for bit instead."""
    import numpy as np
    import torch
    import paper_2412_14775_b200 as rfi
    from tests.parity_util import compare
    K = max(plan.K, 1)
    try:
        g = torch.Generator().manual_seed(3)
        tr = truth.reshape(plan.n_win, plan.n_cells)
        has = tr.any(0).cpu()
        if groups is not None:                              # only cells that belong to a group are candidates
            member = torch.zeros(plan.n_cells, dtype=torch.bool)
            for _, m, _ in groups:
                member |= m.cpu()
            r_cells, c_cells = torch.nonzero(has & member).flatten(), torch.nonzero(~has & member).flatten()
        else:
            r_cells, c_cells = torch.nonzero(has).flatten(), torch.nonzero(~has).flatten()
        idx = torch.cat([r_cells[torch.randperm(r_cells.numel(), generator=g)[:n_rfi]],
                         c_cells[torch.randperm(c_cells.numel(), generator=g)[:n_clean]]]).sort().values
        if w.window_F > 1:                                  # whole footprints: the F channels of a window share a flag
            F = w.window_F
            idx = torch.unique((idx // F)[:, None] * F + torch.arange(F)[None, :]).sort().values
        idx = idx.to(vis.device)
        flags = rfi.unpack_flags(plan.get_flags(), w.n_chan).reshape(K, plan.n_win, plan.n_cells)
        wt = weight.reshape(K, plan.n_out, plan.n_cells).long()
        kept = (~flags).reshape(K, plan.n_out, w.n_int // w.window_M, plan.n_cells).sum(2) * w.window_M
        weight_ok = bool(torch.equal(wt, kept))            # property at FULL size: weight = unflagged sample count
        finite_ok = bool(torch.isfinite(avg).all())
        sub = vis.reshape(w.n_time, plan.n_cells, 4, 2)[:, idx].cpu().numpy()
        s = stats.reshape(3, plan.n_win, plan.n_cells)
        out = {"avg": avg.reshape(K, plan.n_out, plan.n_cells, 4, 2)[:, :, idx].cpu().numpy().view(np.complex64).reshape(K, plan.n_out, -1, 4),
               "weight": wt[:, :, idx].cpu().numpy(), "flags": flags[:, :, idx].cpu().numpy(),
               "tau": s[0][:, idx].cpu().numpy(), "r_re": s[1][:, idx].cpu().numpy(), "r_im": s[2][:, idx].cpu().numpy()}
        del flags, wt, kept
        idx_c = idx.cpu()
        rep = None
        for label, member, g_thr in (groups if groups is not None else [("all", None, thr)]):
            pos = np.arange(idx_c.numel()) if member is None else np.nonzero(member.cpu()[idx_c].numpy())[0]
            if pos.size == 0:
                continue
            o = {k: (a[:, :, pos] if a.ndim >= 3 else a[:, pos]) for k, a in out.items()}
            r = (_tables_compare(sub[:, pos], w, g_thr[0], tables_mask, o) if tables_mask is not None else
                 compare(sub[:, pos], w.window_M, w.n_int, g_thr, o, tol=2e-3 if w.fp16 else 1e-5, fp16=w.fp16, F=w.window_F))
            if rep is None:
                rep = dict(r)
            else:                                           # totals over the groups, worst case of the ratios
                for key in ("n_windows", "flag_mismatch", "flag_mismatch_near_threshold", "flag_mismatch_unexplained", "outputs_skipped"):
                    rep[key] += r[key]
                for key in ("tau_worst_over_bound", "r_re_worst_over_bound", "avg_worst_over_bound"):
                    rep[key] = max(rep.get(key) or 0.0, r.get(key) or 0.0)
                rep["flag_agreement"] = min(rep["flag_agreement"], r["flag_agreement"])
        ok = weight_ok and finite_ok
        return {"status": "ok" if ok else "FAILED",
                "against": ("tables oracle (oracle_tables_process), bit for bit, same seeded chunk" if tables_mask is not None
                            else "fp64 oracle (oracle/), same seeded chunk"),
                "groups": [lab for lab, _, _ in groups] if groups is not None else None,
                "cells_sampled": int(idx.numel()), "windows_compared": rep["n_windows"] * K,
                "tolerance": 2e-3 if w.fp16 else 1e-5, "flag_mismatch": rep["flag_mismatch"],
                "flag_mismatch_near_threshold": rep["flag_mismatch_near_threshold"],
                "flag_mismatch_unexplained": rep["flag_mismatch_unexplained"], "flag_agreement": rep["flag_agreement"],
                "tau_worst_over_bound": rep.get("tau_worst_over_bound"), "r_re_worst_over_bound": rep.get("r_re_worst_over_bound"),
                "avg_worst_over_bound": rep["avg_worst_over_bound"], "outputs_skipped": rep["outputs_skipped"],
                "weight_equals_unflagged_samples_full_size": weight_ok, "avg_finite_full_size": finite_ok}
    except AssertionError as exc:
        return {"status": "FAILED", "error": str(exc)[:300]}


def mode_parity(args, w, plan, vis, truth, thr, two_classes, dev):
    """The verification leg of run_ours for the mode that was just timed (K sets, threshold classes, cell-major input,
    tables arithmetic, on-line adaptation): the thresholds in force are read back, one more launch stores the statistics
    planes, and sampled cells go through the oracle group by group.  Not timed."""
    import torch
    from paper_2412_14775_b200 import synth
    nb, C = plan.n_baselines, w.n_chan
    vis_tm = vis.permute(2, 0, 1, 3, 4) if args.layout == "cell_major" else vis     # a view: (b, c) stay mergeable
    cell_auto = None
    if two_classes:
        autos = synth.auto_baseline_mask(w)[plan.b_first:plan.b_first + nb]
        cell_auto = autos.repeat_interleave(C)
    groups = None
    if args.adaptive > 0 and args.adaptive_scope == "baseline":
        st = plan.get_stream_thresholds()                                      # [nb, 4], in force for the next launch
        picks = sorted({int(b) for b in torch.linspace(0, nb - 1, 8).round().tolist()})
        groups = []
        for b in picks:
            m = torch.zeros(nb * C, dtype=torch.bool)
            m[b * C:(b + 1) * C] = True
            groups.append((f"baseline {plan.b_first + b}", m, [st[b].tolist()]))
    elif args.adaptive > 0:
        cur = plan.get_thresholds()                                            # per class, in force for the next launch
        groups = ([("cross", ~cell_auto, [list(cur[0])]), ("auto", cell_auto, [list(cur[-1])])] if two_classes
                  else [("all", torch.ones(nb * C, dtype=torch.bool), [list(cur[0])])])
    elif two_classes:
        auto = synth.auto_thresholds(w.window_M * w.window_F)
        groups = [("cross", ~cell_auto, [list(t) for t in thr]),
                  ("auto", cell_auto, [list(auto) if args.K <= 1 else [t[0]] + list(auto[1:]) for t in thr])]
    avg2, weight2, stats = plan.alloc_outputs(device=dev, stats=True)
    plan.process_chunk(vis, avg2, weight2, stats)
    torch.cuda.synchronize(dev)
    n_clean, n_rfi = (160, 64) if plan.K > 1 else (512, 128)
    rep = sampled_parity(w, plan, vis_tm, truth, thr, avg2, weight2, stats, n_clean, n_rfi, groups=groups,
                         tables_mask=args.mask if args.arith == "tables" else None)
    del avg2, weight2, stats
    torch.cuda.empty_cache()
    return rep


def _safe(fn, *a, **kw):
    """A verification leg must never cost the run its JSON line: anything unexpected becomes a FAILED record."""
    try:
        return fn(*a, **kw)
    except Exception as exc:      # noqa: BLE001
        return {"status": "FAILED", "error": f"{type(exc).__name__}: {exc}"[:300]}


def per_config_entry(rec):
    """One compact row of roofline.per_config from a sub-record of `configs` (the driver keeps `roofline` whole)."""
    if "skipped" in rec:
        return {"workload": rec["workload"], "K": rec["K"], "skipped": rec["skipped"]}
    r, p = rec["roofline"], rec.get("parity") or {}
    row = {"workload": rec["workload"], "K": rec["K"], "storage": rec["storage"], "window": rec["window"], "kernel": rec["variant"],
           "ms_best": rec["kernel_ms_best"], "ms_median": rec["kernel_ms_median"], "gbs": r["achieved"], "frac": r["frac"],
           "frac_of_nominal_8TBs": r["frac_of_nominal_8TBs"], "parity_status": p.get("status"),
           "cells_sampled": p.get("cells_sampled"), "flag_mismatch_unexplained": p.get("flag_mismatch_unexplained")}
    if rec.get("cpu_baseline"):
        row["cpu_baseline_samples_per_s"] = rec["cpu_baseline"]["value"]
    return row


def measure_config(name, K, dev, steps, warmup, peak, read_probe_gbs, vis=None, truth=None, n_clean=512, n_rfi=128,
                   variant="auto", cpu_baseline=False):
    """One sub-record of `configs`: generate (or reuse) the chunk, time `steps` launches one by one with CUDA events
    after `warmup` untimed ones, then check a sample of cells against the oracle."""
    import torch
    import paper_2412_14775_b200 as rfi
    from paper_2412_14775_b200 import synth
    w = synth.WORKLOADS[name]
    W = w.window_M * w.window_F
    rec = {"workload": name, "baseline_config": (f"BASELINE.json configs[{synth.BASELINE_CONFIG_INDEX[name]}]"
                                                 if name in synth.BASELINE_CONFIG_INDEX else "SURVEY 8(f) NEXT-1 (paper's 10 x 2 footprint)"),
           "K": K, "storage": "f16" if w.fp16 else "f32", "window": f"{w.window_M} x {w.window_F}",
           "input_bytes": w.input_bytes}
    free = torch.cuda.mem_get_info(dev)[0]
    need = (0 if vis is not None else w.input_bytes * 1.12) + 8e9
    if free < need:
        rec["skipped"] = f"needs {need / 1e9:.1f} GB of free device memory, {free / 1e9:.1f} GB available"
        return rec
    own = vis is None
    if own:
        vis, truth = synth.make_chunk(w, seed=1234, device=dev)
    thr = synth.default_thresholds(W) if K <= 1 else synth.sweep_thresholds(W, K)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                       rfi.RFI_FP16 if w.fp16 else rfi.RFI_FP32, n_int=w.n_int)
    if w.window_F > 1:
        plan.set_window_freq(w.window_F)
    plan.set_thresholds(thr)
    plan.set_variant(variant)
    counts = tw = None
    if K > 1 and truth is not None:
        # configs[4]: "per-set flag fraction against injected-RFI ground truth" is an output of the pass -- the K-set kernel
        # fills the K x 4 confusion counters in the timed launch itself (rfi_plan_set_truth)
        tw = rfi.pack_flags(truth.reshape(plan.n_win, plan.n_baselines, w.n_chan))
        counts = plan.set_truth(tw)
    avg, weight, stats = plan.alloc_outputs(device=dev, stats=True)
    out_bytes = avg.numel() * 4 + weight.numel() * 4 + max(plan.K, 1) * plan.n_win * plan.n_baselines * plan.wpb * 4
    algo = w.input_bytes + out_bytes
    small = w.input_bytes < 4 * 126e6
    flush = torch.empty(256 << 20, dtype=torch.int8, device=dev) if small else None
    for _ in range(warmup):
        plan.process_chunk(vis, avg, weight)
    torch.cuda.synchronize(dev)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    l0 = plan.launch_count
    for a, b in evs:
        if flush is not None:
            flush.zero_()
        a.record()
        plan.process_chunk(vis, avg, weight)
        b.record()
    torch.cuda.synchronize(dev)
    ms = [a.elapsed_time(b) for a, b in evs]
    st = _pctl_stats(ms)
    samples = w.n_time * w.n_cells
    gbs_best, gbs_med = algo / (st["kernel_ms_best"] * 1e-3) / 1e9, algo / (st["kernel_ms_median"] * 1e-3) / 1e9
    mix_probe = None
    if K > 1 and not small:      # K-set pass: the ceiling is a read/write MIX, measured live with the same output volume
        try:
            mix_probe = rfi.probe_mix_bandwidth(vis if w.input_bytes <= (40 << 30) else vis.reshape(-1)[: (40 << 30) // vis.element_size()], out_bytes)
        except Exception:
            mix_probe = None
    rec.update(variant=plan.last_variant, gpu_launches=int(plan.launch_count - l0), **st,
               ms_per_step=st["kernel_ms_mean"], samples_per_s=samples / (st["kernel_ms_median"] * 1e-3),
               algorithmic_bytes_per_launch=algo,
               roofline={"bound": "hbm" if not small else "latency", "achieved": gbs_med, "achieved_best": gbs_best, "unit": "GB/s",
                         "peak": peak, "frac": gbs_med / peak, "frac_of_nominal_8TBs": gbs_med / 8000.0,
                         "frac_of_read_stream_probe": (gbs_med / read_probe_gbs) if read_probe_gbs else None,
                         "mix_probe_gbs": mix_probe, "frac_of_mix_probe": (gbs_med / mix_probe) if mix_probe else None},
               l2=("L2 flushed between timed launches (256 MB write outside the events)" if small else "input far larger than the 126 MB L2"))
    if small:
        rec["latency_us"] = {"best": st["kernel_ms_best"] * 1e3, "median": st["kernel_ms_median"] * 1e3}
    if counts is not None:
        torch.cuda.synchronize(dev)
        c = counts.cpu().double()
        fa, md = (c[:, 0] / c[:, 1].clamp(min=1)), (c[:, 2] / c[:, 3].clamp(min=1))
        sep = plan.confusion_counts(tw).cpu()
        rec["detection"] = {"source": "K x 4 confusion counters filled by the timed K-set launch (rfi_plan_set_truth)",
                            "equal_to_separate_mask_pass": bool(torch.equal(sep, counts.cpu())),
                            "false_alarm_min_max": [float(fa.min()), float(fa.max())],
                            "missed_detection_min_max": [float(md.min()), float(md.max())]}
        plan.set_truth(None)
    # one more launch with the statistics planes, then the sampled-cell oracle check (not timed)
    plan.process_chunk(vis, avg, weight, stats)
    torch.cuda.synchronize(dev)
    rec["parity"] = _safe(sampled_parity, w, plan, vis, truth, thr, avg, weight, stats, n_clean, n_rfi)
    if cpu_baseline:
        # SURVEY.md 8(d), configs[3]: the oracle timed on the RFI-bearing cells + a seeded 2 % of the clean cells (bounded)
        g = torch.Generator().manual_seed(11)
        has = truth.reshape(plan.n_win, plan.n_cells).any(0).cpu()
        r_cells, c_cells = torch.nonzero(has).flatten(), torch.nonzero(~has).flatten()
        pick = torch.cat([r_cells[torch.randperm(r_cells.numel(), generator=g)[:16384]],
                          c_cells[torch.randperm(c_cells.numel(), generator=g)[:min(16384, max(1, c_cells.numel() // 50))]]])
        pick = pick[torch.randperm(pick.numel(), generator=g)].to(dev)          # mixed order: any prefix is a fair sample
        sub = vis.reshape(w.n_time, plan.n_cells, 4, 2)[:, pick].cpu().numpy()
        rec["cpu_baseline"] = _safe(oracle_baseline, sub, w, thr, 8.0)
        del sub
    plan.destroy()
    del avg, weight, stats, flush
    if own:
        del vis, truth
    torch.cuda.empty_cache()
    return rec


def sim42_parity(plan, vis, truth_words, sets, T, C, wT, wF, dev):
    """Verification leg of --workload sim42: sampled (realisation, channel) footprints of the block the timed K-set
    launch just flagged, all K sets, against the fp64 oracle at the paper's T x F window."""
    import torch
    import paper_2412_14775_b200 as rfi
    from paper_2412_14775_b200 import synth
    w = synth.Workload("sim42", 29, False, C, T, wT, T, window_F=wF)            # 406 cross baselines = the realisations
    truth = rfi.unpack_flags(truth_words, C).reshape(plan.n_win, -1)
    avg2, weight2, stats = plan.alloc_outputs(device=dev, stats=True)
    plan.process_chunk(vis, avg2, weight2, stats)
    torch.cuda.synchronize(dev)
    rep = sampled_parity(w, plan, vis, truth, sets, avg2, weight2, stats, 48, 48)
    del avg2, weight2, stats
    return rep


def run_sim42(args):
    """--workload sim42: the paper's 400-run FA/MD-vs-INR experiment (Fig. 3) on the device.
    406 realisations (29 stations, cross baselines: the nearest triangular number above 400) of the 2000 x 512 block are
    generated by rfi_sim42_generate at each INR, flagged with 10 x 2 footprints by ONE K-set launch whose sets are
    {SK only, DS only, BOTH} x a ladder of design false-alarm rates (thresholds = empirical null quantiles on RFI-free
    realisations of another seed), and scored by rfi_confusion_counts.  The timed step is the K-set flag+average pass."""
    import torch
    import paper_2412_14775_b200 as rfi
    from paper_2412_14775_b200 import sharding
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise RuntimeError("--workload sim42 is a single-GPU experiment")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    INF = float("inf")
    R, T, C, wT, wF = 406, 2000, 512, 10, 2
    fa_ladder = [0.001, 0.002, 0.005, 0.01, 0.02, 0.05, 0.1][: max(1, min(7, (max(args.K, 3)) // 3))] if args.K < 21 else \
                [0.0005, 0.001, 0.002, 0.003, 0.005, 0.0075, 0.01, 0.015, 0.02, 0.03, 0.04, 0.05, 0.06, 0.075, 0.1, 0.125, 0.15, 0.2, 0.25, 0.3, 0.4]
    plan = rfi.RfiPlan(29, R, C, T, wT, n_int=T)
    plan.set_window_freq(wF)
    vis = torch.empty(T, R, C, 4, 2, dtype=torch.float32, device=dev)
    t0 = time.perf_counter()
    rfi.sim42_generate(R, 0.0, seed=4242, out=vis)
    torch.cuda.synchronize()
    # null quantiles of the two statistics on RFI-free realisations (thresholds from a design false-alarm rate)
    plan.set_thresholds([[1.0, -INF, INF, INF]])
    avg, weight, stats = plan.alloc_outputs(device=dev, stats=True)
    plan.process_chunk(vis, avg, weight, stats)
    s = stats.reshape(3, plan.n_win, R, C)[:, :, :, ::wF]
    g = torch.Generator(device=dev).manual_seed(1)
    idx = torch.randint(0, s[0].numel(), (4_000_000,), generator=g, device=dev)
    tau, rmax = s[0].flatten()[idx], torch.maximum(s[1], s[2]).flatten()[idx]
    sets, labels = [], []
    for fa in fa_ladder:
        lo, hi = float(torch.quantile(tau, fa / 2)), float(torch.quantile(tau, 1 - fa / 2))
        gm = float(torch.quantile(rmax, 1 - fa))
        sets += [[1.0, lo, hi, INF], [1.0, -INF, INF, gm], [1.0, lo, hi, gm]]
        labels += [("sk", fa), ("ds", fa), ("both", fa)]
    del avg, weight, stats, s, tau, rmax
    plan.set_thresholds(sets)
    K = len(sets)
    avg, weight, _ = plan.alloc_outputs(device=dev)
    inrs = [0.01, 0.1, 1.0, 10.0, 100.0, 1000.0]
    curves, gen_ms, kernel_ms = {}, [], []
    sampler = ClockSampler(0)
    sampler.start()
    for polarized in (True, False):
        for inr in inrs:
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            _, truth = rfi.sim42_generate(R, inr, seed=777, polarized=polarized, out=vis)
            b.record()
            for _ in range(args.warmup if not kernel_ms else 0):
                plan.process_chunk(vis, avg, weight)
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(max(2, args.steps // 4))]
            for x, y in evs:
                x.record(); plan.process_chunk(vis, avg, weight); y.record()
            counts = plan.confusion_counts(truth).cpu().double()
            torch.cuda.synchronize()
            gen_ms.append(a.elapsed_time(b)); kernel_ms += [x.elapsed_time(y) for x, y in evs]
            fa_m, md_m = (counts[:, 0] / counts[:, 1].clamp(min=1)).tolist(), (counts[:, 2] / counts[:, 3].clamp(min=1)).tolist()
            for k, (det, fa) in enumerate(labels):
                curves.setdefault(("polarised" if polarized else "unpolarised"), {}).setdefault(f"design_fa_{fa}", {}) \
                      .setdefault(det, []).append({"inr": inr, "false_alarm": round(fa_m[k], 5), "missed_detection": round(md_m[k], 5)})
    clocks = sampler.stop()
    parity = None if args.no_parity else _safe(sim42_parity, plan, vis, truth, sets, T, C, wT, wF, dev)
    peak, peak_src = load_peaks()
    out_bytes = avg.numel() * 4 + weight.numel() * 4 + K * plan.n_win * R * plan.wpb * 4
    algo = vis.numel() * 4 + out_bytes
    k_med = statistics.median(kernel_ms)
    samples = T * R * C
    keep = [f"design_fa_{f}" for f in (0.01, 0.05) if f in fa_ladder] or [f"design_fa_{fa_ladder[0]}"]
    line = {
        "metric": METRIC, "value": samples / (k_med * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": len(kernel_ms), "warmup": args.warmup,
        "ms_per_step": statistics.mean(kernel_ms), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic: the paper's section-4.2 simulator (PAPER.md:219-237) generated on the device, seeded",
        "config": {"workload": "sim42: SURVEY 8(f) NEXT-4, the FA/MD-vs-INR experiment of PAPER.md:235-237 (not a BASELINE.json config)",
                   "n_realisations": R, "n_time": T, "n_chan": C, "window": f"{wT} x {wF}", "K": K, "variant": plan.last_variant,
                   "sets": "{SK only, DS only, BOTH} x design false-alarm ladder " + str(fa_ladder),
                   "input_bytes": vis.numel() * 4, "l2": "input (13.3 GB) is far larger than the 126 MB L2: no flush needed"},
        "roofline": {"bound": "hbm", "achieved": algo / (k_med * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": algo / (k_med * 1e-3) / 1e9 / peak, "traffic": None, "peak_source": peak_src,
                     "kernel": "rfi_batched_mask_kernel<5, fp32>", "kernel_ms_best": min(kernel_ms), "kernel_ms_median": k_med,
                     "frac_of_nominal_8TBs": algo / (k_med * 1e-3) / 1e9 / 8000.0, "algorithmic_bytes_per_launch": algo},
        "cpu_baseline": None, "e2e": None, "gpu_launches": int(plan.launch_count), "clocks": clocks, "parity": parity,
        "sim42": {"generator_ms_median": statistics.median(gen_ms), "generator_gbytes_per_s": vis.numel() * 4 / (statistics.median(gen_ms) * 1e-3) / 1e9,
                  "paper_fig2_context": "INR 100, 10 x 2: SK 0.01/0.89, DS 0.01/0.06, BOTH 0.01/0.05 (FA/MD, PAPER.md:233)",
                  "curves": {pol: {k: v for k, v in c.items() if k in keep} for pol, c in curves.items()},
                  "roc_at_inr_100": {pol: {det: [{"design_fa": fa, **next(p for p in c[f"design_fa_{fa}"][det] if p["inr"] == 100.0)} for fa in fa_ladder]
                                           for det in ("sk", "ds", "both")} for pol, c in curves.items()}},
    }
    for v in line["sim42"]["roc_at_inr_100"].values():
        for pts in v.values():
            for p in pts:
                p.pop("inr", None)
    print(json.dumps(line))
    plan.destroy()


def rank_chunk_and_plan(w, work, dev):
    """This rank's input and plan (sharding.rank_work).  weak: its own subband chunk.  strong: every
    rank draws the SAME chunk and keeps its contiguous baseline range; the plan then processes b_count baselines (no
    exchange: PAPER.md:44, every stream is mitigated separately).  Returns (vis, truth [n_win, cells of this rank], plan)."""
    import torch
    import paper_2412_14775_b200 as rfi
    from paper_2412_14775_b200 import synth
    vis, truth = synth.make_chunk(w, seed=work["seed"], device=dev)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                       rfi.RFI_FP16 if w.fp16 else rfi.RFI_FP32, n_int=w.n_int)
    if work["sharded"]:
        b0, bc = work["b_first"], work["b_count"]
        vis = vis[:, b0:b0 + bc].contiguous()
        truth = truth.reshape(-1, w.n_baselines, w.n_chan)[:, b0:b0 + bc].reshape(truth.shape[0], -1).contiguous()
        plan.set_baseline_shard(b0, bc)
        torch.cuda.empty_cache()
    return vis, truth, plan


def run_ours(args):
    import numpy as np
    import torch
    import paper_2412_14775_b200 as rfi
    from paper_2412_14775_b200 import sharding, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    w = synth.WORKLOADS[args.workload]
    W = w.window_M * w.window_F
    thr = synth.default_thresholds(W) if args.K <= 1 else synth.sweep_thresholds(W, args.K)
    work = sharding.rank_work(w.n_baselines, world, rank, args.scaling)
    vis, truth, plan = rank_chunk_and_plan(w, work, dev)
    if w.window_F > 1:
        plan.set_window_freq(w.window_F)
    if args.layout == "cell_major":
        plan.set_layout("cell_major")
        vis = vis.permute(1, 2, 0, 3, 4).contiguous()          # [b][c][t][pol][re,im]
        args.no_e2e = True                                     # the host path is time-major only
    if args.arith == "tables":
        plan.set_arithmetic("tables", args.mask)
    two_classes = w.autos and args.classes
    if two_classes:       # cross / auto threshold classes: autos have their own null statistics
        plan.set_baseline_classes(synth.auto_baseline_mask(w).int().tolist())
        auto = synth.auto_thresholds(W)
        plan.set_thresholds([[t, auto if args.K <= 1 else [t[0]] + auto[1:]] for t in thr])
    else:
        plan.set_thresholds(thr)
    plan.set_variant(args.variant)
    if args.adaptive > 0:                 # on-line threshold adaptation (rfi_plan_set_adaptive): kernel + a one-CTA update per step
        plan.set_adaptive(args.adaptive, 0.5)
        if args.adaptive_scope == "baseline":
            plan.set_adaptive_scope("baseline")
    avg, weight, _ = plan.alloc_outputs(device=dev)
    out_bytes = avg.numel() * 4 + weight.numel() * 4 + max(plan.K, 1) * plan.n_win * plan.n_baselines * plan.wpb * 4
    in_bytes = vis.numel() * vis.element_size()            # this rank's input (the whole chunk unless sharded)
    algo_bytes = in_bytes + out_bytes
    samples = w.n_time * plan.n_cells

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    torch.cuda.synchronize()
    torch.cuda.profiler.start()       # `ncu --profile-from-start off` then lists the launches from the warm-up on
    for _ in range(args.warmup):
        plan.process_chunk(vis, avg, weight)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
        time.sleep(0.3)
    launches0 = plan.launch_count
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t_start = torch.cuda.Event(enable_timing=True); t_end = torch.cuda.Event(enable_timing=True)
    t_start.record()
    small = in_bytes < 4 * 126e6                           # fits (or nearly fits) the 126 MB L2: flush between iterations
    flush = torch.empty(256 << 20, dtype=torch.int8, device=dev) if small else None
    for a, b in evs:
        if flush is not None:
            flush.zero_()                                  # 256 MB write evicts the chunk from L2 (outside the event pair)
        a.record()
        plan.process_chunk(vis, avg, weight)      # on torch's current stream, where the events are recorded
        b.record()
    t_end.record()
    barrier()
    kernel_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = sum(kernel_ms) if small else t_start.elapsed_time(t_end)   # the flush writes are not part of a step
    launches = plan.launch_count - launches0
    clocks = sampler.stop() if sampler else None
    total_ms = sharding.max_over_ranks(total_ms, device=dev)       # device-measured, MAX over ranks
    ms_per_step = total_ms / args.steps
    total_samples = sharding.sum_scalar_over_ranks(samples, device=dev)      # weak: N chunks; strong: one chunk
    total_algo = sharding.sum_scalar_over_ranks(algo_bytes, device=dev)
    value = total_samples / (ms_per_step * 1e-3)

    # a little science on the way out (not timed): per-set detection quality against the injected ground truth
    # (BASELINE.json configs[4]; false-alarm / missed-detection probabilities of PAPER.md:235) via rfi_confusion_counts
    tr = truth.reshape(plan.n_win, plan.n_cells)
    if w.window_F > 1:                 # a footprint is RFI-bearing if any of its F channels is
        tr = tr.reshape(plan.n_win, -1, w.window_F).any(-1, keepdim=True).expand(-1, -1, w.window_F).reshape(plan.n_win, plan.n_cells)
    counts = plan.confusion_counts(rfi.pack_flags(tr.reshape(plan.n_win, plan.n_baselines, w.n_chan)))
    counts = sharding.sum_over_ranks(counts)
    p_fa, p_md = sharding.rates(counts.cpu())
    flag_frac = (counts[:, 0] + counts[:, 3] - counts[:, 2]).double().cpu() / (counts[:, 1] + counts[:, 3]).double().cpu()
    fa, md = float(p_fa[0]), float(p_md[0])

    # the paper's SK-only / DS-only / BOTH comparison in one batched pass: disabling a detector is
    # a threshold at infinity (include/rfi.h).  Not timed.
    by_detector = None
    if plan.K == 1 and args.arith == "fast" and rank == 0 and not two_classes and args.layout == "time_major" and not work["sharded"] and args.adaptive == 0:
        INF = float("inf")
        d0, lo0, hi0, g0 = thr[0]
        plan3 = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                            rfi.RFI_FP16 if w.fp16 else rfi.RFI_FP32, n_int=w.n_int)
        if w.window_F > 1:
            plan3.set_window_freq(w.window_F)
        plan3.set_thresholds([[d0, lo0, hi0, g0], [d0, lo0, hi0, INF], [d0, -INF, INF, g0]])
        a3, w3, _ = plan3.alloc_outputs(device=dev)
        plan3.process_chunk(vis, a3, w3)
        c3 = plan3.confusion_counts(rfi.pack_flags(tr.reshape(plan.n_win, plan.n_baselines, w.n_chan))).cpu()
        fa3, md3 = sharding.rates(c3)
        by_detector = {name: {"false_alarm": float(fa3[i]), "missed_detection": float(md3[i])}
                       for i, name in enumerate(("both", "sk_only", "ds_only"))}
        plan3.destroy()
        del a3, w3

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    peak, peak_src = load_peaks()
    k_ms = statistics.mean(kernel_ms)
    achieved = algo_bytes / (k_ms * 1e-3) / 1e9
    variant = plan.last_variant
    # like-for-like denominator for a one-touch READ stream, measured live on this device (rfi_probe_read_bandwidth):
    # `peak` (MEASURED_PEAKS.json) is a read+write copy, which a read-only stream can exceed -- so `frac` may read > 1
    try:
        read_probe = rfi.probe_read_bandwidth(vis if in_bytes <= (40 << 30) else vis.reshape(-1)[: (40 << 30) // vis.element_size()])
    except Exception:
        read_probe = None
    mix_probe = None
    if plan.K > 1 and algo_bytes > in_bytes:     # zero-arithmetic stream with the same read/write volumes (rfi_probe_mix_bandwidth)
        try:
            mix_probe = rfi.probe_mix_bandwidth(vis if in_bytes <= (40 << 30) else vis.reshape(-1)[: (40 << 30) // vis.element_size()],
                                                algo_bytes - in_bytes)
        except Exception:
            mix_probe = None
    traffic = load_ncu_traffic(w.name, variant)
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic,
                "traffic_source": ("profiles/ncu_traffic.json (committed ncu --set full capture of this kernel on this workload; "
                                   "not re-measured by this run)" if traffic is not None else None),
                "peak_source": peak_src,
                "kernel": f"rfi_{variant}_kernel", "kernel_ms_mean": k_ms, "kernel_ms_min": min(kernel_ms),
                "kernel_ms_best": min(kernel_ms), "kernel_ms_median": statistics.median(kernel_ms),
                "launches_timed": len(kernel_ms),
                "algorithmic_bytes_per_launch": algo_bytes,
                "frac_of_nominal_8TBs": achieved / 8000.0,
                "read_stream_probe_gbs": read_probe,
                "frac_of_read_stream_probe": (achieved / read_probe) if read_probe else None,
                "mix_probe_gbs": mix_probe, "frac_of_mix_probe": (achieved / mix_probe) if mix_probe else None,
                "note": "frac = achieved / MEASURED_PEAKS hbm_gbs, a read+write copy_ figure; this kernel is a read-only "
                        "stream, so frac_of_read_stream_probe (same-device read-only probe) and frac_of_nominal_8TBs are the "
                        "fractions that cannot exceed 1"}

    # verification of the mode that was timed, against the oracle, in this same run (not timed)
    parity = None if args.no_parity else _safe(mode_parity, args, w, plan, vis, truth, thr, two_classes, dev)

    # end to end through the C ABI with HOST buffers (H2D of the inputs and D2H of the results inside the timed region)
    e2e = None
    if args.no_e2e:
        pass
    elif work["sharded"]:
        e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": out_bytes,
               "skipped": "strong-scaling run: the end-to-end host path is measured by the N = 1 run"}
    elif w.input_bytes > 32e9:
        e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": w.input_bytes, "d2h_bytes_per_step": out_bytes,
               "skipped": "chunk larger than the pinned host memory this bench allows itself (32 GB)"}
    else:
        try:
            h_vis = torch.empty(vis.shape, dtype=vis.dtype, pin_memory=True)
            h_vis.copy_(vis)
            K = max(plan.K, 1)
            h_avg = torch.empty(avg.shape, dtype=torch.float32, pin_memory=True)
            h_weight = torch.empty(weight.shape, dtype=torch.int32, pin_memory=True)
            h_flags = torch.empty(K, plan.n_win, plan.n_baselines, plan.wpb, dtype=torch.int32, pin_memory=True)
            plan.process_chunk_host_into(h_vis, h_avg, h_weight, h_flags)          # warm-up (allocates staging)
            n_e2e = max(5, min(args.steps, 6))               # >= 5 timed end-to-end steps (333 ms each on the lofar shape)
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                plan.process_chunk_host_into(h_vis, h_avg, h_weight, h_flags)      # synchronises before returning
            dt = (time.perf_counter() - t0) / n_e2e
            same = bool(torch.equal(h_avg, avg.cpu()) and torch.equal(h_weight, weight.cpu()))
            # what the link itself does: a plain pinned host-to-device copy of 2 GiB of the same buffer (not part of the step)
            n_probe = min(h_vis.numel(), (2 << 30) // h_vis.element_size())
            src, dst = h_vis.reshape(-1)[:n_probe], vis.reshape(-1)[:n_probe]
            keep = dst.clone()
            dst.copy_(src, non_blocking=True)
            ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ea.record()
            for _ in range(3):
                dst.copy_(src, non_blocking=True)
            eb.record()
            torch.cuda.synchronize(dev)
            link_gbs = 3 * n_probe * h_vis.element_size() / (ea.elapsed_time(eb) * 1e-3) / 1e9
            dst.copy_(keep)
            del keep
            # N > 1: measured on rank 0 alone (pinning N x 18.5 GB of host memory is not safe on every box), so the
            # figure is ONE GPU's end-to-end rate and is not multiplied by N
            e2e = {"value": samples / dt, "unit": UNIT, "ranks_measured": 1, "h2d_bytes_per_step": w.input_bytes,
                   "d2h_bytes_per_step": out_bytes, "ms_per_step": dt * 1e3, "steps": n_e2e,
                   "h2d_gbs": w.input_bytes / dt / 1e9, "h2d_link_probe_gbs": link_gbs,
                   "frac_of_h2d_link": (w.input_bytes / dt / 1e9) / link_gbs, "matches_device_path": same,
                   "api": "rfi_process_chunk_host (pinned host buffers; per-integration H2D overlapped with the kernel)"}
            del h_vis
        except Exception as exc:  # e.g. not enough pinnable host memory on the box
            e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": w.input_bytes, "d2h_bytes_per_step": out_bytes,
                   "error": str(exc)[:200]}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        g = torch.Generator().manual_seed(7)
        n_s = min(w.n_cells, 24576)           # ~12 CPU-seconds of oracle work on the lofar shape
        idx = torch.randperm(w.n_cells, generator=g)[:n_s].sort().values.to(dev)
        sub = vis.reshape(w.n_time, w.n_cells, 4, 2)[:, idx].cpu().numpy()
        cpu = oracle_baseline(sub, w, thr)
        del sub

    # every BASELINE.json config in the SAME run: sub-records, each timed launch by launch with
    # CUDA events (best and median over the launches) and parity-checked on sampled cells
    configs = None
    if (world == 1 and not args.no_configs and args.workload == "lofar" and args.K == 1 and args.arith == "fast"
            and args.layout == "time_major" and not two_classes and args.variant == "auto" and args.adaptive == 0):
        configs = []
        n_sub = max(args.steps, 20)
        plan.destroy()
        del avg, weight
        torch.cuda.empty_cache()
        # configs[4] re-uses the resident lofar chunk (it IS "config 2 data")
        configs.append(measure_config("sweep", 64, dev, n_sub, 3, peak, read_probe, vis=vis, truth=truth, n_clean=160, n_rfi=64))
        del vis, truth
        torch.cuda.empty_cache()
        for name in ("lofar_fp16", "lofar_tf10x2"):          # K = 1 and the K = 64 sweep on the same resident chunk
            v2, t2 = synth.make_chunk(synth.WORKLOADS[name], seed=1234, device=dev)
            configs.append(measure_config(name, 1, dev, n_sub, 3, peak, read_probe, vis=v2, truth=t2))
            configs.append(measure_config(name, 64, dev, n_sub, 3, peak, read_probe, vis=v2, truth=t2, n_clean=160, n_rfi=64))
            del v2, t2
            torch.cuda.empty_cache()
        configs.append(measure_config("large", 1, dev, n_sub, 3, peak, read_probe, n_clean=256, n_rfi=256, cpu_baseline=True))
        configs.append(measure_config("tiny", 1, dev, max(n_sub, 50), 5, peak, read_probe, n_clean=96, n_rfi=6))
        # the same small chunk through the low-latency variant (RFI_VARIANT_SPLIT: a unit's rows split over 16 warps)
        configs.append(measure_config("tiny", 1, dev, max(n_sub, 50), 5, peak, read_probe, n_clean=96, n_rfi=6, variant="split"))

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None,
        "dtype": "f32" if not w.fp16 else "f32 (f16 storage)", "data": "synthetic (seeded; stands in for LOFAR data)",
        "config": {"workload": (f"{w.name}: BASELINE.json configs[{synth.BASELINE_CONFIG_INDEX[w.name]}]"
                                if w.name in synth.BASELINE_CONFIG_INDEX else f"{w.name}: SURVEY 8(f) NEXT-1, not a BASELINE.json config"),
                   "n_stations": w.n_stations, "n_baselines": w.n_baselines, "n_chan": w.n_chan, "n_time": w.n_time,
                   "window_M": w.window_M, "window_F": w.window_F, "n_int": w.n_int, "K": max(plan.K, 1), "variant": variant,
                   "arithmetic": args.arith if args.arith == "fast" else f"tables, mask {args.mask:#06x}",
                   "threshold_classes": 2 if two_classes else 1, "layout": args.layout,
                   "adaptive_false_alarm": args.adaptive if args.adaptive > 0 else None,
                   "adaptive_scope": args.adaptive_scope if args.adaptive > 0 else None,
                   "input_bytes": w.input_bytes,
                   "l2": ("L2 flushed between timed iterations (256 MB write, outside the timed events)" if small
                          else "input (>= 9 GB) is far larger than the 126 MB L2: no flush needed"),
                   "sharding": (("ONE chunk partitioned by baseline (rfi_plan_set_baseline_shard), no collective" if work["sharded"]
                                 else "one subband chunk per rank, no collective") if world > 1 else "single GPU")},
        "gbytes_per_s": total_algo / (ms_per_step * 1e-3) / 1e9,
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "detection": {"false_alarm": fa, "missed_detection": md, "flag_fraction": float(flag_frac[0]), "by_detector": by_detector,
                      "per_set": {"K": int(counts.shape[0]), "false_alarm_min_max": [float(p_fa.min()), float(p_fa.max())],
                                  "missed_detection_min_max": [float(p_md.min()), float(p_md.max())],
                                  "flag_fraction_min_max": [float(flag_frac.min()), float(flag_frac.max())]}},
    }
    line["parity"] = parity
    head = {"workload": w.name, "K": max(args.K, 1), "storage": "f16" if w.fp16 else "f32", "window": f"{w.window_M} x {w.window_F}",
            "kernel": variant, "ms_best": min(kernel_ms), "ms_median": statistics.median(kernel_ms),
            "gbs": algo_bytes / (statistics.median(kernel_ms) * 1e-3) / 1e9,
            "frac": algo_bytes / (statistics.median(kernel_ms) * 1e-3) / 1e9 / peak,
            "frac_of_nominal_8TBs": algo_bytes / (statistics.median(kernel_ms) * 1e-3) / 1e9 / 8000.0,
            "parity_status": (parity or {}).get("status"), "cells_sampled": (parity or {}).get("cells_sampled"),
            "flag_mismatch_unexplained": (parity or {}).get("flag_mismatch_unexplained")}
    if cpu:
        head["cpu_baseline_samples_per_s"] = cpu["value"]
    roofline["per_config"] = [head] + [per_config_entry(c) for c in (configs or [])]
    if configs is not None:
        line["configs"] = configs
    torch.cuda.profiler.stop()        # `ncu --profile-from-start off` lists every launch of the run, sub-records included
    print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def self_launch(args) -> int:
    """`python bench.py --gpus N` without torchrun around it: start the N ranks here, one process per GPU, the way the
    driver's own command does (torch.distributed.run, one node, rendezvous on 127.0.0.1), with the same arguments.
    Returns the launcher's exit code.  Refuses, loudly, a box with fewer than N GPUs (--dry-launch needs none)."""
    import socket
    if not args.dry_launch:
        import torch
        found = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if found < args.gpus:
            sys.stderr.write(f"bench.py: --gpus {args.gpus} needs {args.gpus} GPUs on this node, found {found}\n")
            return 2
    with socket.socket() as sk:                                # a free rendezvous port
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                       # the communicator lines show which ranks / devices joined
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    env.setdefault("OMP_NUM_THREADS", "1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd, env=env)


def run_dry_launch(args):
    """--dry-launch: the N-rank plumbing of run_ours without a GPU (CPU test of the launcher): ranks join a gloo group,
    take their share of the work from sharding.rank_work, reduce a time (MAX) and a sample count (SUM) with the helpers
    the timed path uses, and rank 0 prints one JSON line."""
    import torch.distributed as dist
    from paper_2412_14775_b200 import sharding, synth
    world, rank = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
    w = synth.WORKLOADS[args.workload]
    work = sharding.rank_work(w.n_baselines, world, rank, args.scaling)
    samples = w.n_time * work["b_count"] * w.n_chan
    total = sharding.sum_scalar_over_ranks(samples)
    slowest = sharding.max_over_ranks(1.0 + rank)              # stands in for the device-measured milliseconds
    shares = [None] * world
    if world > 1:
        dist.all_gather_object(shares, work)
    else:
        shares = [work]
    if rank == 0:
        print(json.dumps({"dry_launch": True, "n_gpus": world, "scaling": args.scaling, "total_samples": total,
                          "max_ms": slowest, "work": shares}))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="lofar")
    ap.add_argument("--variant", default="auto", choices=["auto", "direct", "tma"])
    ap.add_argument("--K", type=int, default=1, help="threshold sets (K > 1: batched sweep)")
    ap.add_argument("--arith", default="fast", choices=["fast", "tables"],
                    help="tables: the paper's Tables 1-2 literally, per-group precision from --mask (DESIGN.md section 11)")
    ap.add_argument("--mask", type=lambda x: int(x, 0), default=0x3C50, help="14-bit half-precision mask for --arith tables")
    ap.add_argument("--layout", default="time_major", choices=["time_major", "cell_major"],
                    help="cell_major: vis[b][c][t][pol] through the transposing tensor map (rfi_plan_set_layout)")
    ap.add_argument("--classes", action="store_true",
                    help="separate threshold class for the auto-correlations (rfi_plan_set_baseline_classes)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one chunk per rank; strong = ONE chunk sharded by baseline (rfi_plan_set_baseline_shard)")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config sub-records of the default run")
    ap.add_argument("--adaptive-scope", default="class", choices=["class", "baseline"],
                    help="with --adaptive: one threshold set per baseline class, or per baseline stream (rfi_plan_set_adaptive_scope)")
    ap.add_argument("--adaptive", type=float, default=0.0,
                    help="hold this false-alarm rate by on-line threshold adaptation (rfi_plan_set_adaptive, DESIGN.md NEXT-3)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-parity", action="store_true", help="skip the sampled-cell oracle check of the timed mode")
    ap.add_argument("--dry-launch", action="store_true",
                    help="exercise the N-rank launch and the rank bookkeeping on CPU (gloo), no kernels: tests/test_sharding.py")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    world_env = os.environ.get("WORLD_SIZE")
    if args.impl == "ours" and args.gpus > 1 and world_env is None:
        sys.exit(self_launch(args))                            # not under torchrun: start the N ranks ourselves
    if args.impl == "ours" and world_env is not None and int(world_env) != args.gpus:
        sys.exit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE = {world_env} ranks")
    if args.dry_launch:
        run_dry_launch(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.workload == "sim42":
        if args.K <= 1:
            args.K = 64
        run_sim42(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
