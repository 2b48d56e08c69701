"""Parity comparators: CUDA path (through the C ABI) vs the fp64 oracle, element by element.

Tolerances (north_star: fp32 statistics and averages to relative 1e-5, flags bit-exact except windows whose
statistic lies within 1e-5 relative of a threshold; fp16: 2e-3 and >= 99.9 % flag agreement).  Both statistics
legitimately reach 0 (tau = 0 for a tone, r_im = 0 for autos), so "relative" carries the floors derived in
DESIGN.md section "Tolerances":
    |d tau| <= tol * max(|tau|, 0.01 c),  c = (W d + 1)/(W - 1)
    |d r|   <= tol * max(r, 1/sqrt(W))
    |d avg| <= tol * max(|avg|, rms(avg))      per real component
The pure-relative maxima are returned as well (reported, not gated).
"""
from __future__ import annotations

import math

import numpy as np

from oracle import rfi_oracle as orc


def near_threshold(tau, r_re, r_im, thr, M, tol):
    """bool mask of windows whose statistic is within `tol` (relative, floored) of one of its thresholds.
    M is the window size W (= T*F for T x F footprints)."""
    d, s_low, s_high, gamma = thr
    c = (M * d + 1) / (M - 1)
    near = np.zeros(tau.shape, bool)
    for s in (s_low, s_high):
        if np.isfinite(s):
            near |= np.abs(tau - s) <= tol * max(abs(s), 0.01 * c)
    if np.isfinite(gamma):
        for r in (r_re, r_im):
            near |= np.abs(r - gamma) <= tol * max(abs(gamma), 1 / math.sqrt(M))
    return near


def compare(vis_np, M, n_int, thresholds, gpu, tol=1e-5, fp16=False, oracle_threads=0, F=1):
    """gpu: dict with numpy arrays avg [K,O,cells,4] complex, weight [K,O,cells], flags [K,W,cells] bool,
    optional tau/r_re/r_im [W,cells] (tau for set 0).  Returns a report dict; raises AssertionError on failure."""
    thresholds = np.asarray(thresholds, np.float64).reshape(-1, 4)
    # the kernel receives the thresholds as float32: the oracle must decide on the same numbers
    thr32 = thresholds.astype(np.float32).astype(np.float64)
    res = orc.process(vis_np, M, n_int, thr32, n_threads=oracle_threads, F=F)
    W = M * F                                            # window size of Eq.(4), Eq.(9)
    K, n_win, n_cells = res.flags.shape
    n_out = res.weight.shape[1]
    wpo = n_int // M
    rep = {"n_windows": int(n_win * n_cells), "K": int(K)}
    def check_stat(name, got, ref, floor):
        """compare where the oracle's statistic is finite; where it is not, the GPU's must not be finite either"""
        fin = np.isfinite(ref)
        assert (~np.isfinite(got[~fin])).all(), f"{name}: oracle is non-finite where the GPU is finite"
        d = np.abs(got.astype(np.float64) - ref)[fin]
        bound = tol * np.maximum(np.abs(ref[fin]), floor)
        rep[name + "_max_abs"] = float(d.max(initial=0))
        rep[name + "_max_rel"] = float((d / np.maximum(np.abs(ref[fin]), 1e-300)).max(initial=0))
        rep[name + "_worst_over_bound"] = float((d / bound).max(initial=0))
        assert (d <= bound).all(), f"{name} mismatch: worst |d|/bound = {rep[name + '_worst_over_bound']:.3g}"

    if gpu.get("tau") is not None:
        d0 = thr32[0, 0]
        c0 = (W * d0 + 1) / (W - 1)
        check_stat("tau", gpu["tau"], res.tau[0], 0.01 * c0)
        check_stat("r_re", gpu["r_re"], res.r_re, 1 / math.sqrt(W))
        check_stat("r_im", gpu["r_im"], res.r_im, 1 / math.sqrt(W))

    n_mismatch, n_exempt, n_unexplained, n_out_skipped = 0, 0, 0, 0
    avg_worst, avg_rel_worst = 0.0, 0.0
    for k in range(K):
        mism = gpu["flags"][k] != res.flags[k].astype(bool)
        near = near_threshold(res.tau[k], res.r_re, res.r_im, thr32[k], W, tol if not fp16 else 0.0)
        n_mismatch += int(mism.sum())
        n_exempt += int((mism & near).sum())
        n_unexplained += int((mism & ~near).sum())
        # outputs: skip (cell, output) pairs that contain a mismatched window
        bad_out = mism.reshape(n_out, wpo, n_cells).any(1)
        ok = ~bad_out
        n_out_skipped += int(bad_out.sum())              # reported: (cell, output) pairs whose average is not compared
        assert (gpu["weight"][k][ok] == res.weight[k][ok]).all(), "weight mismatch on outputs with identical flags"
        ref = res.avg[k].view(np.float64).reshape(n_out, n_cells, 8)
        got = gpu["avg"][k].astype(np.complex128).view(np.float64).reshape(n_out, n_cells, 8)
        rms = math.sqrt(float((ref ** 2).mean())) if ref.size else 0.0
        da = np.abs(got - ref)[ok]
        bound = tol * np.maximum(np.abs(ref[ok]), rms)
        if da.size:
            avg_worst = max(avg_worst, float((da / np.maximum(bound, 1e-300)).max()))
            nz = np.abs(ref[ok]) > 0
            if nz.any():
                avg_rel_worst = max(avg_rel_worst, float((da[nz] / np.abs(ref[ok][nz])).max()))
        assert (da <= bound).all(), f"avg mismatch (set {k}): worst |d|/bound = {(da / np.maximum(bound, 1e-300)).max():.3g}"
    total = K * n_win * n_cells
    rep.update(flag_mismatch=n_mismatch, flag_mismatch_near_threshold=n_exempt, flag_mismatch_unexplained=n_unexplained,
               flag_agreement=1.0 - n_mismatch / max(total, 1), avg_worst_over_bound=avg_worst,
               avg_max_rel=avg_rel_worst, oracle_flag_fraction=float(res.flags.mean()),
               outputs_skipped=n_out_skipped, outputs_total=int(K * n_out * n_cells))
    if fp16:
        assert rep["flag_agreement"] >= 0.999, f"fp16 flag agreement {rep['flag_agreement']:.5f} < 0.999"
    else:
        assert n_unexplained == 0, f"{n_unexplained} flag mismatches away from any threshold"
    return rep


def fp16_vs_fp32_original(vis32_np, M, n_int, thresholds, gpu, F=1, oracle_threads=0):
    """SURVEY.md 8(c)-T / PAPER.md:251,269 ("< 1 % of the flags change"): the fp16-STORAGE kernel against the oracle
    run on the ORIGINAL fp32 values (before rounding to half).  Returns the flag agreement (gated by the caller at
    >= 99.9 %) and the statistic deltas the quantisation causes (reported, not gated)."""
    thr32 = np.asarray(thresholds, np.float64).reshape(-1, 4).astype(np.float32).astype(np.float64)
    res = orc.process(vis32_np, M, n_int, thr32, n_threads=oracle_threads, F=F)
    K = res.flags.shape[0]
    mism = sum(int((gpu["flags"][k] != res.flags[k].astype(bool)).sum()) for k in range(K))
    rep = {"flag_agreement_vs_fp32_original": 1.0 - mism / max(res.flags.size, 1), "flag_mismatch_vs_fp32_original": mism}
    if gpu.get("tau") is not None:
        fin = np.isfinite(res.tau[0])
        rep["quantisation_dtau_max"] = float(np.abs(gpu["tau"].astype(np.float64) - res.tau[0])[fin].max(initial=0))
        rep["quantisation_dr_max"] = float(max(np.abs(gpu["r_re"].astype(np.float64) - res.r_re)[fin].max(initial=0),
                                               np.abs(gpu["r_im"].astype(np.float64) - res.r_im)[fin].max(initial=0)))
    return rep


def gpu_outputs_to_numpy(plan, avg, weight, stats, flags_unpacked):
    """torch device outputs -> the dict `compare` expects."""
    K = max(plan.K, 1)
    out = {
        "avg": avg.cpu().numpy().reshape(K, plan.n_out, plan.n_cells, 4, 2).view(np.complex64).reshape(K, plan.n_out, plan.n_cells, 4),
        "weight": weight.cpu().numpy().reshape(K, plan.n_out, plan.n_cells).astype(np.int64),
        "flags": flags_unpacked.cpu().numpy().reshape(K, plan.n_win, plan.n_cells),
    }
    if stats is not None:
        s = stats.cpu().numpy().reshape(3, plan.n_win, plan.n_cells)
        out.update(tau=s[0], r_re=s[1], r_im=s[2])
    return out
