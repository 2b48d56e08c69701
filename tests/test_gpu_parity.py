"""GPU parity: the CUDA path through the C ABI against the fp64 oracle, element by element, on the same
seeded inputs.  Sizes span several 32-cell tiles, ragged tails, both kernel variants and both storage types."""
import math

import numpy as np
import pytest
import torch

import paper_2412_14775_b200 as rfi
from paper_2412_14775_b200 import synth
from tests.parity_util import compare, fp16_vs_fp32_original, gpu_outputs_to_numpy

pytestmark = pytest.mark.gpu
INF = float("inf")


def run_gpu(w, vis, thresholds, variant="auto", stats=True, layout="time_major"):
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                       rfi.RFI_FP16 if w.fp16 else rfi.RFI_FP32, n_int=w.n_int)
    if w.window_F > 1:
        plan.set_window_freq(w.window_F)
    plan.set_thresholds(thresholds)
    plan.set_variant(variant)
    avg, weight, st = plan.alloc_outputs(stats=stats)
    avg.fill_(float("nan")); weight.fill_(-1)
    if st is not None:
        st.fill_(float("nan"))
    d_vis = vis.cuda()
    if layout == "cell_major":                           # vis[b][c][t][pol] behind the transposing tensor map
        plan.set_layout("cell_major")
        d_vis = d_vis.permute(1, 2, 0, 3, 4).contiguous()
    plan.process_chunk(d_vis, avg, weight, st)
    torch.cuda.synchronize()
    flags = rfi.unpack_flags(plan.get_flags(), w.n_chan)
    out = gpu_outputs_to_numpy(plan, avg, weight, st, flags)
    used = plan.last_variant
    assert plan.launch_count >= 1
    plan.destroy()
    return out, used


def check(w, thresholds, variant, seed=1234, tol=None, mutate=None, layout="time_major"):
    vis, truth = synth.make_chunk(w, seed=seed, device="cpu")
    if mutate is not None:
        mutate(vis)
    out, used = run_gpu(w, vis, thresholds, variant, layout=layout)
    if variant != "auto":
        assert used == variant
    v = vis.numpy().reshape(w.n_time, w.n_cells, 4, 2)
    rep = compare(v, w.window_M, w.n_int, thresholds, out, tol=tol or (2e-3 if w.fp16 else 1e-5), fp16=w.fp16,
                  F=w.window_F)
    return rep, out, truth


@pytest.mark.parametrize("variant", ["direct", "tma", "split"])
def test_tiny_config(variant):
    """BASELINE.json configs[0]: 4 stations, 6 baselines, 16 channels, 1024 samples, M=64, 16 outputs."""
    w = synth.WORKLOADS["tiny"]
    thr = synth.default_thresholds(w.window_M)
    rep, out, truth = check(w, thr, variant)
    assert rep["n_windows"] == 16 * 96
    # the injected burst (10x noise power, fully polarised) must be caught where it fills most of a window
    flagged = out["flags"][0]
    assert flagged[truth.numpy()].mean() > 0.5
    assert flagged[~truth.numpy()].mean() < 0.1


@pytest.mark.parametrize("variant", ["direct", "tma", "split"])
def test_mini_lofar_several_tiles_autos_gain_bursts(variant):
    w = synth.WORKLOADS["lofar"].scaled(n_stations=6, n_time=1024, n_int=256, burst_cell_frac=0.1)
    assert w.n_cells == 21 * 64
    rep, out, truth = check(w, synth.default_thresholds(16), variant)
    assert 0.001 < rep["oracle_flag_fraction"] < 0.2


@pytest.mark.parametrize("variant", ["direct", "tma", "split"])
@pytest.mark.parametrize("M,n_int,n_time", [(20, 100, 400), (10, 50, 200), (2, 8, 64), (3, 12, 48), (7, 28, 56),
                                              (64, 128, 256), (128, 256, 256), (16, 16, 64)])
def test_window_sizes_and_ragged_channels(variant, M, n_int, n_time):
    """n_chan = 20: 200 cells = 6.25 tiles, flag words shared between warps (atomic path); the paper's W = 20."""
    w = synth.Workload("ragged", 5, False, 20, n_time, M, n_int, burst_cell_frac=0.2, channel_gain=True)
    assert w.n_cells == 200
    thr = synth.default_thresholds(M) if M >= 8 else [[1.0, 0.02, 1.5, 0.9]]
    check(w, thr, variant, seed=7 + M)


def test_cells_not_multiple_of_four_cannot_use_tma():
    w = synth.Workload("odd", 3, False, 13, 128, 16, 64, burst_cell_frac=0.3)
    assert w.n_cells == 39
    vis, _ = synth.make_chunk(w, seed=3)
    out, used = run_gpu(w, vis, synth.default_thresholds(16), "auto")
    assert used == "direct"
    compare(vis.numpy().reshape(w.n_time, w.n_cells, 4, 2), 16, 64, synth.default_thresholds(16), out)
    plan = rfi.RfiPlan(3, 3, 13, 128, 16)
    plan.set_thresholds(synth.default_thresholds(16)); plan.set_variant("tma")
    avg, weight, _ = plan.alloc_outputs()
    with pytest.raises(rfi.RfiError):
        plan.process_chunk(vis.cuda(), avg, weight)
    plan.destroy()


@pytest.mark.parametrize("n_chan", [1, 8, 16, 32, 48, 96])
def test_flag_word_layouts(n_chan):
    w = synth.Workload("words", 4, True, n_chan, 128, 8, 32, burst_cell_frac=0.3)
    for variant in ("direct", "tma", "split"):
        if variant == "tma" and w.n_cells % 4:
            continue
        check(w, [[1.0, 0.05, 1.0, 0.7]], variant, seed=n_chan)


@pytest.mark.parametrize("variant", ["direct", "tma", "split"])
def test_fp16_storage(variant):
    """configs[2] in miniature: fp16 storage, fp32 accumulation, CW tones on one channel.  Statistics against the
    oracle on the SAME fp16-rounded values at 2e-3; flag agreement >= 99.9 %."""
    w = synth.WORKLOADS["lofar_fp16"].scaled(n_stations=6, n_time=1024, n_int=256, burst_cell_frac=0.1, tone_chan_frac=0.02)
    rep, out, truth = check(w, synth.default_thresholds(16), variant)
    assert rep["flag_agreement"] >= 0.999
    # and the fp32-accumulate path on fp16 data is in fact as tight as the fp32 one
    vis, _ = synth.make_chunk(w, seed=1234)
    compare(vis.numpy().reshape(w.n_time, w.n_cells, 4, 2), 16, 256, synth.default_thresholds(16), out, tol=1e-5)
    # against the oracle on the ORIGINAL fp32 values (the same seeded chunk before
    # it is rounded to half) the flags must agree to >= 99.9 %; the statistic shifts are reported
    vis32, _ = synth.make_chunk(w.scaled(fp16=False), seed=1234)
    assert torch.equal(vis32.to(torch.float16), vis)
    q = fp16_vs_fp32_original(vis32.numpy().reshape(w.n_time, w.n_cells, 4, 2), 16, 256, synth.default_thresholds(16), out)
    print(f"fp16 storage vs fp32 originals [{variant}]: {q}; outputs skipped in the fp16 comparison: "
          f"{rep['outputs_skipped']} of {rep['outputs_total']}")
    assert q["flag_agreement_vs_fp32_original"] >= 0.999


@pytest.mark.parametrize("variant", ["direct", "tma", "split"])
def test_degenerate_inputs(variant):
    """All-zero cell, NaN / Inf samples, Hermitian (auto) cells, tiny and huge amplitudes, disabled detectors."""
    w = synth.Workload("degenerate", 4, True, 16, 256, 16, 64, burst_cell_frac=0.2)

    def mutate(vis):
        v = vis.view(w.n_time, w.n_cells, 4, 2)
        v[:, 5] = 0.0                      # all-zero cell: tau = -c, r = 0
        v[40:48, 7] = 0.0                  # zero samples inside a window
        v[17, 9, 2, 1] = float("nan")
        v[100, 11, 0, 0] = float("inf")
        v[:, 20] *= 1e-12                  # scale invariance at the edges of the documented range
        v[:, 21] *= 1e12

    thr = [[1.0, 0.1, 0.62, 0.52]]
    rep, out, _ = check(w, thr, variant, mutate=mutate)
    f = out["flags"][0]
    assert f[17 // 16, 9] and f[100 // 16, 11]            # non-finite windows are flagged
    assert np.isfinite(out["avg"]).all()
    c = (16 * 1.0 + 1) / 15
    assert np.allclose(out["tau"][:, 5], -c) and (out["r_re"][:, 5] == 0).all()
    assert f[:, 5].all() and (out["weight"][0][:, 5] == 0).all() and (out["avg"][0][:, 5] == 0).all()
    # detectors disabled: only the non-finite windows are flagged
    rep2, out2, _ = check(w, [[1.0, -INF, INF, INF]], variant, mutate=mutate)
    assert out2["flags"].sum() == 2


# Reading G6 (non-finite input: the window is flagged by every set and contributes nothing) on every kernel family
# that has its own code for it: the batched TMA kernel zeroes non-finite window sums before its fma-masked add
# (whole-word and per-word flag stores), the register-staged batched kernel predicates its adds, fp16 storage widens
# half NaN / Inf, the cell-major kernels read through the transposing map.  (name, n_stations, autos, n_chan, fp16, K, layout)
_G6_CASES = [
    ("batched_tma_fullword_K5", 4, True, 32, False, 5, "time_major"),
    ("batched_tma_fullword_K64", 4, True, 32, False, 64, "time_major"),
    ("batched_tma_perword_K5", 4, True, 16, False, 5, "time_major"),
    ("batched_register_staged_ragged_K5", 3, False, 13, False, 5, "time_major"),     # 39 cells: n_cells % 4 != 0
    ("batched_register_staged_ragged_K64", 3, False, 13, False, 64, "time_major"),
    ("fp16_direct_K1", 4, True, 16, True, 1, "time_major"),
    ("fp16_batched_K5", 4, True, 32, True, 5, "time_major"),
    ("fp16_batched_K64", 4, True, 32, True, 64, "time_major"),
    ("cell_major_K1", 4, True, 16, False, 1, "cell_major"),
    ("cell_major_K5", 4, True, 32, False, 5, "cell_major"),
    ("cell_major_fp16_K1", 4, True, 16, True, 1, "cell_major"),
    ("cell_major_fp16_K17", 4, True, 32, True, 17, "cell_major"),
]


@pytest.mark.parametrize("name,n_st,autos,n_chan,fp16,K,layout", _G6_CASES, ids=[c[0] for c in _G6_CASES])
def test_non_finite_and_degenerate_inputs_every_kernel_family(name, n_st, autos, n_chan, fp16, K, layout):
    w = synth.Workload(name, n_st, autos, n_chan, 512, 16, 128, fp16=fp16, burst_cell_frac=0.2)
    nc = w.n_cells

    def mutate(vis):
        v = vis.view(w.n_time, nc, 4, 2)
        v[:, 5 % nc] = 0.0                                # all-zero cell
        v[40:48, 7 % nc] = 0.0                            # zero samples inside a window
        v[17, 9 % nc, 2, 1] = float("nan")
        v[100, 11 % nc, 0, 0] = float("inf")
        v[200, 12 % nc, 3, 1] = float("-inf")
        v[300:303, 13 % nc] = float("nan")                # a run of NaN samples across all pols
        v[317, nc - 1, 1, 0] = float("nan")               # last cell of the last (possibly ragged) tile
        if fp16:
            v[:, 20 % nc] *= 1e-3                         # subnormal halves (|x| < 6.1e-5)
            v[64:80, 21 % nc, 0, 0] = 65504.0             # largest finite half
            v[80:96, 21 % nc, 3, 0] = -65504.0
            v[96, 22 % nc, 0, 0] = 65504.0                # one maximal sample among noise
        else:
            v[:, 20 % nc] *= 1e-12
            v[:, 21 % nc] *= 1e12

    bad = sorted({(17 // 16, 9 % nc), (100 // 16, 11 % nc), (200 // 16, 12 % nc), (300 // 16, 13 % nc), (317 // 16, nc - 1)})
    thr = synth.sweep_thresholds(16, K, seed=3) if K > 1 else [[1.0, 0.1, 0.62, 0.52]]
    rep, out, _ = check(w, thr, "auto", mutate=mutate, layout=layout)
    assert rep["K"] == K
    for k in range(K):
        for (wi, c) in bad:
            assert out["flags"][k][wi, c], f"set {k}: non-finite window ({wi}, cell {c}) not flagged"
    assert np.isfinite(out["avg"]).all()                  # a non-finite window contributes nothing to any average
    assert (out["weight"][:, :, 5 % nc] == 0).all()       # all-zero cell: tau = -c is below every s_low -> all flagged
    # detectors disabled (thresholds at infinity): ONLY the non-finite windows are flagged, in every set
    rep2, out2, _ = check(w, [[1.0, -INF, INF, INF]] * K, "auto", mutate=mutate, layout=layout)
    assert out2["flags"].sum() == K * len(bad)


@pytest.mark.parametrize("variant", ["direct", "tma", "split"])
def test_exact_ties_are_not_flagged(variant):
    """r = |16 - 2*4|/16 = 0.5 exactly and tau = 0 exactly: thresholds equal to the statistic do not flag (Eq.(5),(10) strict)."""
    M = 16
    w = synth.Workload("ties", 2, True, 16, M, M, M)
    vis = torch.zeros(M, 3, 16, 4, 2)
    sign = torch.ones(M); sign[:4] = -1
    vis[:, :, :, 0, 0] = 2.0 * sign[:, None, None]        # xx = +-2, everything else 0: Stokes direction (1,0,0), |I| = 2
    for thr, expect in (([1.0, -INF, INF, 0.5], False), ([1.0, -INF, INF, float(np.nextafter(np.float32(0.5), np.float32(0)))], True),
                        ([1.0, 0.0, INF, INF], False), ([1.0, 1e-30, INF, INF], True), ([1.0, -INF, 0.0, INF], False)):
        out, _ = run_gpu(w, vis, [thr], variant)
        assert out["tau"].max() == 0.0 and out["tau"].min() == 0.0
        assert (out["r_re"] == 0.5).all() and (out["r_im"] == 0.0).all()
        assert out["flags"].all() == expect and out["flags"].any() == expect


def test_host_path_equals_device_path():
    w = synth.WORKLOADS["lofar"].scaled(n_stations=5, n_time=1024, n_int=256, burst_cell_frac=0.1)
    vis, _ = synth.make_chunk(w, seed=11)
    thr = synth.default_thresholds(16)
    out_dev, _ = run_gpu(w, vis, thr, "auto")
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
    plan.set_thresholds(thr)
    for _ in range(2):                                   # twice: staging buffers and tensor maps are reused
        avg, weight, flags, stats = plan.process_chunk_host(vis.pin_memory(), want_stats=True)
    out_host = gpu_outputs_to_numpy(plan, avg, weight, stats, rfi.unpack_flags(flags, w.n_chan))
    assert plan.launch_count == 2 * w.n_out
    plan.destroy()
    for key in ("avg", "weight", "flags", "tau", "r_re", "r_im"):
        np.testing.assert_array_equal(out_dev[key], out_host[key])


def test_host_path_staging_regrows_with_the_slab(K=1):
    """VERDICT r01 / ADVICE: the host path's staging slabs hold one integration of the CURRENT shape.  A host call at
    n_int = 256, then rfi_plan_set_integration(1024) (4x larger slab), then a shard that grows from 2 baselines to all:
    every host call must equal the device path bit for bit (before the fix the second call copied past the slab)."""
    w = synth.WORKLOADS["lofar"].scaled(n_stations=5, n_time=1024, n_int=256, burst_cell_frac=0.1)
    vis, _ = synth.make_chunk(w, seed=21)
    thr = synth.default_thresholds(16)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=256)
    plan.set_thresholds(thr)
    plan.set_baseline_shard(0, 2)                         # smallest slab first: 2 baselines x 256 samples
    shapes = [(0, 2, 256), (0, 2, 1024), (0, w.n_baselines, 1024), (3, 7, 512), (0, w.n_baselines, 256)]
    for b0, bc, n_int in shapes:
        plan.set_baseline_shard(b0, bc)
        plan.set_integration(n_int)
        sub = vis[:, b0:b0 + bc].contiguous()
        ws = synth.Workload("host_regrow", w.n_stations, True, w.n_chan, w.n_time, w.window_M, n_int)
        avg, weight, flags, stats = plan.process_chunk_host(sub.pin_memory(), want_stats=True)
        host = gpu_outputs_to_numpy(plan, avg, weight, stats, rfi.unpack_flags(flags, w.n_chan))
        d_avg, d_weight, d_stats = plan.alloc_outputs(stats=True)
        plan.process_chunk(sub.cuda(), d_avg, d_weight, d_stats)
        torch.cuda.synchronize()
        dev = gpu_outputs_to_numpy(plan, d_avg, d_weight, d_stats, rfi.unpack_flags(plan.get_flags(), w.n_chan))
        for key in ("avg", "weight", "flags", "tau", "r_re", "r_im"):
            np.testing.assert_array_equal(host[key], dev[key], err_msg=f"{key} at shard ({b0},{bc}), n_int {n_int}")
        compare(sub.numpy().reshape(w.n_time, bc * w.n_chan, 4, 2), 16, n_int, thr, host)
    plan.destroy()


def test_tma_variant_rejection_has_a_message():
    plan = rfi.RfiPlan(3, 3, 13, 128, 16)
    plan.set_thresholds(synth.default_thresholds(16)); plan.set_variant("tma")
    avg, weight, _ = plan.alloc_outputs()
    vis = torch.zeros(128, 3, 13, 4, 2, device="cuda")
    with pytest.raises(rfi.RfiError) as e:
        plan.process_chunk(vis, avg, weight)
    assert e.value.code == -1 and "% 4" in rfi.load_library().rfi_last_cuda_error().decode()
    plan.destroy()


@pytest.mark.parametrize("K", [1, 5])
def test_baseline_shards_equal_slices_of_the_full_run(K):
    """shard by baseline with no exchange -- two shard plans reproduce the full run bit for bit."""
    from paper_2412_14775_b200 import sharding
    w = synth.WORKLOADS["lofar"].scaled(n_stations=6, n_time=512, n_int=256, burst_cell_frac=0.1)
    vis, _ = synth.make_chunk(w, seed=17)
    thr = synth.default_thresholds(16) if K == 1 else synth.sweep_thresholds(16, K, seed=2)
    full, _ = run_gpu(w, vis, thr, "auto")
    B, C = w.n_baselines, w.n_chan
    for rank in range(2):
        b0, bc = sharding.shard_baselines(B, 2, rank)
        plan = rfi.RfiPlan(w.n_stations, B, C, w.n_time, w.window_M, n_int=w.n_int)
        plan.set_baseline_shard(b0, bc)
        plan.set_thresholds(thr)
        avg, weight, stats = plan.alloc_outputs(stats=True)
        plan.process_chunk(vis[:, b0:b0 + bc].contiguous().cuda(), avg, weight, stats)
        torch.cuda.synchronize()
        out = gpu_outputs_to_numpy(plan, avg, weight, stats, rfi.unpack_flags(plan.get_flags(), C))
        plan.destroy()
        sl = slice(b0 * C, (b0 + bc) * C)
        for key in ("avg", "weight", "flags"):
            np.testing.assert_array_equal(out[key], full[key][:, :, sl])
        for key in ("tau", "r_re", "r_im"):
            np.testing.assert_array_equal(out[key], full[key][:, sl])


def test_split_variant_against_the_direct_kernel_and_its_limits():
    """RFI_VARIANT_SPLIT (small chunks, low latency): the SK statistic is bit-identical to the direct kernel (same block
    statistics merged in the same order); alignment statistics and averages are summed block-wise: equal within the
    parity tolerance.  Units with more than 96 blocks are rejected with a message; AUTO never picks it."""
    w = synth.WORKLOADS["tiny"]
    vis, _ = synth.make_chunk(w, seed=1234)
    thr = synth.default_thresholds(w.window_M)
    a, used_a = run_gpu(w, vis, thr, "direct")
    b, used_b = run_gpu(w, vis, thr, "split")
    c, used_c = run_gpu(w, vis, thr, "auto")
    assert (used_a, used_b, used_c) == ("direct", "split", "direct")
    np.testing.assert_array_equal(a["tau"], b["tau"])
    assert np.abs(a["r_re"] - b["r_re"]).max() < 2e-6 and np.abs(a["r_im"] - b["r_im"]).max() < 2e-6
    assert np.abs(a["avg"] - b["avg"]).max() <= 1e-5 * np.abs(a["avg"]).max()
    big = synth.Workload("too_long", 4, True, 16, 1024, 16, 1024)             # 1024 / 4 = 256 blocks per unit
    plan = rfi.RfiPlan(big.n_stations, big.n_baselines, big.n_chan, big.n_time, 16, n_int=1024)
    plan.set_thresholds(thr); plan.set_variant("split")
    avg, weight, _ = plan.alloc_outputs()
    with pytest.raises(rfi.RfiError) as e:
        plan.process_chunk(torch.zeros(1024, 10, 16, 4, 2, device="cuda"), avg, weight)
    assert "small chunks" in str(e.value)
    plan.destroy()


def test_variants_agree_bit_for_bit(monkeypatch):
    """Same block length R (rows merged at a time) -> the two load paths feed identical arithmetic."""
    monkeypatch.setenv("RFI_DIRECT_ROWS", "4")
    monkeypatch.setenv("RFI_TMA_ROWS", "4")
    w = synth.WORKLOADS["lofar"].scaled(n_stations=7, n_time=512, n_int=256, burst_cell_frac=0.1)
    vis, _ = synth.make_chunk(w, seed=13)
    thr = synth.default_thresholds(16)
    a, _ = run_gpu(w, vis, thr, "direct")
    b, _ = run_gpu(w, vis, thr, "tma")
    for key in ("avg", "weight", "flags", "tau", "r_re", "r_im"):
        np.testing.assert_array_equal(a[key], b[key])


# ------------------------------------------------------------------------------------------------------
# batched-threshold mode (K > 1): BASELINE.json configs[4] in miniature
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [2, 16, 17, 64, 70])
def test_batched_sets_match_oracle_and_single_set_runs(K):
    """K sets in one pass: parity with the oracle per set, and bit-for-bit equal to K single-set runs."""
    w = synth.WORKLOADS["sweep"].scaled(n_stations=5, n_time=1536, n_int=768, burst_cell_frac=0.1)
    thr = synth.sweep_thresholds(w.window_M, K, seed=K)
    rep, out, truth = check(w, thr, "auto")
    assert rep["K"] == K
    fracs = out["flags"].reshape(K, -1).mean(1)
    assert fracs.min() < fracs.max()                      # the sets really differ
    vis, _ = synth.make_chunk(w, seed=1234)
    for k in sorted({0, 1, K // 2, K - 1}):
        single, used = run_gpu(w, vis, [thr[k]], "direct", stats=False)
        assert used == "direct"
        np.testing.assert_array_equal(single["flags"][0], out["flags"][k])
        np.testing.assert_array_equal(single["weight"][0], out["weight"][k])
        np.testing.assert_array_equal(single["avg"][0], out["avg"][k])


@pytest.mark.parametrize("M,n_int,n_time,n_chan", [(20, 100, 400, 20), (3, 12, 48, 13), (64, 1024, 2048, 16), (8, 8, 64, 96)])
def test_batched_ragged_shapes(M, n_int, n_time, n_chan):
    """windows per output not a multiple of the 16 warps, ragged tiles, shared flag words, one window per output"""
    w = synth.Workload("ragged_k", 5, False, n_chan, n_time, M, n_int, burst_cell_frac=0.2, channel_gain=True)
    K = 5
    thr = synth.sweep_thresholds(M, K, seed=M) if M >= 8 else [[1.0, 0.02 * (k + 1), 1.5, 0.9 - 0.02 * k] for k in range(K)]
    check(w, thr, "auto", seed=M)


@pytest.mark.parametrize("n_st,autos,n_chan,fp16,K,group,M,n_int,n_time,F,layout", [
    (8, True, 64, False, 64, 8, 16, 256, 512, 1, "time_major"),      # 36 baselines x 2 words = 72 words = 9 full groups
    (7, True, 64, False, 40, 8, 16, 768, 768, 1, "time_major"),      # 56 words: 7 groups; 48 windows = 3 rounds
    (6, False, 96, False, 33, 8, 16, 128, 256, 1, "time_major"),     # 15 baselines x 3 words = 45 words: row % 8 != 0 -> G falls to 1
    (9, False, 32, False, 64, 4, 16, 256, 512, 1, "time_major"),     # 36 words: G = 4, 9 groups
    (6, True, 64, False, 17, 8, 10, 200, 400, 2, "time_major"),      # 10 x 2 footprints (R = 5), 42 words: row % 8 != 0, G = 2
    (5, True, 128, True, 64, 8, 16, 256, 512, 1, "time_major"),      # fp16 storage, 60 words -> G = 4
    (8, True, 64, False, 64, 8, 16, 256, 512, 1, "cell_major"),
    (8, True, 64, True, 20, 8, 16, 256, 512, 1, "cell_major"),
])
def test_batched_tile_groups_in_tensor_memory(monkeypatch, n_st, autos, n_chan, fp16, K, group, M, n_int, n_time, F, layout):
    """The K-set kernel parks the flag words of G adjacent tiles in tensor memory and stores them as whole sectors
    (rfi_batched_mask.cuh).  Small chunks would not be grouped (every SM is to get two groups), so the rule is lifted
    here; outputs must match the oracle and, bit for bit, the ungrouped run (G = 1) of the same kernel."""
    w = synth.Workload("groups", n_st, autos, n_chan, n_time, M, n_int, window_F=F, fp16=fp16, burst_cell_frac=0.15,
                       channel_gain=True)
    thr = synth.sweep_thresholds(M * F, K, seed=K + group)
    monkeypatch.setenv("RFI_BT_GROUP_ANY", "1")
    monkeypatch.setenv("RFI_BT_GROUP", str(group))
    rep, grouped, _ = check(w, thr, "auto", seed=group, layout=layout)
    assert rep["K"] == K
    monkeypatch.setenv("RFI_BT_GROUP", "1")
    vis, _ = synth.make_chunk(w, seed=group)
    plain, used = run_gpu(w, vis, thr, "auto", layout=layout)
    assert used == "batched"
    for key in ("avg", "weight", "flags", "tau", "r_re", "r_im"):
        np.testing.assert_array_equal(grouped[key], plain[key], err_msg=key)
    assert 0 < grouped["flags"].mean() < 1


def test_batched_fp16_and_host_path():
    w = synth.WORKLOADS["lofar_fp16"].scaled(n_stations=5, n_time=1024, n_int=256, burst_cell_frac=0.1, tone_chan_frac=0.02)
    thr = synth.sweep_thresholds(16, 8, seed=3)
    rep, out, _ = check(w, thr, "auto")
    vis, _ = synth.make_chunk(w, seed=1234)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, rfi.RFI_FP16, n_int=w.n_int)
    plan.set_thresholds(thr)
    avg, weight, flags, stats = plan.process_chunk_host(vis.pin_memory(), want_stats=True)
    assert plan.last_variant == "batched"
    host = gpu_outputs_to_numpy(plan, avg, weight, stats, rfi.unpack_flags(flags, w.n_chan))
    plan.destroy()
    for key in ("avg", "weight", "flags", "tau", "r_re", "r_im"):
        np.testing.assert_array_equal(out[key], host[key])


# ------------------------------------------------------------------------------------------------------
# T x F window footprints (the paper's 10 x 2 and 5 x 4, W = 20)
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", ["direct", "tma", "split"])
@pytest.mark.parametrize("T,F,n_chan", [(10, 2, 64), (5, 4, 64), (16, 2, 20), (4, 8, 24), (2, 32, 64), (8, 16, 48)])
def test_tf_footprints(variant, T, F, n_chan):
    w = synth.Workload("tf", 5, True, n_chan, T * 24, T, T * 6, window_F=F, burst_cell_frac=0.15, channel_gain=True)
    W = T * F
    thr = [[0.8, 0.25 * (W * 0.8 + 1) / (W - 1) * 0.4, (W * 0.8 + 1) / (W - 1) * 0.45, 2.2 / math.sqrt(W)]]
    if variant == "tma" and w.n_cells % 4:
        pytest.skip("TMA variant needs n_cells % 4 == 0")
    rep, out, _ = check(w, thr, variant, seed=T * 100 + F)
    f = out["flags"][0].reshape(w.n_win, w.n_baselines, n_chan // F, F)
    assert (f == f[..., :1]).all()                        # one flag per footprint
    assert 0.0 < f.mean() < 0.9


@pytest.mark.parametrize("fp16", [False, True])
def test_tf_footprints_batched(fp16):
    w = synth.Workload("tf_k", 5, True, 64, 10 * 32, 10, 10 * 16, fp16=fp16, window_F=2, burst_cell_frac=0.15)
    thr = synth.sweep_thresholds(20, 9, seed=4)
    rep, out, _ = check(w, thr, "auto")
    assert rep["K"] == 9
    w2 = synth.Workload("tf_k2", 5, False, 12, 5 * 16, 5, 5 * 8, fp16=fp16, window_F=4, burst_cell_frac=0.15)   # ragged: old batched kernel
    check(w2, synth.sweep_thresholds(20, 5, seed=5), "auto")


# ------------------------------------------------------------------------------------------------------
# per-set confusion counters against the injected ground truth (BASELINE.json configs[4])
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_chan,K", [(64, 7), (45, 3), (16, 1)])
def test_confusion_counts_are_exact(n_chan, K):
    from oracle import rfi_oracle as orc
    w = synth.Workload("conf", 5, True, n_chan, 256, 16, 64, burst_cell_frac=0.2, channel_gain=True)
    thr = synth.sweep_thresholds(16, K, seed=8) if K > 1 else synth.default_thresholds(16)
    vis, truth = synth.make_chunk(w, seed=77)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
    plan.set_thresholds(thr)
    avg, weight, _ = plan.alloc_outputs()
    plan.process_chunk(vis.cuda(), avg, weight)
    tw = rfi.pack_flags(truth.reshape(plan.n_win, w.n_baselines, n_chan).cuda())
    counts = plan.confusion_counts(tw).cpu().numpy()
    torch.cuda.synchronize()
    flags = rfi.unpack_flags(plan.get_flags(), n_chan).reshape(K, plan.n_win, plan.n_cells).cpu().numpy()
    plan.destroy()
    t = truth.numpy().reshape(plan.n_win, plan.n_cells)
    # the oracle's flags on the same data (thresholds as float32, like the kernel's)
    ref = orc.process(vis.numpy().reshape(w.n_time, w.n_cells, 4, 2), 16, w.n_int,
                      np.asarray(thr, np.float32).astype(np.float64), want_stats=False).flags.astype(bool)
    for k in range(K):
        want = [(flags[k] & ~t).sum(), (~t).sum(), (~flags[k] & t).sum(), t.sum()]
        assert counts[k].tolist() == [int(x) for x in want]
        if (flags[k] == ref[k]).all():
            assert counts[k].tolist() == [int((ref[k] & ~t).sum()), int((~t).sum()), int((~ref[k] & t).sum()), int(t.sum())]
    assert counts[:, 1].min() > 0 and counts[:, 3].min() > 0


@pytest.mark.parametrize("n_chan,K,fp16,layout,group", [(64, 64, False, "time_major", 8), (64, 5, False, "time_major", 1),
                                                        (32, 40, True, "time_major", 4), (64, 70, False, "time_major", 8),
                                                        (64, 33, False, "cell_major", 8), (48, 6, False, "time_major", 1),
                                                        (64, 1, False, "time_major", 1)])
def test_in_kernel_confusion_counters_equal_the_mask_pass(monkeypatch, n_chan, K, fp16, layout, group):
    """rfi_plan_set_truth: the counters filled by rfi_process_chunk itself (the K-set kernel counts while it packs the
    flag words; ragged channel counts and K = 1 are followed by the mask pass) equal rfi_confusion_counts, which
    test_confusion_counts_are_exact pins against the flags and the oracle.  Refilled, not accumulated, by a second call."""
    monkeypatch.setenv("RFI_BT_GROUP_ANY", "1")
    monkeypatch.setenv("RFI_BT_GROUP", str(group))
    w = synth.Workload("conf2", 8, True, n_chan, 512, 16, 256, fp16=fp16, burst_cell_frac=0.2, channel_gain=True)
    thr = synth.sweep_thresholds(16, K, seed=K) if K > 1 else synth.default_thresholds(16)
    vis, truth = synth.make_chunk(w, seed=21)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, rfi.RFI_FP16 if fp16 else rfi.RFI_FP32,
                       n_int=w.n_int)
    plan.set_thresholds(thr)
    d_vis = vis.cuda()
    if layout == "cell_major":
        plan.set_layout("cell_major")
        d_vis = d_vis.permute(1, 2, 0, 3, 4).contiguous()
    tw = rfi.pack_flags(truth.reshape(plan.n_win, w.n_baselines, n_chan).cuda())
    counts = plan.set_truth(tw)
    avg, weight, _ = plan.alloc_outputs()
    for _ in range(2):
        plan.process_chunk(d_vis, avg, weight)
    torch.cuda.synchronize()
    fused = counts.cpu().numpy().copy()
    plan.set_truth(None)
    plan.process_chunk(d_vis, avg, weight)
    separate = plan.confusion_counts(tw).cpu().numpy()
    plan.destroy()
    np.testing.assert_array_equal(fused, separate)
    if layout == "time_major" and K in (1, 40):            # the host path fills the same counters
        plan3 = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                            rfi.RFI_FP16 if fp16 else rfi.RFI_FP32, n_int=w.n_int)
        plan3.set_thresholds(thr)
        c3 = plan3.set_truth(tw)
        plan3.process_chunk_host(vis.pin_memory())
        np.testing.assert_array_equal(c3.cpu().numpy(), separate)
        plan3.destroy()
    if K == 5:                                             # the counter buffer was sized for K sets: a new K needs a new one
        plan2 = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
        plan2.set_thresholds(thr)
        plan2.set_truth(tw)
        plan2.set_thresholds(thr[:3])
        avg3, weight3, _ = plan2.alloc_outputs()
        with pytest.raises(rfi.RfiError):
            plan2.process_chunk(d_vis, avg3, weight3)
        plan2.destroy()
    assert fused[:, 1].min() > 0 and fused[:, 3].min() > 0 and (fused[:, 0] + fused[:, 2]).max() > 0


# ------------------------------------------------------------------------------------------------------
# guard bands: compute-sanitizer is not available on the pool, so out-of-bounds stores are caught by canaries
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", ["direct", "tma", "batched", "batched_ragged", "tables", "tf", "fp16"])
def test_no_writes_outside_the_output_buffers(mode):
    n_chan = 45 if mode == "batched_ragged" else 64
    w = synth.Workload("guard", 5, True, n_chan, 320, 16 if mode != "tf" else 10, 160, fp16=(mode == "fp16"),
                       burst_cell_frac=0.2, window_F=2 if mode == "tf" else 1)
    vis, _ = synth.make_chunk(w, seed=5)
    K = 5 if mode.startswith("batched") else 1
    thr = synth.sweep_thresholds(16, K, seed=1) if K > 1 else synth.default_thresholds(w.window_M * w.window_F)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                       rfi.RFI_FP16 if w.fp16 else rfi.RFI_FP32, n_int=w.n_int)
    if w.window_F > 1:
        plan.set_window_freq(w.window_F)
    if mode == "tables":
        plan.set_arithmetic("tables", 0x3C50)
    plan.set_thresholds(thr)
    if mode in ("direct", "tma"):
        plan.set_variant(mode)
    G = 4096                                                   # guard elements on each side
    n_avg = K * plan.n_out * plan.n_cells * 8
    n_wt = K * plan.n_out * plan.n_cells
    n_st = 3 * plan.n_win * plan.n_cells
    fbuf = torch.full((G + n_avg + G + n_st + G,), -777.0, device="cuda")
    ibuf = torch.full((G + n_wt + G,), -777, dtype=torch.int32, device="cuda")
    avg = fbuf[G:G + n_avg]
    stats = fbuf[G + n_avg + G:G + n_avg + G + n_st]
    weight = ibuf[G:G + n_wt]
    # the input sits between guards too: a stray READ cannot be seen, but the guards make sure it stays in bounds of an allocation
    vbuf = torch.zeros(G + vis.numel() + G, dtype=vis.dtype, device="cuda")
    vbuf[G:G + vis.numel()] = vis.flatten().cuda()
    plan.process_chunk(vbuf[G:G + vis.numel()], avg, weight, stats)
    torch.cuda.synchronize()
    assert (fbuf[:G] == -777).all() and (fbuf[G + n_avg:G + n_avg + G] == -777).all() and (fbuf[-G:] == -777).all()
    assert (ibuf[:G] == -777).all() and (ibuf[-G:] == -777).all()
    assert (avg != -777).all() and (weight != -777).all() and (stats != -777).all()      # and everything inside was written
    assert (vbuf[:G] == 0).all() and (vbuf[-G:] == 0).all()
    plan.destroy()


# ------------------------------------------------------------------------------------------------------
# per-baseline threshold classes (cross / auto): each cell against the oracle run with its class's thresholds
# ------------------------------------------------------------------------------------------------------
def _run_classes(w, vis, classes, pairs, variant="auto", shard=None):
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                       rfi.RFI_FP16 if w.fp16 else rfi.RFI_FP32, n_int=w.n_int)
    if w.window_F > 1:
        plan.set_window_freq(w.window_F)
    plan.set_baseline_classes(classes)
    v = vis
    if shard is not None:
        plan.set_baseline_shard(*shard)
        v = vis[:, shard[0]:shard[0] + shard[1]].contiguous()
    plan.set_thresholds(pairs)
    plan.set_variant(variant)
    avg, weight, st = plan.alloc_outputs(stats=True)
    plan.process_chunk(v.cuda(), avg, weight, st)
    torch.cuda.synchronize()
    out = gpu_outputs_to_numpy(plan, avg, weight, st, rfi.unpack_flags(plan.get_flags(), w.n_chan))
    used = plan.last_variant
    plan.destroy()
    return out, used


@pytest.mark.parametrize("mode", ["direct", "tma", "batched", "batched_ragged", "fp16", "tf", "shard"])
def test_baseline_classes(mode):
    n_chan = 24 if mode == "batched_ragged" else 64
    F = 2 if mode == "tf" else 1
    w = synth.Workload("cls", 6, True, n_chan, 512, 16, 256, fp16=(mode == "fp16"), window_F=F,
                       burst_cell_frac=0.15, channel_gain=True)
    vis, _ = synth.make_chunk(w, seed=91)
    autos = synth.auto_baseline_mask(w).numpy()
    classes = autos.astype(int).tolist()
    W = 16 * F
    K = 6 if mode.startswith("batched") else 1
    cross_sets = synth.sweep_thresholds(W, K, seed=2) if K > 1 else synth.default_thresholds(W)
    c = (W * 0.7 + 1) / (W - 1)
    auto_sets = [[0.7, -float("inf"), c * (0.02 + 0.01 * k), 0.9 - 0.02 * k] for k in range(K)]   # autos: tau ~ 0, r_re ~ 1
    pairs = [[cross_sets[k], auto_sets[k]] for k in range(K)]
    shard = (5, 9) if mode == "shard" else None
    out, used = _run_classes(w, vis, classes, pairs, variant=mode if mode in ("direct", "tma") else "auto", shard=shard)
    b0, bc = shard if shard else (0, w.n_baselines)
    v = vis[:, b0:b0 + bc].numpy().reshape(w.n_time, bc * n_chan, 4, 2)
    cell_auto = np.repeat(autos[b0:b0 + bc], n_chan)
    tol = 2e-3 if w.fp16 else 1e-5
    n_flagged = 0
    for cls, sets in ((0, cross_sets), (1, auto_sets)):
        sel = np.nonzero(cell_auto == bool(cls))[0]
        sub = {"avg": out["avg"][:, :, sel], "weight": out["weight"][:, :, sel], "flags": out["flags"][:, :, sel],
               "tau": out["tau"][:, sel], "r_re": out["r_re"][:, sel], "r_im": out["r_im"][:, sel]}
        rep = compare(v[:, sel], 16, w.n_int, sets, sub, tol=tol, fp16=w.fp16, F=F)
        n_flagged += rep["oracle_flag_fraction"] > 0
    assert n_flagged >= 1
    # the classes really matter: the same data with the cross thresholds everywhere differs on the autos only
    if shard is None:
        single, _ = run_gpu(w, vis, cross_sets[:1], "auto")
        assert (single["flags"][0][:, ~cell_auto] == out["flags"][0][:, ~cell_auto]).all()
        assert (single["flags"][0][:, cell_auto] != out["flags"][0][:, cell_auto]).mean() > 0.05


# ------------------------------------------------------------------------------------------------------
# CUDA graphs: after one warm-up call (lazy allocations), rfi_process_chunk is pure stream work and can be captured
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [1, 6])
def test_process_chunk_is_cuda_graph_capturable(K):
    w = synth.WORKLOADS["tiny"]
    thr = synth.default_thresholds(w.window_M) if K == 1 else synth.sweep_thresholds(w.window_M, K, seed=1)
    vis_a, _ = synth.make_chunk(w, seed=1)
    vis_b, _ = synth.make_chunk(w, seed=2)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
    plan.set_thresholds(thr)
    avg, weight, stats = plan.alloc_outputs(stats=True)
    d_vis = vis_a.cuda()
    plan.process_chunk(d_vis, avg, weight, stats)                 # warm-up: flag buffer, tensor map, attributes
    torch.cuda.synchronize()
    ref_a = (avg.clone(), weight.clone(), plan.get_flags().clone())
    d_vis.copy_(vis_b.cuda())
    plan.process_chunk(d_vis, avg, weight, stats)
    torch.cuda.synchronize()
    ref_b = (avg.clone(), weight.clone(), plan.get_flags().clone())
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            plan.process_chunk(d_vis, avg, weight, stats, stream=side)
    for vis, ref in ((vis_a, ref_a), (vis_b, ref_b), (vis_a, ref_a)):
        d_vis.copy_(vis.cuda())
        avg.zero_(); weight.zero_()
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(avg, ref[0]) and torch.equal(weight, ref[1]) and torch.equal(plan.get_flags(), ref[2])
    plan.destroy()


# ------------------------------------------------------------------------------------------------------
# cell-major input layout vis[b][c][t][pol] (rfi_plan_set_layout): same arithmetic behind a transposing tensor map
# ------------------------------------------------------------------------------------------------------
def _run_cell_major(w, vis, thr, classes=None):
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                       rfi.RFI_FP16 if w.fp16 else rfi.RFI_FP32, n_int=w.n_int)
    if w.window_F > 1:
        plan.set_window_freq(w.window_F)
    plan.set_layout("cell_major")
    plan.set_thresholds(thr)
    avg, weight, st = plan.alloc_outputs(stats=True)
    avg.fill_(float("nan")); weight.fill_(-1); st.fill_(float("nan"))
    cm = vis.permute(1, 2, 0, 3, 4).contiguous().cuda()            # [b][c][t][pol][re,im]
    plan.process_chunk(cm, avg, weight, st)
    torch.cuda.synchronize()
    out = gpu_outputs_to_numpy(plan, avg, weight, st, rfi.unpack_flags(plan.get_flags(), w.n_chan))
    assert plan.last_variant == "tma" and plan.launch_count == 1
    plan.destroy()
    return out


@pytest.mark.parametrize("fp16,M,n_chan,F", [(False, 16, 64, 1), (False, 4, 13 * 4, 1), (False, 64, 16, 1), (True, 16, 64, 1),
                                            (True, 8, 24, 1), (False, 8, 20, 2), (False, 12, 45, 1)])
def test_cell_major_layout(fp16, M, n_chan, F):
    w = synth.Workload("cm", 5, True, n_chan, M * 24, M, M * 8, fp16=fp16, window_F=F, burst_cell_frac=0.15, channel_gain=True)
    W = M * F
    thr = synth.default_thresholds(W) if W >= 8 else [[1.0, 0.01, 2.0, 0.95]]
    vis, _ = synth.make_chunk(w, seed=M + n_chan)
    out = _run_cell_major(w, vis, thr)
    v = vis.numpy().reshape(w.n_time, w.n_cells, 4, 2)
    compare(v, M, w.n_int, thr, out, tol=2e-3 if fp16 else 1e-5, fp16=fp16, F=F)
    # bit-identical to the time-major TMA kernel with the same block length
    import os
    os.environ["RFI_TMA_ROWS"] = "8" if fp16 else "4"
    try:
        if w.fp16 or w.n_cells % 4 == 0:
            tm, used = run_gpu(w, vis, thr, "tma")
            for key in ("avg", "weight", "flags", "tau", "r_re", "r_im"):
                np.testing.assert_array_equal(out[key], tm[key])
    finally:
        del os.environ["RFI_TMA_ROWS"]


def test_cell_major_rejects_unsupported_plans():
    plan = rfi.RfiPlan(4, 10, 32, 60, 6)                            # window_M = 6 is not a multiple of 4
    plan.set_layout("cell_major")
    plan.set_thresholds([[1.0, 0.1, 1.0, 0.5]])
    avg, weight, _ = plan.alloc_outputs()
    vis = torch.zeros(10, 32, 60, 4, 2, device="cuda")
    with pytest.raises(rfi.RfiError) as e:
        plan.process_chunk(vis, avg, weight)
    assert e.value.code == -1
    plan.destroy()


@pytest.mark.parametrize("fp16,n_chan,K", [(False, 64, 5), (True, 64, 20), (False, 24, 40)])
def test_cell_major_layout_batched(fp16, n_chan, K):
    """K > 1 behind the transposing tensor map: parity with the oracle and bit-identical to the time-major batched run."""
    w = synth.Workload("cm_k", 5, True, n_chan, 16 * 40, 16, 16 * 20, fp16=fp16, burst_cell_frac=0.15, channel_gain=True)
    thr = synth.sweep_thresholds(16, K, seed=K)
    vis, _ = synth.make_chunk(w, seed=K)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M,
                       rfi.RFI_FP16 if fp16 else rfi.RFI_FP32, n_int=w.n_int)
    plan.set_layout("cell_major")
    plan.set_thresholds(thr)
    avg, weight, st = plan.alloc_outputs(stats=True)
    plan.process_chunk(vis.permute(1, 2, 0, 3, 4).contiguous().cuda(), avg, weight, st)
    torch.cuda.synchronize()
    out = gpu_outputs_to_numpy(plan, avg, weight, st, rfi.unpack_flags(plan.get_flags(), w.n_chan))
    assert plan.last_variant == "batched"
    plan.destroy()
    compare(vis.numpy().reshape(w.n_time, w.n_cells, 4, 2), 16, w.n_int, thr, out, tol=2e-3 if fp16 else 1e-5, fp16=fp16)
    tm, _ = run_gpu(w, vis, thr, "auto")
    for key in ("avg", "weight", "flags", "tau", "r_re", "r_im"):
        np.testing.assert_array_equal(out[key], tm[key])


def test_bench_strong_scaling_shards_reproduce_the_full_chunk():
    """bench.py --gpus N --scaling strong on ONE GPU: the per-rank preparation (`bench.rank_chunk_and_plan` with
    `sharding.rank_work`) run for every rank of a world of 3 in turn -- the shards' outputs are the slices of the
    unsharded run bit for bit, and their sample counts add up to the one chunk (no multi-GPU box is available)."""
    import bench
    from paper_2412_14775_b200 import sharding
    w = synth.WORKLOADS["lofar"].scaled(n_stations=7, n_time=512, n_int=256, burst_cell_frac=0.1)
    thr = synth.default_thresholds(16)
    dev = torch.device("cuda")
    vis_full, _, plan_full = bench.rank_chunk_and_plan(w, sharding.rank_work(w.n_baselines, 1, 0, "strong"), dev)
    plan_full.set_thresholds(thr)
    avg_f, wt_f, _ = plan_full.alloc_outputs()
    plan_full.process_chunk(vis_full, avg_f, wt_f)
    torch.cuda.synchronize()
    flags_f = plan_full.get_flags().clone()
    world, total = 3, 0
    for rank in range(world):
        work = sharding.rank_work(w.n_baselines, world, rank, "strong")
        vis, truth, plan = bench.rank_chunk_and_plan(w, work, dev)
        assert work["sharded"] and vis.shape[1] == work["b_count"] and truth.shape[1] == work["b_count"] * w.n_chan
        plan.set_thresholds(thr)
        avg, wt, _ = plan.alloc_outputs()
        plan.process_chunk(vis, avg, wt)
        torch.cuda.synchronize()
        b0, bc = work["b_first"], work["b_count"]
        assert torch.equal(avg, avg_f[:, :, b0:b0 + bc]) and torch.equal(wt, wt_f[:, :, b0:b0 + bc])
        assert torch.equal(plan.get_flags(), flags_f[:, :, b0:b0 + bc])
        total += w.n_time * plan.n_cells
        plan.destroy()
    assert total == w.n_time * w.n_cells
    weak = sharding.rank_work(w.n_baselines, world, 2, "weak")
    assert not weak["sharded"] and weak["seed"] == 1236
    plan_full.destroy()


def test_mix_probe_moves_the_bytes_it_reports():
    """rfi_probe_mix_bandwidth (diagnostics): reads every 1 KiB row once, writes one row per `reads_per_write` rows --
    the XOR of the rows read -- and rejects an output buffer that is too small."""
    import ctypes
    lib = rfi.load_library()
    g = torch.Generator().manual_seed(5)
    rows, rpw = 4096 * 9, 9
    buf = torch.randint(-2**31, 2**31 - 1, (rows, 256), dtype=torch.int32, generator=g).cuda()
    out = torch.zeros(rows // rpw, 256, dtype=torch.int32, device="cuda")
    ms, moved = ctypes.c_float(), ctypes.c_size_t()
    rc = lib.rfi_probe_mix_bandwidth(buf.data_ptr(), buf.numel() * 4, out.data_ptr(), out.numel() * 4, rpw, 2,
                                     ctypes.byref(ms), ctypes.byref(moved), None)
    assert rc == 0 and ms.value > 0 and moved.value == (rows + rows // rpw) * 1024
    want = buf.view(rows // rpw, rpw, 256)[:, 0].clone()
    for r in range(1, rpw):
        want ^= buf.view(rows // rpw, rpw, 256)[:, r]
    assert torch.equal(out, want)
    rc = lib.rfi_probe_mix_bandwidth(buf.data_ptr(), buf.numel() * 4, out.data_ptr(), out.numel() * 4 - 1024, rpw, 2,
                                     ctypes.byref(ms), ctypes.byref(moved), None)
    assert rc != 0
    assert rfi.probe_mix_bandwidth(buf, out.numel() * 4, repeats=2) > 0


@pytest.mark.parametrize("what", ["K", "tables", "cell_major"])
def test_split_variant_is_refused_where_it_cannot_run(what):
    """RFI_VARIANT_SPLIT exists for K = 1, fast arithmetic, time-major input only: a plan in any other mode refuses
    the request with a message instead of quietly running another kernel."""
    w = synth.WORKLOADS["tiny"]
    vis, _ = synth.make_chunk(w, seed=3)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
    plan.set_thresholds(synth.sweep_thresholds(w.window_M, 3, seed=1) if what == "K" else synth.default_thresholds(w.window_M))
    d_vis = vis.cuda()
    if what == "tables":
        plan.set_arithmetic("tables", 0x3C50)
    if what == "cell_major":
        plan.set_layout("cell_major")
        d_vis = d_vis.permute(1, 2, 0, 3, 4).contiguous()
    plan.set_variant("split")
    avg, weight, _ = plan.alloc_outputs()
    n0 = plan.launch_count
    with pytest.raises(rfi.RfiError) as e:
        plan.process_chunk(d_vis, avg, weight)
    assert e.value.code == -1 and "RFI_VARIANT_SPLIT needs K = 1" in str(e.value)
    assert plan.launch_count == n0
    plan.set_variant("auto")                                   # the same plan runs once the request is withdrawn
    plan.process_chunk(d_vis, avg, weight)
    torch.cuda.synchronize()
    plan.destroy()


def test_host_path_refuses_a_changed_K_before_it_enqueues_anything():
    """rfi_plan_set_truth sized the counters for K sets; with another K rfi_process_chunk_host returns RFI_ESTATE
    up front: no kernel launched, the flags of the previous chunk still in place."""
    w = synth.Workload("hostK", 6, True, 64, 256, 16, 128, burst_cell_frac=0.2)
    vis, truth = synth.make_chunk(w, seed=8)
    thr = synth.sweep_thresholds(16, 5, seed=2)
    plan = rfi.RfiPlan(w.n_stations, w.n_baselines, w.n_chan, w.n_time, w.window_M, n_int=w.n_int)
    plan.set_thresholds(thr)
    tw = rfi.pack_flags(truth.reshape(plan.n_win, w.n_baselines, w.n_chan).cuda())
    counts = plan.set_truth(tw)
    h = vis.pin_memory()
    plan.process_chunk_host(h)
    before, n0 = counts.cpu().numpy().copy(), plan.launch_count
    plan.set_thresholds(thr[:3])
    with pytest.raises(rfi.RfiError) as e:
        plan.process_chunk_host(h)
    assert e.value.code == -4 and "rfi_plan_set_truth was called with K = 5" in str(e.value)
    assert plan.launch_count == n0
    np.testing.assert_array_equal(counts.cpu().numpy(), before)
    plan.destroy()
