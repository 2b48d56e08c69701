"""CPU tests of the seeded input generators (paper_2412_14775_b200/synth.py)."""
import math

import numpy as np
import torch

from paper_2412_14775_b200 import synth


def test_workload_shapes_match_baseline_configs():
    W = synth.WORKLOADS
    assert (W["tiny"].n_baselines, W["tiny"].n_cells, W["tiny"].n_win, W["tiny"].n_out) == (6, 96, 16, 16)
    assert (W["lofar"].n_baselines, W["lofar"].n_cells, W["lofar"].n_win, W["lofar"].n_out) == (1176, 75264, 480, 10)
    assert W["lofar"].input_bytes == 18_496_880_640 and W["lofar_fp16"].input_bytes == 9_248_440_320
    assert W["tiny"].input_bytes == 3_145_728
    assert (W["large"].n_baselines, W["large"].n_cells) == (2926, 749056)
    assert W["large"].input_bytes == 73_635_201_024


def test_seeded_and_deterministic():
    w = synth.WORKLOADS["lofar"].scaled(n_stations=4, n_time=256, n_int=128)
    a, ta = synth.make_chunk(w, seed=5)
    b, tb = synth.make_chunk(w, seed=5)
    c, _ = synth.make_chunk(w, seed=6)
    assert torch.equal(a, b) and torch.equal(ta, tb) and not torch.equal(a, c)
    assert a.shape == (256, 10, 64, 4, 2) and a.dtype == torch.float32


def test_noise_statistics_and_autos():
    w = synth.Workload("n", 6, True, 32, 2048, 16, 2048)
    vis, truth = synth.make_chunk(w, seed=1)
    assert not truth.any()
    v = torch.view_as_complex(vis)
    autos = synth.auto_baseline_mask(w)
    cross = v[:, ~autos]
    assert abs(cross.abs().pow(2).mean().item() - 1.0) < 0.01                   # unit variance per pol
    assert abs((cross[..., 0] * cross[..., 3].conj()).mean().real.item() - synth.RHO ** 2) < 0.01
    au = v[:, autos]
    assert au[..., 0].imag.abs().max() == 0 and au[..., 3].imag.abs().max() == 0    # Hermitian
    assert torch.allclose(au[..., 2], au[..., 1].conj())
    assert abs(au[..., 0].real.mean().item() - 1.0) < 0.01


def test_tiny_burst_recipe():
    w = synth.WORKLOADS["tiny"]
    vis, truth = synth.make_chunk(w, seed=1234)
    clean, _ = synth.make_chunk(w.scaled(fixed_burst=False), seed=1234)
    diff = torch.view_as_complex(vis - clean).reshape(w.n_time, w.n_cells, 4)
    hit = diff.abs().sum(-1) > 0
    assert hit.sum().item() == 40 * 6                                           # 40 samples on 2 channels x 3 baselines
    power = diff[hit].abs().pow(2).sum(-1)
    assert torch.allclose(power, torch.full_like(power, 10.0), rtol=1e-4)        # 10x noise power, rank-1 coherency
    cells = hit.any(0).nonzero().flatten().tolist()
    assert cells == [3, 7, 19, 23, 35, 39]
    n_flagged_windows = truth.sum(0)[cells].tolist()
    assert n_flagged_windows == [1, 1, 2, 2, 1, 1]                               # inside / straddling / ending at a boundary


def test_burst_truth_mask_matches_injection():
    w = synth.WORKLOADS["lofar"].scaled(n_stations=5, n_time=512, n_int=256, burst_cell_frac=0.1, channel_gain=False)
    vis, truth = synth.make_chunk(w, seed=9)
    clean, _ = synth.make_chunk(w.scaled(burst_cell_frac=0.0), seed=9)
    # the RNG stream differs once bursts are drawn, so compare structure instead: duty cycle and cell count
    n_aff = int(round(0.1 * w.n_cells))
    assert truth.any(0).sum().item() <= n_aff
    frac = truth[:, truth.any(0)].float().mean().item()
    assert 0.15 < frac < 0.35                                                    # ~25 % of windows carry a burst


def test_fp16_and_thresholds():
    w = synth.WORKLOADS["lofar_fp16"].scaled(n_stations=4, n_time=256, n_int=128)
    vis, truth = synth.make_chunk(w, seed=2)
    assert vis.dtype == torch.float16 and torch.isfinite(vis).all()
    assert truth[:, :].any()
    sets = synth.sweep_thresholds(16, 64)
    assert len(sets) == 64 and all(0.5 <= s[0] <= 1 and s[1] < s[2] and 0 < s[3] < 1 for s in sets)
    d, lo, hi, g = synth.default_thresholds(20)[0]
    assert lo < hi and 0 < g < 1


def test_auto_null_quantiles_are_reproduced_by_the_committed_script():
    """provenance of synth._NULL_Q_AUTO: tests/golden/make_null_quantiles.py (oracle/ + synth only) re-derives W = 16
    on a smaller sample within Monte-Carlo tolerance"""
    from tests.golden.make_null_quantiles import null_quantiles_auto
    xq, rq, n = null_quantiles_auto(16, n_stations=16, n_windows=256, seed=5)
    ref_x, ref_r = synth._NULL_Q_AUTO[16]
    assert n == 16 * 16 * 256
    for got, want, tol in zip(xq[1:5], ref_x[1:5], (0.06, 0.04, 0.04, 0.06)):     # 1, 5, 95, 99 %
        assert abs(got / want - 1) < tol, (xq, ref_x)
    assert abs(rq[0] / ref_r[0] - 1) < 0.03 and abs(rq[1] / ref_r[1] - 1) < 0.04


def test_fp16_chunk_is_the_rounded_fp32_chunk():
    """the fp16 gate against the ORIGINAL fp32 data relies on make_chunk rounding as its last step"""
    w = synth.WORKLOADS["lofar_fp16"].scaled(n_stations=4, n_time=256, n_int=128, burst_cell_frac=0.1, tone_chan_frac=0.05)
    v16, t16 = synth.make_chunk(w, seed=9)
    v32, t32 = synth.make_chunk(w.scaled(fp16=False), seed=9)
    assert v16.dtype == torch.float16 and v32.dtype == torch.float32
    assert torch.equal(v32.to(torch.float16), v16) and torch.equal(t16, t32)


def test_rl_windows_recipe():
    """scale factors in [0.01, 1000], RFI with probability 0.4 inside a rectangular footprint"""
    w = synth.rl_windows(4000, 10, 2, seed=3)
    assert w.shape == (4000, 20, 4, 2) and w.dtype == torch.float32
    assert torch.equal(w, synth.rl_windows(4000, 10, 2, seed=3))
    rms = w.pow(2).mean((1, 2, 3)).sqrt()
    assert rms.min() > 0.005 and rms.max() < 3000
    clean = synth.rl_windows(4000, 10, 2, seed=3, rfi_prob=0.0)
    changed = (w != clean).flatten(1).any(1).float().mean()
    assert abs(changed - 0.4) < 0.03
